"""Pins for the oracle's HITRAN-style line parameters (Eq. 4, pressure shift L238 / Table 4,
isotopologue table; R23, R24)."""
import numpy as np
import pytest

from oracle import hk_oracle as O

GRID, CUT = (0.0, 100.0, 0.05), 8.0


def _exomol(n=200, seed=0):
    rng = np.random.default_rng(seed)
    return dict(nu0=rng.uniform(10, 90, n), A=10 ** rng.uniform(-3, 1, n), g_up=rng.integers(1, 9, n).astype(float),
                E_low=rng.uniform(0, 3000, n), gamma_ref=rng.uniform(0.02, 0.1, n), n_exp=rng.uniform(0.5, 0.75, n))


def _hitran(L, gamma_self=None, delta=None, iso=None):
    n = L["nu0"].size
    H = {k: L[k] for k in ("nu0", "A", "g_up", "E_low", "n_exp")}
    H["gamma_air"] = L["gamma_ref"]
    H["gamma_self"] = L["gamma_ref"] if gamma_self is None else gamma_self
    H["delta"] = np.zeros(n) if delta is None else delta
    H["iso"] = np.zeros(n, dtype=np.int32) if iso is None else iso
    return H


def _close(a, b, tol):
    m = np.maximum(np.abs(a), np.abs(b)) > 0
    return np.abs(a[m] - b[m]).max() <= tol * np.abs(b).max()


def test_reduces_to_eq5_when_air_equals_self_and_no_shift():
    L = _exomol()
    cond = dict(T=900.0, P_atm=0.8, mass_amu=28.0, Q=250.0)
    k0, e0 = O.opacity_grid(L, cond, GRID, CUT)
    k1, e1 = O.opacity_grid_hitran(_hitran(L), dict(T=900.0, P_atm=0.8, P_self_atm=0.3, isos=[(28.0, 250.0, 1.0)]), GRID, CUT)
    assert e0 == e1 and _close(k1, k0, 1e-12)


def test_pure_self_gas_uses_gamma_self_only_and_pure_air_gamma_air_only():
    L = _exomol(seed=1)
    gs = L["gamma_ref"] * 3.7
    H = _hitran(L, gamma_self=gs)
    base = dict(T=700.0, P_atm=1.3, isos=[(18.0, 100.0, 1.0)])
    k_self, _ = O.opacity_grid_hitran(H, dict(base, P_self_atm=1.3), GRID, CUT)
    k_air, _ = O.opacity_grid_hitran(H, dict(base, P_self_atm=0.0), GRID, CUT)
    cond = dict(T=700.0, P_atm=1.3, mass_amu=18.0, Q=100.0)
    assert _close(k_self, O.opacity_grid(dict(L, gamma_ref=gs), cond, GRID, CUT)[0], 1e-12)
    assert _close(k_air, O.opacity_grid(L, cond, GRID, CUT)[0], 1e-12)
    # Eq. 4 by hand for one line at a mixed composition
    S, gL, aD, ctr, valid = O.line_params_hitran(H, dict(base, P_self_atm=0.4))
    want = L["A"][0] / (4 * np.pi * 2.99792458e10) + (700.0 / 296.0) ** (-L["n_exp"][0]) * (L["gamma_ref"][0] * 0.9 + gs[0] * 0.4)
    assert gL[0] == pytest.approx(want, rel=1e-13)


def test_pressure_shift_moves_the_profile_not_the_strength():
    L = dict(nu0=np.array([50.0]), A=np.array([1.0]), g_up=np.array([3.0]), E_low=np.array([200.0]),
             gamma_ref=np.array([0.05]), n_exp=np.array([0.6]))
    grid = (40.0, 60.0, 0.001)
    cond = dict(T=500.0, P_atm=2.0, P_self_atm=0.0, isos=[(30.0, 50.0, 1.0)])
    k0, _ = O.opacity_grid_hitran(_hitran(L), cond, grid, 0.0)
    k1, _ = O.opacity_grid_hitran(_hitran(L, delta=np.array([-0.0125])), cond, grid, 0.0)   # shift = -0.025 = 25 bins
    assert np.argmax(k1) == np.argmax(k0) - 25
    assert np.abs(k1[1000:-1025] / k0[1025:-1000] - 1.0).max() <= 1e-9                       # same curve, moved
    S0, _, a0, c0, _ = O.line_params_hitran(_hitran(L), cond)
    S1, _, a1, c1, _ = O.line_params_hitran(_hitran(L, delta=np.array([-0.0125])), cond)
    assert S0[0] == S1[0] and a0[0] == a1[0] and c1[0] == pytest.approx(50.0 - 0.025, rel=1e-15)


def test_isotopologues_abundance_mass_and_partition_function():
    L = _exomol(n=120, seed=2)
    iso = (np.arange(120) % 2).astype(np.int32)
    isos = [(18.0, 170.0, 0.997), (20.0, 176.0, 0.002)]
    cond = dict(T=800.0, P_atm=0.5, P_self_atm=0.1, isos=isos)
    k, _ = O.opacity_grid_hitran(_hitran(L, iso=iso), cond, GRID, CUT)
    parts = []
    for j, (m, Q, ab) in enumerate(isos):
        sel = iso == j
        Lj = {f: v[sel] for f, v in L.items()}
        kj, _ = O.opacity_grid(Lj, dict(T=800.0, P_atm=0.5, mass_amu=m, Q=Q), GRID, CUT)
        parts.append(ab * kj)
    assert _close(k, parts[0] + parts[1], 1e-12)
    S, gL, aD, ctr, valid = O.line_params_hitran(_hitran(L, iso=iso), cond)
    assert (aD[0] / L["nu0"][0]) / (aD[1] / L["nu0"][1]) == pytest.approx(np.sqrt(20.0 / 18.0), rel=1e-14)
    bad = _hitran(L, iso=np.where(np.arange(120) == 5, 7, iso).astype(np.int32))            # index outside the table
    kb, _ = O.opacity_grid_hitran(bad, cond, GRID, CUT)
    keep = np.arange(120) != 5
    kk, _ = O.opacity_grid_hitran({f: v[keep] for f, v in _hitran(L, iso=iso).items()}, cond, GRID, CUT)
    assert _close(kb, kk, 1e-13)
