"""Pins for the oracle's plinth removal (section 2.1.1; R21): every line's own value at
the cutting length position is subtracted from every bin of its extent."""
import numpy as np
import pytest

from oracle import hk_oracle as O

scipy_special = pytest.importorskip("scipy.special")

COND = dict(T=900.0, P_atm=0.8, mass_amu=28.0, Q=250.0)


def _lines(nu0, rng):
    n = len(nu0)
    return dict(nu0=np.asarray(nu0, dtype=np.float64), A=10 ** rng.uniform(-3, 2, n), g_up=rng.integers(1, 9, n).astype(float),
                E_low=rng.uniform(0, 3000, n), gamma_ref=rng.uniform(0.02, 0.2, n), n_exp=rng.uniform(0.5, 0.75, n))


def test_bins_at_the_cut_get_nothing_and_terms_are_nonnegative():
    rng = np.random.default_rng(0)
    grid, cut = (0.0, 200.0, 0.25), 10.0                      # cut and centre on grid points: |nu_i - nu0| = cut exists
    L = _lines([100.0], rng)
    k, _ = O.opacity_grid(L, COND, grid, cut, plinth=True)
    k0, _ = O.opacity_grid(L, COND, grid, cut)
    jc = 400
    assert abs(k[jc - 40]) <= 1e-12 * k0[jc - 40] and abs(k[jc + 40]) <= 1e-12 * k0[jc + 40]
    assert k[jc - 41] == 0.0 and k[jc + 41] == 0.0           # outside the extent: nothing, as without plinth removal
    assert (k >= -1e-18 * k0.max()).all() and (k <= k0).all()
    assert k[jc] == pytest.approx(k0[jc] - k0[jc + 40], rel=1e-12)   # symmetric line: V(cut) is the value at +-cut


def test_removed_part_is_the_box_sum_of_plinths_third_opinion():
    """k - k_plinth at bin i = sum over lines covering i of S V(cut), with V from scipy's wofz and the oracle's own
    line parameters; coverage from the integer extents."""
    rng = np.random.default_rng(1)
    grid, cut = (50.0, 120.0, 0.05), 7.3
    L = _lines(rng.uniform(40.0, 130.0, 300), rng)
    k0, ev0 = O.opacity_grid(L, COND, grid, cut)
    k1, ev1 = O.opacity_grid(L, COND, grid, cut, plinth=True)
    assert ev0 == ev1
    S, gL, aD, valid = O.line_params(L, COND["T"], COND["P_atm"], COND["mass_amu"], COND["Q"])
    N = O.grid_size(*grid)
    ilo, ihi, _ = O.extents(L["nu0"], valid, grid[0], grid[2], N, cut)
    pl = S * scipy_special.wofz((cut + 1j * gL) / aD).real / (aD * np.sqrt(np.pi))
    box = np.zeros(N + 1)
    for a, b, p in zip(ilo, ihi, pl):
        if a <= b:
            box[a] += p
            box[b + 1] -= p
    box = np.cumsum(box)[:N]
    assert np.abs((k0 - k1) - box).max() <= 1e-9 * box.max()


def test_integrated_opacity_with_plinth_removed_closed_form():
    """Resolved grid: sum k dnu = S (1 - wing loss beyond the cut - 2 cut V(cut)), wing loss and V(cut) from the
    two-term asymptotic series (independent of the oracle's w)."""
    grid, cut = (0.0, 60.0, 0.002), 20.0
    L = dict(nu0=np.array([30.0]), A=np.array([5.0]), g_up=np.array([3.0]), E_low=np.array([500.0]),
             gamma_ref=np.array([0.09]), n_exp=np.array([0.6]))
    k, _ = O.opacity_grid(L, COND, grid, cut, plinth=True)
    S, gL, aD, _ = O.line_params(L, COND["T"], COND["P_atm"], COND["mass_amu"], COND["Q"])
    S, G, a, c = S[0], gL[0], aD[0], cut
    loss = 1.0 - (2.0 / np.pi) * np.arctan(c / G) + (G / np.pi) * a * a * c / (c * c + G * G) ** 2
    q = c * c + G * G
    v_cut = G / (np.pi * q) * (1.0 + a * a * (1.5 - 2.0 * G * G / q) / q)
    assert k.sum() * grid[2] == pytest.approx(S * (1.0 - loss - 2.0 * c * v_cut), rel=2e-6)


def test_uncut_has_no_plinth_and_linearity_holds():
    rng = np.random.default_rng(2)
    grid = (0.0, 40.0, 0.1)
    L = _lines(rng.uniform(1.0, 39.0, 40), rng)
    ka, _ = O.opacity_grid(L, COND, grid, 0.0, plinth=True)
    kb, _ = O.opacity_grid(L, COND, grid, 0.0)
    assert np.array_equal(ka, kb)
    k, _ = O.opacity_grid(L, COND, grid, 5.0, plinth=True)
    k1, _ = O.opacity_grid({f: v[:15] for f, v in L.items()}, COND, grid, 5.0, plinth=True)
    k2, _ = O.opacity_grid({f: v[15:] for f, v in L.items()}, COND, grid, 5.0, plinth=True)
    assert np.abs(k - (k1 + k2)).max() <= 1e-12 * k.max()
