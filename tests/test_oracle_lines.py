"""Pins for the oracle's per-line parameters, integer extents and the sum over
lines (Eq. 3, Eq. 5, Eq. 9, Eq. 13, Eq. 14,
Eq. 15-16; cut from the centre L239/L262; R1-R18)."""
import math
from decimal import Decimal, getcontext

import numpy as np
import pytest
from scipy import special

from oracle import hk_oracle as O

C_CM = 2.99792458e10
KB = 1.380649e-16
H = 6.62607015e-27
NA = 6.02214076e23


def _lines(**kw):
    n = len(kw["nu0"])
    d = dict(A=np.ones(n), g_up=np.ones(n), E_low=np.zeros(n),
             gamma_ref=np.full(n, 0.05), n_exp=np.full(n, 0.6))
    d.update({k: np.asarray(v, dtype=np.float64) for k, v in kw.items()})
    return d


def test_eq9_hand_calculation_decimal():
    """Eq. 9 (L127) evaluated with 50-digit decimal arithmetic for three lines."""
    getcontext().prec = 50
    D = Decimal
    pi = D("3.14159265358979323846264338327950288419716939937510")
    cases = [(1234.5, 3.2e-3, 7.0, 2500.0, 900.0, 18.0, 321.0),
             (31.25, 1.5e2, 33.0, 12000.0, 2500.0, 55.845, 50.0),
             (25000.0, 7.7e-9, 1.0, 0.0, 296.0, 1.008, 2.5)]
    for nu0, A, g, E, T, mass, Q in cases:
        c2 = D(H) * D(C_CM) / D(KB)
        m = D(mass) / D(NA)
        S = (D(A) * D(g) / (8 * pi * D(C_CM) * m * D(nu0) ** 2 * D(Q))
             * (-c2 * D(E) / D(T)).exp() * (1 - (-c2 * D(nu0) / D(T)).exp()))
        got, _, _, valid = O.line_params(_lines(nu0=[nu0], A=[A], g_up=[g], E_low=[E]), T, 1.0, mass, Q)
        assert valid[0] == 1
        assert got[0] == pytest.approx(float(S), rel=5e-14)


def test_widths_against_eq3_eq5():
    L = _lines(nu0=[2000.0, 10.0], A=[1e9, 0.0], gamma_ref=[0.08, 0.02], n_exp=[0.5, 0.75])
    T, P, mass = 1184.0, 3.0, 18.015
    _, gL, aD, _ = O.line_params(L, T, P, mass, 100.0)
    # Eq. 3: Gamma_D = (nu0/c) sqrt(2 ln2 kB T / m) = sqrt(ln 2) alpha_D
    m = mass / NA
    gD = 2000.0 / C_CM * math.sqrt(2 * math.log(2) * KB * T / m)
    assert aD[0] * math.sqrt(math.log(2)) == pytest.approx(gD, rel=1e-14)
    assert aD[1] / aD[0] == pytest.approx(10.0 / 2000.0, rel=1e-14)          # alpha_D ~ nu0
    # Eq. 5 with T = 4 T_ref and n = 1/2: (T_ref/T)^n = 1/2 exactly
    assert gL[0] == pytest.approx(1e9 / (4 * math.pi * C_CM) + 0.08 * 0.5 * 3.0, rel=1e-14)
    assert gL[1] == pytest.approx(0.02 * 0.25 ** 0.75 * 3.0, rel=1e-14)
    # natural width of A = 1e9 1/s: 2.65e-3 cm^-1 (R6)
    assert 1e9 / (4 * math.pi * C_CM) == pytest.approx(2.654e-3, rel=1e-3)


def test_scaling_laws():
    base = _lines(nu0=[1500.0, 40.0], A=[0.3, 5.0], g_up=[9.0, 2.0], E_low=[4000.0, 100.0])
    S0, g0, a0, _ = O.line_params(base, 1200.0, 0.0, 18.0, 700.0)
    S1, _, _, _ = O.line_params(base, 1200.0, 0.0, 18.0, 1400.0)
    np.testing.assert_allclose(S1, S0 / 2, rtol=1e-15)                        # k ~ 1/Q
    S2, _, a2, _ = O.line_params(base, 1200.0, 0.0, 72.0, 700.0)
    np.testing.assert_allclose(S2, S0 / 4, rtol=1e-15)                        # S ~ 1/m
    np.testing.assert_allclose(a2, a0 / 2, rtol=1e-15)                        # alpha_D ~ m^-1/2
    dbl = dict(base, A=base["A"] * 2, g_up=base["g_up"] * 3)
    S3, g3, _, _ = O.line_params(dbl, 1200.0, 0.0, 18.0, 700.0)
    np.testing.assert_allclose(S3, S0 * 6, rtol=1e-15)                        # S ~ A g'
    np.testing.assert_allclose(g3, g0 * 2, rtol=1e-15)                        # P = 0: Gamma_L = A/(4 pi c)
    # Eq. 15 x Eq. 16 == Eq. 9: S' = g' A/(8 pi c nu0^2 m), T-part = e^{-E hc/kT}(1-e^{-hc nu0/kT})/Q
    c2 = H * C_CM / KB
    m = 18.0 / NA
    Sp = base["g_up"] * base["A"] / (8 * math.pi * C_CM * base["nu0"] ** 2 * m)
    Tpart = np.exp(-c2 * base["E_low"] / 1200.0) * (1 - np.exp(-c2 * base["nu0"] / 1200.0)) / 700.0
    np.testing.assert_allclose(S0, Sp * Tpart, rtol=1e-13)
    # high-temperature limit of the stimulated-emission factor (needs expm1, R15)
    tiny = _lines(nu0=[1e-6])
    St, _, _, _ = O.line_params(tiny, 1000.0, 1.0, 18.0, 1.0)
    lim = 1.0 / (8 * math.pi * C_CM * m * 1e-12) * (c2 * 1e-6 / 1000.0)
    assert St[0] == pytest.approx(lim, rel=1e-8)


def test_invalid_lines_are_skipped():
    L = _lines(nu0=[0.0, -5.0, np.nan, 100.0, 100.0, 100.0], A=[1, 1, 1, -1.0, np.inf, 1.0])
    S, gL, aD, valid = O.line_params(L, 1000.0, 1.0, 18.0, 10.0)
    assert valid.tolist() == [0, 0, 0, 0, 0, 1]
    assert np.all(S[:5] == 0.0) and S[5] > 0
    k, ev = O.opacity_bins(L, dict(T=1000.0, P_atm=1.0, mass_amu=18.0, Q=10.0), (0.0, 200.0, 1.0), 25.0,
                           np.arange(200))
    assert ev == 51 and k[100] > 0 and k[10] == 0.0


def test_grid_size_and_extents_brute_force():
    assert O.grid_size(0.0, 2000.0, 0.1) == 20000
    assert O.grid_size(0.0, 10000.0, 0.01) == 1000000
    assert O.grid_size(0.0, 30000.0, 0.01) == 3000000
    assert O.grid_size(0.0, 50000.0, 0.01) == 5000000
    rng = np.random.default_rng(7)
    numin, dnu, N, cut = 50.0, 0.25, 400, 7.3
    nu0 = rng.uniform(30.0, 170.0, 500)                  # some centres off the grid on both sides
    ilo, ihi, jc = O.extents(nu0, None, numin, dnu, N, cut)
    nu = numin + np.arange(N) * dnu
    for l in range(nu0.size):
        inside = np.nonzero(np.abs(nu - nu0[l]) <= cut)[0]
        if inside.size == 0:
            assert ilo[l] > ihi[l]
        else:
            assert (ilo[l], ihi[l]) == (inside[0], inside[-1])
        assert jc[l] == math.floor((nu0[l] - numin) / dnu)
    ilo, ihi, _ = O.extents(nu0, None, numin, dnu, N, 0.0)   # uncut
    assert np.all(ilo == 0) and np.all(ihi == N - 1)
    ilo, ihi, _ = O.extents(nu0, None, numin, dnu, N, np.inf)
    assert np.all(ilo == 0) and np.all(ihi == N - 1)


def test_three_lines_eleven_bins_written_out():
    """k_i = sum_l S_l V_l(nu_i) with S from Eq. 9 typed here and V through scipy's wofz."""
    T, P, mass, Q = 800.0, 0.5, 28.0, 150.0
    numin, dnu, N, cut = 99.5, 0.1, 11, 0.35
    L = _lines(nu0=[99.93, 100.0, 100.41], A=[2.0, 0.5, 30.0], g_up=[3.0, 5.0, 1.0],
               E_low=[120.0, 0.0, 900.0], gamma_ref=[0.09, 0.03, 0.06], n_exp=[0.5, 0.7, 0.62])
    m = mass / NA
    c2 = H * C_CM / KB
    expect = np.zeros(N)
    for l in range(3):
        nu0, A, g, E, gam, nx = (L[k][l] for k in O.FIELDS)
        S = A * g / (8 * math.pi * C_CM * m * nu0 ** 2 * Q) * math.exp(-c2 * E / T) * (1 - math.exp(-c2 * nu0 / T))
        aD = nu0 / C_CM * math.sqrt(2 * KB * T / m)
        gL = A / (4 * math.pi * C_CM) + gam * (296.0 / T) ** nx * P
        for i in range(N):
            nu = numin + i * dnu
            if abs(nu - nu0) <= cut:
                expect[i] += S * special.wofz(((nu - nu0) + 1j * gL) / aD).real / (aD * math.sqrt(math.pi))
    k, ev = O.opacity_bins(L, dict(T=T, P_atm=P, mass_amu=mass, Q=Q), (numin, numin + N * dnu, dnu), cut,
                           np.arange(N))
    np.testing.assert_allclose(k, expect, rtol=1e-11)
    assert ev == 7 + 7 + 5          # bins within 0.35 of 99.93, 100.0, 100.41 on 99.5..100.5


def test_linearity_and_permutation():
    from workload import linelists as W
    L = W.to_numpy(W.make_lines(1, n=600))
    cond, grid = W.conditions(1), W.CONFIGS[1]["grid"]
    bins = np.arange(0, 20000, 37)
    k, _ = O.opacity_bins(L, cond, grid, 25.0, bins)
    A = {f: v[:250] for f, v in L.items()}
    B = {f: v[250:] for f, v in L.items()}
    ka, _ = O.opacity_bins(A, cond, grid, 25.0, bins)
    kb, _ = O.opacity_bins(B, cond, grid, 25.0, bins)
    np.testing.assert_allclose(ka + kb, k, rtol=1e-13)
    perm = np.random.default_rng(3).permutation(600)
    kp, _ = O.opacity_bins({f: v[perm] for f, v in L.items()}, cond, grid, 25.0, bins)
    np.testing.assert_allclose(kp, k, rtol=1e-13)
    # the windowed driver (sorted lines, narrowed range) equals the plain definition
    kg, _ = O.opacity_grid(L, cond, grid, 25.0)
    np.testing.assert_allclose(kg[bins], k, rtol=1e-13)


def test_integrated_opacity_equals_sum_S_minus_wing_loss():
    """Resolved lines on a fine grid: sum_i k_i dnu = sum_l S_l (1 - loss_l)."""
    rng = np.random.default_rng(11)
    n = 12
    L = _lines(nu0=rng.uniform(2990.0, 3010.0, n), A=10 ** rng.uniform(-2, 1, n), g_up=rng.integers(1, 9, n),
               E_low=rng.uniform(0, 3000, n), gamma_ref=rng.uniform(0.05, 0.1, n), n_exp=rng.uniform(0.5, 0.75, n))
    cond = dict(T=700.0, P_atm=1.0, mass_amu=18.0, Q=200.0)
    cut, dnu = 12.0, 2.5e-4
    grid = (2970.0, 3030.0, dnu)
    k, _ = O.opacity_grid(L, cond, grid, cut, block=4096)
    S, gL, aD, _ = O.line_params(L, **cond)
    assert gL.min() / dnu > 50 and aD.min() / dnu > 15
    loss = 1 - 2 / np.pi * np.arctan(cut / gL) + gL / np.pi * aD ** 2 * cut / (cut ** 2 + gL ** 2) ** 2
    assert k.sum() * dnu == pytest.approx(np.sum(S * (1 - loss)), rel=2e-6)
