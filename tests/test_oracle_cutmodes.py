"""Pins for the oracle's width-relative cutting lengths ("a fixed cutting length, a fraction of the
Doppler half-width, or a fraction of the Lorentzian half-width"; R25)."""
import numpy as np
import pytest

from oracle import hk_oracle as O

COND = dict(T=900.0, P_atm=0.8, mass_amu=28.0, Q=250.0)
GRID = (0.0, 100.0, 0.01)


def _lines(n=300, seed=0):
    rng = np.random.default_rng(seed)
    return dict(nu0=rng.uniform(10, 90, n), A=10 ** rng.uniform(-3, 1, n), g_up=rng.integers(1, 9, n).astype(float),
                E_low=rng.uniform(0, 3000, n), gamma_ref=rng.uniform(0.02, 0.1, n), n_exp=rng.uniform(0.5, 0.75, n))


@pytest.mark.parametrize("mode,factor", [("lorentz", 50.0), ("doppler", 400.0)])
def test_each_line_is_cut_at_its_own_multiple_of_its_half_width(mode, factor):
    """One line at a time: the support of k is exactly the bins within factor x half-width of the centre, and inside it
    the values are those of the fixed-cut run with that cutting length."""
    L = _lines(12, seed=3)
    S, gL, aD, _ = O.line_params(L, **COND)
    hw = gL if mode == "lorentz" else aD * np.sqrt(np.log(2.0))
    nu = GRID[0] + np.arange(O.grid_size(*GRID)) * GRID[2]
    for l in range(12):
        one = {f: v[l:l + 1] for f, v in L.items()}
        k, ev = O.opacity_grid(one, COND, GRID, factor, cut_mode=mode)
        c = factor * hw[l]
        inside = np.abs(nu - L["nu0"][l]) <= c
        edge = np.abs(np.abs(nu - L["nu0"][l]) - c) < 1e-9          # bins exactly at the cut may round either way
        assert np.array_equal((k > 0)[~edge], inside[~edge]) and ev == int((k > 0).sum())
        kf, _ = O.opacity_grid(one, COND, GRID, c)
        assert np.array_equal(k[~edge], kf[~edge])


def test_sum_over_lines_and_fixed_mode_unchanged():
    L = _lines()
    k, ev = O.opacity_grid(L, COND, GRID, 60.0, cut_mode="lorentz")
    parts = [O.opacity_grid({f: v[a:b] for f, v in L.items()}, COND, GRID, 60.0, cut_mode="lorentz") for a, b in ((0, 100), (100, 300))]
    assert ev == parts[0][1] + parts[1][1]
    assert np.abs(k - (parts[0][0] + parts[1][0])).max() <= 1e-12 * k.max()
    k0, e0 = O.opacity_grid(L, COND, GRID, 5.0)
    k1, e1 = O.opacity_grid(L, COND, GRID, 5.0, cut_mode="fixed")
    assert e0 == e1 and np.array_equal(k0, k1)
    ku, eu = O.opacity_grid(L, COND, GRID, 0.0, cut_mode="doppler")       # no cut: the mode is irrelevant
    assert eu == 300 * O.grid_size(*GRID)


def test_plinth_is_taken_at_the_lines_own_cut():
    L = {f: v[:1] for f, v in _lines(1, seed=5).items()}
    S, gL, aD, _ = O.line_params(L, **COND)
    k0, _ = O.opacity_grid(L, COND, GRID, 30.0, cut_mode="lorentz")
    k1, _ = O.opacity_grid(L, COND, GRID, 30.0, cut_mode="lorentz", plinth=True)
    c = 30.0 * gL[0]
    inside = k0 > 0
    assert np.abs((k0 - k1)[inside] - S[0] * O.profile(L["nu0"][0] + c, L["nu0"][0], gL[0], aD[0])).max() <= 1e-12 * k0.max()
