"""Pins for the oracle's Lorentz and Doppler profile options (section 2.1: "pure Doppler and Lorentzian
profiles"), against closed forms and against the (separately pinned) Voigt oracle in its limits."""
import numpy as np
import pytest

from oracle import hk_oracle as O

COND = dict(T=1100.0, P_atm=0.5, mass_amu=44.0, Q=300.0)


def _one(nu0=500.0, gamma_ref=0.08, A=2.0):
    return dict(nu0=np.array([nu0]), A=np.array([A]), g_up=np.array([5.0]), E_low=np.array([800.0]),
                gamma_ref=np.array([gamma_ref]), n_exp=np.array([0.7]))


def test_lorentz_half_width_area_and_peak():
    L = _one()
    S, gL, aD, _ = O.line_params(L, **COND)
    dnu = gL[0] / 64.0                                         # Gamma_L = 64 bins exactly, centre on grid point 16384
    grid = (500.0 - 16384 * dnu, 500.0 + 16384 * dnu, dnu)
    k, _ = O.opacity_grid(L, COND, grid, 0.0, profile="lorentz")
    jc = 16384
    assert k[jc] == pytest.approx(S[0] / (np.pi * gL[0]), rel=1e-12)              # peak S/(pi Gamma_L)
    assert k[jc + 64] / k[jc] == pytest.approx(0.5, rel=1e-9)                       # half maximum at Delta = Gamma_L
    c = 8000 * dnu
    kc, _ = O.opacity_grid(L, COND, grid, c, profile="lorentz")
    area = kc.sum() * grid[2] / S[0]
    assert area == pytest.approx((2.0 / np.pi) * np.arctan(c / gL[0]), rel=3e-4)    # trapezoid sum of a resolved line


def test_doppler_half_width_area_and_peak():
    L = _one()
    S, gL, aD, _ = O.line_params(L, **COND)
    hwhm = aD[0] * np.sqrt(np.log(2.0))                        # Gamma_D of Eq. 3 (L77-81)
    dnu = hwhm / 32.0
    grid = (500.0 - 1024 * dnu, 500.0 + 1024 * dnu, dnu)
    k, _ = O.opacity_grid(L, COND, grid, 0.0, profile="doppler")
    jc = 1024
    assert k[jc] == pytest.approx(S[0] / (aD[0] * np.sqrt(np.pi)), rel=1e-9)
    assert k[jc + 32] / k[jc] == pytest.approx(0.5, rel=1e-6)
    assert k.sum() * grid[2] == pytest.approx(S[0], rel=1e-9)                       # unit area (Gaussian: spectral accuracy)


def test_voigt_limits_reach_both_profiles():
    """alpha_D -> 0 (heavy, cold emitter far from the centre): Voigt -> Lorentz; Gamma_L -> 0 (no pressure, weak A):
    Voigt -> Doppler.  Ties the new options to the pinned w(z)."""
    grid = (480.0, 520.0, 0.05)
    L = _one()
    cold = dict(COND, mass_amu=4.0e9)                          # alpha_D 1e4 times smaller, S still finite
    kv, _ = O.opacity_grid(L, cold, grid, 0.0)
    kl, _ = O.opacity_grid(L, cold, grid, 0.0, profile="lorentz")
    far = np.abs(np.arange(kv.size) * 0.05 + 480.0 - 500.0) > 0.02
    assert np.abs(kv[far] / kl[far] - 1.0).max() <= 1e-6
    Lw = _one(gamma_ref=1e-8, A=1e-12)                         # y = Gamma_L/alpha_D ~ 1e-6
    fine = (499.95, 500.05, 2e-4)
    S, gL, aD, _ = O.line_params(Lw, **COND)
    assert 1e-7 < gL[0] / aD[0] < 1e-5
    kv, _ = O.opacity_grid(Lw, COND, fine, 0.0)
    kd, _ = O.opacity_grid(Lw, COND, fine, 0.0, profile="doppler")
    x = (fine[0] + np.arange(kv.size) * fine[2] - 500.0) / aD[0]
    core = np.abs(x) <= 1.5                                    # further out the Lorentz wing y/(sqrt(pi) x^2) shows
    assert core.sum() > 10
    assert np.abs(kv[core] / kd[core] - 1.0).max() <= 5e-5


def test_plinth_uses_the_selected_profile():
    L = _one()
    grid, cut = (490.0, 510.0, 0.01), 4.0
    S, gL, aD, _ = O.line_params(L, **COND)
    k0, _ = O.opacity_grid(L, COND, grid, cut, profile="lorentz")
    k1, _ = O.opacity_grid(L, COND, grid, cut, profile="lorentz", plinth=True)
    inside = k0 > 0
    assert np.abs((k0 - k1)[inside] - S[0] * gL[0] / (np.pi * (cut * cut + gL[0] ** 2))).max() <= 1e-12 * k0.max()


def test_binned_gaussian_conserves_the_integral_and_reaches_its_limits():
    """Bin average of the Doppler profile (R26): sum_i V_i dnu = 1 at ANY resolution (the erf differences
    telescope), the Doppler profile when the line is resolved, one bin of height 1/dnu when it is not."""
    L = _one()
    S, gL, aD, _ = O.line_params(L, **COND)
    a = aD[0]
    for dnu in (a / 40.0, a / 3.0, a * 2.5, a * 300.0):
        n = 2000
        grid = (500.0 - (n + 0.3) * dnu, 500.0 + (n - 0.3) * dnu, dnu)       # centre 0.3 bins off a grid point
        k, _ = O.opacity_grid(L, COND, grid, 0.0, profile="binned_gaussian")
        assert k.sum() * dnu == pytest.approx(S[0], rel=1e-10)
        if dnu < a / 30.0:
            kd, _ = O.opacity_grid(L, COND, grid, 0.0, profile="doppler")
            x = (grid[0] + np.arange(k.size) * dnu - 500.0) / a
            m = np.abs(x) < 3.0
            h = dnu / (2 * a)
            assert np.abs(k[m] / kd[m] - (1.0 + h * h * (2 * x[m] ** 2 - 1) / 3.0)).max() <= 1e-6   # second-order bin average
        if dnu > 100.0 * a:
            jc = int(np.argmax(k))
            assert k[jc] * dnu == pytest.approx(S[0], rel=1e-10) and np.count_nonzero(k > 1e-30 * k[jc]) == 1
    # symmetric about the centre when it sits on a grid point
    grid = (500.0 - 50 * a, 500.0 + 50 * a, a / 4.0)
    k, _ = O.opacity_grid(L, COND, grid, 0.0, profile="binned_gaussian")
    assert np.abs(k[1:] - k[1:][::-1]).max() <= 1e-9 * k.max()         # (grid points round differently left and right)
