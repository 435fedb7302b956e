"""Pins for the oracle's line profile V(nu) = Re w(x+iy)/(alpha_D sqrt(pi))
(R1; Eq. 1-2, Eq. 11-13)."""
import math

import numpy as np
import pytest
from scipy import integrate

from oracle import hk_oracle as O


def test_unit_area():
    for gL, aD in [(0.05, 0.02), (0.004, 0.03), (0.3, 0.001)]:
        f = lambda nu: O.profile(nu, 100.0, gL, aD)
        w = max(gL, aD)
        core, _ = integrate.quad(f, 100.0 - 200 * w, 100.0 + 200 * w, points=[100.0],
                                 epsabs=0, epsrel=1e-11, limit=4000)
        # beyond +-200 w the profile is Lorentzian to ~1e-5 relative of a ~1e-3 tail
        tail = 1.0 - 2.0 / math.pi * math.atan(200 * w / gL)
        assert core + tail == pytest.approx(1.0, abs=3e-7)


def test_pure_lorentz_limit():
    gL = 0.07
    for d in [0.0, 0.01, 0.07, 0.5, 25.0]:
        v = O.profile(1000.0 + d, 1000.0, gL, 1e-9)
        assert v == pytest.approx(gL / (math.pi * (d * d + gL * gL)), rel=1e-9)


def test_pure_gauss_limit():
    aD = 0.03
    for d in [0.0, 0.01, 0.05, 0.1]:
        v = O.profile(1000.0 + d, 1000.0, 0.0, aD)
        assert v == pytest.approx(math.exp(-(d / aD) ** 2) / (aD * math.sqrt(math.pi)), rel=1e-11)  # nu0+d rounds
        v2 = O.profile(1000.0 + d, 1000.0, 1e-12, aD)
        assert v2 == pytest.approx(v, rel=1e-6)     # Lorentz wing term y/(sqrt(pi) x^2) is real


def test_mirror_symmetry_on_grid_point():
    for d in [0.125, 0.5, 3.0]:                      # exactly representable offsets
        a = O.profile(512.0 + d, 512.0, 0.031, 0.017)
        b = O.profile(512.0 - d, 512.0, 0.031, 0.017)
        assert a == pytest.approx(b, rel=1e-13)


def test_wing_loss_formula():
    """area beyond +-c = 1 - (2/pi) atan(c/G) + (G/pi) aD^2 c/(c^2+G^2)^2 + O(aD^4/c^4)
    (derived from the second asymptotic term) vs quadrature."""
    gL, aD, c = 0.05, 0.02, 25.0
    f = lambda nu: O.profile(nu, 0.0, gL, aD)
    far, _ = integrate.quad(f, c, np.inf, epsabs=0, epsrel=1e-12, limit=2000)
    loss = 1.0 - 2.0 / math.pi * math.atan(c / gL) + gL / math.pi * aD ** 2 * c / (c * c + gL * gL) ** 2
    assert 2.0 * far == pytest.approx(loss, rel=1e-9)
