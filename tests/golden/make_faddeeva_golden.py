"""Writes tests/golden/faddeeva_mpmath.txt: Re w(x + i y) = Re[exp(-z^2) erfc(-i z)] on a small lattice, computed
with mpmath at 60 significant digits -- a definition-level value (Faddeeva function; the Voigt profile is its real
part, Eq. 1-2) that depends on neither oracle/ nor the CUDA library.

    python tests/golden/make_faddeeva_golden.py
"""
import os

import mpmath as mp

mp.mp.dps = 60
XS = ["0", "0.1", "0.5", "0.75", "1", "1.7", "2.5", "4", "6.3", "10", "24.9", "25.1", "80", "299", "301", "5000", "1e6"]
YS = ["0.001", "0.02", "0.13", "0.5", "1", "2.2", "8", "30", "400"]


def K(x, y):
    z = mp.mpc(mp.mpf(x), mp.mpf(y))
    return mp.re(mp.exp(-z * z) * mp.erfc(-1j * z))


def main():
    out = os.path.join(os.path.dirname(os.path.abspath(__file__)), "faddeeva_mpmath.txt")
    with open(out, "w") as f:
        f.write("# x y Re_w(x+iy)   (mpmath 60 digits, printed to 20; made by make_faddeeva_golden.py)\n")
        for x in XS:
            for y in YS:
                f.write(f"{x} {y} {mp.nstr(K(x, y), 20)}\n")
    print(out)


if __name__ == "__main__":
    main()
