"""Writes tests/golden/slab_rt_analytic.txt: |R|, |T| of a homogeneous Drude slab in vacuum.

Closed form only (no oracle, no CUDA path): the characteristic (ABCD) matrix of one layer
at normal incidence, evaluated in 40-digit arithmetic with mpmath.  This is the "analytical
solution" the paper compares against in Figs. 2-3 without printing it;
parameters are the paper's: wp = 2 pi 28.7e9 rad/s, nu = 2e10 1/s, and a
slab thickness of 9 mm (BASELINE config 1: 120 cells of 75 um).

    python tests/golden/make_slab_rt.py
"""
import os

import mpmath as mp

mp.mp.dps = 40
C0 = mp.mpf(299792458)
WP = 2 * mp.pi * mp.mpf("28.7e9")
NU = mp.mpf("2.0e10")
D = mp.mpf("9e-3")


def rt(f_ghz):
    w = 2 * mp.pi * mp.mpf(f_ghz) * 1e9
    eps = 1 - WP ** 2 / (w ** 2 - 1j * w * NU)          # e^{+jwt}: eps = 1 - wp^2/(w (w - j nu))
    n = mp.sqrt(eps)
    delta = n * w / C0 * D                               # phase thickness
    # layer matrix [[cos d, j sin d / n], [j n sin d, cos d]] between two vacuum half-spaces
    A, B, Cc, Dd = mp.cos(delta), 1j * mp.sin(delta) / n, 1j * n * mp.sin(delta), mp.cos(delta)
    den = A + B + Cc + Dd
    return abs((A + B - Cc - Dd) / den), abs(2 / den)


if __name__ == "__main__":
    out = os.path.join(os.path.dirname(os.path.abspath(__file__)), "slab_rt_analytic.txt")
    with open(out, "w") as fh:
        fh.write("# f_GHz  |R|  |T|   homogeneous Drude slab, wp=2pi*28.7e9, nu=2e10, d=9mm (PAPER.md:123; BASELINE config 1)\n")
        fh.write("# written by tests/golden/make_slab_rt.py (closed form, mpmath 40 digits)\n")
        for f in ["1.0", "2.5", "5.0", "10.0", "15.0", "20.0", "25.0", "28.7", "30.0", "40.0", "60.0"]:
            R, T = rt(f)
            fh.write(f"{f} {mp.nstr(R, 12)} {mp.nstr(T, 12)}\n")
