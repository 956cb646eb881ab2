"""The R/T parameter sweep of BASELINE config 3 done end to end on the device (second half;
PAPER.md:130-132: reflection and transmission coefficients by Fourier transform of the probe records) — `-m gpu`.

The probe records are reduced on the device to complex DFT accumulators (row a7); a second, all-vacuum run gives the
incident spectrum; |R| = |X_slab - X_vac| / |X_vac| at the reflected probe, |T| = |X_slab| / |X_vac| at the transmitted
one.  Checked against (i) the oracle's accumulators, (ii) the closed-form slab solution for every grid's drawn
(thickness, wp, nu) — north_star check (c), here across the sweep.
"""
import numpy as np
import pytest

import oracle
from paper_1709_00821_b200 import workloads as wl

pytestmark = pytest.mark.gpu
C0 = 299792458.0
NB = 64
FREQS = np.linspace(2e9, 26e9, 13)          # inside the pulse band (1.3-28 GHz)


def _slab_rt(f, wp, nu, d):
    w = 2 * np.pi * f
    n = np.sqrt(1 - wp ** 2 / (w ** 2 - 1j * w * nu))
    n = np.where(n.imag > 0, -n, n)
    k = n * w / C0
    r = (1 - n) / (1 + n)
    P = np.exp(-2j * k * d)
    return np.abs(r * (1 - P) / (1 - r ** 2 * P)), np.abs((1 - r ** 2) * np.exp(-1j * k * d) / (1 - r ** 2 * P))


@pytest.mark.parametrize("dtype,tol_x,tol_rt", [("f64", 1e-12, 1e-3), ("f32", 1e-5, 1e-3)])
def test_config3_sweep_reflection_transmission(dtype, tol_x, tol_rt):
    from paper_1709_00821_b200 import rketd
    w = wl.config3(nbatch=NB)
    w.dft_freqs = FREQS
    wv = wl.config3(nbatch=1)
    wv.dft_freqs = FREQS
    wv.media = lambda lo=0, hi=w.ncells, b0=0, b1=1: (np.zeros((b1 - b0, hi - lo)), np.zeros((b1 - b0, hi - lo)))
    X = {}
    for key, ww in (("slab", w), ("vac", wv)):
        s = rketd.Sim.from_workload(ww, dtype)
        s.run(ww.nsteps)
        X[key] = s.read_probe_dft()
        mag = s.read_probes().astype(np.float64)
        s.close()
        assert np.max(np.abs(np.abs(X[key]) - mag)) <= 1e-6 * np.max(mag)        # read_probes = |read_probe_dft|
    # (i) against the oracle's accumulators, per grid, relative to the grid's largest bin
    ref = oracle.run_workload(w, omp=True)["dft"]
    err = np.abs(X["slab"] - ref).reshape(NB, -1).max(1) / np.abs(ref).reshape(NB, -1).max(1)
    assert err.max() <= tol_x, err.max()
    # (ii) against the closed form, every grid of the sweep
    inc = X["vac"][0]
    R = np.abs(X["slab"][:, 0] - inc[0]) / np.abs(inc[0])
    T = np.abs(X["slab"][:, 1]) / np.abs(inc[1])
    wp, nu = w.media(2000, 2001, 0, NB)
    thick = (w.media(0, w.ncells, 0, NB)[0] > 0).sum(1)
    worst = 0.0
    for g in range(NB):
        Ra, Ta = _slab_rt(FREQS, wp[g, 0], nu[g, 0], thick[g] * w.dz)
        worst = max(worst, np.abs(R[g] - Ra).max(), np.abs(T[g] - Ta).max())
    print(f"sweep of {NB} slabs, {dtype}: worst |R|, |T| error against the closed form {worst:.2e}")
    assert worst <= tol_rt
