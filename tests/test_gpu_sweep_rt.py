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
    X, sims = {}, {}
    for key, ww in (("slab", w), ("vac", wv)):
        s = rketd.Sim.from_workload(ww, dtype)
        s.run(ww.nsteps)
        X[key] = s.read_probe_dft()
        mag = s.read_probes().astype(np.float64)
        sims[key] = s
        assert np.max(np.abs(np.abs(X[key]) - mag)) <= 1e-6 * np.max(mag)        # read_probes = |read_probe_dft|
    R_dev, T_dev = sims["slab"].read_sweep_rt(sims["vac"], 0, 1)                 # |R|, |T| formed on the device
    for s in sims.values():
        s.close()
    # (i) against the oracle's accumulators, per grid, relative to the grid's largest bin
    ref = oracle.run_workload(w, omp=True)["dft"]
    err = np.abs(X["slab"] - ref).reshape(NB, -1).max(1) / np.abs(ref).reshape(NB, -1).max(1)
    assert err.max() <= tol_x, err.max()
    # (ii) against the closed form, every grid of the sweep
    inc = X["vac"][0]
    R = np.abs(X["slab"][:, 0] - inc[0]) / np.abs(inc[0])
    T = np.abs(X["slab"][:, 1]) / np.abs(inc[1])
    assert np.max(np.abs(R_dev - R)) <= 1e-13 and np.max(np.abs(T_dev - T)) <= 1e-13     # the same two quotients
    R, T = R_dev, T_dev
    wp, nu = w.media(2000, 2001, 0, NB)
    thick = (w.media(0, w.ncells, 0, NB)[0] > 0).sum(1)
    worst = 0.0
    for g in range(NB):
        Ra, Ta = _slab_rt(FREQS, wp[g, 0], nu[g, 0], thick[g] * w.dz)
        worst = max(worst, np.abs(R[g] - Ra).max(), np.abs(T[g] - Ta).max())
    print(f"sweep of {NB} slabs, {dtype}: worst |R|, |T| error against the closed form {worst:.2e}")
    assert worst <= tol_rt


def test_on_device_rt_of_the_config1_slab_against_the_golden_table():
    """north_star check (c) through the CUDA path alone: config 1's slab (9 mm, wp = 2 pi 28.7e9, nu = 2e10) and an
    all-vacuum grid, probe DFT at the frequencies of tests/golden/slab_rt_analytic.txt that lie in the pulse band,
    |R| and |T| formed on the device by rketd_read_sweep_rt, within 1e-2 of the analytic values."""
    import os
    from paper_1709_00821_b200 import rketd
    tab = np.loadtxt(os.path.join(os.path.dirname(__file__), "golden", "slab_rt_analytic.txt"))
    tab = tab[(tab[:, 0] >= 2.0) & (tab[:, 0] <= 26.0)]              # the band where the incident spectrum is >= 1e-2 of its peak
    assert len(tab) >= 5
    freqs = tab[:, 0] * 1e9
    sims = []
    for vacuum in (False, True):
        w = wl.config1(nsteps=12000)
        s = rketd.Sim(w.ncells, 1, w.dz, w.dt, "f64")
        wp, nu = w.media_full()
        s.set_media(wp * (0.0 if vacuum else 1.0), nu * (0.0 if vacuum else 1.0))
        s.set_source(w.src_kind, w.src_params, w.src_cell)
        s.set_probes(w.probes)
        s.set_probe_dft(freqs)
        s.run(w.nsteps)
        sims.append(s)
    R, T = sims[0].read_sweep_rt(sims[1], 0, 1)
    for s in sims:
        s.close()
    print("f GHz, |R| device / analytic, |T| device / analytic")
    for f, r, t, ra, ta in zip(tab[:, 0], R[0], T[0], tab[:, 1], tab[:, 2]):
        print(f"{f:5.1f}  {r:.6f} / {ra:.6f}   {t:.6f} / {ta:.6f}")
    assert np.max(np.abs(R[0] - tab[:, 1])) <= 1e-2 and np.max(np.abs(T[0] - tab[:, 2])) <= 1e-2
