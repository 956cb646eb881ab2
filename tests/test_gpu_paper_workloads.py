"""The paper's own two workloads on the GPU — `-m gpu`.

Experiment A: probe records against the oracle at the north_star tolerance, and |R|, |T| from the
GPU records against the closed-form slab solution.  Table 2: every line length of the sweep,
1000 steps, probe records and final fields against the oracle (the lengths above 4096 cells run the temporal-
blocking kernel on a handful of tiles, the shorter ones the resident kernel).
"""
import math

import numpy as np
import pytest

import oracle
from paper_1709_00821_b200 import workloads as wl

pytestmark = pytest.mark.gpu
C0 = 299792458.0


@pytest.fixture(scope="module")
def rk():
    from paper_1709_00821_b200 import rketd
    return rketd


def _slab_rt(f, wp, nu, d):
    w = 2 * np.pi * f
    n = np.sqrt(1 - wp ** 2 / (w ** 2 - 1j * w * nu))
    n = np.where(n.imag > 0, -n, n)
    k = n * w / C0
    r = (1 - n) / (1 + n)
    P = np.exp(-2j * k * d)
    return np.abs(r * (1 - P) / (1 - r ** 2 * P)), np.abs((1 - r ** 2) * np.exp(-1j * k * d) / (1 - r ** 2 * P))


def _gpu_records(rk, w, dtype="f64", kernel=0):
    s = rk.Sim.from_workload(w, dtype)
    s.set_plan(kernel, 0, -1)
    s.run(w.nsteps)
    rec = s.read_probes().astype(np.float64)
    used = s.counter(rk.CTR_KERNEL_USED)
    s.close()
    return rec[0], used


@pytest.mark.parametrize("dtype,tol", [("f64", 1e-12), ("f32", 1e-5)])
def test_experiment_A_parity_and_RT(rk, dtype, tol):
    w = wl.paper_exp_a()
    ref = oracle.run_workload(w)["rec"][0]
    tot, used = _gpu_records(rk, w, dtype)
    assert used == rk.KERNEL_RESIDENT
    assert np.max(np.abs(tot - ref)) <= tol * np.max(np.abs(ref))
    wv = wl.paper_exp_a()
    wv.media = lambda lo=0, hi=w.ncells, b0=0, b1=1: (np.zeros((b1 - b0, hi - lo)), np.zeros((b1 - b0, hi - lo)))
    inc, _ = _gpu_records(rk, wv, dtype)
    freqs = np.fft.rfftfreq(w.nsteps, w.dt)
    Ir, It = np.fft.rfft(inc[0]), np.fft.rfft(inc[1])
    R = np.abs(np.fft.rfft(tot[0] - inc[0])) / np.abs(Ir)
    T = np.abs(np.fft.rfft(tot[1])) / np.abs(It)
    band = (np.abs(Ir) >= 1e-2 * np.max(np.abs(Ir))) & (freqs <= 150e9)
    Ra, Ta = _slab_rt(freqs[band], 2 * math.pi * 28.7e9, 2.0e10, 1200 * w.dz)
    assert np.max(np.abs(R[band] - Ra)) < 1e-2 and np.max(np.abs(T[band] - Ta)) < 1e-2     # north_star (c)


@pytest.mark.parametrize("ncells", wl.PAPER_TABLE2_CELLS)
def test_table2_lengths_match_oracle(rk, ncells):
    w = wl.paper_table2(ncells)
    o = oracle.run_workload(w)
    ref, st = o["rec"][0], o["state"]
    s = rk.Sim.from_workload(w, "f64")
    s.run(w.nsteps)
    rec = s.read_probes()[0]
    used = s.counter(rk.CTR_KERNEL_USED)
    E, H, J = s.get_fields()
    s.close()
    assert used == (rk.KERNEL_RESIDENT if ncells <= 20480 else rk.KERNEL_TBLOCK)     # a cluster's registers hold up to ~24 K nodes
    assert np.max(np.abs(ref)) > 0
    assert np.max(np.abs(rec - ref)) <= 1e-12 * np.max(np.abs(ref))
    for g, r in ((E, st.E), (H, st.H), (J, st.J)):
        assert np.max(np.abs(g[0] - r[0])) <= 1e-12 * np.max(np.abs(r))
