"""Parity at BASELINE.json's FULL sizes, in the launch configuration bench.py times — `-m gpu`.

The oracle cannot run 2.7e11 cell updates in seconds, so it computes sampled outputs one by one:
  - long lines (configs 2, 4): pin P7 (domain of dependence, tests/test_oracle_pins.py) makes a
    windowed oracle run around a probe bit-identical to the full-line oracle, so every probe record
    and 64 random 4096-node windows of the final state are checked against windowed runs;
  - batches (configs 3, 5): grids are independent, so a seeded sample of whole grids is checked
    (including the grids with the extreme drawn parameters).
"""
import numpy as np
import pytest

import oracle
from paper_1709_00821_b200 import workloads as wl

pytestmark = pytest.mark.gpu
TOL = {"f64": 1e-12, "f32": 1e-5}
UNIT_ROUNDOFF = {"f64": 2.0 ** -53, "f32": 2.0 ** -24}
# Linear worst-case drift per step, in unit roundoffs of the LOCAL field amplitude: the kernels round
# 7 times per node and step and read 4 stored coefficients that are each rounded once (11 sites); the fp64 oracle
# rounds 9 times and reads 6 rounded coefficients (15 sites, which only count when the GPU also runs in fp64).  The
# lossless leapfrog does not amplify an injected error, so after n steps |gpu - oracle| <= K n u x local amplitude.
DRIFT_K = {"f64": 11 + 15, "f32": 11}


@pytest.fixture(scope="module")
def rk():
    from paper_1709_00821_b200 import rketd
    return rketd


def _line_parity(rk, w, dtype, nwindows=64, wlen=4096):
    import torch
    n = w.nsteps
    s = rk.Sim.from_workload(w, dtype)
    s.run(n)
    rec = s.read_probes().astype(np.float64)
    assert s.counter(rk.CTR_KERNEL_USED) == rk.KERNEL_TBLOCK
    tdt = torch.float64 if dtype == "f64" else torch.float32
    E, H, J = (torch.empty((1, w.ncells), dtype=tdt, device="cuda") for _ in range(3))
    rk.rketd_get_fields(s.h, E, H, J)
    s.close()
    # every probe record against a windowed oracle run (light cone of n steps + 1)
    worst = 0.0
    peak = 0.0
    worst_rel = 0.0
    for i, p in enumerate(w.probes):
        lo, hi = max(0, int(p) - n - 1), min(w.ncells, int(p) + n + 2)
        o = oracle.run_workload(w, cells=(lo, hi))
        j = o["probe_cells"].index(int(p))
        pk = np.max(np.abs(o["rec"][0][j]))
        d = np.max(np.abs(rec[0][i] - o["rec"][0][j]))
        assert pk > 0, ("vacuous: oracle record identically zero at probe", int(p))
        peak, worst, worst_rel = max(peak, pk), max(worst, d), max(worst_rel, d / pk)
    # north_star tolerance: error over every probe sample against the field peak of the grid (SURVEY §8(c)
    # tolerance rule; the source node is a probe of config 4, so the peak is the driven field, ~1)
    assert worst <= TOL[dtype] * peak, (worst, peak)
    # per-probe figure (not gated by the north_star), held to the drift bound above.
    # Observed on B200, n = 1000: 2.3e-13 (fp64, = 2 n u), 6.9e-5 (fp32, = 1.2 n u).
    print(f"{w.name} {dtype}: worst |gpu-oracle|/grid peak {worst / peak:.3e}, worst per-probe {worst_rel:.3e}")
    assert worst_rel <= DRIFT_K[dtype] * n * UNIT_ROUNDOFF[dtype], worst_rel
    # random windows of the final state
    rng = np.random.default_rng(99)
    worst_win = 0.0
    starts = list(rng.integers(0, w.ncells - wlen, nwindows - 3)) + [0, w.ncells - wlen, w.src_cell - wlen // 2]
    for a in starts:
        a = min(max(int(a), 0), w.ncells - wlen)
        lo, hi = max(0, a - n - 1), min(w.ncells, a + wlen + n + 1)
        st = oracle.run_workload(w, cells=(lo, hi))["state"]
        for name, dev, ref in (("E", E, st.E), ("H", H, st.H), ("J", J, st.J)):
            r = ref[0][a - lo:a - lo + wlen].copy()
            g = dev[0, a:a + wlen].cpu().numpy().astype(np.float64)
            if name == "H" and a + wlen == w.ncells:
                r[-1] = 0.0
            # north_star tolerance is relative to the FIELD PEAK of the grid; a window far from the source holds only
            # the 1e-3 noise, so the check here is the stricter window-local one: 1e-12 of the window's own peak in
            # fp64, the drift bound K n u of the window's own peak in fp32 (1e-5 of a 2e-3 local peak is below what
            # 1000 fp32 steps can hold: observed 1.1e-5)
            scale = max(np.max(np.abs(ref)), 1e-300)
            err = np.max(np.abs(g - r))
            worst_win = max(worst_win, err / scale)
            assert err <= max(TOL[dtype], DRIFT_K[dtype] * n * UNIT_ROUNDOFF[dtype] if dtype == "f32" else 0.0) * scale, (name, a, err / scale)
            if name == "E":
                assert err <= TOL[dtype] * peak, (name, a, err, peak)      # the north_star gate itself
    print(f"{w.name} {dtype}: worst final-state window error / window peak {worst_win:.3e}")


def test_config2_full(rk):
    """1e7 nodes, 2000 steps, periodic random slabs (fp64)."""
    _line_parity(rk, wl.config2(), "f64")


@pytest.mark.parametrize("dtype", ["f64", "f32"])
def test_config4_full(rk, dtype):
    """2^28 nodes, 1000 steps, tanh profile, six per-node coefficient arrays — the bench.py workload."""
    _line_parity(rk, wl.config4(), dtype)


def test_config3_full(rk):
    """4096 grids x 4096 nodes x 20 000 steps, full probe time series; 10 sampled grids vs the oracle."""
    w = wl.config3()
    s = rk.Sim.from_workload(w, "f64")
    s.run(w.nsteps)
    rec = s.read_probes()
    assert s.counter(rk.CTR_KERNEL_USED) == rk.KERNEL_RESIDENT and rec.shape == (4096, 2, 20000)
    s.close()
    wp, nu = w.media(2000, 2001, 0, 4096)      # the slab's first node carries each grid's drawn (wp, nu)
    sample = {0, 4095, int(np.argmax(wp)), int(np.argmin(wp)), int(np.argmax(nu)), int(np.argmin(nu))}
    sample |= {int(g) for g in np.random.default_rng(3).integers(0, 4096, 4)}
    for g in sorted(sample):
        ref = oracle.run_workload(w, b0=g, b1=g + 1)["rec"]
        d = np.max(np.abs(rec[g] - ref[0])) / np.max(np.abs(ref))
        assert d <= 1e-12, (g, d)


@pytest.mark.parametrize("dtype", ["f64", "f32"])
def test_config5_full(rk, dtype):
    """65 536 grids x 1024 nodes x 5000 steps, |DFT| at 64 frequencies; 16 sampled grids vs the oracle."""
    w = wl.config5()
    s = rk.Sim.from_workload(w, dtype)
    s.run(w.nsteps)
    mag = s.read_probes().astype(np.float64)
    assert mag.shape == (65536, 2, 64) and s.counter(rk.CTR_KERNEL_USED) == rk.KERNEL_RESIDENT
    s.close()
    sample = sorted({0, 65535} | {int(g) for g in np.random.default_rng(5).integers(0, 65536, 14)})
    for g in sample:
        ref = oracle.run_workload(w, b0=g, b1=g + 1)["dft_mag"]
        d = np.max(np.abs(mag[g] - ref[0])) / np.max(np.abs(ref))
        assert d <= TOL[dtype], (g, d)
