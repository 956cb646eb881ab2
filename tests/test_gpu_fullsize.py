"""Parity at BASELINE.json's FULL sizes, in the launch configuration bench.py times — `-m gpu`.

The oracle cannot run 2.7e11 cell updates in seconds, so it computes sampled outputs one by one:
  - long lines (configs 2, 4): pin P7 (domain of dependence, tests/test_oracle_pins.py) makes a
    windowed oracle run around a probe bit-identical to the full-line oracle, so every probe record
    and 64 random 4096-node windows of the final state are checked against windowed runs;
  - batches (configs 3, 5): grids are independent; EVERY grid is compared with the OpenMP oracle (in chunks), the grids
    with the extreme drawn parameters first.
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
    wp_max = max(float(w.media(lo, hi)[0].max()) for lo, hi in ((0, min(w.ncells, 1 << 21)), (w.ncells // 2, w.ncells // 2 + 1)))
    floors = {"E": peak, "H": peak / 376.73, "J": 8.854e-12 * wp_max ** 2 * 20e-12 * peak}
    worst_ns = {"E": 0.0, "H": 0.0, "J": 0.0}
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
            # the north_star gate itself, for all three fields: error against the field peak of the GRID — E: the
            # record peak; H: that over the vacuum impedance; J: eps0 wp_max^2 tau x peak (tau = 20 ps, the source
            # width) — the floors of tests/test_gpu_parity.py::check_fields
            assert err <= TOL[dtype] * floors[name], (name, a, err, floors[name])
            worst_ns[name] = max(worst_ns[name], err / floors[name])
    print(f"{w.name} {dtype}: worst final-state window error / window peak {worst_win:.3e}; against the grid peak "
          f"E {worst_ns['E']:.3e}, H {worst_ns['H']:.3e}, J {worst_ns['J']:.3e}")


def test_config2_full(rk):
    """1e7 nodes, 2000 steps, periodic random slabs (fp64)."""
    _line_parity(rk, wl.config2(), "f64")


@pytest.mark.parametrize("dtype", ["f64", "f32"])
def test_config4_full(rk, dtype):
    """2^28 nodes, 1000 steps, tanh profile, six per-node coefficient arrays — the bench.py workload."""
    _line_parity(rk, wl.config4(), dtype)


# ---- batches (configs 3, 5): EVERY grid against the OpenMP build of the oracle (pin P9: bit-identical to the serial
# build), in chunks so that host memory stays bounded.  SURVEY §8(d) "CPU baseline plan" / BASELINE.md §3: all grids when
# the oracle finishes in time, else >= 512 grids that include the extremes of every drawn parameter.  The grids are
# therefore visited in the order: extremes first, then all grids in contiguous chunks; the loop stops early only when
# BATCH_BUDGET_S of oracle time are spent (a slow host), never before 512 grids, and the test prints exactly how many
# grids were compared.
BATCH_BUDGET_S = 330.0
_ORACLE_CACHE = {}


def _oracle_batch(w, key, extremes, field, chunk):
    """oracle results [nbatch, ...] (NaN rows where the budget ran out), cached per workload so that the fp32 and fp64
    cases share one oracle run.  Order: the extreme grids one by one, then contiguous chunks of `chunk` grids from grid 0
    (the draws are i.i.d. per grid, so a prefix is as good a seeded sample as any)."""
    import time
    if key in _ORACLE_CACHE:
        return _ORACLE_CACHE[key]
    out, done = None, np.zeros(w.nbatch, bool)
    t0 = time.perf_counter()
    groups = [(int(g), int(g) + 1) for g in dict.fromkeys(extremes)]
    groups += [(b0, min(w.nbatch, b0 + chunk)) for b0 in range(0, w.nbatch, chunk)]
    for b0, b1 in groups:
        if done[b0:b1].all():
            continue
        if done.sum() >= 512 and time.perf_counter() - t0 > BATCH_BUDGET_S:
            break
        r = oracle.run_workload(w, b0=b0, b1=b1, omp=b1 - b0 > 1)[field]
        if out is None:
            out = np.full((w.nbatch,) + r.shape[1:], np.nan)
        out[b0:b1] = r
        done[b0:b1] = True
    _ORACLE_CACHE[key] = (out, done, time.perf_counter() - t0)
    return _ORACLE_CACHE[key]


def _batch_check(name, dtype, gpu, ref, done, extremes, secs):
    assert done[list(extremes)].all() and done.sum() >= min(512, len(done))
    idx = np.flatnonzero(done)
    d = np.abs(gpu[idx].astype(np.float64) - ref[idx]).reshape(len(idx), -1).max(1)
    pk = np.abs(ref[idx]).reshape(len(idx), -1).max(1)
    assert np.all(pk > 0), "vacuous: an oracle record is identically zero"
    err = d / pk
    worst = int(idx[np.argmax(err)])
    print(f"{name} {dtype}: {len(idx)} of {len(done)} grids compared with the oracle ({secs:.0f} s of OpenMP oracle time), "
          f"worst per-grid error {err.max():.3e} at grid {worst}, median {np.median(err):.3e}")
    assert err.max() <= TOL[dtype], (worst, err.max())


def test_config3_full(rk):
    """4096 grids x 4096 nodes x 20 000 steps, full probe time series (the R/T sweep): every grid."""
    w = wl.config3()
    s = rk.Sim.from_workload(w, "f64")
    s.run(w.nsteps)
    rec = s.read_probes()
    assert s.counter(rk.CTR_KERNEL_USED) == rk.KERNEL_RESIDENT and rec.shape == (4096, 2, 20000)
    s.close()
    wp, nu = w.media(2000, 2401, 0, 4096)      # the slab starts at node 2000 and is 40..400 nodes thick
    M = (wp > 0).sum(1)
    assert M.min() >= 40 and M.max() <= 400
    extremes = [0, 4095] + [int(f(a)) for a in (M, wp[:, 0], nu[:, 0]) for f in (np.argmin, np.argmax)]
    ref, done, secs = _oracle_batch(w, "config3", extremes, "rec", 128)
    _batch_check(w.name, "f64", rec, ref, done, extremes, secs)


def _config5_extremes(w):
    """grids holding the smallest / largest of each of the 8 layer widths, layer wp, layer nu, and of the total thickness"""
    ex = [0, w.nbatch - 1]
    widths, wps, nus = [], [], []
    for b0 in range(0, w.nbatch, 8192):
        wp, nu = w.media(319, 722, b0, min(w.nbatch, b0 + 8192))      # node 319 is vacuum; 8 layers of <= 50 nodes
        key = wp + 1e-3 * nu
        edges = np.nonzero(np.diff(key, axis=1) != 0)
        e = edges[1].reshape(wp.shape[0], 9)                           # 9 interfaces per grid
        widths.append(np.diff(e, axis=1))
        rows = np.arange(wp.shape[0])[:, None]
        wps.append(wp[rows, e[:, :8] + 1])
        nus.append(nu[rows, e[:, :8] + 1])
    widths, wps, nus = np.concatenate(widths), np.concatenate(wps), np.concatenate(nus)
    assert widths.min() >= 5 and widths.max() <= 50
    for a in (widths, wps, nus):
        for l in range(8):
            ex += [int(np.argmin(a[:, l])), int(np.argmax(a[:, l]))]
    tot = widths.sum(1)
    ex += [int(np.argmin(tot)), int(np.argmax(tot))]
    return ex


@pytest.mark.parametrize("dtype", ["f64", "f32"])
def test_config5_full(rk, dtype):
    """65 536 grids x 1024 nodes x 5000 steps, |DFT| at 64 frequencies: every grid (one oracle run serves both types)."""
    w = wl.config5()
    s = rk.Sim.from_workload(w, dtype)
    s.run(w.nsteps)
    mag = s.read_probes().astype(np.float64)
    assert mag.shape == (65536, 2, 64) and s.counter(rk.CTR_KERNEL_USED) == rk.KERNEL_RESIDENT
    s.close()
    extremes = _config5_extremes(w)
    ref, done, secs = _oracle_batch(w, "config5", extremes, "dft_mag", 2048)
    _batch_check(w.name, dtype, mag, ref, done, extremes, secs)
