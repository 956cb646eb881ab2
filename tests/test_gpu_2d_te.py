"""GPU parity of the 2-D TEz path (include/rketd2d.h second half; SURVEY §8(f) NEXT-3 "2-D TMz/TEz") against the CPU
oracle (oracle2d_te_run), through the C ABI.  fp64: max |gpu - oracle| / max |oracle| <= 1e-12 over every probe sample
and over the final fields; fp32: <= 1e-5."""
import numpy as np
import pytest

import oracle
from paper_1709_00821_b200 import workloads as wl

pytestmark = pytest.mark.gpu
TOL = {"f64": 1e-12, "f32": 1e-5}
C0 = 299792458.0
DX = 75e-6
DT = DX / (2 * C0)
SRC = (20e-12, 30e-12, 1.0)


def _mod():
    from paper_1709_00821_b200 import rketd2d
    return rketd2d


def _err(a, b, floor=0.0):
    s = max(np.max(np.abs(b)), floor)
    return float(np.max(np.abs(np.asarray(a, np.float64) - b)) / s) if s > 0 else float(np.max(np.abs(a)))


def _case(nx, ny, nsteps, boundary, dy_over_dx, src, comp, dtype, seed=1, splits=None):
    """random media and initial fields (all five), a source on `comp`, probes on both components incl. edge cells"""
    m = _mod()
    rng = np.random.default_rng(seed)
    dx, dy = DX, DX * dy_over_dx
    dt = DX * min(1.0, dy_over_dx) / (2 * C0)
    wp = rng.uniform(0, 2 * np.pi * 40e9, (ny, nx)) * (rng.uniform(size=(ny, nx)) > 0.4)
    nu = rng.uniform(0, 5e10, (ny, nx))
    Ex0 = 1e-2 * rng.uniform(-1, 1, (ny, nx)); Ex0[:, -1] = 0.0
    Ey0 = 1e-2 * rng.uniform(-1, 1, (ny, nx)); Ey0[-1, :] = 0.0
    Hz0 = 1e-5 * rng.uniform(-1, 1, (ny, nx)); Hz0[-1, :] = 0.0; Hz0[:, -1] = 0.0
    Jx0 = 1e-1 * rng.uniform(-1, 1, (ny, nx)) * (wp > 0); Jx0[:, -1] = 0.0
    Jy0 = 1e-1 * rng.uniform(-1, 1, (ny, nx)) * (wp > 0); Jy0[-1, :] = 0.0
    if boundary == wl.BC_PEC:
        Ex0[0, :] = Ex0[-1, :] = 0.0; Ey0[:, 0] = Ey0[:, -1] = 0.0
    probes = [(src[0], src[1], comp), (0, ny // 2, 1), (nx - 1, ny // 3, 1), (nx // 2, 0, 0), (nx // 3, ny - 1, 0),
              (1, 1, 0), (nx - 2, ny - 2, 1), (nx // 2, ny // 2, 0), (nx // 2, ny // 2, 1)]
    st = oracle.State2DTE(nx, ny, Ex0, Ey0, Hz0, Jx0, Jy0)
    ref = oracle.run2d_te(st, wp, nu, dx, dy, dt, nsteps, src_kind=0, src_params=SRC, src_ij=src, src_comp=comp,
                          probes=probes, boundary=boundary)
    sim = m.Sim2DTE(nx, ny, dx, dy, dt, dtype)
    cast = lambda a: np.ascontiguousarray(a, sim.np_dtype)
    sim.set_fields(cast(Ex0), cast(Ey0), cast(Hz0), cast(Jx0), cast(Jy0))       # before the media: J is kept as J
    sim.set_media(wp, nu)
    sim.set_boundary(boundary)
    sim.set_source(0, SRC, src[0], src[1], comp)
    sim.set_probes(probes)
    for part in (splits or [nsteps]):
        sim.run(part)
    rec = sim.read_probes().astype(np.float64)
    fields = [f.astype(np.float64) for f in sim.get_fields()]
    assert sim.counter(m.CTR_STEPS_DONE) == nsteps and sim.counter(m.CTR_STEP_LAUNCHES) == nsteps
    sim.close()
    tol = TOL[dtype]
    assert np.max(np.abs(ref)) > 0 and _err(rec, ref) <= tol
    peakE = max(np.max(np.abs(st.Ex)), np.max(np.abs(st.Ey)))
    for g, o, floor in zip(fields, (st.Ex, st.Ey, st.Hz, st.Jx, st.Jy), (peakE, peakE, peakE / 376.73, 0.0, 0.0)):
        assert _err(g, o, floor) <= tol


@pytest.mark.parametrize("dtype", ["f64", "f32"])
@pytest.mark.parametrize("boundary", [wl.BC_MUR, wl.BC_PEC])
def test_random_media_all_fields(dtype, boundary):
    _case(150, 110, 90, boundary, 1.0, (40, 60), 1, dtype)


@pytest.mark.parametrize("nx,ny", [(3, 3), (4, 7), (33, 5), (129, 64), (257, 31)])
def test_ragged_sizes_and_anisotropic_steps(nx, ny):
    _case(nx, ny, 40, wl.BC_MUR, 1.3, (nx // 2, ny // 2), 0, "f64", seed=nx * 100 + ny)


@pytest.mark.parametrize("src,comp", [((0, 10), 1), ((59, 10), 1), ((20, 0), 0), ((20, 39), 0), ((1, 1), 0), ((58, 38), 1)])
def test_source_on_and_next_to_the_edges(src, comp):
    _case(60, 40, 50, wl.BC_MUR, 0.8, src, comp, "f64", seed=7, splits=[1, 20, 29])


def test_reduces_to_the_1d_library_along_x():
    """fields uniform along y: (Ey, Hz) of the TEz kernel are (E, H) of the 1-D kernels (same operation sequence)"""
    from paper_1709_00821_b200 import rketd
    m = _mod()
    n, nother, nsteps = 300, 2 * 70 + 9, 60
    k = np.arange(n, dtype=np.float64)
    wp1 = np.zeros(n); nu1 = np.zeros(n); wp1[140:190] = 2 * np.pi * 28.7e9; nu1[140:190] = 2e10
    E1 = np.exp(-((k - 100.0) / 12.0) ** 2)
    s1 = rketd.Sim(n, 1, DX, DT, "f64")
    s1.set_media(wp1[None], nu1[None]); s1.set_fields(E=E1[None]); s1.set_probes([60, 150, 189]); s1.set_plan(rketd.KERNEL_STEP, 0, -1)
    s1.run(nsteps)
    rec1 = s1.read_probes()[0]
    E1n, H1n, J1n = (a[0] for a in s1.get_fields())
    s1.close()
    rep = lambda a: np.ascontiguousarray(np.repeat(a[None, :], nother, 0))
    s2 = m.Sim2DTE(n, nother, DX, 1.7 * DX, DT, "f64")
    s2.set_media(rep(wp1), rep(nu1)); s2.set_fields(Ey=rep(E1))
    mid = nother // 2
    s2.set_probes([(60, mid, 1), (150, mid, 1), (189, mid, 1)])
    s2.run(nsteps)
    rec2 = s2.read_probes()
    Ex, Ey, Hz, Jx, Jy = s2.get_fields()
    s2.close()
    assert np.max(np.abs(rec1)) > 0.1 and np.array_equal(rec2, rec1)
    assert np.array_equal(Ey[mid], E1n) and np.array_equal(Hz[mid], H1n) and not np.any(Ex[mid])
    assert np.max(np.abs(Jy[mid] - J1n)) <= 1e-13 * np.max(np.abs(J1n))


def test_media_change_with_live_fields_and_error_codes():
    m = _mod()
    from paper_1709_00821_b200.rketd import RketdError, EINVAL, ESTATE
    nx, ny = 70, 50
    rng = np.random.default_rng(4)
    wpA, wpB = (rng.uniform(0, 2 * np.pi * 40e9, (ny, nx)) for _ in range(2))
    nuA, nuB = (rng.uniform(0, 5e10, (ny, nx)) for _ in range(2))
    Ey0 = rng.uniform(-1, 1, (ny, nx)); Ey0[-1, :] = 0.0
    st = oracle.State2DTE(nx, ny, Ey0=Ey0)
    r1 = oracle.run2d_te(st, wpA, nuA, DX, DX, DT, 30, probes=[(20, 20, 1), (30, 25, 0)])
    r2 = oracle.run2d_te(st, wpB, nuB, DX, DX, DT, 30, probes=[(20, 20, 1), (30, 25, 0)])
    s = m.Sim2DTE(nx, ny, DX, DX, DT)
    with pytest.raises(RketdError) as e:
        s.run(1)
    assert e.value.code == ESTATE
    s.set_media(wpA, nuA); s.set_fields(Ey=Ey0); s.set_probes([(20, 20, 1), (30, 25, 0)])
    s.run(30)
    bad = wpB.copy(); bad[3, 3] = -1.0
    with pytest.raises(RketdError) as e:
        s.set_media(bad, nuB)                       # rejected before anything changes
    assert e.value.code == EINVAL
    s.set_media(wpB, nuB)                           # live fields: the physical J is kept
    s.run(30)
    assert _err(s.read_probes(), np.concatenate([r1, r2], 1)) <= 1e-12
    for g, o in zip(s.get_fields(), (st.Ex, st.Ey, st.Hz, st.Jx, st.Jy)):
        assert _err(g, o) <= 1e-12
    for call in (lambda: s.set_probes([(nx, 0, 0)]), lambda: s.set_probes([(0, 0, 2)]), lambda: s.set_source(0, SRC, 0, ny, 1),
                 lambda: s.set_source(0, SRC, 0, 0, 5), lambda: s.set_boundary(7), lambda: s.run(-1)):
        with pytest.raises(RketdError) as e:
            call()
        assert e.value.code == EINVAL
    s.close()
    with pytest.raises(RketdError):
        m.Sim2DTE(2, 5, DX, DX, DT)
    with pytest.raises(RketdError):
        m.Sim2DTE(10, 10, DX, DX, 2 * DT)           # unstable


@pytest.mark.parametrize("dtype", ["f64", "f32"])
def test_column_workload_sampled_against_windowed_oracle(dtype):
    """the plasma-column workload at 4096 x 4096 cells x 300 steps in the TEz polarisation; every probe against an oracle
    run on the window that can influence it (pin R6)"""
    m = _mod()
    w = wl.tm2d_column(nx=4096, ny=4096, nsteps=300, nprobes=14)
    sim = m.Sim2DTE.from_workload(w, dtype)
    sim.run(w.nsteps)
    rec = sim.read_probes().astype(np.float64)
    sim.close()
    r = w.nsteps + 2
    peak, worst = 0.0, 0.0
    for q, (pi, pj) in enumerate(w.probes):
        pi, pj = int(pi), int(pj)
        win = (max(0, pi - r), min(w.nx, pi + r + 1), max(0, pj - r), min(w.ny, pj + r + 1))
        o = oracle.run_workload2d_te(w, window=win, omp=True)
        kk = [tuple(p) for p in o["probe_ij"]].index((pi, pj))
        peak = max(peak, np.max(np.abs(o["rec"][kk])))
        worst = max(worst, np.max(np.abs(rec[q] - o["rec"][kk])))
    print(f"TEz column {dtype}: worst |gpu - oracle| / grid peak {worst / peak:.3e}")
    assert peak > 1e-3 and worst / peak <= TOL[dtype]
