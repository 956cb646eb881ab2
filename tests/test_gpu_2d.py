"""GPU parity of the 2-D TMz path (include/rketd2d.h) against the CPU oracle (oracle2d_*), through
the C ABI.  fp64: max |gpu - oracle| / max |oracle| <= 1e-12 over every probe sample and over the final fields;
fp32: <= 1e-5.  The one-step kernel (K1) and the streaming kernel (K2, every depth) must agree bit for bit."""
import math

import numpy as np
import pytest

import oracle
from paper_1709_00821_b200 import workloads as wl

pytestmark = pytest.mark.gpu

TOL = {"f64": 1e-12, "f32": 1e-5}
C0 = 299792458.0
DX = 75e-6
DT = DX / (2 * C0)
SRC = (20e-12, 80e-12, 1.0)


def _mod():
    from paper_1709_00821_b200 import rketd2d
    return rketd2d


def _gpu_run(w, dtype="f64", kernel=None, depth=0, nsteps=None, splits=None, fields=None):
    m = _mod()
    sim = m.Sim2D.from_workload(w, dtype)
    if fields is not None:
        sim.set_fields(*[None if f is None else np.ascontiguousarray(f, sim.np_dtype) for f in fields])
    sim.set_plan(m.KERNEL_AUTO if kernel is None else kernel, depth)
    n = w.nsteps if nsteps is None else nsteps
    for part in (splits or [n]):
        sim.run(part)
    rec = sim.read_probes()
    out = dict(rec=rec, fields=sim.get_fields(), launches=sim.counter(m.CTR_STEP_LAUNCHES),
               kernel=sim.counter(m.CTR_KERNEL_USED))
    sim.close()
    return out


def _oracle_run(w, nsteps=None, fields=None):
    n = w.nsteps if nsteps is None else nsteps
    wp, nu = w.media()
    if fields is None:
        st = oracle.State2D(w.nx, w.ny, Ez0=w.initial_E())
    else:
        st = oracle.State2D(w.nx, w.ny, *fields)
    rec, _ = oracle.run2d(st, wp, nu, w.dx, w.dy, w.dt, n, src_kind=w.src_kind, src_params=w.src_params, src_ij=w.src_ij,
                          probes=w.probes, boundary=w.boundary)
    return dict(rec=rec, fields=(st.Ez, st.Hx, st.Hy, st.Jz))


def _err(a, b):
    s = np.max(np.abs(b))
    return float(np.max(np.abs(np.asarray(a, np.float64) - b)) / s) if s > 0 else float(np.max(np.abs(a)))


def _check(g, o, tol):
    assert np.max(np.abs(o["rec"])) > 0
    assert _err(g["rec"], o["rec"]) <= tol
    for gf, of in zip(g["fields"], o["fields"]):
        assert _err(gf, of) <= tol


def _edge_workload(nx, ny, nsteps, boundary=wl.BC_MUR, dy_over_dx=1.0, src=None):
    """tm2d_column with probes on every edge, next to every edge, in the corners, and on the source."""
    w = wl.tm2d_column(nx, ny, nsteps, boundary=boundary, dy_over_dx=dy_over_dx, nprobes=24)
    pts = {(0, 0), (nx - 1, 0), (0, ny - 1), (nx - 1, ny - 1), (0, ny // 2), (nx - 1, ny // 2), (nx // 2, 0), (nx // 2, ny - 1),
           (1, 1), (nx - 2, ny - 2), (1, ny // 2), (nx // 2, 1), (nx // 2, ny // 2), (nx - 2, 1), (min(2, nx - 1), ny - 2)}
    if src is not None:
        w.src_ij = src
    pts.add(tuple(w.src_ij))
    w.probes = np.array(sorted(pts), np.int64)
    return w


# ----------------------------------------------------------------------------- K1 vs oracle, K2 == K1
@pytest.mark.parametrize("dtype", ["f64", "f32"])
def test_reduced_column_all_kernels(dtype):
    m = _mod()
    w = _edge_workload(530, 310, 150)
    o = _oracle_run(w)
    k1 = _gpu_run(w, dtype, m.KERNEL_STEP)
    assert k1["kernel"] == m.KERNEL_STEP and k1["launches"] == 150
    _check(k1, o, TOL[dtype])
    for T in (1, 2, 4, 6, 8) + ((16,) if dtype == "f32" else ()):
        k2 = _gpu_run(w, dtype, m.KERNEL_STREAM, T)
        assert k2["kernel"] == m.KERNEL_STREAM
        assert np.array_equal(k2["rec"], k1["rec"]), T
        for a, b in zip(k2["fields"], k1["fields"]):
            assert np.array_equal(a, b), T
    auto = _gpu_run(w, dtype)
    assert auto["kernel"] == m.KERNEL_STREAM and np.array_equal(auto["rec"], k1["rec"])


# sizes: one node inside; strips whose last column falls on lane 0 (57, 249, 265: the shifted last strip); a last strip
# of one column (241); several strips and segments; rows fewer than the depth
@pytest.mark.parametrize("nx,ny", [(3, 3), (4, 3), (3, 7), (5, 4), (33, 17), (57, 40), (249, 33), (241, 9), (265, 70),
                                   (481, 5), (700, 333), (64, 1200), (369, 9), (393, 70), (800, 40)])
def test_ragged_sizes_mur(nx, ny):
    m = _mod()
    nsteps = 37
    w = _edge_workload(nx, ny, nsteps, src=(nx // 2, ny // 2))
    o = _oracle_run(w)
    k1 = _gpu_run(w, "f64", m.KERNEL_STEP)
    _check(k1, o, 1e-12)
    for T in (8, 6, 2):
        k2 = _gpu_run(w, "f64", m.KERNEL_STREAM, T)
        assert np.array_equal(k2["rec"], k1["rec"]), (T, np.max(np.abs(k2["rec"] - k1["rec"])))
        for a, b in zip(k2["fields"], k1["fields"]):
            assert np.array_equal(a, b), T


@pytest.mark.parametrize("src", ["edge_x0", "edge_y0", "edge_x1", "edge_y1", "next_to_x0", "next_to_y0", "next_to_y1"])
@pytest.mark.parametrize("boundary", [wl.BC_MUR, wl.BC_PEC])
def test_source_on_and_next_to_the_edges(src, boundary):
    m = _mod()
    nx, ny = 270, 90
    pos = {"edge_x0": (0, 40), "edge_y0": (100, 0), "edge_x1": (nx - 1, 33), "edge_y1": (250, ny - 1),
           "next_to_x0": (1, 50), "next_to_y0": (120, 1), "next_to_y1": (7, ny - 2)}[src]
    w = _edge_workload(nx, ny, 45, boundary=boundary, dy_over_dx=1.3, src=pos)
    w.src_kind, w.src_params = wl.SRC_TABLE, tuple(np.sin(0.3 * np.arange(45)) + 0.5)
    o = _oracle_run(w)
    k1 = _gpu_run(w, "f64", m.KERNEL_STEP)
    _check(k1, o, 1e-12)
    k2 = _gpu_run(w, "f64", m.KERNEL_STREAM, 8)
    assert np.array_equal(k2["rec"], k1["rec"])
    for a, b in zip(k2["fields"], k1["fields"]):
        assert np.array_equal(a, b)


def test_initial_fields_restart_and_anisotropic_steps():
    m = _mod()
    nx, ny = 300, 260
    w = _edge_workload(nx, ny, 64, dy_over_dx=0.8)
    rng = np.random.default_rng(3)
    wp, _ = w.media()
    f0 = (1e-3 * rng.uniform(-1, 1, (ny, nx)), 1e-6 * rng.uniform(-1, 1, (ny, nx)), 1e-6 * rng.uniform(-1, 1, (ny, nx)),
          1e-2 * rng.uniform(-1, 1, (ny, nx)) * (wp > 0))
    f0[1][-1, :] = 0.0                                       # padding row / column of Hx / Hy
    f0[2][:, -1] = 0.0
    o = _oracle_run(w, fields=f0)
    g = _gpu_run(w, "f64", m.KERNEL_STREAM, 8, fields=f0, splits=[13, 1, 30, 20])
    _check(g, o, 1e-12)
    g1 = _gpu_run(w, "f64", m.KERNEL_STEP, fields=f0)
    assert np.array_equal(g["rec"], g1["rec"])
    g32 = _gpu_run(w, "f32", m.KERNEL_STREAM, 16, fields=f0)
    _check(g32, o, 1e-5)


def test_fields_before_media_and_media_change_with_live_fields():
    """The kernels carry G = cj Jz - cj kc Ez, which depends on the media: Jz given before the media, and a change of
    media in the middle of a run, must both go through the physical Jz."""
    m = _mod()
    nx, ny = 120, 90
    w = _edge_workload(nx, ny, 40)
    wp, nu = w.media()
    rng = np.random.default_rng(9)
    E0 = 1e-3 * rng.uniform(-1, 1, (ny, nx)); J0 = 1e-2 * rng.uniform(-1, 1, (ny, nx)) * (wp > 0)
    wp2, nu2 = wp * 0.5 + 1e10, nu * 2.0 + 1e9
    kw = dict(src_kind=w.src_kind, src_params=w.src_params, src_ij=w.src_ij, probes=w.probes, boundary=w.boundary)
    st = oracle.State2D(nx, ny, Ez0=E0, Jz0=J0)
    r1, _ = oracle.run2d(st, wp, nu, w.dx, w.dy, w.dt, 25, **kw)
    r2, _ = oracle.run2d(st, wp2, nu2, w.dx, w.dy, w.dt, 15, **kw)
    sim = m.Sim2D(nx, ny, w.dx, w.dy, w.dt)
    sim.set_fields(Ez=E0, Jz=J0)                       # before any media
    sim.set_media(wp, nu)
    sim.set_source(w.src_kind, w.src_params, *w.src_ij)
    sim.set_probes(w.probes)
    sim.run(25)
    sim.set_media(wp2, nu2)                            # live fields
    sim.run(15)
    rec = sim.read_probes()
    ref = np.concatenate([r1, r2], 1)
    assert _err(rec, ref) <= 1e-12
    for gf, of in zip(sim.get_fields(), (st.Ez, st.Hx, st.Hy, st.Jz)):
        assert _err(gf, of) <= 1e-12
    sim.discard_records()
    sim.run(3)
    assert sim.read_probes().shape == (len(w.probes), 3) and sim.counter(m.CTR_STEPS_DONE) == 43
    sim.reset()
    assert not np.any(sim.get_fields()[0]) and sim.counter(m.CTR_STEPS_DONE) == 0
    sim.close()


def test_cavity_mode_on_the_gpu_follows_the_dispersion_recurrence():
    """Pin Q3 through the CUDA path: conducting box, one eigenmode, dx != dy."""
    m = _mod()
    nx, ny, mm, nn, nsteps = 41, 31, 2, 3, 400
    dx, dy, dt = DX, 1.3 * DX, 0.9 * DT
    i = np.arange(nx)[None, :]; j = np.arange(ny)[:, None]
    mode = np.sin(mm * math.pi * i / (nx - 1)) * np.sin(nn * math.pi * j / (ny - 1))
    mode[0, :] = mode[-1, :] = 0.0; mode[:, 0] = mode[:, -1] = 0.0
    L = 4.0 * ((C0 * dt / dx) ** 2 * math.sin(mm * math.pi / (2 * (nx - 1))) ** 2 +
               (C0 * dt / dy) ** 2 * math.sin(nn * math.pi / (2 * (ny - 1))) ** 2)
    a = [1.0, 1.0 - L]
    for _ in range(nsteps - 1):
        a.append((2.0 - L) * a[-1] - a[-2])
    a = np.array(a)
    sim = m.Sim2D(nx, ny, dx, dy, dt)
    z = np.zeros((ny, nx))
    sim.set_media(z, z)
    sim.set_boundary(m.BC_PEC)
    sim.set_fields(Ez=mode)
    probes = [(7, 5), (20, 15), (33, 22), (12, 26)]
    sim.set_probes(probes)
    sim.run(nsteps)
    rec = sim.read_probes()
    for p, (pi, pj) in enumerate(probes):
        assert np.max(np.abs(rec[p] - a[1:] * mode[pj, pi])) < 5e-12
    assert np.max(np.abs(sim.get_fields()[0] - a[-1] * mode)) < 5e-12
    sim.close()


def test_kernel_coefficients_against_the_oracle_in_ulps():
    m = _mod()
    w = wl.tm2d_column(96, 80, 1, dy_over_dx=1.25)
    sim = m.Sim2D.from_workload(w)
    kc = sim.get_kernel_coefficients()
    wp, nu = w.media()
    c = oracle.coefficients2d(wp, nu, w.dx, w.dy, w.dt)
    ref = {"P": c["ca"] - c["cj"] * c["kc"], "ce": c["cex"], "ka": c["ka"], "Q": c["ka"] * c["cj"] * c["kc"] + c["cj"] * c["kb"]}
    for k, r in ref.items():
        scale = np.max(np.abs(r))
        assert np.max(np.abs(kc[k] - r)) <= 8 * np.finfo(np.float64).eps * scale, k
    assert kc["chx"] == pytest.approx(c["chx"], rel=1e-15) and kc["chy"] == pytest.approx(c["chy"], rel=1e-15)
    assert kc["mx"] == pytest.approx(c["mx"], rel=1e-15) and kc["my"] == pytest.approx(c["my"], rel=1e-15)
    assert np.max(np.abs(c["cey"] - c["cex"] * (w.dx / w.dy))) <= 4 * np.finfo(np.float64).eps * np.max(c["cey"])
    sim.close()


def test_error_codes_2d():
    m = _mod()
    from paper_1709_00821_b200.rketd import RketdError, EINVAL, ESTATE
    with pytest.raises(RketdError) as e:
        m.Sim2D(2, 10, DX, DX, DT)
    assert e.value.code == EINVAL
    with pytest.raises(RketdError) as e:
        m.Sim2D(10, 10, DX, DX, 1.5 * DT)                    # c dt sqrt(2)/dx = 1.06
    assert e.value.code == EINVAL
    sim = m.Sim2D(10, 12, DX, DX, DT)
    with pytest.raises(RketdError) as e:
        sim.run(1)
    assert e.value.code == ESTATE
    for bad in ([(10, 0)], [(0, 12)], [(-1, 3)]):
        with pytest.raises(RketdError) as e:
            sim.set_probes(bad)
        assert e.value.code == EINVAL
    with pytest.raises(RketdError) as e:
        sim.set_source(0, SRC, 3, 12)
    assert e.value.code == EINVAL
    with pytest.raises(RketdError) as e:
        sim.set_plan(m.KERNEL_STREAM, 3)
    assert e.value.code == EINVAL
    wp = np.zeros((12, 10)); nu = np.zeros((12, 10)); wp[3, 3] = -1.0
    with pytest.raises(RketdError) as e:
        sim.set_media(wp, nu)
    assert e.value.code == EINVAL
    sim.close()


# ----------------------------------------------------------------------------- the size bench.py times
# Rounding sites per node and step (DESIGN.md §5, 2-D count).  Kernels: 13 rounded operations + 4 stored coefficients
# + the two global H coefficients = 19.  Oracle: Hx 3, Hy 3, Ez 9, Jz 5 operations + 7 stored coefficients + the two
# global ones = 29 (they only count when the GPU also runs in fp64).  The leapfrog does not amplify an injected error
# (pin Q2), so |gpu - oracle| <= K n u x the local field amplitude.
DRIFT_K_2D = {"f64": 19 + 29, "f32": 19}
_ORACLE_2D = {}


def _oracle_windows_2d(w, half):
    """per probe: its record and the final fields on the (2 half + 1)^2 box around it, from one oracle run on the window
    of nodes that can influence that box (pin Q7: bit-exact domain of dependence); cached: one oracle pass serves the
    three parametrisations below"""
    key = (w.name, w.nsteps, len(w.probes), half)
    if key in _ORACLE_2D:
        return _ORACLE_2D[key]
    r = w.nsteps + 1 + half
    out = []
    for pi, pj in w.probes:
        pi, pj = int(pi), int(pj)
        win = (max(0, pi - r), min(w.nx, pi + r + 1), max(0, pj - r), min(w.ny, pj + r + 1))
        o = oracle.run_workload2d(w, window=win, omp=True)
        k = [tuple(p) for p in o["probe_ij"]].index((pi, pj))
        bi0, bi1, bj0, bj1 = max(0, pi - half), min(w.nx, pi + half + 1), max(0, pj - half), min(w.ny, pj + half + 1)
        st = o["state"]
        box = tuple(np.array(f[bj0 - win[2]:bj1 - win[2], bi0 - win[0]:bi1 - win[0]]) for f in (st.Ez, st.Hx, st.Hy, st.Jz))
        out.append(dict(rec=o["rec"][k].copy(), box=(bi0, bi1, bj0, bj1), fields=box))
    _ORACLE_2D[key] = out
    return out


@pytest.mark.parametrize("dtype,kernel", [("f64", 2), ("f32", 2), ("f64", 1)])
def test_full_size_sampled_against_windowed_oracle(dtype, kernel):
    """16384 x 16384 nodes x the 1000 steps `bench.py --workload tm2d` times, in its launch configuration (streaming
    kernel, default depth; and the one-step kernel): every probe record and the final Ez, Hx, Hy, Jz on a 65 x 65 box
    around each of the 20 probes (source node, column centre, nodes on and next to every edge, seeded random nodes)."""
    import torch
    m = _mod()
    half = 32
    w = wl.tm2d_column(nprobes=20)
    nsteps = w.nsteps
    assert nsteps == 1000
    sim = m.Sim2D(w.nx, w.ny, w.dx, w.dy, w.dt, dtype)
    wp, nu = w.media()
    wp_max = float(wp.max())
    sim.set_media(wp, nu)
    del wp, nu
    sim.set_fields(Ez=np.ascontiguousarray(w.initial_E(), sim.np_dtype))
    sim.set_source(w.src_kind, w.src_params, *w.src_ij)
    sim.set_probes(w.probes)
    sim.set_plan(kernel, 0)                                  # 2: the streaming kernel at its default depth; 1: one launch per step
    sim.run(nsteps)
    rec = sim.read_probes().astype(np.float64)
    assert sim.counter(m.CTR_KERNEL_USED) == kernel
    assert sim.counter(m.CTR_DEPTH_USED) == (8 if kernel == m.KERNEL_STREAM else 1)
    tdt = torch.float64 if dtype == "f64" else torch.float32
    dev = [torch.empty((w.ny, w.nx), dtype=tdt, device="cuda") for _ in range(4)]
    m.rketd2d_get_fields(sim.h, *dev)
    sim.close()
    refs = _oracle_windows_2d(w, half)
    peak = max(np.max(np.abs(o["rec"])) for o in refs)
    assert peak > 2e-2                                        # the source node is a probe: the driven field (a line source in 2-D: 0.04)
    u = 2.0 ** -53 if dtype == "f64" else 2.0 ** -24
    floors = (peak, peak / 376.73, peak / 376.73, 8.854e-12 * wp_max ** 2 * 20e-12 * peak)
    worst, worst_rel, worst_f = 0.0, 0.0, [0.0] * 4
    for q, o in enumerate(refs):
        d = np.max(np.abs(rec[q] - o["rec"]))
        own = np.max(np.abs(o["rec"]))
        assert own > 0, ("vacuous: oracle record identically zero at probe", q)
        worst, worst_rel = max(worst, d), max(worst_rel, d / max(own, 1e-3))
        # per probe, relative to the probe's own peak (not gated by the north_star): the drift bound K n u
        assert d <= DRIFT_K_2D[dtype] * nsteps * u * max(own, 1e-3), (q, d, own)
        bi0, bi1, bj0, bj1 = o["box"]
        for a in range(4):
            g = dev[a][bj0:bj1, bi0:bi1].cpu().numpy().astype(np.float64)
            ref = o["fields"][a].copy()
            if a == 1 and bj1 == w.ny:
                ref[-1, :] = 0.0                              # row ny-1 of Hx / column nx-1 of Hy are padding: reported as 0
            if a == 2 and bi1 == w.nx:
                ref[:, -1] = 0.0
            e = np.max(np.abs(g - ref))
            worst_f[a] = max(worst_f[a], e / floors[a])
            assert e <= TOL[dtype] * floors[a], (q, "Ez Hx Hy Jz".split()[a], e, floors[a])     # the north_star gate
    del dev
    torch.cuda.empty_cache()
    print(f"tm2d {dtype} kernel {kernel}: {len(refs)} probes x {nsteps} steps: worst |gpu-oracle| / grid peak {worst / peak:.3e}, "
          f"per probe {worst_rel:.3e}; final fields on {len(refs)} boxes of {2 * half + 1}^2 nodes against the grid peak: "
          + ", ".join(f"{n} {v:.3e}" for n, v in zip("Ez Hx Hy Jz".split(), worst_f)))
    assert worst / peak <= TOL[dtype]


# ----------------------------------------------------------------------------- the paper's boundary: split-field PML
@pytest.mark.parametrize("dtype", ["f64", "f32"])
def test_pml_layer_against_the_oracle(dtype):
    """rketd2d_set_boundary_pml: random media, a source next to a corner inside the layer region's
    reach, probes inside the layers, on the conductor and in the interior; records and final Ez, Hx, Hy, Jz against
    oracle2d_run_pml; then back to Mur."""
    m = _mod()
    nx, ny, nsteps = 150, 110, 160
    pml = (8, 2.0, 1e-4)
    rng = np.random.default_rng(21)
    wp = rng.uniform(0, 2 * np.pi * 40e9, (ny, nx)) * (rng.uniform(size=(ny, nx)) > 0.5)
    nu = rng.uniform(0, 5e10, (ny, nx))
    src = (20, 15)
    probes = [src, (3, 50), (nx - 4, 60), (70, 2), (75, ny - 3), (0, 30), (nx // 2, ny // 2), (9, 9), (nx - 9, ny - 9)]
    st = oracle.State2D(nx, ny)
    ref = oracle.run2d_pml(st, wp, nu, DX, 1.2 * DX, 0.9 * DT, nsteps, pml=pml, src_kind=0, src_params=(20e-12, 30e-12, 1.0),
                           src_ij=src, probes=probes)
    sim = m.Sim2D(nx, ny, DX, 1.2 * DX, 0.9 * DT, dtype)
    sim.set_boundary_pml(*pml)
    sim.set_media(wp, nu)
    sim.set_source(0, (20e-12, 30e-12, 1.0), *src)
    sim.set_probes(probes)
    for part in (1, 59, 100):
        sim.run(part)
    rec = sim.read_probes().astype(np.float64)
    assert sim.counter(m.CTR_KERNEL_USED) == m.KERNEL_STEP            # the layer runs in the one-step kernel
    Ez, Hx, Hy, Jz = (f.astype(np.float64) for f in sim.get_fields())
    tol = TOL[dtype]
    assert np.max(np.abs(ref)) > 0.1 and _err(rec, ref) <= tol
    pk = np.max(np.abs(st.Ez))
    assert np.max(np.abs(Ez - st.Ez)) <= tol * pk and np.max(np.abs(Hx - st.Hx)) <= tol * pk / 376.73
    assert np.max(np.abs(Hy - st.Hy)) <= tol * pk / 376.73 and np.max(np.abs(Jz - st.Jz)) <= tol * np.max(np.abs(st.Jz))
    assert not np.any(Jz[:pml[0]]) and not np.any(Jz[:, -pml[0]:])       # layer nodes carry no current
    # back to first-order Mur (takes effect with the next media), fields reset
    sim.set_boundary(m.BC_MUR)
    sim.set_media(wp, nu)
    sim.reset()
    sim.run(40)
    st2 = oracle.State2D(nx, ny)
    ref2, _ = oracle.run2d(st2, wp, nu, DX, 1.2 * DX, 0.9 * DT, 40, src_kind=0, src_params=(20e-12, 30e-12, 1.0), src_ij=src, probes=probes)
    assert _err(sim.read_probes(), ref2) <= tol
    from paper_1709_00821_b200.rketd import RketdError
    for bad in ((0, 2.0, 1e-4), (60, 2.0, 1e-4), (5, 2.0, 0.0), (5, -1.0, 1e-4)):
        with pytest.raises(RketdError):
            sim.set_boundary_pml(*bad)
    sim.close()


def test_pml_reflection_floor_on_the_gpu():
    """the oblique-pulse experiment of oracle pin U3 through the CUDA path: what comes back to the probe with the layer
    is a small fraction of what first-order Mur returns"""
    m = _mod()
    nx = ny = 161
    z = np.zeros((ny, nx))
    i = np.arange(nx)[None, :]; j = np.arange(ny)[:, None]
    E0 = np.exp(-((i - 40.0) / 3.0) ** 2 - ((j - 40.0) / 3.0) ** 2)
    big = oracle.State2D(3 * nx, 3 * ny, Ez0=np.pad(E0, ((ny, ny), (nx, nx))))
    rr = oracle.run2d(big, np.zeros((3 * ny, 3 * nx)), np.zeros((3 * ny, 3 * nx)), DX, DX, DT, 700, probes=[(80 + nx, 80 + ny)],
                      boundary=oracle.BOUNDARY_PEC)[0][0]
    back = {}
    for kind in ("pml", "mur"):
        sim = m.Sim2D(nx, ny, DX, DX, DT)
        if kind == "pml":
            sim.set_boundary_pml(10, 3.0, 1e-6)
        sim.set_media(z, z)
        sim.set_fields(Ez=E0)
        sim.set_probes([(80, 80)])
        sim.set_plan(m.KERNEL_STEP, 0)
        sim.run(700)
        back[kind] = np.max(np.abs(sim.read_probes()[0] - rr)) / np.max(np.abs(rr))
        sim.close()
    print(f"reflection seen at the probe (GPU): PML(10) {back['pml']:.2e}, Mur-1 {back['mur']:.2e}")
    assert back["pml"] < 0.25 * back["mur"] and back["pml"] < 5e-3
