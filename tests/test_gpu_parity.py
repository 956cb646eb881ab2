"""Parity of the CUDA path (librketd, through its C ABI) against the CPU oracle — `-m gpu`.

Tolerances (BASELINE.json north_star; SURVEY.md §8(c) "Tolerance rule"):
  fp64: per grid, max over all probes and samples of |gpu - oracle| / max |oracle|  <= 1e-12
  fp32: the same ratio against the fp64 oracle                                       <= 1e-5
Final fields are held to the same bars (normalised by the field's own max).  K1, K2 (all launch
variants and depths) and K3 must agree BIT FOR BIT with each other: they run the same correctly
rounded operation sequence per node, only the schedule differs.
"""
import numpy as np
import pytest

import oracle
from paper_1709_00821_b200 import workloads as wl

pytestmark = pytest.mark.gpu

TOL = {"f64": 1e-12, "f32": 1e-5}
C0 = 299792458.0


@pytest.fixture(scope="module")
def rk():
    from paper_1709_00821_b200 import rketd
    return rketd


def grid_err(gpu, ref):
    """max over grids of (max |gpu-ref| over probes, samples) / (max |ref| over probes, samples)"""
    gpu = np.asarray(gpu, np.float64)
    d = np.abs(gpu - ref).reshape(ref.shape[0], -1).max(1)
    s = np.abs(ref).reshape(ref.shape[0], -1).max(1)
    assert np.all(s > 0), "vacuous comparison: oracle record is identically zero"
    return float(np.max(d / s))


def run_gpu(rk, w, dtype="f64", kernel=0, depth=0, variant=-1, nsteps=None, chunks=None, fields=True):
    s = rk.Sim.from_workload(w, dtype)
    s.set_plan(kernel, depth, variant)
    n = w.nsteps if nsteps is None else nsteps
    for c in (chunks or [n]):
        s.run(c)
    out = {"rec": s.read_probes(), "kernel": s.counter(rk.CTR_KERNEL_USED), "launches": s.counter(rk.CTR_STEP_LAUNCHES)}
    if fields:
        out["E"], out["H"], out["J"] = s.get_fields()
    s.close()
    return out


def floors_of(w, ref):
    return np.max(np.abs(ref["rec"])), float(np.max(w.media(0, w.ncells, 0, min(w.nbatch, 64))[0]))


def check_fields(gpu, st, tol, peak=0.0, wp_max=0.0):
    """Final fields.  Errors scale with the largest amplitude the run has seen, not with what is left in
    the grid at the end, hence the floors from the probe peak: E ~ peak, H ~ peak/eta0,
    J ~ eps0 wp^2 tau peak (tau = 20 ps, the source width)."""
    floors = {"E": peak, "H": peak / 376.73, "J": 8.854e-12 * wp_max ** 2 * 20e-12 * peak}
    for k, ref in (("E", st.E), ("H", st.H), ("J", st.J)):
        ref = ref.copy()
        if k == "H":
            ref[:, -1] = 0.0            # H[ncells-1] is padding: the library reports 0
        scale = max(np.max(np.abs(ref)), floors[k])
        if scale > 0:
            assert np.max(np.abs(np.asarray(gpu[k], np.float64) - ref)) <= tol * scale, k


def WT(nw=0, nc=0, k=0):
    """rketd_set_plan variant of the resident warp-tile kernel: k grids per chunk on a cluster of nc CTAs x nw warps"""
    return 0x40000000 | (k << 16) | (nc << 8) | nw


LEAN, NOLEAN = 0x10000000, 0x20000000      # the 168- / 232-register instantiation of k3_wtile (default: by batch size)
HALF, NOHALF = 0x08000000, 0x04000000      # a lane holds half a 64-B row / a whole one (default: half rows for a few grids)


# K1; the resident kernel K3: warp tiles with the library's packing at several depths (steps between halo refreshes),
# explicit packings (one CTA, clusters of 2..9 CTAs over DSMEM), the older one-barrier-per-step kernel; K2 variants
ALL_PLANS = [(1, 0, -1)] + [(3, d, -1) for d in (0, 1, 3, 8, 13, 16)] + \
            [(3, 8, WT(8, 2)), (3, 8, WT(5, 2)), (3, 8, WT(1, 9)), (3, 5, WT(2, 5)), (3, 16, WT(4, 3)), (3, 0, WT(3, 3))] + \
            [(3, 8, WT(8, 2) | LEAN), (3, 7, WT(9, 1) | LEAN), (3, 16, WT(2, 5) | LEAN), (3, 0, WT(3, 3) | LEAN), (3, 0, WT(5, 2) | NOLEAN)] + \
            [(3, 16, WT() | HALF), (3, 8, WT(3, 0) | HALF), (3, 4, WT(8, 0) | HALF), (3, 13, WT(2, 11) | HALF), (3, 0, WT() | NOHALF), (3, 5, WT() | NOHALF)] + \
            [(3, 0, 0), (3, 0, 2)] + [(2, 0, v) for v in (0, 2, 6)] + [(2, d, 0) for d in (1, 7, 16, 33)] + \
            [(2, d, 6) for d in (1, 2, 9, 32, 40)] + [(2, 5, 0), (2, 40, 2)]


# ------------------------------------------------------------------------------------------ config 1
@pytest.mark.parametrize("dtype", ["f64", "f32"])
def test_config1_full_all_kernels(rk, dtype):
    """BASELINE config 1 at full size (2000 nodes, 6000 steps), every kernel, variant and a few depths."""
    w = wl.config1()
    ref = oracle.run_workload(w)
    first = None
    for kernel, depth, variant in ALL_PLANS:
        g = run_gpu(rk, w, dtype, kernel, depth, variant)
        assert g["kernel"] == kernel
        assert grid_err(g["rec"], ref["rec"]) <= TOL[dtype], (kernel, depth, variant)
        check_fields(g, ref["state"], TOL[dtype], *floors_of(w, ref))
        if first is None:
            first = g
        else:
            for k in ("rec", "E", "H", "J"):
                assert np.array_equal(first[k], g[k]), f"{k}: plan {(kernel, depth, variant)} differs from K1"


def test_coefficients_match_oracle_in_ulps(rk):
    """T1: the six per-node coefficients vs the oracle's S0, random media incl. nu = 0, tiny nu."""
    rng = np.random.default_rng(5)
    n = 5000
    wp = rng.uniform(0, 2 * np.pi * 60e9, (3, n))
    nu = rng.uniform(0, 1e11, (3, n))
    wp[0, :100] = 0.0
    nu[1, :100] = 0.0
    nu[2, :200] = 10.0 ** rng.uniform(-3, 13, 200)        # includes x = nu dt > 0.5 (formula branch)
    s = rk.Sim(n, 3, wl.DZ, wl.DT, "f64")
    s.set_media(wp, nu)
    c = s.get_coefficients()
    o = oracle.coefficients(wp, nu, wl.DZ, wl.DT)
    small = nu * wl.DT < 0.02           # every BASELINE config has nu dt <= 1.25e-2
    for k in ("ca", "cj", "ch", "ka", "kb", "kc"):
        ulp = np.abs(c[k] - o[k]) / np.maximum(np.spacing(np.abs(o[k])), 1e-300)
        # kb = b - c ~ b/2: one ulp of b (expm1 of glibc vs CUDA) is two ulps of kb
        assert ulp[small].max() <= (4.0 if k == "kb" else 2.0), (k, ulp[small].max())
        assert (ulp[small] > 0).mean() < 0.05, (k, "more than 5 % of nodes differ by an ulp")
        # larger nu dt: kb = b - c cancels (b - c ~ c / (nu dt) for large nu dt), so the 1-ulp freedom of
        # exp / expm1 between glibc and CUDA is amplified
        assert np.all(np.abs(c[k] - o[k])[~small] <= 1e-12 * np.abs(o[k])[~small]), k
    assert c["chh"] == o["chh"] and c["m"] == o["m"]
    # the four arrays the kernels read: P = ca - cj kc, ch, ka, Q = ka cj kc + cj kb (rketd_device.cuh)
    kc4 = s.get_kernel_coefficients()
    s.close()
    kcp = o["cj"] * o["kc"]
    want = {"P": o["ca"] - kcp, "ch": o["ch"], "ka": o["ka"], "Q": o["ka"] * kcp + o["cj"] * o["kb"]}
    for k in ("P", "ch", "ka", "Q"):
        ulp = np.abs(kc4[k] - want[k]) / np.maximum(np.spacing(np.abs(want[k])), 1e-300)
        assert ulp[small].max() <= (8.0 if k == "Q" else 2.0), (k, ulp[small].max())
        assert np.all(np.abs(kc4[k] - want[k])[~small] <= 1e-12 * np.abs(want[k])[~small] + 1e-300), k
    # fp32 mode: the fp64 values rounded once; the six reported coefficients stay fp64
    s = rk.Sim(n, 3, wl.DZ, wl.DT, "f32")
    s.set_media(wp, nu)
    c32 = s.get_coefficients()
    for k in ("ca", "cj", "ch", "ka", "kb", "kc"):
        assert np.array_equal(c32[k], c[k]), k
    k32 = s.get_kernel_coefficients()
    for k in ("P", "ch", "ka", "Q"):
        assert np.array_equal(k32[k], kc4[k].astype(np.float32).astype(np.float64)), k
    s.close()


def test_media_and_fields_in_any_order(rk):
    """The kernels carry G = cj J - cj kc E: set_fields before set_media, and a change of media with live
    fields, must both keep E, H, J (checked against the oracle, which is called once per media)."""
    rng = np.random.default_rng(11)
    n, nb = 777, 2
    wpA, wpB = (rng.uniform(0, 2 * np.pi * 40e9, (nb, n)) for _ in range(2))
    nuA, nuB = (rng.uniform(0, 5e10, (nb, n)) for _ in range(2))
    E0, H0, J0 = (rng.uniform(-1, 1, (nb, n)) for _ in range(3))
    H0 /= 376.73
    H0[:, -1] = 0.0
    st = oracle.State(n, nb, E0, H0, J0)
    rec1, _ = oracle.run(st, wpA, nuA, wl.DZ, wl.DT, 150, probes=[5, 700])
    rec2, _ = oracle.run(st, wpB, nuB, wl.DZ, wl.DT, 150, probes=[5, 700])
    ref = np.concatenate([rec1, rec2], axis=2)
    for kernel in (1, 2, 3):
        s = rk.Sim(n, nb, wl.DZ, wl.DT, "f64")
        s.set_fields(E0, H0, J0)              # before the media
        E, H, J = s.get_fields()
        assert np.array_equal(J, J0) and np.array_equal(E, E0)
        s.set_media(wpA, nuA)
        E, H, J = s.get_fields()              # J -> G -> J round trip
        assert np.max(np.abs(J - J0)) <= 4e-16 * np.max(np.abs(J0)) + 4e-16 * np.abs(E0).max() * 1e-2
        s.set_probes([5, 700])
        s.set_plan(kernel, 0, -1)
        s.run(150)
        s.set_media(wpB, nuB)                 # live fields: J is kept, G is re-derived
        s.run(150)
        assert grid_err(s.read_probes(), ref) <= 1e-12
        E, H, J = s.get_fields()
        assert np.max(np.abs(J - st.J)) <= 1e-12 * np.max(np.abs(st.J))
        assert np.max(np.abs(E - st.E)) <= 1e-12 * np.max(np.abs(st.E))
        s.close()


def test_rejected_media_leaves_live_fields_alone(rk):
    """rketd_set_media validates before it touches anything: after an EINVAL on live fields (the kernels' third array
    holds G of the OLD media) the run continues exactly as if the call had not happened, and a following valid
    change of media still converts J correctly."""
    rng = np.random.default_rng(12)
    n, nb = 515, 2
    wpA, wpB = (rng.uniform(0, 2 * np.pi * 40e9, (nb, n)) for _ in range(2))
    nuA, nuB = (rng.uniform(0, 5e10, (nb, n)) for _ in range(2))
    E0 = rng.uniform(-1, 1, (nb, n))
    st = oracle.State(n, nb, E0)
    recs = [oracle.run(st, wpA, nuA, wl.DZ, wl.DT, 120, probes=[7, 400])[0]]
    stA = (st.E.copy(), st.J.copy())
    recs.append(oracle.run(st, wpA, nuA, wl.DZ, wl.DT, 60, probes=[7, 400])[0])
    recs.append(oracle.run(st, wpB, nuB, wl.DZ, wl.DT, 120, probes=[7, 400])[0])
    ref = np.concatenate(recs, axis=2)
    bad = wpB.copy()
    bad[1, 300] = np.nan
    for kernel in (1, 2, 3):
        s = rk.Sim(n, nb, wl.DZ, wl.DT, "f64")
        s.set_media(wpA, nuA)
        s.set_fields(E0)
        s.set_probes([7, 400])
        s.set_plan(kernel, 0, -1)
        s.run(120)
        with pytest.raises(rk.RketdError) as ei:
            s.set_media(bad, nuB)
        assert ei.value.code == rk.EINVAL
        E, H, J = s.get_fields()                       # still E, J under media A
        assert np.max(np.abs(J - stA[1])) <= 1e-12 * np.max(np.abs(stA[1]))
        assert np.max(np.abs(E - stA[0])) <= 1e-12 * np.max(np.abs(stA[0]))
        s.run(60)                                      # media A still in force
        s.set_media(wpB, nuB)
        s.run(120)
        assert grid_err(s.read_probes(), ref) <= 1e-12
        E, H, J = s.get_fields()
        assert np.max(np.abs(J - st.J)) <= 1e-12 * np.max(np.abs(st.J))
        s.close()


# ------------------------------------------------------------------------------------------ reduced configs 2-5
@pytest.mark.parametrize("dtype", ["f64", "f32"])
def test_config2_reduced(rk, dtype):
    """Periodic random slabs, noise start; several tiles and a ragged tail (200 003 nodes)."""
    w = wl.config2(ncells=200_003, nsteps=700)
    ref = oracle.run_workload(w, omp=True)
    for plan in [(0, 0, -1), (2, 24, 0), (1, 0, -1)]:
        g = run_gpu(rk, w, dtype, *plan)
        assert grid_err(g["rec"], ref["rec"]) <= TOL[dtype], plan
        check_fields(g, ref["state"], TOL[dtype], *floors_of(w, ref))


@pytest.mark.parametrize("dtype", ["f64", "f32"])
def test_config3_reduced(rk, dtype):
    """Batched 4096-node grids (K3 with coefficients in shared memory in fp64), 24 grids, 6000 steps."""
    w = wl.config3(nbatch=24, nsteps=6000)
    ref = oracle.run_workload(w, omp=True)
    g = run_gpu(rk, w, dtype)
    assert g["kernel"] == 3 and g["launches"] == 1
    assert grid_err(g["rec"], ref["rec"]) <= TOL[dtype]
    check_fields(g, ref["state"], TOL[dtype], *floors_of(w, ref))
    # the same batch through temporal blocking, the one-barrier-per-step resident kernel, and other packings of the
    # warp-tile kernel: 2 grids per chunk on a cluster of 3 CTAs, one grid on 4 CTAs, deeper rounds
    for plan in [(2, 16, 0), (3, 0, 0), (3, 0, WT(8, 5, 2)), (3, 0, WT(0, 4, 1)), (3, 16, -1), (3, 5, WT(0, 3, 1)),
                 (3, 8, WT(12, 3, 2) | LEAN), (3, 0, WT(0, 2, 1) | LEAN), (3, 9, WT(0, 4, 1) | LEAN)]:
        g2 = run_gpu(rk, w, dtype, *plan)
        assert np.array_equal(g["rec"], g2["rec"]) and np.array_equal(g["J"], g2["J"]), plan


@pytest.mark.parametrize("dtype", ["f64", "f32"])
def test_config4_reduced(rk, dtype):
    """tanh density profile, per-node coefficients, source inside the plasma, noise start (2^20 nodes)."""
    w = wl.config4(ncells=1 << 20, nsteps=300)
    ref = oracle.run_workload(w, omp=True)
    g = run_gpu(rk, w, dtype)
    assert g["kernel"] == 2
    assert grid_err(g["rec"], ref["rec"]) <= TOL[dtype]
    check_fields(g, ref["state"], TOL[dtype], *floors_of(w, ref))


@pytest.mark.parametrize("dtype", ["f64", "f32"])
def test_config5_reduced_dft(rk, dtype):
    """Random multilayers, probes reduced on the device to |DFT| at 64 frequencies (48 grids, 5000 steps)."""
    w = wl.config5(nbatch=48)
    ref = oracle.run_workload(w, omp=True)
    s = rk.Sim.from_workload(w, dtype)
    s.run(2000)
    s.run(3000)
    mag = s.read_probes()
    s.close()
    assert mag.shape == (48, 2, 64)
    assert grid_err(mag, ref["dft_mag"]) <= TOL[dtype]
    # time-series mode of the same workload
    w2 = wl.config5(nbatch=48, dft=False)
    ref2 = oracle.run_workload(w2, omp=True)
    outs = []
    # 48 grids: chunks of 1, 2, 3, 4, 5 and 7 whole grids (7 does not divide 48: a ragged last chunk), clusters, and the
    # one-barrier-per-step kernel
    for depth, variant in [(0, -1), (0, WT(0, 1, 1)), (0, WT(0, 2, 2)), (0, WT(0, 2, 3)), (0, WT(0, 3, 4)), (0, WT(0, 3, 5)),
                           (0, WT(0, 4, 7)), (3, WT(0, 2, 2)), (0, 0), (0, 2),
                           (0, WT(0, 1, 1) | LEAN), (0, WT(0, 1, 2) | LEAN), (5, WT(0, 2, 5) | LEAN), (0, WT(0, 1, 1) | NOLEAN),
                           (0, WT(0, 0, 1) | HALF), (5, WT(0, 6, 5) | HALF), (0, WT(8, 0, 2) | HALF)]:
        g = run_gpu(rk, w2, dtype, 3, depth, variant)
        assert grid_err(g["rec"], ref2["rec"]) <= TOL[dtype], (depth, variant)
        check_fields(g, ref2["state"], TOL[dtype], *floors_of(w2, ref2))
        outs.append(g)
    for g in outs[1:]:
        for k in ("rec", "E", "H", "J"):
            assert np.array_equal(outs[0][k], g[k]), k


# ------------------------------------------------------------------------------------------ edge cases
@pytest.mark.parametrize("ncells", [3, 4, 5, 8, 9, 16, 17, 33, 127, 1025, 4093, 4097])
def test_small_and_ragged_grids(rk, ncells):
    """Smallest legal grid, grids around row boundaries, both layout offsets; source and probes ON the Mur nodes."""
    rng = np.random.default_rng(ncells)
    nb = 3
    wp = rng.uniform(0, 2 * np.pi * 40e9, (nb, ncells))
    nu = rng.uniform(0, 5e10, (nb, ncells))
    E0, H0, J0 = (rng.uniform(-1, 1, (nb, ncells)) for _ in range(3))
    H0 /= 376.73
    J0 *= 10.0
    H0[:, -1] = 0.0
    probes = sorted({0, 1, ncells // 2, ncells - 2, ncells - 1})
    tab = rng.uniform(-1, 1, 50)
    for src_cell in (0, ncells - 1, ncells // 2):
        st = oracle.State(ncells, nb, E0, H0, J0)
        rec, _ = oracle.run(st, wp, nu, wl.DZ, wl.DT, 60, src_kind=1, src_params=tab, src_cell=src_cell, probes=probes)
        outs = []
        plans = [(1, 0, -1), (0, 0, -1), (2, 7, 0), (2, 7, 6), (2, 3, 2), (3, 0, -1), (3, 5, -1), (3, 0, WT(0, 0, 2)), (3, 0, WT(0, 0, 3))]
        if ncells > 300:
            plans += [(3, 0, WT(0, 3, 1)), (3, 0, WT(2, 0, 1)), (3, 2, WT(0, 0, 3)), (3, 0, WT(0, 0, 3) | LEAN)]
        plans += [(3, 0, WT(0, 0, 1) | LEAN), (3, 3, WT(0, 0, 2) | LEAN)]
        plans += [(3, 0, WT(0, 0, 2) | HALF), (3, 3, WT(0, 0, 3) | HALF), (3, 0, WT() | NOHALF)]
        for kernel, depth, variant in plans:
            s = rk.Sim(ncells, nb, wl.DZ, wl.DT, "f64")
            s.set_media(wp, nu)
            s.set_fields(E0, H0, J0)
            s.set_source(rk.SRC_TABLE, tab, src_cell)
            s.set_probes(probes)
            s.set_plan(kernel, depth, variant)
            s.run(60)
            outs.append((s.read_probes(),) + s.get_fields())
            s.close()
            assert grid_err(outs[-1][0], rec) <= 1e-12
            assert np.max(np.abs(outs[-1][1] - st.E)) <= 1e-12 * np.max(np.abs(st.E))
            assert np.max(np.abs(outs[-1][3] - st.J)) <= 1e-12 * np.max(np.abs(st.J))
            assert np.all(outs[-1][2][:, -1] == 0.0)
        for o in outs[1:]:
            assert all(np.array_equal(a, b) for a, b in zip(outs[0], o))


def test_repeated_runs_continue_time(rk):
    w = wl.config1(nsteps=900)
    one = run_gpu(rk, w, "f64")
    for plan in [(0, 0, -1), (2, 16, 0), (1, 0, -1), (3, 0, 0), (3, 0, WT(5, 2, 1))]:
        parts = run_gpu(rk, w, "f64", *plan, chunks=[1, 0, 299, 17, 583])
        assert parts["rec"].shape == one["rec"].shape
        for k in ("rec", "E", "H", "J"):
            assert np.array_equal(one[k], parts[k]), (plan, k)


def test_P1_courant_one_translation_on_gpu(rk):
    """North_star pin (a) on the CUDA path: wp = 0, S = 1, a pulse moves one node per step; Mur (m = 0) absorbs."""
    N, n1 = 3000, 1200
    dt = wl.DZ / C0
    eta0 = 4e-7 * np.pi * C0
    k = np.arange(N, dtype=np.float64)
    f = lambda x: np.exp(-((x - 300.0) / 25.0) ** 2) * np.sin(0.2 * x)
    for kernel, variant in [(0, -1), (2, 6), (2, 0), (3, 0)]:
        s = rk.Sim(N, 1, wl.DZ, dt, "f64")
        z = np.zeros((1, N))
        s.set_media(z, z)
        s.set_fields(f(k)[None, :].copy(), (f(k + 1.0) / eta0)[None, :].copy(), None)
        s.set_plan(kernel, 0, variant)
        s.run(n1)
        E, _, _ = s.get_fields()
        assert np.max(np.abs(E[0] - f(k - n1))) < 2e-13
        s.run(2500)
        E, _, _ = s.get_fields()
        assert np.max(np.abs(E)) < 1e-12
        s.close()


def test_gauss_deriv_source_and_reset(rk):
    w = wl.config1(nsteps=400)
    s = rk.Sim.from_workload(w, "f64")
    s.run(400)
    a = s.read_probes()
    s.reset()
    s.set_fields(E=np.ascontiguousarray(w.initial_E_full()))
    s.run(400)
    b = s.read_probes()
    assert b.shape == a.shape and np.array_equal(a, b)
    assert s.counter(rk.CTR_STEPS_DONE) == 400
    s.close()


def test_device_pointers_and_stream(rk):
    """set_media / set_fields / read_probes / get_fields with torch CUDA tensors on a non-default stream."""
    import torch
    w = wl.config1(nsteps=300)
    ref = oracle.run_workload(w)
    stream = torch.cuda.Stream()
    with torch.cuda.stream(stream):
        wp, nu = (torch.from_numpy(np.ascontiguousarray(a)).cuda() for a in w.media_full())
        E0 = torch.from_numpy(w.initial_E_full()).cuda()
        stream.synchronize()
        s = rk.Sim(w.ncells, 1, w.dz, w.dt, "f64", stream=stream.cuda_stream)
        s.set_media(wp, nu)
        s.set_fields(E=E0)
        s.set_source(w.src_kind, w.src_params, w.src_cell)
        s.set_probes(w.probes)
        s.run(300)
        out = torch.empty((1, 2, 300), dtype=torch.float64, device="cuda")
        s.read_probes(out)
        assert grid_err(out.cpu().numpy(), ref["rec"]) <= 1e-12
        s.close()


def test_error_codes(rk):
    with pytest.raises(rk.RketdError) as e:
        rk.Sim(2, 1, wl.DZ, wl.DT)
    assert e.value.code == rk.EINVAL
    with pytest.raises(rk.RketdError):
        rk.Sim(100, 1, wl.DZ, 2.1 * wl.DT)              # c dt/dz > 1
    s = rk.Sim(100, 2, wl.DZ, wl.DT)
    with pytest.raises(rk.RketdError) as e:
        s.run(1)
    assert e.value.code == rk.ESTATE
    bad = np.zeros((2, 100))
    bad[1, 7] = -1.0
    with pytest.raises(rk.RketdError) as e:
        s.set_media(bad, np.zeros((2, 100)))
    assert e.value.code == rk.EINVAL
    bad[1, 7] = np.nan
    with pytest.raises(rk.RketdError):
        s.set_media(np.zeros((2, 100)), bad)
    s.set_media(np.zeros((2, 100)), np.zeros((2, 100)))
    for call in (lambda: s.set_probes([100]), lambda: s.set_probes([-1]), lambda: s.set_source(0, (1e-11, 0, 1), 100),
                 lambda: s.set_source(0, (0.0, 0, 1), 5), lambda: s.set_source(7, (), 5), lambda: s.set_plan(9, 0, -1),
                 lambda: s.set_plan(2, 100000, 4), lambda: s.run(-1)):
        with pytest.raises(rk.RketdError) as e:
            call()
        assert e.value.code == rk.EINVAL
    s.run(0)
    s.set_probes([3, 4])
    assert s.read_probes().shape == (2, 2, 0)
    big = rk.Sim(5000, 1, wl.DZ, wl.DT)
    with pytest.raises(rk.RketdError):
        big.set_plan(rk.KERNEL_RESIDENT, 0, 0)           # 5000 fp64 nodes do not fit the one-CTA resident kernel
    big.set_plan(rk.KERNEL_RESIDENT, 0, -1)              # ... but the registers of a cluster hold them (warp tiles)
    big.close()
    huge = rk.Sim(100000, 1, wl.DZ, wl.DT)
    with pytest.raises(rk.RketdError):
        huge.set_plan(rk.KERNEL_RESIDENT, 0, -1)         # 12 500 rows: more than 16 CTAs x 8 warp tiles hold
    huge.close()
    s.close()


# ---- first-order ETD, eq. (9): only the coefficient precompute differs
def test_ETD1_coefficients_and_parity_all_kernels(rk):
    rng = np.random.default_rng(9)
    n = 3000
    wp = rng.uniform(0, 2 * np.pi * 60e9, (2, n))
    nu = rng.uniform(0, 1e11, (2, n))
    wp[0, :50] = 0.0
    nu[1, :50] = 0.0
    s = rk.Sim(n, 2, wl.DZ, wl.DT, "f64")
    s.set_scheme(rk.SCHEME_ETD1)
    s.set_media(wp, nu)
    c = s.get_coefficients()
    s.close()
    o = oracle.coefficients(wp, nu, wl.DZ, wl.DT, oracle.SCHEME_ETD1)
    assert np.all(c["kc"] == 0.0)
    for k in ("ca", "cj", "ch", "ka", "kb"):
        ulp = np.abs(c[k] - o[k]) / np.maximum(np.spacing(np.abs(o[k])), 1e-300)
        # kb = eps0 wp^2 dt phi1(x): expm1 of glibc vs CUDA (1 ulp each way) plus two products
        assert ulp.max() <= (4.0 if k == "kb" else 2.0), (k, ulp.max())
    # config 1 at full size through K1, K2, K3: parity with the scheme-1 oracle, bit-identical among the kernels,
    # and NOT equal to the scheme-0 result (the switch really changes the recurrence)
    w = wl.config1()
    ref = oracle.run_workload(w, scheme=oracle.SCHEME_ETD1)
    ref0 = oracle.run_workload(w)["rec"]
    assert np.max(np.abs(ref["rec"] - ref0)) > 1e-6 * np.max(np.abs(ref0))
    first = None
    for kernel in (rk.KERNEL_STEP, rk.KERNEL_TBLOCK, rk.KERNEL_RESIDENT):
        s = rk.Sim.from_workload(w, "f64", scheme=rk.SCHEME_ETD1)
        s.set_plan(kernel, 0, -1)
        s.run(w.nsteps)
        rec = s.read_probes()
        s.close()
        assert grid_err(rec, ref["rec"]) <= 1e-12, kernel
        if first is None:
            first = rec
        else:
            assert np.array_equal(first, rec), kernel
    # fields (J through the G <-> J conversion with kc = 0) while the pulse is still on the line
    ref = oracle.run_workload(w, nsteps=1500, scheme=oracle.SCHEME_ETD1)["state"]
    s = rk.Sim.from_workload(w, "f64", scheme=rk.SCHEME_ETD1)
    s.set_plan(rk.KERNEL_TBLOCK, 0, -1)
    s.run(1500)
    E, H, J = s.get_fields()
    s.close()
    for g, r in ((E, ref.E), (H, ref.H), (J, ref.J)):
        assert np.max(np.abs(r)) > 0 and np.max(np.abs(g - r)) <= 1e-12 * np.max(np.abs(r))


def test_set_scheme_errors(rk):
    s = rk.Sim(64, 1, wl.DZ, wl.DT, "f64")
    with pytest.raises(rk.RketdError) as e:
        s.set_scheme(7)
    assert e.value.code == 1
    s.close()
