"""The fixed-index instantiations of the resident kernels (SF_FAST, DESIGN.md section 16 item 13) against the oracle and the
per-step kernel K1 — `-m gpu`.

A warp takes them when node ncells-1 is the last node of its lane, the source and every probe the first of theirs, and no
lane records two probes (WarpSpecial::fast); any other layout keeps the general select arithmetic.  Each case below sits on
one side of one of those conditions, so that both code paths and every mixture inside one grid (a warp on the fast path
next to a warp on the general one) are compared: records and final fields within 1e-12 / 1e-5 of the oracle, and K3 (both
variants of k3_resident, warp tiles whole-row and half-row) bit for bit equal to K1.
"""
import numpy as np
import pytest

import oracle
from paper_1709_00821_b200 import workloads as wl

pytestmark = pytest.mark.gpu

TOL = {"f64": 1e-12, "f32": 1e-5}
WTILE, HALF, NOHALF = 0x40000000, 0x08000000, 0x04000000


@pytest.fixture(scope="module")
def rk():
    from paper_1709_00821_b200 import rketd
    return rketd


# (ncells, source cell, probes): rows hold 8 fp64 / 16 fp32 nodes
CASES = [
    (1024, 64, (192, 832)),            # config 5's layout: everything on the fast path
    (1024, 64, (192, 832, 1008)),      # a third probe, first of its lane, in the warp with node ncells-1
    (1024, 65, (192, 832)),            # source second in its lane: its warp general, the last warp fast
    (1024, 64, (195, 832)),            # one probe mid-lane
    (1024, 64, (192, 196, 832)),       # two probes among one lane's nodes (192 and 196: lane 24 of fp64 rows, lane 12 of fp32 rows)
    (1024, 0, (0, 1023)),              # source and probes ON the Mur nodes (node 0 first of its lane, node 1023 last: a probe that is not first)
    (1023, 64, (192, 832)),            # node ncells-1 not last in its lane (general right end), the rest aligned
    (1032, 64, (192, 832)),            # aligned for fp64 rows only (1032 = 129 x 8)
    (2048, 512, (256, 1536)),          # 8 / 4 warps per grid
    (4096, 400, (1200, 3200)),         # config 3's layout
]


@pytest.mark.parametrize("dtype", ["f64", "f32"])
@pytest.mark.parametrize("ncells,src_cell,probes", CASES)
def test_fixed_index_and_general_paths(rk, dtype, ncells, src_cell, probes):
    rng = np.random.default_rng(ncells * 7919 + src_cell * 31 + len(probes))
    nb, nsteps = 5, 257
    # piecewise-constant media with two slabs (uniform and non-uniform warps), random initial fields
    wp = np.zeros((nb, ncells)); nu = np.zeros((nb, ncells))
    for g in range(nb):
        a, b = sorted(rng.integers(ncells // 4, 3 * ncells // 4, 2))
        wp[g, a:b + 1] = rng.uniform(2 * np.pi * 5e9, 2 * np.pi * 60e9)
        nu[g, a:b + 1] = rng.uniform(0, 1e11)
        c = int(rng.integers(8, ncells // 8))
        wp[g, c:c + 13] = rng.uniform(2 * np.pi * 5e9, 2 * np.pi * 60e9)
        nu[g, c:c + 13] = rng.uniform(0, 1e11)
    E0 = rng.uniform(-1, 1, (nb, ncells))
    H0 = rng.uniform(-1, 1, (nb, ncells)) / 376.73
    H0[:, -1] = 0.0
    tab = rng.uniform(-1, 1, nsteps)
    probes = list(probes)
    st = oracle.State(ncells, nb, E0, H0, np.zeros((nb, ncells)))
    rec, _ = oracle.run(st, wp, nu, wl.DZ, wl.DT, nsteps, src_kind=1, src_params=tab, src_cell=src_cell, probes=probes)
    npd = np.float64 if dtype == "f64" else np.float32
    outs = []
    plans = [(1, 0, -1), (3, 0, -1), (3, 0, 0), (3, 0, 2), (3, 0, WTILE | (2 << 16)), (3, 4, WTILE | (1 << 16) | HALF),
             (3, 0, WTILE | NOHALF)]
    for kernel, depth, variant in plans:
        s = rk.Sim(ncells, nb, wl.DZ, wl.DT, dtype)
        s.set_media(wp, nu)
        s.set_fields(E0.astype(npd), H0.astype(npd), None)
        s.set_source(rk.SRC_TABLE, tab, src_cell)
        s.set_probes(probes)
        try:
            s.set_plan(kernel, depth, variant)
        except rk.RketdError:
            s.close()              # a packing this grid size cannot take
            continue
        s.run(100)
        s.run(nsteps - 100)
        outs.append((s.read_probes(),) + s.get_fields())
        s.close()
    assert len(outs) >= 4
    g = np.asarray(outs[0][0], np.float64)
    scale = np.abs(rec).reshape(nb, -1).max(1)
    assert np.all(scale > 0)
    assert float((np.abs(g - rec).reshape(nb, -1).max(1) / scale).max()) <= TOL[dtype]
    assert np.max(np.abs(np.asarray(outs[0][1], np.float64) - st.E)) <= TOL[dtype] * max(np.max(np.abs(st.E)), float(scale.max()))
    for o in outs[1:]:
        for a, b in zip(outs[0], o):
            assert np.array_equal(a, b)
