"""rketd_run_from_host (include/rketd.h): the one-call job with host inputs, whose copies overlap the steps and whose K2
passes run in a time-skewed order over pieces of the line.  It must give, BIT FOR BIT, what the sequence
rketd_reset + rketd_set_media + rketd_set_fields(E0) + rketd_run gives — for any number of pieces, any temporal depth
(also depths whose halo is wider than what a tile writes: boundaries then move k > 1 tiles per pass), Mur ends and
absorbing layers, source and probes anywhere (next to piece boundaries too) — and agree with the CPU oracle."""
import numpy as np
import pytest

import oracle

pytestmark = pytest.mark.gpu
C0 = 299792458.0
DZ = 75e-6
DT = DZ / (2 * C0)
SRC = (20e-12, 30e-12, 1.0)


@pytest.fixture(scope="module")
def rk():
    from paper_1709_00821_b200 import rketd
    return rketd


def _inputs(n, dtype, seed):
    rng = np.random.default_rng(seed)
    wp = rng.uniform(0, 2 * np.pi * 40e9, n) * (rng.uniform(size=n) > 0.3)
    nu = rng.uniform(0, 5e10, n)
    E0 = (1e-2 * rng.uniform(-1, 1, n)).astype(np.float64 if dtype == "f64" else np.float32)
    return wp, nu, E0


def _setup(rk, n, dtype, depth, probes, src_cell, pml):
    s = rk.Sim(n, 1, DZ, DT, dtype)
    s.set_plan(rk.KERNEL_TBLOCK, depth, -1)
    if pml:
        s.set_boundary(1, pml)                       # RKETD_BC_PML
    s.set_source(rk.SRC_GAUSS_DERIV, SRC, src_cell)
    s.set_probes(probes)
    return s


def _sequence(rk, n, dtype, depth, probes, src_cell, pml, wp, nu, E0, nsteps):
    s = _setup(rk, n, dtype, depth, probes, src_cell, pml)
    s.reset(); s.set_media(wp[None], nu[None]); s.set_fields(E=E0[None]); s.run(nsteps)
    out = (s.read_probes(), *s.get_fields())
    s.close()
    return out


@pytest.mark.parametrize("dtype,depth,pml", [("f64", 16, 0), ("f32", 32, 0), ("f64", 100, 0), ("f64", 7, 6), ("f32", 200, 4)])
def test_bit_identical_to_the_sequence_of_calls(rk, dtype, depth, pml):
    n, nsteps = 150_001, 333
    wp, nu, E0 = _inputs(n, dtype, 5)
    C = 8 if dtype == "f64" else 16
    rows_out = 32 - 2 * ((depth + C - 1) // C)
    tile = rows_out * C
    probes = [0, 1, n - 1, n // 2, 7 * tile - 1, 7 * tile, 7 * tile + 1, 3 * tile - 2, n - 2 * tile, 11 * tile + 30]
    src_cell = 11 * tile - 1                       # on a tile boundary: a piece boundary for npieces that divide so
    ref = _sequence(rk, n, dtype, depth, probes, src_cell, pml, wp, nu, E0, nsteps)
    assert np.max(np.abs(ref[0])) > 0.1 and np.sum(np.max(np.abs(ref[0]), axis=-1) > 1e-4) >= 8     # (layer ends read 0)
    s = _setup(rk, n, dtype, depth, probes, src_cell, pml)
    for npieces in (1, 2, 5, 13, 64, 0):
        s.run_from_host(wp, nu, E0, nsteps, npieces)
        got = (s.read_probes(), *s.get_fields())
        assert s.counter(rk.CTR_STEPS_DONE) == nsteps and s.counter(rk.CTR_KERNEL_USED) == rk.KERNEL_TBLOCK
        if npieces:
            assert 1 <= s.counter(rk.CTR_PIECES) <= npieces
            assert npieces == 1 or s.counter(rk.CTR_PIECES) > 1
        for g, r, name in zip(got, ref, ("rec", "E", "H", "J")):
            assert np.array_equal(g, r), (name, npieces)
    s.close()


def test_pinned_and_device_inputs_and_no_initial_field(rk):
    import torch
    n, nsteps = 90_000, 150
    wp, nu, _ = _inputs(n, "f64", 9)
    probes, src_cell = [10, n // 3, n - 5], n // 2
    s0 = _setup(rk, n, "f64", 16, probes, src_cell, 0)
    s0.reset(); s0.set_media(wp[None], nu[None]); s0.run(nsteps)
    ref = s0.read_probes()
    s0.close()
    s = _setup(rk, n, "f64", 16, probes, src_cell, 0)
    wp_pin, nu_pin = torch.from_numpy(wp).pin_memory(), torch.from_numpy(nu).pin_memory()
    s.run_from_host(wp_pin, nu_pin, None, nsteps, 6)
    assert np.array_equal(s.read_probes(), ref)
    s.run_from_host(wp_pin.cuda(), nu_pin.cuda(), None, nsteps, 3)      # device pointers work too (no overlap to gain)
    assert np.array_equal(s.read_probes(), ref)
    s.run(50)                                                          # the job leaves a handle that simply goes on
    assert s.counter(rk.CTR_STEPS_DONE) == nsteps + 50 and s.read_probes().shape[-1] == nsteps + 50
    s.close()


def test_against_the_oracle(rk):
    n, nsteps = 20_000, 260
    wp, nu, E0 = _inputs(n, "f64", 21)
    probes, src_cell = [3, 9_950, 10_060, n - 1], 10_000
    st = oracle.State(n, 1, E0=E0[None])
    ref, _ = oracle.run(st, wp[None], nu[None], DZ, DT, nsteps, src_kind=0, src_params=SRC, src_cell=src_cell, probes=probes)
    s = _setup(rk, n, "f64", 16, probes, src_cell, 0)
    s.run_from_host(wp, nu, E0, nsteps, 9)
    rec = s.read_probes()
    E, H, J = s.get_fields()
    s.close()
    peak = np.max(np.abs(ref))
    assert peak > 0.1 and np.max(np.abs(rec - ref)) <= 1e-12 * peak
    assert np.max(np.abs(E - st.E)) <= 1e-12 * max(peak, np.max(np.abs(st.E)))
    assert np.max(np.abs(J - st.J)) <= 1e-12 * np.max(np.abs(st.J))


def test_other_shapes_run_as_the_plain_sequence(rk):
    """batches, resident kernels and DFT probes: same call, same result, CTR_PIECES = 0"""
    n, nb, nsteps = 700, 5, 120
    rng = np.random.default_rng(2)
    wp = rng.uniform(0, 2 * np.pi * 40e9, (nb, n)); nu = rng.uniform(0, 5e10, (nb, n))
    E0 = 1e-2 * rng.uniform(-1, 1, (nb, n))
    a = rk.Sim(n, nb, DZ, DT, "f64"); b = rk.Sim(n, nb, DZ, DT, "f64")
    for s in (a, b):
        s.set_source(rk.SRC_GAUSS_DERIV, SRC, 300); s.set_probes([100, 500])
    a.set_media(wp, nu); a.set_fields(E=E0); a.run(nsteps)
    b.run_from_host(wp, nu, E0, nsteps)
    assert b.counter(rk.CTR_PIECES) == 0 and np.array_equal(a.read_probes(), b.read_probes())
    for x, y in zip(a.get_fields(), b.get_fields()):
        assert np.array_equal(x, y)
    a.close(); b.close()


def test_rejected_media_leave_a_reset_handle_without_media(rk):
    n = 60_000
    wp, nu, E0 = _inputs(n, "f64", 3)
    s = _setup(rk, n, "f64", 16, [5, n - 9], n // 2, 0)
    s.run_from_host(wp, nu, E0, 64, 4)
    good = s.read_probes()
    bad = wp.copy(); bad[n - 100] = -1.0             # in the last piece: the earlier ones have long been stepping
    with pytest.raises(rk.RketdError) as e:
        s.run_from_host(bad, nu, E0, 64, 4)
    assert e.value.code == rk.EINVAL
    with pytest.raises(rk.RketdError) as e:
        s.run(1)
    assert e.value.code == rk.ESTATE and s.counter(rk.CTR_STEPS_DONE) == 0
    assert rk.rketd_read_probes(s.h) == 0
    s.run_from_host(wp, nu, E0, 64, 4)               # and works again
    assert np.array_equal(s.read_probes(), good)
    for call in (lambda: s.run_from_host(wp, nu, E0, -1), lambda: s.run_from_host(wp, nu, E0, 10, -2), lambda: s.run_from_host(None, nu, E0, 10)):
        with pytest.raises(rk.RketdError) as e:
            call()
        assert e.value.code == rk.EINVAL
    s.close()
