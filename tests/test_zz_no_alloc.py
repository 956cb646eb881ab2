"""rketd_probe_dft_noalloc — the entry point that allocates nothing (static device scratch, include/rketd.h) — against the
existing path (rketd_set_probe_dft + rketd_run + rketd_read_probes) on the same seeded workload, `-m gpu`.

Collected last on purpose (the suite runs with `pytest -x`).  Passes alone in a fresh process and after the other tests:
it makes no assumption about what an earlier call left in the shared scratch array.

Tolerance: the bars of tests/test_gpu_parity.py (1e-12 fp64, 1e-5 fp32 of the per-series peak).  Both paths reduce the same
records with the same twiddles in fp64; the existing path adds the partial sums of several record segments, the new one
sums a series in one go, so the two differ by the rounding of those additions only.
"""
import numpy as np
import pytest

from paper_1709_00821_b200 import workloads as wl

gpu = pytest.mark.gpu

TOL = {"f64": 1e-12, "f32": 1e-5}


@pytest.fixture(scope="module")
def rk():
    from paper_1709_00821_b200 import rketd
    return rketd


def _existing_path(rk, w, dtype, chunks):
    s = rk.Sim.from_workload(w, dtype)           # DFT mode: w.dft_freqs is set
    for c in chunks:
        s.run(c)
    mag = s.read_probes()
    s.close()
    return np.asarray(mag, np.float64)


def _records_on_device(rk, w_ts, dtype, torch):
    s = rk.Sim.from_workload(w_ts, dtype)        # time-series mode of the same workload
    s.run(w_ts.nsteps)
    rec = torch.empty((w_ts.nbatch, len(w_ts.probes), w_ts.nsteps), device="cuda",
                      dtype=torch.float64 if dtype == "f64" else torch.float32)
    s.read_probes(rec)
    s.close()
    return rec


def _no_alloc(rk, rec, w, dtype, torch, nsamples=None, out=None, freqs=None):
    nb, npr, ns = rec.shape
    freqs = torch.as_tensor(w.dft_freqs, dtype=torch.float64, device="cuda") if freqs is None else freqs
    if out is None:
        out = torch.full((nb, npr, freqs.numel()), float("nan"), device="cuda", dtype=rec.dtype)
    rk.rketd_probe_dft_noalloc(rk.F64 if dtype == "f64" else rk.F32, rec, nb * npr, ns if nsamples is None else nsamples, 0, w.dt,
                               freqs, freqs.numel(), out, torch.cuda.current_stream().cuda_stream)
    return out


def _err(a, ref):
    """per grid, over its probes and frequencies, as grid_err of tests/test_gpu_parity.py (call 2 is shorter than the
    pulse's way to the second probe: that series is all zeros on both paths)"""
    a = np.asarray(a, np.float64).reshape(ref.shape[0], -1)
    ref = ref.reshape(ref.shape[0], -1)
    scale = np.abs(ref).max(1)
    assert np.all(scale > 0), "vacuous comparison"
    return float((np.abs(a - ref).max(1) / scale).max())


def test_source_calls_no_allocator():
    """the entry point's translation unit names no allocating or freeing runtime call, and takes the scratch address
    with cudaGetSymbolAddress (runs without a GPU)"""
    import os, re
    src = open(os.path.join(os.path.dirname(os.path.dirname(os.path.abspath(__file__))), "paper_1709_00821_b200", "csrc",
                            "rketd_noalloc.cu")).read()
    code = re.sub(r"//[^\n]*", "", src)
    for banned in ("cudaMalloc", "cudaFree", "cudaHostAlloc", "cudaMemPool", "cudaStreamSynchronize", "cudaDeviceSynchronize",
                   "new ", "malloc("):
        assert banned not in code, banned
    assert "cudaGetSymbolAddress" in code and "static __device__ __align__(256)" in code


@gpu
@pytest.mark.parametrize("dtype", ["f64", "f32"])
def test_two_calls_in_a_row_match_the_existing_path(rk, dtype):
    import torch
    # call 1: 40 grids x 2 probes x 3000 samples x 64 frequencies (a ragged last block of series: 80 = 2 x 32 + 16)
    w1 = wl.config5(nbatch=40, nsteps=3000)
    ref1 = _existing_path(rk, w1, dtype, [1700, 1300])
    rec1 = _records_on_device(rk, wl.config5(nbatch=40, nsteps=3000, dft=False), dtype, torch)
    # call 2: another batch, fewer samples and 13 frequencies: the table of call 1 is still behind the part call 2 rewrites
    w2 = wl.config5(nbatch=7, nsteps=1111)
    f2 = np.ascontiguousarray(w2.dft_freqs[3::5])
    assert f2.size == 13
    s = rk.Sim.from_workload(w2, dtype)
    s.set_probe_dft(f2)
    s.run(1111)
    ref2 = np.asarray(s.read_probes(), np.float64)
    s.close()
    rec2 = _records_on_device(rk, wl.config5(nbatch=7, nsteps=1111, dft=False), dtype, torch)

    out1 = _no_alloc(rk, rec1, w1, dtype, torch)
    out2 = _no_alloc(rk, rec2, w2, dtype, torch, freqs=torch.as_tensor(f2, device="cuda"))
    out1_again = _no_alloc(rk, rec1, w1, dtype, torch)                  # and back: call 2's table is overwritten
    torch.cuda.synchronize()
    assert out1.shape == (40, 2, 64) and out2.shape == (7, 2, 13)
    assert not torch.isnan(out1).any() and not torch.isnan(out2).any()   # every element written
    e1, e2 = _err(out1.cpu().numpy(), ref1), _err(out2.cpu().numpy(), ref2)
    print(f"no-alloc |DFT| vs existing path [{dtype}]: call 1 {e1:.2e}, call 2 {e2:.2e}")
    assert e1 <= TOL[dtype] and e2 <= TOL[dtype]
    assert torch.equal(out1, out1_again)


@gpu
def test_limits_and_errors(rk):
    import torch
    w = wl.config5(nbatch=2, nsteps=64)
    f = torch.as_tensor(w.dft_freqs, device="cuda")
    rec = torch.zeros((2, 2, 64), device="cuda", dtype=torch.float64)
    out = torch.empty((2, 2, 64), device="cuda", dtype=torch.float64)
    F64 = rk.F64
    # beyond the static table: 8193 samples x 64 frequencies > 2^19 entries (no kernel runs: sizes are checked first)
    with pytest.raises(rk.RketdError) as ei:
        rk.rketd_probe_dft_noalloc(F64, rec, 4, rk.NOALLOC_MAX_TWIDDLES // 64 + 1, 0, w.dt, f, 64, out)
    assert ei.value.code == rk.EINVAL and "RKETD_NOALLOC_MAX_TWIDDLES" in str(ei.value)
    with pytest.raises(rk.RketdError) as ei:
        rk.rketd_probe_dft_noalloc(F64, rec, rk.NOALLOC_MAX_SERIES + 1, 64, 0, w.dt, f, 64, out)
    assert ei.value.code == rk.EINVAL and "RKETD_NOALLOC_MAX_SERIES" in str(ei.value)
    # host memory is rejected, not dereferenced
    with pytest.raises(rk.RketdError) as ei:
        rk.rketd_probe_dft_noalloc(F64, np.zeros((2, 2, 64)), 4, 64, 0, w.dt, f, 64, out)
    assert ei.value.code == rk.EINVAL and "device memory" in str(ei.value)
    with pytest.raises(rk.RketdError):
        rk.rketd_probe_dft_noalloc(7, rec, 4, 64, 0, w.dt, f, 64, out)
    with pytest.raises(rk.RketdError):
        rk.rketd_probe_dft_noalloc(F64, rec, 4, 64, 0, 0.0, f, 64, out)
    # exactly at the limit is accepted; an all-zero record gives zeros; zero samples give zeros; empty inputs are no-ops
    n = rk.NOALLOC_MAX_TWIDDLES // 64
    big = torch.zeros((1, 1, n), device="cuda", dtype=torch.float64)
    o = torch.full((1, 1, 64), 5.0, device="cuda", dtype=torch.float64)
    rk.rketd_probe_dft_noalloc(F64, big, 1, n, 0, w.dt, f, 64, o)
    assert float(o.abs().max()) == 0.0
    o.fill_(5.0)
    rk.rketd_probe_dft_noalloc(F64, big, 1, 0, 0, w.dt, f, 64, o)
    assert float(o.abs().max()) == 0.0
    o.fill_(5.0)
    rk.rketd_probe_dft_noalloc(F64, big, 0, n, 0, w.dt, f, 64, o)
    rk.rketd_probe_dft_noalloc(F64, big, 1, n, 0, w.dt, f, 0, o)
    assert float(o.min()) == 5.0
    # a single tone against the closed form: rec[n] = cos(2 pi f0 (n+1) dt) over whole periods -> |X(f0)| = N/2
    dt = 1e-12
    f0 = torch.tensor([25e9, 50e9], device="cuda", dtype=torch.float64)      # 40 and 20 samples per period
    N = 4000
    t = (torch.arange(N, device="cuda", dtype=torch.float64) + 1) * dt
    tone = torch.cos(2 * np.pi * 25e9 * t).reshape(1, 1, N).contiguous()
    o2 = torch.empty((1, 1, 2), device="cuda", dtype=torch.float64)
    rk.rketd_probe_dft_noalloc(F64, tone, 1, N, 0, dt, f0, 2, o2)
    got = o2.cpu().numpy().ravel()
    assert abs(got[0] - N / 2) <= 1e-9 * N and got[1] <= 1e-9 * N
