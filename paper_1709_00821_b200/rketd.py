"""Thin ctypes binding of librketd (include/rketd.h): argument marshalling only.

Same names as the C ABI (``rketd_create`` ... ``rketd_read_probes``), plus the small ``Sim``
convenience class that tests and bench.py use.  Pointers may be numpy arrays (host), torch
tensors (host or CUDA) or raw integers.  PyTorch is used only by callers, for device memory and
streams.  The library must exist: there is no fallback path (ImportError / OSError otherwise).
"""
from __future__ import annotations

import ctypes
import os
from typing import Optional, Sequence

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "librketd.so")

F64, F32 = 0, 1
OK, EINVAL, ENOMEM, ECUDA, ESTATE = 0, 1, 2, 3, 4
SRC_NONE, SRC_GAUSS_DERIV, SRC_TABLE = -1, 0, 1
KERNEL_AUTO, KERNEL_STEP, KERNEL_TBLOCK, KERNEL_RESIDENT = 0, 1, 2, 3
CTR_LAUNCHES, CTR_STEP_LAUNCHES, CTR_KERNEL_USED, CTR_DEPTH_USED, CTR_STEPS_DONE, CTR_TILE_CELLS, \
    CTR_HALO_CELLS, CTR_STATE_BYTES, CTR_PIECES = range(9)

EXPORTS = ["rketd_create", "rketd_set_media", "rketd_set_source", "rketd_set_probes", "rketd_set_probe_dft",
           "rketd_set_fields", "rketd_reset", "rketd_discard_records", "rketd_set_plan", "rketd_run", "rketd_run_from_host",
           "rketd_read_probes",
           "rketd_get_fields", "rketd_get_coefficients", "rketd_get_kernel_coefficients", "rketd_set_scheme",
           "rketd_set_boundary", "rketd_read_probe_dft",
           "rketd_read_sweep_rt", "rketd_measure_peak", "rketd_probe_dft_noalloc", "rketd_noalloc_last_error",
           "rketd_get_counter", "rketd_destroy", "rketd_last_error"]
PEAK_NAMES = ("dfma_1reg", "dfma_2reg", "dfma_3reg", "dfma_2reg_const", "ffma_1reg", "ffma_2reg", "ffma_3reg",
              "ffma_2reg_const", "mix_f64", "mix_f32", "lds128", "lat_dfma", "lat_shfl64", "lat_step_f64", "lat_step_f32",
              "lat_bar_sync_256", "lat_cluster_barrier_8x128")      # index = RKETD_PEAK_* / RKETD_LAT_*
RESIDENT_WTILE_FLAG = 0x40000000
RESIDENT_WTILE_NOLEAN, RESIDENT_WTILE_LEAN, RESIDENT_WTILE_HALF, RESIDENT_WTILE_NOHALF = 0x20000000, 0x10000000, 0x08000000, 0x04000000


def RESIDENT_WTILE(nw: int = 0, nc: int = 0, k: int = 0) -> int:
    """rketd_set_plan variant for KERNEL_RESIDENT: k grids per chunk on a cluster of nc CTAs x nw warps (0 = library's choice)"""
    return RESIDENT_WTILE_FLAG | (k << 16) | (nc << 8) | nw


SCHEME_ETD2, SCHEME_ETD1 = 0, 1
BC_MUR, BC_PML = 0, 1

if not os.path.exists(LIB_PATH):
    raise ImportError(f"{LIB_PATH} is missing: build it with `python -m paper_1709_00821_b200.build` "
                      "(librketd has no CPU fallback)")
_lib = ctypes.CDLL(LIB_PATH)

_vp, _i64, _i32, _dbl = ctypes.c_void_p, ctypes.c_int64, ctypes.c_int, ctypes.c_double
_lib.rketd_create.argtypes = [ctypes.POINTER(_vp), _i64, _i64, _dbl, _dbl, _i32, _vp]
_lib.rketd_set_media.argtypes = [_vp, _vp, _vp]
_lib.rketd_set_source.argtypes = [_vp, _i32, _vp, _i64, _i64]
_lib.rketd_set_probes.argtypes = [_vp, _vp, _i32]
_lib.rketd_set_probe_dft.argtypes = [_vp, _vp, _i32]
_lib.rketd_set_fields.argtypes = [_vp, _vp, _vp, _vp]
_lib.rketd_reset.argtypes = [_vp]
_lib.rketd_discard_records.argtypes = [_vp]
_lib.rketd_set_plan.argtypes = [_vp, _i32, _i32, _i32]
_lib.rketd_run.argtypes = [_vp, _i64]
_lib.rketd_run_from_host.argtypes = [_vp, _vp, _vp, _vp, _i64, _i32]
_lib.rketd_read_probes.argtypes = [_vp, _vp, _i64, ctypes.POINTER(_i64)]
_lib.rketd_get_fields.argtypes = [_vp, _vp, _vp, _vp]
_lib.rketd_get_coefficients.argtypes = [_vp, _vp, _vp]
_lib.rketd_get_kernel_coefficients.argtypes = [_vp, _vp]
_lib.rketd_set_scheme.argtypes = [_vp, _i32]
_lib.rketd_set_boundary.argtypes = [_vp, _i32, _i32, _dbl, _dbl]
_lib.rketd_read_probe_dft.argtypes = [_vp, _vp, _vp, _i64]
_lib.rketd_get_counter.argtypes = [_vp, _i32]
_lib.rketd_get_counter.restype = _i64
_lib.rketd_destroy.argtypes = [_vp]
_lib.rketd_destroy.restype = None
_lib.rketd_last_error.argtypes = [_vp]
_lib.rketd_last_error.restype = ctypes.c_char_p
_lib.rketd_measure_peak.argtypes = [_i32, _i32, _vp, _vp]
_lib.rketd_read_sweep_rt.argtypes = [_vp, _vp, _i32, _i32, _vp, _vp, _i64]
_lib.rketd_probe_dft_noalloc.argtypes = [_i32, _vp, _i64, _i64, _i64, _dbl, _vp, _i32, _vp, _vp]
_lib.rketd_probe_dft_noalloc.restype = _i32
_lib.rketd_noalloc_last_error.argtypes = []
_lib.rketd_noalloc_last_error.restype = ctypes.c_char_p
for _n in EXPORTS[:19]:
    getattr(_lib, _n).restype = _i32


class RketdError(RuntimeError):
    def __init__(self, code: int, msg: str):
        super().__init__(f"librketd error {code}: {msg}")
        self.code = code


def _ptr(a) -> Optional[int]:
    """address of a numpy array / torch tensor / int / None (the caller keeps the object alive)"""
    if a is None:
        return None
    if isinstance(a, int):
        return a
    if isinstance(a, np.ndarray):
        assert a.flags.c_contiguous
        return a.ctypes.data
    if hasattr(a, "data_ptr"):
        assert a.is_contiguous()
        return a.data_ptr()
    raise TypeError(type(a))


def _check(h, rc: int):
    if rc != OK:
        raise RketdError(rc, (_lib.rketd_last_error(h) or b"").decode())


# ---- the C ABI, one to one -------------------------------------------------------------------
def rketd_create(ncells: int, nbatch: int, dz: float, dt: float, dtype: int = F64, cuda_stream: int = 0):
    h = _vp()
    _check(None, _lib.rketd_create(ctypes.byref(h), ncells, nbatch, dz, dt, dtype, cuda_stream or None))
    return h


def rketd_set_media(h, wp, nu):
    _check(h, _lib.rketd_set_media(h, _ptr(wp), _ptr(nu)))


def rketd_set_source(h, kind: int, params: Sequence[float], cell: int):
    prm = np.ascontiguousarray(params, np.float64)
    _check(h, _lib.rketd_set_source(h, kind, _ptr(prm) if prm.size else None, prm.size, cell))


def rketd_set_probes(h, cells: Sequence[int]):
    c = np.ascontiguousarray(cells, np.int64)
    _check(h, _lib.rketd_set_probes(h, _ptr(c) if c.size else None, c.size))


def rketd_set_probe_dft(h, freqs_hz: Optional[Sequence[float]]):
    f = np.ascontiguousarray([] if freqs_hz is None else freqs_hz, np.float64)
    _check(h, _lib.rketd_set_probe_dft(h, _ptr(f) if f.size else None, f.size))


def rketd_set_fields(h, E=None, H=None, J=None):
    _check(h, _lib.rketd_set_fields(h, _ptr(E), _ptr(H), _ptr(J)))


def rketd_reset(h):
    _check(h, _lib.rketd_reset(h))


def rketd_discard_records(h):
    _check(h, _lib.rketd_discard_records(h))


def rketd_set_scheme(h, scheme: int):
    _check(h, _lib.rketd_set_scheme(h, scheme))


def rketd_read_probe_dft(h, re, im):
    _check(h, _lib.rketd_read_probe_dft(h, _ptr(re), _ptr(im), re.size if isinstance(re, np.ndarray) else re.numel()))


def rketd_read_sweep_rt(h, h_vacuum, probe_r: int, probe_t: int, R, T):
    _check(h, _lib.rketd_read_sweep_rt(h, h_vacuum, probe_r, probe_t, _ptr(R), _ptr(T),
                                       R.size if isinstance(R, np.ndarray) else R.numel()))


def rketd_set_boundary(h, kind: int, npml: int = 5, grading: float = 3.0, R0: float = 1e-6):
    _check(h, _lib.rketd_set_boundary(h, kind, npml, grading, R0))


def rketd_set_plan(h, kernel: int = KERNEL_AUTO, depth: int = 0, variant: int = -1):
    _check(h, _lib.rketd_set_plan(h, kernel, depth, variant))


def rketd_run(h, nsteps: int):
    _check(h, _lib.rketd_run(h, nsteps))


def rketd_run_from_host(h, wp, nu, E0, nsteps: int, npieces: int = 0):
    _check(h, _lib.rketd_run_from_host(h, _ptr(wp), _ptr(nu), _ptr(E0), nsteps, npieces))


def rketd_read_probes(h, out=None, out_bytes: int = 0) -> int:
    n = _i64()
    _check(h, _lib.rketd_read_probes(h, _ptr(out), out_bytes, ctypes.byref(n)))
    return n.value


def rketd_get_fields(h, E=None, H=None, J=None):
    _check(h, _lib.rketd_get_fields(h, _ptr(E), _ptr(H), _ptr(J)))


def rketd_get_coefficients(h, out, chh_m=None):
    _check(h, _lib.rketd_get_coefficients(h, _ptr(out), _ptr(chh_m)))


def rketd_get_kernel_coefficients(h, out):
    _check(h, _lib.rketd_get_kernel_coefficients(h, _ptr(out)))


def rketd_get_counter(h, which: int) -> int:
    return _lib.rketd_get_counter(h, which)


def rketd_measure_peak(what: int, iters: int = 4000, cuda_stream: int = 0):
    """(per ns over the device, per clock and SM, SM MHz held, SMs) of microbenchmark RKETD_PEAK_* `what`"""
    out = np.zeros(4, np.float64)
    _check(None, _lib.rketd_measure_peak(what, iters, _ptr(out), cuda_stream or None))
    return {"name": PEAK_NAMES[what], "per_ns": float(out[0]), "per_clk_sm": float(out[1]), "sm_mhz": float(out[2]),
            "sms": int(out[3])}


NOALLOC_MAX_TWIDDLES, NOALLOC_MAX_SERIES = 1 << 19, 1 << 24


def rketd_probe_dft_noalloc(dtype: int, rec, nseries: int, nsamples: int, step0: int, dt: float, freqs_hz, nfreq: int, out,
                            cuda_stream: int = 0):
    """records -> |DFT| without any allocation (include/rketd.h); rec, freqs_hz, out: DEVICE tensors or raw addresses"""
    rc = _lib.rketd_probe_dft_noalloc(dtype, _ptr(rec), nseries, nsamples, step0, dt, _ptr(freqs_hz), nfreq, _ptr(out),
                                      cuda_stream or None)
    if rc != OK:
        raise RketdError(rc, rketd_noalloc_last_error())


def rketd_noalloc_last_error() -> str:
    return (_lib.rketd_noalloc_last_error() or b"").decode()


def rketd_destroy(h):
    _lib.rketd_destroy(h)


def rketd_last_error(h=None) -> str:
    return (_lib.rketd_last_error(h) or b"").decode()


# ---- convenience wrapper (still marshalling only) --------------------------------------------
class Sim:
    """Owns one rketd_sim handle.  Arrays in/out are numpy (host) unless a torch tensor is given."""

    def __init__(self, ncells: int, nbatch: int, dz: float, dt: float, dtype: str = "f64", stream: int = 0):
        self.ncells, self.nbatch = ncells, nbatch
        self.dtype = dtype
        self.np_dtype = np.float64 if dtype == "f64" else np.float32
        self.nprobes = 0
        self.nfreq = 0
        self.h = rketd_create(ncells, nbatch, dz, dt, F64 if dtype == "f64" else F32, stream)

    @classmethod
    def from_workload(cls, w, dtype: str = "f64", stream: int = 0, b0: int = 0, b1: Optional[int] = None,
                      scheme: int = SCHEME_ETD2, pml=None):
        b1 = w.nbatch if b1 is None else b1
        s = cls(w.ncells, b1 - b0, w.dz, w.dt, dtype, stream)
        s.set_scheme(scheme)
        if pml is not None:                      # (npml, grading, R0)
            s.set_boundary(BC_PML, int(pml[0]), float(pml[1]), float(pml[2]))
        wp, nu = w.media(0, w.ncells, b0, b1)
        s.set_media(np.ascontiguousarray(wp), np.ascontiguousarray(nu))
        E0 = w.initial_E(0, w.ncells, b0, b1)
        if E0 is not None:
            s.set_fields(E=np.ascontiguousarray(E0, s.np_dtype))
        s.set_source(w.src_kind, w.src_params, w.src_cell)
        s.set_probes(w.probes)
        if w.dft_freqs is not None:
            s.set_probe_dft(w.dft_freqs)
        return s

    def set_media(self, wp, nu): rketd_set_media(self.h, wp, nu)
    def set_source(self, kind, params, cell): rketd_set_source(self.h, kind, params, cell)

    def set_probes(self, cells):
        rketd_set_probes(self.h, cells)
        self.nprobes = len(cells)

    def set_probe_dft(self, freqs):
        rketd_set_probe_dft(self.h, freqs)
        self.nfreq = 0 if freqs is None else len(freqs)

    def set_fields(self, E=None, H=None, J=None): rketd_set_fields(self.h, E, H, J)
    def reset(self): rketd_reset(self.h)
    def discard_records(self): rketd_discard_records(self.h)
    def set_plan(self, kernel=KERNEL_AUTO, depth=0, variant=-1): rketd_set_plan(self.h, kernel, depth, variant)

    def set_scheme(self, scheme): rketd_set_scheme(self.h, scheme)

    def set_boundary(self, kind, npml=5, grading=3.0, R0=1e-6): rketd_set_boundary(self.h, kind, npml, grading, R0)
    def run(self, nsteps): rketd_run(self.h, nsteps)

    def run_from_host(self, wp, nu, E=None, nsteps=0, npieces=0):
        """reset + set_media + set_fields(E) + run in one call, copies overlapped with the steps (one long line)"""
        rketd_run_from_host(self.h, wp, nu, E, nsteps, npieces)

    def counter(self, which): return rketd_get_counter(self.h, which)

    def read_probes(self, out=None):
        n = rketd_read_probes(self.h)
        if out is None:
            out = np.empty((self.nbatch, self.nprobes, n), self.np_dtype)
        nbytes = out.nbytes if isinstance(out, np.ndarray) else out.numel() * out.element_size()
        rketd_read_probes(self.h, out, nbytes)
        return out

    def read_probe_dft(self):
        """complex [nbatch][nprobes][nfreq] accumulators of the device DFT"""
        nf = rketd_read_probes(self.h)
        re = np.empty((self.nbatch, self.nprobes, nf), np.float64)
        im = np.empty_like(re)
        rketd_read_probe_dft(self.h, re, im)
        return re + 1j * im

    def read_sweep_rt(self, vacuum: "Sim", probe_r: int = 0, probe_t: int = 1):
        """(|R|, |T|) [nbatch][nfreq] of this slab batch against the vacuum handle, formed on the device"""
        nf = rketd_read_probes(self.h)
        R = np.empty((self.nbatch, nf), np.float64)
        T = np.empty_like(R)
        rketd_read_sweep_rt(self.h, vacuum.h, probe_r, probe_t, R, T)
        return R, T

    def get_fields(self):
        E, H, J = (np.empty((self.nbatch, self.ncells), self.np_dtype) for _ in range(3))
        rketd_get_fields(self.h, E, H, J)
        return E, H, J

    def get_coefficients(self):
        out = np.empty((6, self.nbatch, self.ncells), np.float64)
        cm = np.empty(2, np.float64)
        rketd_get_coefficients(self.h, out, cm)
        d = {k: out[i] for i, k in enumerate(("ca", "cj", "ch", "ka", "kb", "kc"))}
        d["chh"], d["m"] = float(cm[0]), float(cm[1])
        return d

    def get_kernel_coefficients(self):
        out = np.empty((4, self.nbatch, self.ncells), np.float64)
        rketd_get_kernel_coefficients(self.h, out)
        return {k: out[i] for i, k in enumerate(("P", "ch", "ka", "Q"))}

    def close(self):
        if self.h is not None:
            rketd_destroy(self.h)
            self.h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass
