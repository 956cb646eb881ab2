"""Thin ctypes binding of the 2-D TMz entry points of librketd (include/rketd2d.h): argument marshalling only.

Same names as the C ABI (``rketd2d_create`` ... ``rketd2d_read_probes``) plus the small ``Sim2D`` convenience class
that tests and bench.py use.  There is no fallback path: the library must exist.
"""
from __future__ import annotations

import ctypes
from typing import Sequence

import numpy as np

from .rketd import (F32, F64, OK, RketdError, _dbl, _i32, _i64, _lib, _ptr, _vp)

BC_MUR, BC_PEC, BC_PML = 0, 1, 2
KERNEL_AUTO, KERNEL_STEP, KERNEL_STREAM = 0, 1, 2
CTR_LAUNCHES, CTR_STEP_LAUNCHES, CTR_KERNEL_USED, CTR_DEPTH_USED, CTR_STEPS_DONE, CTR_STRIP_COLS, CTR_HALO_COLS, \
    CTR_SEG_ROWS, CTR_STATE_BYTES = range(9)

EXPORTS = ["rketd2d_create", "rketd2d_set_media", "rketd2d_set_boundary_pml", "rketd2d_set_boundary", "rketd2d_set_source", "rketd2d_set_probes",
           "rketd2d_set_fields", "rketd2d_get_fields", "rketd2d_reset", "rketd2d_set_plan", "rketd2d_run",
           "rketd2d_read_probes", "rketd2d_get_kernel_coefficients", "rketd2d_discard_records", "rketd2d_get_counter",
           "rketd2d_destroy", "rketd2d_last_error"]
TE_EXPORTS = ["rketd2d_te_create", "rketd2d_te_set_media", "rketd2d_te_set_boundary", "rketd2d_te_set_source",
              "rketd2d_te_set_probes", "rketd2d_te_set_fields", "rketd2d_te_get_fields", "rketd2d_te_run",
              "rketd2d_te_read_probes", "rketd2d_te_get_counter", "rketd2d_te_destroy", "rketd2d_te_last_error"]
EXPORTS += TE_EXPORTS
EX, EY = 0, 1                # component ids of TEz sources and probes

_lib.rketd2d_create.argtypes = [ctypes.POINTER(_vp), _i64, _i64, _dbl, _dbl, _dbl, _i32, _vp]
_lib.rketd2d_set_media.argtypes = [_vp, _vp, _vp]
_lib.rketd2d_set_boundary.argtypes = [_vp, _i32]
_lib.rketd2d_set_boundary_pml.argtypes = [_vp, _i32, _dbl, _dbl]
_lib.rketd2d_set_source.argtypes = [_vp, _i32, _vp, _i64, _i64, _i64]
_lib.rketd2d_set_probes.argtypes = [_vp, _vp, _i32]
_lib.rketd2d_set_fields.argtypes = [_vp, _vp, _vp, _vp, _vp]
_lib.rketd2d_get_fields.argtypes = [_vp, _vp, _vp, _vp, _vp]
_lib.rketd2d_reset.argtypes = [_vp]
_lib.rketd2d_discard_records.argtypes = [_vp]
_lib.rketd2d_set_plan.argtypes = [_vp, _i32, _i32]
_lib.rketd2d_run.argtypes = [_vp, _i64]
_lib.rketd2d_read_probes.argtypes = [_vp, _vp, _i64, ctypes.POINTER(_i64)]
_lib.rketd2d_get_kernel_coefficients.argtypes = [_vp, _vp, _vp]
_lib.rketd2d_get_counter.argtypes = [_vp, _i32]
_lib.rketd2d_get_counter.restype = _i64
_lib.rketd2d_destroy.argtypes = [_vp]
_lib.rketd2d_destroy.restype = None
_lib.rketd2d_last_error.argtypes = [_vp]
_lib.rketd2d_last_error.restype = ctypes.c_char_p
for _n in EXPORTS[:14]:
    getattr(_lib, _n).restype = _i32
_lib.rketd2d_te_create.argtypes = [ctypes.POINTER(_vp), _i64, _i64, _dbl, _dbl, _dbl, _i32, _vp]
_lib.rketd2d_te_set_media.argtypes = [_vp, _vp, _vp]
_lib.rketd2d_te_set_boundary.argtypes = [_vp, _i32]
_lib.rketd2d_te_set_source.argtypes = [_vp, _i32, _vp, _i64, _i64, _i64, _i32]
_lib.rketd2d_te_set_probes.argtypes = [_vp, _vp, _i32]
_lib.rketd2d_te_set_fields.argtypes = [_vp] + [_vp] * 5
_lib.rketd2d_te_get_fields.argtypes = [_vp] + [_vp] * 5
_lib.rketd2d_te_run.argtypes = [_vp, _i64]
_lib.rketd2d_te_read_probes.argtypes = [_vp, _vp, _i64, ctypes.POINTER(_i64)]
_lib.rketd2d_te_get_counter.argtypes = [_vp, _i32]
_lib.rketd2d_te_get_counter.restype = _i64
_lib.rketd2d_te_destroy.argtypes = [_vp]
_lib.rketd2d_te_destroy.restype = None
_lib.rketd2d_te_last_error.argtypes = [_vp]
_lib.rketd2d_te_last_error.restype = ctypes.c_char_p
for _n in TE_EXPORTS[:9]:
    getattr(_lib, _n).restype = _i32


def _check(h, rc: int):
    if rc != OK:
        raise RketdError(rc, (_lib.rketd2d_last_error(h) or b"").decode())


# ---- the C ABI, one to one -------------------------------------------------------------------
def rketd2d_create(nx: int, ny: int, dx: float, dy: float, dt: float, dtype: int = F64, cuda_stream: int = 0):
    h = _vp()
    _check(None, _lib.rketd2d_create(ctypes.byref(h), nx, ny, dx, dy, dt, dtype, cuda_stream or None))
    return h


def rketd2d_set_media(h, wp, nu):
    _check(h, _lib.rketd2d_set_media(h, _ptr(wp), _ptr(nu)))


def rketd2d_set_boundary(h, kind: int):
    _check(h, _lib.rketd2d_set_boundary(h, kind))


def rketd2d_set_boundary_pml(h, npml: int = 5, grading: float = 3.0, R0: float = 1e-6):
    _check(h, _lib.rketd2d_set_boundary_pml(h, npml, grading, R0))


def rketd2d_set_source(h, kind: int, params: Sequence[float], i: int, j: int):
    prm = np.ascontiguousarray(params, np.float64)
    _check(h, _lib.rketd2d_set_source(h, kind, _ptr(prm) if prm.size else None, prm.size, i, j))


def rketd2d_set_probes(h, ij):
    c = np.ascontiguousarray(ij, np.int64).reshape(-1, 2)
    _check(h, _lib.rketd2d_set_probes(h, _ptr(c) if c.size else None, c.shape[0]))


def rketd2d_set_fields(h, Ez=None, Hx=None, Hy=None, Jz=None):
    _check(h, _lib.rketd2d_set_fields(h, _ptr(Ez), _ptr(Hx), _ptr(Hy), _ptr(Jz)))


def rketd2d_get_fields(h, Ez=None, Hx=None, Hy=None, Jz=None):
    _check(h, _lib.rketd2d_get_fields(h, _ptr(Ez), _ptr(Hx), _ptr(Hy), _ptr(Jz)))


def rketd2d_reset(h):
    _check(h, _lib.rketd2d_reset(h))


def rketd2d_discard_records(h):
    _check(h, _lib.rketd2d_discard_records(h))


def rketd2d_set_plan(h, kernel: int = KERNEL_AUTO, depth: int = 0):
    _check(h, _lib.rketd2d_set_plan(h, kernel, depth))


def rketd2d_run(h, nsteps: int):
    _check(h, _lib.rketd2d_run(h, nsteps))


def rketd2d_read_probes(h, out=None, out_bytes: int = 0) -> int:
    n = _i64()
    _check(h, _lib.rketd2d_read_probes(h, _ptr(out), out_bytes, ctypes.byref(n)))
    return n.value


def rketd2d_get_kernel_coefficients(h, out=None, globals_=None):
    _check(h, _lib.rketd2d_get_kernel_coefficients(h, _ptr(out), _ptr(globals_)))


def rketd2d_get_counter(h, which: int) -> int:
    return _lib.rketd2d_get_counter(h, which)


def rketd2d_destroy(h):
    _lib.rketd2d_destroy(h)


def rketd2d_last_error(h=None) -> str:
    return (_lib.rketd2d_last_error(h) or b"").decode()


# ---- convenience wrapper (still marshalling only) --------------------------------------------
class Sim2D:
    """Owns one rketd2d_sim handle.  Arrays in/out are numpy (host) unless a torch tensor is given."""

    def __init__(self, nx: int, ny: int, dx: float, dy: float, dt: float, dtype: str = "f64", stream: int = 0):
        self.nx, self.ny, self.dtype = nx, ny, dtype
        self.np_dtype = np.float64 if dtype == "f64" else np.float32
        self.nprobes = 0
        self.h = rketd2d_create(nx, ny, dx, dy, dt, F64 if dtype == "f64" else F32, stream)

    @classmethod
    def from_workload(cls, w, dtype: str = "f64", stream: int = 0):
        s = cls(w.nx, w.ny, w.dx, w.dy, w.dt, dtype, stream)
        wp, nu = w.media()
        s.set_media(np.ascontiguousarray(wp), np.ascontiguousarray(nu))
        E0 = w.initial_E()
        if E0 is not None:
            s.set_fields(Ez=np.ascontiguousarray(E0, s.np_dtype))
        s.set_boundary(w.boundary)
        s.set_source(w.src_kind, w.src_params, *w.src_ij)
        s.set_probes(w.probes)
        return s

    def set_media(self, wp, nu): rketd2d_set_media(self.h, wp, nu)
    def set_boundary(self, kind): rketd2d_set_boundary(self.h, kind)
    def set_boundary_pml(self, npml=5, grading=3.0, R0=1e-6): rketd2d_set_boundary_pml(self.h, npml, grading, R0)
    def set_source(self, kind, params, i, j): rketd2d_set_source(self.h, kind, params, i, j)

    def set_probes(self, ij):
        rketd2d_set_probes(self.h, ij)
        self.nprobes = len(ij)

    def set_fields(self, Ez=None, Hx=None, Hy=None, Jz=None): rketd2d_set_fields(self.h, Ez, Hx, Hy, Jz)
    def reset(self): rketd2d_reset(self.h)
    def discard_records(self): rketd2d_discard_records(self.h)
    def set_plan(self, kernel=KERNEL_AUTO, depth=0): rketd2d_set_plan(self.h, kernel, depth)
    def run(self, nsteps): rketd2d_run(self.h, nsteps)
    def counter(self, which): return rketd2d_get_counter(self.h, which)

    def read_probes(self, out=None):
        n = rketd2d_read_probes(self.h)
        if out is None:
            out = np.empty((self.nprobes, n), self.np_dtype)
        nbytes = out.nbytes if isinstance(out, np.ndarray) else out.numel() * out.element_size()
        rketd2d_read_probes(self.h, out, nbytes)
        return out

    def get_fields(self):
        Ez, Hx, Hy, Jz = (np.empty((self.ny, self.nx), self.np_dtype) for _ in range(4))
        rketd2d_get_fields(self.h, Ez, Hx, Hy, Jz)
        return Ez, Hx, Hy, Jz

    def get_kernel_coefficients(self):
        out = np.empty((4, self.ny, self.nx), np.float64)
        g = np.empty(4, np.float64)
        rketd2d_get_kernel_coefficients(self.h, out, g)
        d = {k: out[i] for i, k in enumerate(("P", "ce", "ka", "Q"))}
        d["chx"], d["chy"], d["mx"], d["my"] = (float(v) for v in g)
        return d

    def close(self):
        if self.h is not None:
            rketd2d_destroy(self.h)
            self.h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


# ---- 2-D TEz (include/rketd2d.h, second half): the C ABI one to one, then the convenience class ----------------------
def _check_te(h, rc: int):
    if rc != OK:
        raise RketdError(rc, (_lib.rketd2d_te_last_error(h) or b"").decode())


def rketd2d_te_create(nx: int, ny: int, dx: float, dy: float, dt: float, dtype: int = F64, cuda_stream: int = 0):
    h = _vp()
    _check_te(None, _lib.rketd2d_te_create(ctypes.byref(h), nx, ny, dx, dy, dt, dtype, cuda_stream or None))
    return h


def rketd2d_te_set_media(h, wp, nu):
    _check_te(h, _lib.rketd2d_te_set_media(h, _ptr(wp), _ptr(nu)))


def rketd2d_te_set_boundary(h, kind: int):
    _check_te(h, _lib.rketd2d_te_set_boundary(h, kind))


def rketd2d_te_set_source(h, kind: int, params: Sequence[float], i: int, j: int, component: int = EY):
    prm = np.ascontiguousarray(params, np.float64)
    _check_te(h, _lib.rketd2d_te_set_source(h, kind, _ptr(prm) if prm.size else None, prm.size, i, j, component))


def rketd2d_te_set_probes(h, ijc):
    c = np.ascontiguousarray(ijc, np.int64).reshape(-1, 3)
    _check_te(h, _lib.rketd2d_te_set_probes(h, _ptr(c) if c.size else None, c.shape[0]))


def rketd2d_te_set_fields(h, Ex=None, Ey=None, Hz=None, Jx=None, Jy=None):
    _check_te(h, _lib.rketd2d_te_set_fields(h, _ptr(Ex), _ptr(Ey), _ptr(Hz), _ptr(Jx), _ptr(Jy)))


def rketd2d_te_get_fields(h, Ex=None, Ey=None, Hz=None, Jx=None, Jy=None):
    _check_te(h, _lib.rketd2d_te_get_fields(h, _ptr(Ex), _ptr(Ey), _ptr(Hz), _ptr(Jx), _ptr(Jy)))


def rketd2d_te_run(h, nsteps: int):
    _check_te(h, _lib.rketd2d_te_run(h, nsteps))


def rketd2d_te_read_probes(h, out=None, out_bytes: int = 0) -> int:
    n = _i64()
    _check_te(h, _lib.rketd2d_te_read_probes(h, _ptr(out), out_bytes, ctypes.byref(n)))
    return n.value


def rketd2d_te_get_counter(h, which: int) -> int:
    return _lib.rketd2d_te_get_counter(h, which)


def rketd2d_te_destroy(h):
    _lib.rketd2d_te_destroy(h)


def rketd2d_te_last_error(h=None) -> str:
    return (_lib.rketd2d_te_last_error(h) or b"").decode()


class Sim2DTE:
    """Owns one rketd2d_te_sim handle (marshalling only)."""

    def __init__(self, nx: int, ny: int, dx: float, dy: float, dt: float, dtype: str = "f64", stream: int = 0):
        self.nx, self.ny, self.dtype = nx, ny, dtype
        self.np_dtype = np.float64 if dtype == "f64" else np.float32
        self.nprobes = 0
        self.h = rketd2d_te_create(nx, ny, dx, dy, dt, F64 if dtype == "f64" else F32, stream)

    @classmethod
    def from_workload(cls, w, dtype: str = "f64", stream: int = 0):
        """a workloads.Workload2D run in the TEz polarisation: initial E on Ey, source on w.src_comp, probes on w.probe_comp"""
        s = cls(w.nx, w.ny, w.dx, w.dy, w.dt, dtype, stream)
        wp, nu = w.media()
        s.set_media(np.ascontiguousarray(wp), np.ascontiguousarray(nu))
        E0 = w.initial_E()
        if E0 is not None:
            s.set_fields(Ey=np.ascontiguousarray(E0, s.np_dtype))
        s.set_boundary(w.boundary)
        s.set_source(w.src_kind, w.src_params, w.src_ij[0], w.src_ij[1], w.src_comp)
        s.set_probes([(int(i), int(j), int(w.probe_comp)) for i, j in w.probes])
        return s

    def set_media(self, wp, nu): rketd2d_te_set_media(self.h, wp, nu)
    def set_boundary(self, kind): rketd2d_te_set_boundary(self.h, kind)
    def set_source(self, kind, params, i, j, component=EY): rketd2d_te_set_source(self.h, kind, params, i, j, component)

    def set_probes(self, ijc):
        rketd2d_te_set_probes(self.h, ijc)
        self.nprobes = len(ijc)

    def set_fields(self, Ex=None, Ey=None, Hz=None, Jx=None, Jy=None): rketd2d_te_set_fields(self.h, Ex, Ey, Hz, Jx, Jy)
    def run(self, nsteps): rketd2d_te_run(self.h, nsteps)
    def counter(self, which): return rketd2d_te_get_counter(self.h, which)

    def read_probes(self, out=None):
        n = rketd2d_te_read_probes(self.h)
        if out is None:
            out = np.empty((self.nprobes, n), self.np_dtype)
        nbytes = out.nbytes if isinstance(out, np.ndarray) else out.numel() * out.element_size()
        rketd2d_te_read_probes(self.h, out, nbytes)
        return out

    def get_fields(self):
        f = [np.empty((self.ny, self.nx), self.np_dtype) for _ in range(5)]
        rketd2d_te_get_fields(self.h, *f)
        return tuple(f)

    def close(self):
        if self.h is not None:
            rketd2d_te_destroy(self.h)
            self.h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass
