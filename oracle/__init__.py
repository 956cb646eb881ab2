"""CPU oracle for the RKETD-FDTD hot path — TEST INFRASTRUCTURE, NOT PRODUCT CODE.

ctypes front-end of ``oracle/rketd_oracle.cpp`` (plain serial C++17, fp64; see
the header of that file for what it states and which pins hold it).  Only
``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s ``cpu_baseline`` /
``--impl reference`` legs may import this package.  It imports nothing from
``paper_1709_00821_b200`` (the CUDA path) and that package never imports this.

Two builds of the one source: ``liboracle_rketd.so`` (serial) and
``liboracle_rketd_omp.so`` (``-fopenmp``); ``run(..., omp=True)`` selects the
latter.  Both are compiled with ``-O2 -ffp-contract=off`` so that the
arithmetic is the plain expression of the source (no fused multiply-add).
"""
from __future__ import annotations

import ctypes
import os
import subprocess
from typing import Optional, Sequence

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "rketd_oracle.cpp")
_LIBS = {False: os.path.join(_HERE, "liboracle_rketd.so"), True: os.path.join(_HERE, "liboracle_rketd_omp.so")}
_loaded = {}

BOUNDARY_MUR = 0
BOUNDARY_PEC = 1
BOUNDARY_PML = 2     # Berenger layer + PEC (reading in DESIGN.md §12): pml = (npml, m, R0)
SRC_NONE = -1
SRC_GAUSS_DERIV = 0
SRC_TABLE = 1
SCHEME_ETD2 = 0      # eq. (11) PAPER.md:68 — the paper's method
SCHEME_ETD1 = 1      # eq. (9) PAPER.md:59 — first-order ETD


_SAN_LIB = os.path.join(_HERE, "liboracle_rketd_asan.so")


def build_sanitized(force: bool = False) -> str:
    """A third build of the same source under AddressSanitizer + UndefinedBehaviorSanitizer, same
    arithmetic flags.  A process that sets RKETD_ORACLE_SANITIZED=1 (and preloads libasan) gets this build from
    every call below; tests/test_oracle_sanitized.py runs the pin suites that way."""
    if force or not os.path.exists(_SAN_LIB) or os.path.getmtime(_SAN_LIB) < os.path.getmtime(_SRC):
        cmd = ["g++", "-fopenmp", "-std=c++17", "-O1", "-g", "-ffp-contract=off", "-fsanitize=address,undefined",
               "-fno-sanitize-recover=all", "-fno-omit-frame-pointer", "-fPIC", "-shared", _SRC, "-o", _SAN_LIB + ".tmp"]
        subprocess.run(cmd, check=True)
        os.replace(_SAN_LIB + ".tmp", _SAN_LIB)
    return _SAN_LIB


def build(force: bool = False) -> None:
    """Compile both builds of the oracle with g++ (a few seconds)."""
    for omp, out in _LIBS.items():
        if not force and os.path.exists(out) and os.path.getmtime(out) >= os.path.getmtime(_SRC):
            continue
        cmd = ["g++", "-std=c++17", "-O2", "-ffp-contract=off", "-fPIC", "-shared", _SRC, "-o", out + ".tmp"]
        if omp:
            cmd.insert(1, "-fopenmp")
        subprocess.run(cmd, check=True)
        os.replace(out + ".tmp", out)


_D = ctypes.POINTER(ctypes.c_double)
_I64 = ctypes.POINTER(ctypes.c_int64)


def _lib(omp: bool = False) -> ctypes.CDLL:
    if omp not in _loaded:
        build()
        lib = ctypes.CDLL(build_sanitized() if os.environ.get("RKETD_ORACLE_SANITIZED") == "1" else _LIBS[omp])
        lib.oracle_constants.argtypes = [_D, _D, _D]
        lib.oracle_constants.restype = None
        lib.oracle_phi.argtypes = [ctypes.c_double, _D, _D]
        lib.oracle_phi.restype = None
        lib.oracle_coefficients.argtypes = [ctypes.c_int64, _D, _D, ctypes.c_double, ctypes.c_double] + [_D] * 8
        lib.oracle_coefficients.restype = ctypes.c_int
        lib.oracle_coefficients_scheme.argtypes = lib.oracle_coefficients.argtypes + [ctypes.c_int]
        lib.oracle_coefficients_scheme.restype = ctypes.c_int
        lib.oracle_source.argtypes = [ctypes.c_int, _D, ctypes.c_int64, ctypes.c_int64, ctypes.c_double]
        lib.oracle_source.restype = ctypes.c_double
        lib.oracle_run.argtypes = [ctypes.c_int64, ctypes.c_int64, ctypes.c_double, ctypes.c_double,
                                   _D, _D, _D, _D, _D,
                                   ctypes.c_int, _D, ctypes.c_int64, ctypes.c_int64,
                                   _I64, ctypes.c_int, ctypes.c_int64, ctypes.c_int64,
                                   _D, _D, _D, ctypes.c_int, _D, _D, ctypes.c_int]
        lib.oracle_run.restype = ctypes.c_int
        lib.oracle_run_scheme.argtypes = lib.oracle_run.argtypes + [ctypes.c_int]
        lib.oracle_run_scheme.restype = ctypes.c_int
        lib.oracle_run_bc.argtypes = lib.oracle_run_scheme.argtypes + [ctypes.c_int, ctypes.c_double, ctypes.c_double]
        lib.oracle_run_bc.restype = ctypes.c_int
        lib.oracle2d_coefficients.argtypes = [ctypes.c_int64, _D, _D, ctypes.c_double, ctypes.c_double, ctypes.c_double,
                                              ctypes.c_int] + [_D] * 8
        lib.oracle2d_coefficients.restype = ctypes.c_int
        lib.oracle2d_run.argtypes = [ctypes.c_int64, ctypes.c_int64, ctypes.c_double, ctypes.c_double, ctypes.c_double,
                                     _D, _D, _D, _D, _D, _D,
                                     ctypes.c_int, _D, ctypes.c_int64, ctypes.c_int64, ctypes.c_int64,
                                     _I64, ctypes.c_int, ctypes.c_int64, ctypes.c_int64, _D, _D, ctypes.c_int, ctypes.c_int]
        lib.oracle2d_run.restype = ctypes.c_int
        lib.oracle2d_te_run.argtypes = [ctypes.c_int64, ctypes.c_int64, ctypes.c_double, ctypes.c_double, ctypes.c_double,
                                        _D, _D, _D, _D, _D, _D, _D,
                                        ctypes.c_int, _D, ctypes.c_int64, ctypes.c_int64, ctypes.c_int64, ctypes.c_int,
                                        _I64, ctypes.c_int, ctypes.c_int64, ctypes.c_int64, _D, ctypes.c_int, ctypes.c_int]
        lib.oracle2d_te_run.restype = ctypes.c_int
        lib.oracle2d_run_pml.argtypes = [ctypes.c_int64, ctypes.c_int64, ctypes.c_double, ctypes.c_double, ctypes.c_double,
                                         _D, _D, _D, _D, _D, _D, _D,
                                         ctypes.c_int, _D, ctypes.c_int64, ctypes.c_int64, ctypes.c_int64,
                                         _I64, ctypes.c_int, ctypes.c_int64, ctypes.c_int64, _D,
                                         ctypes.c_int, ctypes.c_double, ctypes.c_double]
        lib.oracle2d_run_pml.restype = ctypes.c_int
        _loaded[omp] = lib
    return _loaded[omp]


def _p(a: Optional[np.ndarray]):
    return None if a is None else a.ctypes.data_as(_D)


def constants():
    """(c0, mu0, eps0) as hard-coded in the oracle."""
    c0, mu0, eps0 = ctypes.c_double(), ctypes.c_double(), ctypes.c_double()
    _lib().oracle_constants(ctypes.byref(c0), ctypes.byref(mu0), ctypes.byref(eps0))
    return c0.value, mu0.value, eps0.value


def phi(x: float):
    p1, p2 = ctypes.c_double(), ctypes.c_double()
    _lib().oracle_phi(float(x), ctypes.byref(p1), ctypes.byref(p2))
    return p1.value, p2.value


def coefficients(wp: np.ndarray, nu: np.ndarray, dz: float, dt: float, scheme: int = SCHEME_ETD2):
    """S0: returns dict(ca, cj, ch, ka, kb, kc [same shape as wp], chh, m)."""
    wp = np.ascontiguousarray(wp, np.float64)
    nu = np.ascontiguousarray(nu, np.float64)
    out = {k: np.empty_like(wp) for k in ("ca", "cj", "ch", "ka", "kb", "kc")}
    chh, m = ctypes.c_double(), ctypes.c_double()
    rc = _lib().oracle_coefficients_scheme(wp.size, _p(wp), _p(nu), dz, dt, *[_p(out[k]) for k in
                                           ("ca", "cj", "ch", "ka", "kb", "kc")], ctypes.byref(chh), ctypes.byref(m),
                                           scheme)
    if rc:
        raise ValueError("oracle_coefficients: invalid argument")
    out["chh"], out["m"] = chh.value, m.value
    return out


def source(kind: int, params: Sequence[float], step_index: int, dt: float) -> float:
    prm = np.ascontiguousarray(params, np.float64)
    return _lib().oracle_source(kind, _p(prm), prm.size, step_index, dt)


class State:
    """E, H, J [nbatch][ncells] fp64 plus the global step counter; advanced in place by run()."""

    def __init__(self, ncells: int, nbatch: int = 1, E0=None, H0=None, J0=None):
        shp = (nbatch, ncells)
        self.E = np.zeros(shp) if E0 is None else np.array(E0, np.float64).reshape(shp).copy()
        self.H = np.zeros(shp) if H0 is None else np.array(H0, np.float64).reshape(shp).copy()
        self.J = np.zeros(shp) if J0 is None else np.array(J0, np.float64).reshape(shp).copy()
        self.step = 0


def run(state: State, wp, nu, dz: float, dt: float, nsteps: int, *, src_kind: int = SRC_NONE,
        src_params: Sequence[float] = (), src_cell: int = 0, probes: Sequence[int] = (),
        freqs=None, dft=None, record_J: bool = False, boundary: int = BOUNDARY_MUR, omp: bool = False,
        scheme: int = SCHEME_ETD2, pml: Sequence[float] = (0, 0.0, 1.0)):
    """Advance ``state`` by nsteps.  Returns (rec, recJ) with rec[nbatch][nprobes][nsteps]
    (recJ None unless record_J).  ``dft`` = (re, im) accumulator arrays [nbatch][nprobes][nfreq],
    updated in place when ``freqs`` is given."""
    nbatch, ncells = state.E.shape
    wp = np.ascontiguousarray(wp, np.float64).reshape(nbatch, ncells)
    nu = np.ascontiguousarray(nu, np.float64).reshape(nbatch, ncells)
    prm = np.ascontiguousarray(src_params, np.float64)
    prb = np.ascontiguousarray(probes, np.int64)
    rec = np.zeros((nbatch, prb.size, nsteps))
    recJ = np.zeros((nbatch, prb.size, nsteps)) if record_J else None
    fr = None if freqs is None else np.ascontiguousarray(freqs, np.float64)
    re = im = None
    if fr is not None:
        re, im = dft
        assert re.shape == (nbatch, prb.size, fr.size) and re.flags.c_contiguous and im.flags.c_contiguous
    rc = _lib(omp).oracle_run_bc(ncells, nbatch, dz, dt, _p(wp), _p(nu), _p(state.E), _p(state.H), _p(state.J),
                              src_kind, _p(prm) if prm.size else None, prm.size, src_cell,
                              prb.ctypes.data_as(_I64) if prb.size else None, prb.size, state.step, nsteps,
                              _p(rec), _p(recJ), _p(fr), 0 if fr is None else fr.size, _p(re), _p(im), boundary, scheme,
                                 int(pml[0]), float(pml[1]), float(pml[2]))
    if rc:
        raise ValueError("oracle_run: invalid argument")
    state.step += nsteps
    return rec, recJ


def run_workload(w, nsteps: Optional[int] = None, b0: int = 0, b1: Optional[int] = None, omp: bool = False,
                 cells: Optional[tuple] = None, scheme: int = SCHEME_ETD2, boundary: int = BOUNDARY_MUR,
                 pml: Sequence[float] = (0, 0.0, 1.0)):
    """Run a ``workloads.Workload`` (duck-typed: only its data attributes are used) on grids
    b0..b1-1.  ``cells=(lo, hi)`` runs the window lo..hi-1 only, with Mur at the window ends
    (pin P7: exact for probes at distance > nsteps from both window ends).
    Returns dict(rec, dft_mag, dft (complex accumulators), state)."""
    b1 = w.nbatch if b1 is None else b1
    lo, hi = (0, w.ncells) if cells is None else cells
    nsteps = w.nsteps if nsteps is None else nsteps
    wp, nu = w.media(lo, hi, b0, b1)
    E0 = w.initial_E(lo, hi, b0, b1)
    st = State(hi - lo, b1 - b0, E0)
    probes = [int(p) - lo for p in w.probes if lo <= p < hi]
    in_src = lo <= w.src_cell < hi
    dft = None
    if w.dft_freqs is not None:
        dft = (np.zeros((b1 - b0, len(probes), len(w.dft_freqs))), np.zeros((b1 - b0, len(probes), len(w.dft_freqs))))
    rec, _ = run(st, wp, nu, w.dz, w.dt, nsteps, src_kind=w.src_kind if in_src else SRC_NONE,
                 src_params=w.src_params, src_cell=w.src_cell - lo if in_src else 0, probes=probes,
                 freqs=w.dft_freqs, dft=dft, omp=omp, scheme=scheme, boundary=boundary, pml=pml)
    mag = None if dft is None else np.hypot(dft[0], dft[1])
    cplx = None if dft is None else dft[0] + 1j * dft[1]
    return {"rec": rec, "dft_mag": mag, "dft": cplx, "state": st, "probe_cells": [p + lo for p in probes]}


# ----------------------------------------------------------------------------------------------------------------
# 2-D TMz: see the second half of rketd_oracle.cpp
# ----------------------------------------------------------------------------------------------------------------
class State2D:
    """Ez, Hx, Hy, Jz [ny][nx] fp64 plus the global step counter; advanced in place by run2d()."""

    def __init__(self, nx: int, ny: int, Ez0=None, Hx0=None, Hy0=None, Jz0=None):
        shp = (ny, nx)
        mk = lambda a: np.zeros(shp) if a is None else np.array(a, np.float64).reshape(shp).copy()
        self.Ez, self.Hx, self.Hy, self.Jz = mk(Ez0), mk(Hx0), mk(Hy0), mk(Jz0)
        self.step = 0


def coefficients2d(wp, nu, dx: float, dy: float, dt: float, scheme: int = SCHEME_ETD2):
    """dict(ca, cj, cex, cey, ka, kb, kc [same shape as wp], chx, chy, mx, my)."""
    wp = np.ascontiguousarray(wp, np.float64)
    nu = np.ascontiguousarray(nu, np.float64)
    names = ("ca", "cj", "cex", "cey", "ka", "kb", "kc")
    out = {k: np.empty_like(wp) for k in names}
    g = np.zeros(4)
    if _lib().oracle2d_coefficients(wp.size, _p(wp), _p(nu), dx, dy, dt, scheme, *[_p(out[k]) for k in names], _p(g)):
        raise ValueError("oracle2d_coefficients: invalid argument")
    out["chx"], out["chy"], out["mx"], out["my"] = (float(v) for v in g)
    return out


def run2d(state: State2D, wp, nu, dx: float, dy: float, dt: float, nsteps: int, *, src_kind: int = SRC_NONE,
          src_params: Sequence[float] = (), src_ij=(0, 0), probes=(), record_J: bool = False,
          boundary: int = BOUNDARY_MUR, omp: bool = False, scheme: int = SCHEME_ETD2):
    """Advance ``state`` by nsteps.  probes = sequence of (i, j).  Returns (rec, recJ), each [nprobes][nsteps]."""
    ny, nx = state.Ez.shape
    wp = np.ascontiguousarray(wp, np.float64).reshape(ny, nx)
    nu = np.ascontiguousarray(nu, np.float64).reshape(ny, nx)
    prm = np.ascontiguousarray(src_params, np.float64)
    prb = np.ascontiguousarray(probes, np.int64).reshape(-1, 2)
    rec = np.zeros((prb.shape[0], nsteps))
    recJ = np.zeros((prb.shape[0], nsteps)) if record_J else None
    rc = _lib(omp).oracle2d_run(nx, ny, dx, dy, dt, _p(wp), _p(nu), _p(state.Ez), _p(state.Hx), _p(state.Hy),
                                _p(state.Jz), src_kind, _p(prm) if prm.size else None, prm.size, int(src_ij[0]),
                                int(src_ij[1]), prb.ctypes.data_as(_I64) if prb.size else None, prb.shape[0],
                                state.step, nsteps, _p(rec), _p(recJ), boundary, scheme)
    if rc:
        raise ValueError("oracle2d_run: invalid argument")
    state.step += nsteps
    return rec, recJ


def run2d_pml(state: State2D, wp, nu, dx: float, dy: float, dt: float, nsteps: int, *, pml=(5, 3.0, 1e-6),
              src_kind: int = SRC_NONE, src_params: Sequence[float] = (), src_ij=(0, 0), probes=(), omp: bool = False):
    """2-D TMz with Berenger's split-field layer on the four sides (oracle2d_run_pml).  The split parts Ezx, Ezy are kept
    on the state (state.Esplit, [2][ny][nx], created as zeros on first use: a field given inside a layer starts as Ezx).
    Returns rec [nprobes][nsteps]."""
    ny, nx = state.Ez.shape
    if not hasattr(state, "Esplit"):
        state.Esplit = np.zeros((2, ny, nx))
        state.Esplit[0] = state.Ez
    wp = np.ascontiguousarray(wp, np.float64).reshape(ny, nx)
    nu = np.ascontiguousarray(nu, np.float64).reshape(ny, nx)
    prm = np.ascontiguousarray(src_params, np.float64)
    prb = np.ascontiguousarray(probes, np.int64).reshape(-1, 2)
    rec = np.zeros((prb.shape[0], nsteps))
    rc = _lib(omp).oracle2d_run_pml(nx, ny, dx, dy, dt, _p(wp), _p(nu), _p(state.Ez), _p(state.Hx), _p(state.Hy),
                                    _p(state.Jz), _p(state.Esplit), src_kind, _p(prm) if prm.size else None, prm.size,
                                    int(src_ij[0]), int(src_ij[1]), prb.ctypes.data_as(_I64) if prb.size else None,
                                    prb.shape[0], state.step, nsteps, _p(rec), int(pml[0]), float(pml[1]), float(pml[2]))
    if rc:
        raise ValueError("oracle2d_run_pml: invalid argument")
    state.step += nsteps
    return rec


def run_workload2d(w, nsteps: Optional[int] = None, window=None, omp: bool = False, boundary: Optional[int] = None):
    """Run a ``workloads.Workload2D`` (duck-typed).  window = (i0, i1, j0, j1) runs nodes i0..i1-1 x j0..j1-1 only,
    with the edge rule at the window edges (pin Q7: exact for probes farther than nsteps from every window edge).
    Returns dict(rec [nprobes][nsteps], probe_ij, state)."""
    i0, i1, j0, j1 = (0, w.nx, 0, w.ny) if window is None else window
    nsteps = w.nsteps if nsteps is None else nsteps
    wp, nu = w.media(i0, i1, j0, j1)
    st = State2D(i1 - i0, j1 - j0, w.initial_E(i0, i1, j0, j1))
    probes = [(int(i) - i0, int(j) - j0) for i, j in w.probes if i0 <= i < i1 and j0 <= j < j1]
    in_src = i0 <= w.src_ij[0] < i1 and j0 <= w.src_ij[1] < j1
    rec, _ = run2d(st, wp, nu, w.dx, w.dy, w.dt, nsteps, src_kind=w.src_kind if in_src else SRC_NONE,
                   src_params=w.src_params, src_ij=(w.src_ij[0] - i0, w.src_ij[1] - j0) if in_src else (0, 0),
                   probes=probes, omp=omp, boundary=w.boundary if boundary is None else boundary)
    return {"rec": rec, "probe_ij": [(i + i0, j + j0) for i, j in probes], "state": st}


# ----------------------------------------------------------------------------------------------------------------
# 2-D TEz (second polarisation): see the last section of rketd_oracle.cpp
# ----------------------------------------------------------------------------------------------------------------
EX, EY = 0, 1        # component ids of sources and probes


class State2DTE:
    """Ex, Ey, Hz, Jx, Jy [ny][nx] fp64 plus the global step counter; advanced in place by run2d_te()."""

    def __init__(self, nx: int, ny: int, Ex0=None, Ey0=None, Hz0=None, Jx0=None, Jy0=None):
        shp = (ny, nx)
        mk = lambda a: np.zeros(shp) if a is None else np.array(a, np.float64).reshape(shp).copy()
        self.Ex, self.Ey, self.Hz, self.Jx, self.Jy = mk(Ex0), mk(Ey0), mk(Hz0), mk(Jx0), mk(Jy0)
        self.step = 0


def run2d_te(state: State2DTE, wp, nu, dx: float, dy: float, dt: float, nsteps: int, *, src_kind: int = SRC_NONE,
             src_params: Sequence[float] = (), src_ij=(0, 0), src_comp: int = EY, probes=(),
             boundary: int = BOUNDARY_MUR, omp: bool = False, scheme: int = SCHEME_ETD2):
    """Advance ``state`` by nsteps.  probes = sequence of (i, j, component).  Returns rec [nprobes][nsteps]."""
    ny, nx = state.Ex.shape
    wp = np.ascontiguousarray(wp, np.float64).reshape(ny, nx)
    nu = np.ascontiguousarray(nu, np.float64).reshape(ny, nx)
    prm = np.ascontiguousarray(src_params, np.float64)
    prb = np.ascontiguousarray(probes, np.int64).reshape(-1, 3)
    rec = np.zeros((prb.shape[0], nsteps))
    rc = _lib(omp).oracle2d_te_run(nx, ny, dx, dy, dt, _p(wp), _p(nu), _p(state.Ex), _p(state.Ey), _p(state.Hz),
                                   _p(state.Jx), _p(state.Jy), src_kind, _p(prm) if prm.size else None, prm.size,
                                   int(src_ij[0]), int(src_ij[1]), int(src_comp),
                                   prb.ctypes.data_as(_I64) if prb.size else None, prb.shape[0], state.step, nsteps,
                                   _p(rec), boundary, scheme)
    if rc:
        raise ValueError("oracle2d_te_run: invalid argument")
    state.step += nsteps
    return rec


def run_workload2d_te(w, nsteps: Optional[int] = None, window=None, omp: bool = False, boundary: Optional[int] = None):
    """Run a ``workloads.Workload2D`` in the TEz polarisation (source on w.src_comp, probes (i, j) on w.probe_comp).
    window = (i0, i1, j0, j1) as in run_workload2d (pin R6).  Returns dict(rec, probe_ij, state)."""
    i0, i1, j0, j1 = (0, w.nx, 0, w.ny) if window is None else window
    nsteps = w.nsteps if nsteps is None else nsteps
    wp, nu = w.media(i0, i1, j0, j1)
    E0 = w.initial_E(i0, i1, j0, j1)
    st = State2DTE(i1 - i0, j1 - j0, Ey0=E0)
    probes = [(int(i) - i0, int(j) - j0, int(w.probe_comp)) for i, j in w.probes if i0 <= i < i1 and j0 <= j < j1]
    in_src = i0 <= w.src_ij[0] < i1 and j0 <= w.src_ij[1] < j1
    rec = run2d_te(st, wp, nu, w.dx, w.dy, w.dt, nsteps, src_kind=w.src_kind if in_src else SRC_NONE,
                   src_params=w.src_params, src_ij=(w.src_ij[0] - i0, w.src_ij[1] - j0) if in_src else (0, 0),
                   src_comp=w.src_comp, probes=probes, omp=omp, boundary=w.boundary if boundary is None else boundary)
    return {"rec": rec, "probe_ij": [(i + i0, j + j0) for i, j, _ in probes], "state": st}
