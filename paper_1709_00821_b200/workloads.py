"""Seeded synthetic inputs for the five BASELINE.json configs.

This module holds NONE of the method's arithmetic: it only draws / lays out the
inputs (plasma frequency wp[b][k], collision frequency nu[b][k], initial E,
source parameters, probe cells, DFT frequencies).  The very same arrays are
handed to the CPU oracle (``oracle/``) and to the CUDA library (``librketd``);
neither of those two contains a random number generator.

Shapes, sizes and value distributions follow the paper's workload
(§IV.B: a Drude slab in vacuum, dz = 75 um, dt ~ dz/(2c),
Gaussian-derivative pulse) with the sizes BASELINE.json ``configs`` gives.
Every generator takes ``scale`` knobs so that tests can run a geometrically
similar, smaller instance; the default arguments are the literal configs.

Large configs (2 and 4) never materialise more than the requested window:
``media(lo, hi)`` / ``initial_E(lo, hi)`` return cells ``lo..hi-1`` only, so
the oracle can be run on windows (pin P7) without a multi-GB host array.

Random streams: ``numpy.random.Generator(PCG64(SeedSequence([SEED0+cfg, tag, block])))``;
per-cell noise is drawn in blocks of 2**20 cells so that any window can be
regenerated bit-for-bit.
"""
from __future__ import annotations

import dataclasses
import math
from typing import Callable, Optional, Sequence, Tuple

import numpy as np

C0 = 299_792_458.0          # m/s, exact (SI); used only to fix dt = dz/(2c)
DZ = 75e-6
DT = DZ / (2.0 * C0)         # BASELINE configs: dt = dz/(2c)
SEED0 = 170900821
_NOISE_BLOCK = 1 << 20

SRC_GAUSS_DERIV = 0          # kind ids mirror include/rketd.h
SRC_TABLE = 1


def _rng(cfg: int, tag: int, block: int = 0) -> np.random.Generator:
    return np.random.Generator(np.random.PCG64(np.random.SeedSequence([SEED0 + cfg, tag, block])))


def _block_noise(cfg: int, tag: int, lo: int, hi: int, amp: float) -> np.ndarray:
    """amp * U(-1,1) per cell, reproducible for any window [lo, hi)."""
    out = np.empty(hi - lo, dtype=np.float64)
    b0, b1 = lo // _NOISE_BLOCK, (hi - 1) // _NOISE_BLOCK if hi > lo else lo // _NOISE_BLOCK
    for b in range(b0, b1 + 1):
        blk = _rng(cfg, tag, b).uniform(-1.0, 1.0, _NOISE_BLOCK)
        s, e = max(lo, b * _NOISE_BLOCK), min(hi, (b + 1) * _NOISE_BLOCK)
        if e > s:
            out[s - lo:e - lo] = amp * blk[s - b * _NOISE_BLOCK:e - b * _NOISE_BLOCK]
    return out


@dataclasses.dataclass
class Workload:
    """One problem instance: everything rketd_create/set_*/run need, as plain data."""
    name: str
    cfg: int
    ncells: int
    nbatch: int
    nsteps: int
    dz: float
    dt: float
    src_kind: int
    src_params: Tuple[float, ...]       # GAUSS_DERIV: (tau, t0, amplitude)
    src_cell: int
    probes: np.ndarray                  # int64 cells, same in every grid
    dft_freqs: Optional[np.ndarray]     # Hz, or None (time series mode)
    # media(lo, hi, b0, b1) -> (wp, nu) float64 arrays of shape [b1-b0, hi-lo]
    media: Callable[..., Tuple[np.ndarray, np.ndarray]]
    # initial_E(lo, hi, b0, b1) -> float64 [b1-b0, hi-lo] or None (zeros)
    initial_E: Callable[..., Optional[np.ndarray]]
    dtypes: Tuple[str, ...] = ("f64",)
    notes: str = ""

    @property
    def cell_updates(self) -> int:
        return self.ncells * self.nbatch * self.nsteps

    def media_full(self):
        return self.media(0, self.ncells, 0, self.nbatch)

    def initial_E_full(self):
        return self.initial_E(0, self.ncells, 0, self.nbatch)


_SRC = (20e-12, 80e-12, 1.0)    # tau ("width 20 ps"), t0 ("delay 80 ps"), unit peak


# ----------------------------------------------------------------------------
# config 1: one 2000-cell grid, 120-cell slab, tiny noise on the initial E
# ----------------------------------------------------------------------------
def config1(ncells: int = 2000, nsteps: int = 6000) -> Workload:
    s = ncells / 2000.0
    slab_lo, slab_hi = int(round(900 * s)), int(round(1020 * s))      # cells 900..1019 inclusive
    wp0, nu0 = 2.0 * math.pi * 28.7e9, 2.0e10

    def media(lo=0, hi=ncells, b0=0, b1=1):
        k = np.arange(lo, hi)
        inside = (k >= slab_lo) & (k < slab_hi)
        wp = np.where(inside, wp0, 0.0)[None, :].repeat(b1 - b0, 0)
        nu = np.where(inside, nu0, 0.0)[None, :].repeat(b1 - b0, 0)
        return np.ascontiguousarray(wp), np.ascontiguousarray(nu)

    def initial_E(lo=0, hi=ncells, b0=0, b1=1):
        return _block_noise(1, 1, lo, hi, 1e-12)[None, :].copy()

    return Workload("config1_slab2000", 1, ncells, 1, nsteps, DZ, DT, SRC_GAUSS_DERIV, _SRC,
                    int(round(200 * s)), np.array([int(round(600 * s)), int(round(1400 * s))], np.int64),
                    None, media, initial_E,
                    notes="paper Exp. A (PAPER.md:123-128) at 1/10 slab thickness; Mur instead of PML")


# ----------------------------------------------------------------------------
# config 2: 1e7 cells, periodic slabs (120 of every 1000 cells), random wp, nu per slab
# ----------------------------------------------------------------------------
def config2(ncells: int = 10_000_000, nsteps: int = 2000, noise: bool = True,
            extra_probes: Sequence[int] = (600, 1400)) -> Workload:
    period, width, first = 1000, 120, 440             # slab p on cells 1000p+440 .. 1000p+559
    nslab = (ncells + period - 1) // period
    r = _rng(2, 1)
    wp_s = r.uniform(2 * math.pi * 10e9, 2 * math.pi * 40e9, nslab)   # draw 1
    nu_s = r.uniform(1e9, 5e10, nslab)                                # draw 2

    def media(lo=0, hi=ncells, b0=0, b1=1):
        k = np.arange(lo, hi)
        p, q = k // period, k % period
        inside = (q >= first) & (q < first + width)
        wp = np.where(inside, wp_s[np.minimum(p, nslab - 1)], 0.0)
        nu = np.where(inside, nu_s[np.minimum(p, nslab - 1)], 0.0)
        return wp[None, :].repeat(b1 - b0, 0), nu[None, :].repeat(b1 - b0, 0)

    def initial_E(lo=0, hi=ncells, b0=0, b1=1):
        if not noise:
            return None
        return _block_noise(2, 3, lo, hi, 1e-3)[None, :].copy()

    probes = [((i + 1) * ncells) // 17 for i in range(16)] + [p for p in extra_probes if p < ncells]
    return Workload("config2_periodic_1e7", 2, ncells, 1, nsteps, DZ, DT, SRC_GAUSS_DERIV, _SRC,
                    min(1000, ncells // 2), np.array(sorted(set(probes)), np.int64), None, media, initial_E,
                    notes="seeded 1e-3 noise on E0 so that far probes are not identically zero (SURVEY H8)")


# ----------------------------------------------------------------------------
# config 3: 4096 grids x 4096 cells, one homogeneous slab per grid (R/T sweep)
# ----------------------------------------------------------------------------
def config3(ncells: int = 4096, nbatch: int = 4096, nsteps: int = 20_000) -> Workload:
    s = ncells / 4096.0
    r = _rng(3, 1)
    M = r.integers(40, 401, 4096)                                        # thickness in cells
    wp_g = r.uniform(2 * math.pi * 5e9, 2 * math.pi * 60e9, 4096)
    nu_g = r.uniform(0.0, 1e11, 4096)
    slab0 = int(round(2000 * s))

    def media(lo=0, hi=ncells, b0=0, b1=nbatch):
        k = np.arange(lo, hi)[None, :]
        g = np.arange(b0, b1) % 4096
        m = np.maximum(1, np.round(M[g] * s).astype(np.int64))[:, None]
        inside = (k >= slab0) & (k < slab0 + m)
        wp = np.where(inside, wp_g[g][:, None], 0.0)
        nu = np.where(inside, nu_g[g][:, None], 0.0)
        return np.ascontiguousarray(wp), np.ascontiguousarray(nu)

    def initial_E(lo=0, hi=ncells, b0=0, b1=nbatch):
        return None

    return Workload("config3_batch4096x4096", 3, ncells, nbatch, nsteps, DZ, DT, SRC_GAUSS_DERIV, _SRC,
                    int(round(400 * s)), np.array([int(round(1200 * s)), int(round(3200 * s))], np.int64),
                    None, media, initial_E, notes="R/T parameter sweep; full probe time series")


# ----------------------------------------------------------------------------
# config 4: one long line (2**28 cells), tanh (Epstein) density profile, per-cell coefficients
# ----------------------------------------------------------------------------
def config4(ncells: int = 1 << 28, nsteps: int = 1000, noise: bool = True) -> Workload:
    N = ncells
    wp_peak, nu0 = 2 * math.pi * 50e9, 1e10

    def media(lo=0, hi=ncells, b0=0, b1=1):
        k = np.arange(lo, hi, dtype=np.float64)
        prof = 0.5 * (np.tanh((k - 0.35 * N) / (0.025 * N)) - np.tanh((k - 0.65 * N) / (0.025 * N)))
        wp = wp_peak * np.sqrt(np.maximum(prof, 0.0))
        nu = np.full(hi - lo, nu0)
        return wp[None, :].repeat(b1 - b0, 0), nu[None, :].repeat(b1 - b0, 0)

    def initial_E(lo=0, hi=ncells, b0=0, b1=1):
        if not noise:
            return None
        return _block_noise(4, 1, lo, hi, 1e-3)[None, :].copy()

    probes = [((2 * i + 1) * N) // 32 for i in range(16)] + [N // 2 - 256, N // 2, N // 2 + 256]   # N/2: the source node
    probes += [int(v) for v in _rng(4, 2).integers(0, N, 16)]
    return Workload("config4_line_2p28" if N == 1 << 28 else f"config4_line_{N}", 4, N, 1, nsteps, DZ, DT,
                    SRC_GAUSS_DERIV, _SRC, N // 2, np.array(sorted(set(probes)), np.int64), None,
                    media, initial_E, dtypes=("f64", "f32"),
                    notes="source inside the plasma plateau; tiny wp at both boundary nodes (SURVEY G11)")


# ----------------------------------------------------------------------------
# config 5: 65536 grids x 1024 cells, 8 random layers per grid, |DFT| at 64 frequencies
# ----------------------------------------------------------------------------
def dft_frequencies(nfreq: int = 64) -> np.ndarray:
    """f_m = 1 GHz + m * (59/63) GHz, m = 0..63 (linear, inclusive) — SURVEY G15."""
    return 1e9 + np.arange(nfreq, dtype=np.float64) * (59e9 / (nfreq - 1))


def config5(ncells: int = 1024, nbatch: int = 65_536, nsteps: int = 5000, dft: bool = True) -> Workload:
    s = ncells / 1024.0
    r = _rng(5, 1)
    w = r.integers(5, 51, (65_536, 8))
    wp_l = r.uniform(2 * math.pi * 5e9, 2 * math.pi * 60e9, (65_536, 8))
    nu_l = r.uniform(0.0, 1e11, (65_536, 8))
    start = int(round(320 * s))

    def media(lo=0, hi=ncells, b0=0, b1=nbatch):
        g = np.arange(b0, b1) % 65_536
        edges = start + np.concatenate([np.zeros((len(g), 1), np.int64),
                                        np.cumsum(np.maximum(1, np.round(w[g] * s).astype(np.int64)), 1)], 1)
        k = np.arange(lo, hi)[None, :]
        wp = np.zeros((len(g), hi - lo))
        nu = np.zeros((len(g), hi - lo))
        for l in range(8):
            inside = (k >= edges[:, l:l + 1]) & (k < edges[:, l + 1:l + 2])
            wp = np.where(inside, wp_l[g][:, l:l + 1], wp)
            nu = np.where(inside, nu_l[g][:, l:l + 1], nu)
        return wp, nu

    def initial_E(lo=0, hi=ncells, b0=0, b1=nbatch):
        return None

    return Workload("config5_batch65536x1024", 5, ncells, nbatch, nsteps, DZ, DT, SRC_GAUSS_DERIV, _SRC,
                    int(round(64 * s)), np.array([int(round(192 * s)), int(round(832 * s))], np.int64),
                    dft_frequencies() if dft else None, media, initial_E, dtypes=("f64", "f32"),
                    notes="random multilayer; probes reduced on device to |DFT| at 64 frequencies")


# ----------------------------------------------------------------------------
# The paper's own two workloads
# ----------------------------------------------------------------------------
PAPER_DT = 125e-15           # "a single time step is taken to be 125 fs"; S = c dt/dz = 0.49965
PAPER_TABLE2_CELLS = (1024, 5120, 10240, 20480, 30720, 40960, 51200, 61440)


def _paper_slab(name: str, cfg: int, ncells: int, nsteps: int, src_cell: int, probes) -> Workload:
    """A slab on the middle 1200/4096 of the line, wp = 2 pi 28.7e9 rad/s, nu = 20e9 1/s, vacuum elsewhere,
    Gaussian-derivative pulse with tau = 15 dt, delay 5 tau.  The paper ends the line in 5-cell
    PMLs whose parameters it does not give; here the ends are Mur-1 like everywhere else (DESIGN.md §2 G10)."""
    m = (ncells * 1200) // 4096
    slab_lo = (ncells - m) // 2
    wp0, nu0 = 2.0 * math.pi * 28.7e9, 2.0e10
    tau = 15.0 * PAPER_DT

    def media(lo=0, hi=ncells, b0=0, b1=1):
        k = np.arange(lo, hi)
        inside = (k >= slab_lo) & (k < slab_lo + m)
        wp = np.where(inside, wp0, 0.0)[None, :].repeat(b1 - b0, 0)
        nu = np.where(inside, nu0, 0.0)[None, :].repeat(b1 - b0, 0)
        return np.ascontiguousarray(wp), np.ascontiguousarray(nu)

    def initial_E(lo=0, hi=ncells, b0=0, b1=1):
        return None

    w = Workload(name, cfg, ncells, 1, nsteps, DZ, PAPER_DT, SRC_GAUSS_DERIV, (tau, 5.0 * tau, 1.0), src_cell,
                 np.array(sorted(probes), np.int64), None, media, initial_E,
                 notes="paper's own workload (PAPER.md:123-128); Mur instead of the unspecified PML")
    w.slab = (slab_lo, m)
    return w


def paper_exp_a(nsteps: int = 16384) -> Workload:
    """Experiment A (Figs. 2-3): 4096 cells, slab = middle 1200 cells (9 cm), R and T by FFT.
    The paper gives neither source nor probe positions nor the run length: source 300, reflected probe 800,
    transmitted probe 3300, 16 384 steps (both records have decayed to < 1e-6 of their peak by then)."""
    return _paper_slab("paper_expA_4096", 11, 4096, nsteps, 300, (800, 3300))


def paper_table2(ncells: int, nsteps: int = 1000) -> Workload:
    """One row of Table 2: `ncells` Yee cells x 1000 steps; the same slab geometry scaled to the
    line (the paper does not say what fills the longer lines, nor where it records)."""
    src = max(2, (ncells * 300) // 4096)
    # the pulse travels 500 cells in 1000 steps (S = 1/2): probes 128 and 400 cells behind the source see it
    return _paper_slab(f"paper_table2_{ncells}", 12, ncells, nsteps, src, (src + 128, src + 400))


CONFIGS = {1: config1, 2: config2, 3: config3, 4: config4, 5: config5}


# ----------------------------------------------------------------------------
# 2-D TMz (the paper's stated next step): a plasma column in vacuum
# ----------------------------------------------------------------------------
BC_MUR = 0
BC_PEC = 1


@dataclasses.dataclass
class Workload2D:
    """One 2-D TMz problem instance as plain data (arrays are [ny][nx], x fastest)."""
    name: str
    cfg: int
    nx: int
    ny: int
    nsteps: int
    dx: float
    dy: float
    dt: float
    src_kind: int
    src_params: Tuple[float, ...]
    src_ij: Tuple[int, int]
    probes: np.ndarray                  # int64 [nprobes][2] = (i, j)
    boundary: int
    # media(i0, i1, j0, j1) -> (wp, nu) float64 [j1-j0][i1-i0];  initial_E(i0, i1, j0, j1) -> same shape or None
    media: Callable[..., Tuple[np.ndarray, np.ndarray]]
    initial_E: Callable[..., Optional[np.ndarray]]
    dtypes: Tuple[str, ...] = ("f64", "f32")
    notes: str = ""
    src_comp: int = 1                   # TEz runs: component the soft source drives / the probes read (0 = Ex, 1 = Ey)
    probe_comp: int = 1

    @property
    def cell_updates(self) -> int:
        return self.nx * self.ny * self.nsteps


def _row_noise(cfg: int, tag: int, i0: int, i1: int, j0: int, j1: int, nx: int, amp: float) -> np.ndarray:
    """amp * U(-1,1) per node, one stream per grid row, so that any window regenerates bit for bit."""
    out = np.empty((j1 - j0, i1 - i0))
    for j in range(j0, j1):
        out[j - j0] = amp * _rng(cfg, tag, j).uniform(-1.0, 1.0, nx)[i0:i1]
    return out


def tm2d_column(nx: int = 16384, ny: int = 16384, nsteps: int = 1000, noise: bool = True, dy_over_dx: float = 1.0,
                boundary: int = BC_MUR, nprobes: int = 16) -> Workload2D:
    """The 2-D counterpart of config 4: a plasma column with a tanh (Epstein) edge in the middle of an nx x ny grid,
    wp^2(r) = (2 pi 50e9)^2 * 1/2 [1 - tanh((r - 0.15 nx)/(0.025 nx))] (r in nodes of dx, measured in physical
    distance / dx), nu = 1e10; per-node coefficient arrays.  Source: the same Gaussian-derivative pulse as the 1-D
    configs, at (nx/4, ny/2), outside the column.  Probes: the source node, nodes around it, on a ring through the
    column and seeded random nodes.  dx = 75 um, dt = dx/(2c) (Courant number 1/2 per axis, 0.707 of the 2-D limit
    when dy = dx).  Initial E: 1e-3 U(-1,1) so that probes the pulse has not reached yet carry a signal."""
    dx, dy = DZ, DZ * dy_over_dx
    dt = DZ * min(1.0, dy_over_dx) / (2.0 * C0)
    wp0, nu0 = 2.0 * math.pi * 50e9, 1.0e10
    ci, cj, R, wd = nx / 2.0, ny / 2.0, 0.15 * nx, 0.025 * nx

    def media(i0=0, i1=nx, j0=0, j1=ny):
        i = np.arange(i0, i1)[None, :] - ci
        j = (np.arange(j0, j1)[:, None] - cj) * dy_over_dx
        r = np.sqrt(i * i + j * j)
        wp = wp0 * np.sqrt(np.clip(0.5 * (1.0 - np.tanh((r - R) / wd)), 0.0, None))
        return np.ascontiguousarray(wp), np.full(wp.shape, nu0)

    def initial_E(i0=0, i1=nx, j0=0, j1=ny):
        return _row_noise(21, 1, i0, i1, j0, j1, nx, 1e-3) if noise else None

    src = (nx // 4, ny // 2)
    pr = [src, (src[0] + 3, src[1]), (src[0], src[1] + 5), (src[0] - 7, src[1] - 2), (nx // 2, ny // 2), (1, ny // 3),
          (nx - 2, ny // 3), (nx // 3, 1), (nx // 3, ny - 2), (0, ny // 2), (nx // 2, 0)]
    rng = _rng(21, 2)
    while len(pr) < nprobes:
        pr.append((int(rng.integers(0, nx)), int(rng.integers(0, ny))))
    pr = np.array(pr[:max(nprobes, 1)], np.int64)
    return Workload2D(f"tm2d_column_{nx}x{ny}", 21, nx, ny, nsteps, dx, dy, dt, SRC_GAUSS_DERIV, _SRC, src, pr, boundary,
                      media, initial_E, notes="2-D TMz plasma column, per-node coefficients")
