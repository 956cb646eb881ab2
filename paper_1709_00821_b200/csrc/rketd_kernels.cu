// rketd_kernels.cu — the three stencil kernels of librketd (sm_100a) and their launchers.
//
//   K1  k1_step      one fused H/E/J step per launch; a thread owns one 64-B row; halos from
//                    global memory; ping-pong buffers.  HBM-bound baseline and cross-check
//                    (this is the paper's H-kernel + E-kernel pair, fused).
//   K2  k2_wtile     temporal blocking, warp tiles (default): every WARP of a persistent CTA owns
//                    a tile of 32 rows x 64 B (halo included) of the seven input arrays (E, H, G,
//                    P, ch, ka, Q), staged into shared memory by 3-D tiled TMA loads (hardware
//                    64-B swizzle -> conflict-free 128-bit reads) on the warp's own mbarrier,
//                    moved into registers, advanced T steps with halos travelling by warp
//                    shuffles only (no block barrier, no shared memory in the time loop), and the
//                    valid interior written back by TMA stores or 256-bit global stores.  Every
//                    HBM byte serves T steps; the next tile's loads fly while this one computes.
//       k2_tblock    the same with one tile per CTA (128/256 rows: less redundant halo work, but
//                    one block barrier per step).
//   K3  k3_resident  one CTA per grid keeps the whole grid on chip (fields in registers,
//                    coefficients in registers or shared memory) for ALL steps of the run and
//                    streams probe samples out; the batched variant of the north_star.
//
// Mur boundaries, the soft source and probe recording are folded into the rows that hold
// those nodes (rowflag) inside the same kernels — see step_fields in rketd_device.cuh.
#include <algorithm>
#include <cstddef>

#include "rketd_device.cuh"
#include "rketd_internal.h"
#include "rketd_wtile.cuh"

namespace rketd {


// ------------------------------------------------------------------------------------ K1
template <typename R, bool PML>
__global__ void __launch_bounds__(128) k1_step(RowPtrs<R> src, RowPtrs<R> dst, CoefPtrs<R> cp,
                                               const __grid_constant__ StepParams<R> p, int64_t nrows,
                                               int64_t total_rows) {
  constexpr int C = kRowBytes / sizeof(R);
  const int64_t r = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (r >= total_rows) return;
  const int64_t g = r / nrows, row = r - g * nrows;
  R E[C], En[C], H[C], G[C];
  CoefRegs<R, C> cf;
  load_nodes_global<R, C>(src.E, r * C, E);
  load_nodes_global<R, C>(src.H, r * C, H);
  load_nodes_global<R, C>(src.J, r * C, G);
#pragma unroll
  for (int a = 0; a < kNumCoef; ++a) load_nodes_global<R, C>(cp.c[a], r * C, cf.c[a]);
  const R El = row > 0 ? src.E[r * C - 1] : R(0);
  const R Hl = row > 0 ? src.H[r * C - 1] : R(0);
  const R Er = row < nrows - 1 ? src.E[(r + 1) * C] : R(0);
  const uint32_t flag = p.rowflag[row];
  const R src_now = (flag & F_SRC) ? p.src_tab[p.n0] : R(0);
  const SpecialIdx sx = make_special<R, C, PML>(p, flag, row * C, g, true);
  step_fields<SF_SLOW, PML, R, C>(E, En, H, G, cf, El, Hl, Er, p.nchh, p, sx, WarpSpecial(), p.n0, src_now);
  step_current<R, C>(G, E, cf);
  store_nodes_global<R, C>(dst.E, r * C, En);
  store_nodes_global<R, C>(dst.H, r * C, H);
  store_nodes_global<R, C>(dst.J, r * C, G);
}

// The time loop shared by K2 and K3: nsteps leapfrog steps of this thread's nodes, halos
// exchanged inside the CTA.  One __syncthreads per step, placed after phase 2.  The loop is
// unrolled by two so that E ping-pongs between two register arrays without copies.
template <int MASK, bool PML, typename R, int C, int NW, typename CF>
__device__ __forceinline__ void time_loop(R (&E)[C], R (&H)[C], R (&J)[C], const CF &cf, HaloSlots<R, NW> &hs,
                                          const StepParams<R> &p, const SpecialIdx &sx, const WarpSpecial &ws,
                                          SourceStream<R> &src, int64_t nsteps, int warp, int lane) {
  constexpr bool SRC = MASK == SF_SLOW || (MASK & SF_SRC) != 0;
  const R nchh = pin_register(p.nchh);
  int64_t nloc = p.n0;
  R El, Hl, Er;
  typedef HaloSlots<R, NW> HS;
  static_assert(offsetof(HS, e_first) == 0 && offsetof(HS, e_last) == 2 * (NW + 2) * sizeof(R) &&
                    offsetof(HS, h_last) == 4 * (NW + 2) * sizeof(R), "halo_off assumes this layout");
  const uint32_t wa = pin_register(smem_u32(&hs) + (uint32_t)warp * (uint32_t)sizeof(R));
  send_halo_a<R, C, NW>(E, H, wa, 0, lane, El, Hl, Er);
  cta_barrier();
  recv_halo_a<R, NW>(wa, 0, lane, El, Hl, Er);
  R Eb[C];
  auto one_step = [&](const R (&Ein)[C], R (&Eout)[C], int par) {
    const R src_now = SRC ? src.sample(p, nloc, lane) : R(0);
    step_fields<MASK, PML, R, C, CF, true>(Ein, Eout, H, J, cf, El, Hl, Er, nchh, p, sx, ws, nloc, src_now);
    send_halo_a<R, C, NW>(Eout, H, wa, par, lane, El, Hl, Er);     // for the next step
    step_current<R, C>(J, Ein, cf);
    cta_barrier();
    recv_halo_a<R, NW>(wa, par, lane, El, Hl, Er);
    if (MASK != 0) ++nloc;
  };
  int64_t left = nsteps;
  for (; left >= 2; left -= 2) {
    one_step(E, Eb, 1);
    one_step(Eb, E, 0);
  }
  if (left) {
    one_step(E, Eb, 1);
#pragma unroll
    for (int i = 0; i < C; ++i) E[i] = Eb[i];
  }
  if constexpr (MASK != 0 && MASK != SF_SLOW) zero_padding_H<R, C>(H, ws);
}

// The warps of a CTA pick the instantiation that matches their features once, before the time loop (the barrier counts
// arriving warps, not program counters).  Four select variants instead of sixteen: Mur only, source/probe only, all.
template <bool PML, typename R, int C, int NW, typename CF>
__device__ __forceinline__ void time_loop_dispatch(R (&E)[C], R (&H)[C], R (&J)[C], const CF &cf, HaloSlots<R, NW> &hs,
                                                   const StepParams<R> &p, uint32_t flag, int64_t k0, int64_t g, bool owner,
                                                   int64_t nsteps, int warp, int lane) {
  const bool special = __any_sync(0xffffffffu, flag != 0u);
  const SpecialIdx sx = special ? make_special<R, C, PML>(p, flag, k0, g, owner) : SpecialIdx();
  const WarpSpecial ws = special ? make_warp_special<R, C, PML>(p, sx) : WarpSpecial();
  SourceStream<R> src;
  src.start(p, special && __any_sync(0xffffffffu, (flag & F_SRC) != 0u), p.n0, lane);
  constexpr int kMur = SF_MURL | SF_MURR, kSrcProbe = SF_SRC | SF_PROBE;
  constexpr int kFastAll = SF_MURR | SF_SRC | SF_PROBE;
  if (PML || ws.mask == SF_SLOW) time_loop<SF_SLOW, PML, R, C, NW>(E, H, J, cf, hs, p, sx, ws, src, nsteps, warp, lane);
  else if (ws.mask == 0) time_loop<0, false, R, C, NW>(E, H, J, cf, hs, p, sx, ws, src, nsteps, warp, lane);
  // every feature at a fixed local index (all BASELINE configs): straight-line selects, no branch in the step
  else if (ws.fast == kFastAll && (ws.mask & SF_SRC)) time_loop<SF_FAST | kMur | kSrcProbe, false, R, C, NW>(E, H, J, cf, hs, p, sx, ws, src, nsteps, warp, lane);
  else if (ws.fast == kFastAll) time_loop<SF_FAST | kMur | SF_PROBE, false, R, C, NW>(E, H, J, cf, hs, p, sx, ws, src, nsteps, warp, lane);
  else if ((ws.mask & kSrcProbe) == 0) time_loop<kMur, false, R, C, NW>(E, H, J, cf, hs, p, sx, ws, src, nsteps, warp, lane);
  else if ((ws.mask & kMur) == 0) time_loop<kSrcProbe, false, R, C, NW>(E, H, J, cf, hs, p, sx, ws, src, nsteps, warp, lane);
  else time_loop<kMur | kSrcProbe, false, R, C, NW>(E, H, J, cf, hs, p, sx, ws, src, nsteps, warp, lane);
}

// ------------------------------------------------------------------------------------ K3
// One CTA per grid; NT threads x C nodes cover the grid (NT * C >= physical nodes per grid).
// Which 32 rows of the grid a hardware warp holds.  The warps of a CTA sit on the SM's four schedulers by warp index
// (consecutive warps on consecutive schedulers, measured), and the warps with a boundary, the source or a probe issue
// 1.5-2.2 x the instructions of a plain one.  `tile[]` (host: k3_balance) deals the heavy tiles of a grid to different
// schedulers: config 3 (16 warps; tiles 0, 4, 12 heavy, all on scheduler 0 in natural order) 1085 -> 1230 Gcell/s.  Across
// the CTAs that share an SM nothing is needed: the hardware starts each CTA on the next scheduler (measured with %warpid:
// of four resident 4-warp CTAs, warp 0 sits once on each scheduler), and a rotation by CTA index changed nothing.
struct K3Map {
  uint8_t tile[16];
};

template <typename R, int C, int NT, bool CSM, int MINB, bool PML>
__global__ void __launch_bounds__(NT, MINB) k3_resident(RowPtrs<R> f, CoefPtrs<R> cp,
                                                        const __grid_constant__ StepParams<R> p, int64_t nrows,
                                                        int64_t nsteps, const K3Map map) {
  typedef Geom<R, C> G;
  constexpr int NW = NT / 32;
  constexpr int ROWS = NT / G::TPR;
  typedef typename Arith<R>::Vec Vec;
  __shared__ HaloSlots<R, NW> hs;
  extern __shared__ uint8_t smem_raw[];

  const int lane = threadIdx.x & 31;
  const int warp = map.tile[threadIdx.x >> 5];      // the tile, from here on
  const int tid = warp * 32 + lane;
  const int64_t g = blockIdx.x;
  const int row = tid / G::TPR;
  const bool valid = row < nrows;
  const int64_t k0 = (int64_t)tid * C;                       // physical in-grid index of the first node
  const int64_t first_node = g * nrows * G::CR + k0;
  hs.clear(tid);

  R E[C], H[C], J[C];
#pragma unroll
  for (int i = 0; i < C; ++i) { E[i] = R(0); H[i] = R(0); J[i] = R(0); }
  if (valid) {
    load_nodes_global<R, C>(f.E, first_node, E);
    load_nodes_global<R, C>(f.H, first_node, H);
    load_nodes_global<R, C>(f.J, first_node, J);
  }
  const uint32_t flag = valid ? p.rowflag[row] : 0u;
  __syncthreads();

  if constexpr (CSM) {
    const uint32_t base = smem_u32(smem_raw);
    CoefSmem<R, C, ROWS> cf;
    cf.init(base + ((1024u - (base & 1023u)) & 1023u), tid);
    // each thread stages its own coefficient chunks (only it reads them back: no barrier needed) and notes
    // whether its C nodes all carry the same values
    R first[kNumCoef];
    bool uniform = true;
    auto stage = [&](auto ac) {
      constexpr int a = decltype(ac)::value;
#pragma unroll
      for (int j = 0; j < G::NCH; ++j) {
        R z[G::V] = {};
        Vec v = vec_pack(z);
        if (valid) v = reinterpret_cast<const Vec *>(cp.c[a] + first_node)[j];
        cf.template store_chunk<a>(j, v);
        vec_unpack(v, z);
        if (j == 0) first[a] = z[0];
#pragma unroll
        for (int u = 0; u < G::V; ++u) uniform = uniform && (z[u] == first[a]);
      }
    };
    stage(std::integral_constant<int, 0>{}); stage(std::integral_constant<int, 1>{});
    stage(std::integral_constant<int, 2>{}); stage(std::integral_constant<int, 3>{});
    // piecewise-constant media: a warp whose rows are all uniform reads its coefficients from four registers and
    // leaves shared memory alone (one 512-row grid would otherwise read 128 KB of coefficients per step: the
    // shared-memory roofline, profiles/r01_ncu_k3_config3.md); warps on a media interface keep the general path
    if (__all_sync(0xffffffffu, uniform)) {
      CoefUniform<R, C> cu;
#pragma unroll
      for (int a = 0; a < kNumCoef; ++a) cu.v[a] = first[a];
      time_loop_dispatch<PML, R, C, NW>(E, H, J, cu, hs, p, flag, k0, g, true, nsteps, warp, lane);
    } else {
      time_loop_dispatch<PML, R, C, NW>(E, H, J, cf, hs, p, flag, k0, g, true, nsteps, warp, lane);
    }
  } else {
    CoefRegs<R, C> cf;
#pragma unroll
    for (int a = 0; a < kNumCoef; ++a) {
#pragma unroll
      for (int i = 0; i < C; ++i) cf.c[a][i] = R(0);
      if (valid) load_nodes_global<R, C>(cp.c[a], first_node, cf.c[a]);
    }
    time_loop_dispatch<PML, R, C, NW>(E, H, J, cf, hs, p, flag, k0, g, true, nsteps, warp, lane);
  }

  if (valid) {
    store_nodes_global<R, C>(f.E, first_node, E);
    store_nodes_global<R, C>(f.H, first_node, H);
    store_nodes_global<R, C>(f.J, first_node, J);
  }
}

// ------------------------------------------------------------------------------------ K2
struct K2Args {
  int T;                  // steps this pass
  int HR;                 // halo rows
  int rows_out;           // ROWS - 2 HR
  uint32_t tiles_per_grid, total_tiles;   // 32-bit on purpose: tile index arithmetic sits between two tiles
  uint32_t tile_first;    // this launch covers the tiles [tile_first, total_tiles) (rketd_run_from_host: pieces of a line)
  int64_t nrows;
  int spread;             // warp tiles: 1 = fewer tiles than one wave of warps: deal them out across the SMs first
};
constexpr int kNumIn = 3 + kNumCoef;      // arrays a tile loads: E, H, G, P, ch, ka, Q

// a thread's chunks of one staged tile: shared memory -> registers
template <typename R, int C>
__device__ __forceinline__ void tile_to_regs(uint32_t sin, const uint32_t (&off)[Geom<R, C>::NCH], uint32_t array_bytes,
                                             R (&E)[C], R (&H)[C], R (&J)[C], CoefRegs<R, C> &cf) {
  typedef typename Arith<R>::Vec Vec;
#pragma unroll
  for (int j = 0; j < Geom<R, C>::NCH; ++j) {
    const uint32_t my = sin + off[j];
    Vec v;
    lds128(my + 0 * array_bytes, v); vec_to_regs<R, C>(v, E, j);
    lds128(my + 1 * array_bytes, v); vec_to_regs<R, C>(v, H, j);
    lds128(my + 2 * array_bytes, v); vec_to_regs<R, C>(v, J, j);
#pragma unroll
    for (int a = 0; a < kNumCoef; ++a) {
      lds128(my + (3 + a) * array_bytes, v);
      vec_to_regs<R, C>(v, cf.c[a], j);
    }
  }
}
template <typename R, int C>
__device__ __forceinline__ void regs_to_tile(uint32_t sout, const uint32_t (&off)[Geom<R, C>::NCH], uint32_t array_bytes,
                                             const R (&E)[C], const R (&H)[C], const R (&J)[C]) {
#pragma unroll
  for (int j = 0; j < Geom<R, C>::NCH; ++j) {
    const uint32_t my = sout + off[j];
    sts128(my + 0 * array_bytes, regs_to_vec<R, C>(E, j));
    sts128(my + 1 * array_bytes, regs_to_vec<R, C>(H, j));
    sts128(my + 2 * array_bytes, regs_to_vec<R, C>(J, j));
  }
}

// Persistent CTAs; tile = ROWS = NT / TPR rows of 64 B (halo of HR rows on each side included).
template <typename R, int C, int NT, int MINB, bool PML>
__global__ void __launch_bounds__(NT, MINB) k2_tblock(const __grid_constant__ K2Maps maps,
                                                      const __grid_constant__ StepParams<R> p, K2Args q) {
  typedef Geom<R, C> G;
  constexpr int NW = NT / 32;
  constexpr int ROWS = NT / G::TPR;
  constexpr uint32_t kArrayBytes = ROWS * kRowBytes;

  __shared__ HaloSlots<R, NW> hs;
  __shared__ __align__(8) uint64_t mbar;
  extern __shared__ uint8_t smem_raw[];
  const uint32_t base = smem_u32(smem_raw);
  const uint32_t sin = base + ((1024u - (base & 1023u)) & 1023u);
  const uint32_t sout = sin + kNumIn * kArrayBytes;

  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int row = tid / G::TPR, sub = tid % G::TPR;

  auto issue_loads = [&](uint32_t tile) {   // one elected thread
    const uint32_t g = tile / q.tiles_per_grid, ti = tile - g * q.tiles_per_grid;
    const int row0 = (int)(ti * q.rows_out) - q.HR;
    mbar_expect_tx(&mbar, (uint32_t)kNumIn * kArrayBytes);
#pragma unroll
    for (int a = 0; a < kNumIn; ++a) tma_load_3d(sin + a * kArrayBytes, &maps.ld[a], &mbar, 0, row0, (int)g);
  };

  hs.clear(tid);
  if (tid == 0) {
    mbar_init(&mbar, 1);
    fence_barrier_init();
  }
  __syncthreads();
  uint32_t tile = q.tile_first + blockIdx.x;
  if (tid == 0 && tile < q.total_tiles) issue_loads(tile);
  uint32_t phase = 0;

  const int r_out = row - q.HR;
  const bool owner = r_out >= 0 && r_out < q.rows_out;
  uint32_t off_in[G::NCH], off_out[G::NCH];
#pragma unroll
  for (int j = 0; j < G::NCH; ++j) {
    off_in[j] = swz_off(row, sub * G::NCH + j);
    off_out[j] = swz_off(owner ? r_out : 0, sub * G::NCH + j);
  }

  for (; tile < q.total_tiles; tile += gridDim.x) {
    const uint32_t g = tile / q.tiles_per_grid, ti = tile - g * q.tiles_per_grid;
    const int64_t rowg = (int64_t)ti * q.rows_out - q.HR + row;     // this thread's row in the grid
    const uint32_t flag = (rowg >= 0 && rowg < q.nrows) ? p.rowflag[rowg] : 0u;

    mbar_wait(&mbar, phase);
    phase ^= 1u;

    R E[C], H[C], J[C];
    CoefRegs<R, C> cf;
    tile_to_regs<R, C>(sin, off_in, kArrayBytes, E, H, J, cf);
    const bool special = __syncthreads_or(flag != 0u);   // barrier: everyone has left the input stage
    if (tid == 0) {
      const uint32_t next = tile + gridDim.x;
      if (next < q.total_tiles) issue_loads(next);   // overlaps with the T steps below
      tma_wait_read0();                    // previous tile's stores have drained the output stage
    }

    if (special)   // tile holds a boundary, source or probe row (a handful of tiles per grid)
      time_loop_dispatch<PML, R, C, NW>(E, H, J, cf, hs, p, flag, rowg * G::CR + sub * C, g, owner, q.T, warp, lane);
    else
      time_loop_dispatch<false, R, C, NW>(E, H, J, cf, hs, p, 0u, 0, g, false, q.T, warp, lane);

    // (the barriers of the time loop order tma_wait_read0 before the writes below)
    if (owner) regs_to_tile<R, C>(sout, off_out, kArrayBytes, E, H, J);
    fence_proxy_async_smem();
    __syncthreads();
    if (tid == 0) {
      const int row_out0 = (int)(ti * q.rows_out);
#pragma unroll 1
      for (int a = 0; a < 3; ++a) tma_store_3d(&maps.st[a], sout + a * kArrayBytes, 0, row_out0, (int)g);
      tma_commit();
    }
  }
  if (tid == 0) tma_wait0();
}

// ------------------------------------------------------------------------------------ K2, warp tiles (warp_step / warp_time_loop: rketd_wtile.cuh)
// DIRECT = false: results leave through a shared-memory stage and TMA stores (10 x 2 KB of shared memory
// per warp).  DIRECT = true: every owner lane writes its 64-B rows with 256-bit global stores (full 32-B
// sectors); 7 x 2 KB per warp, which lets 12 warps (3 per scheduler) share an SM.
template <typename R, int NW, int MINB, bool DIRECT, bool PML>
__global__ void __launch_bounds__(NW * 32, MINB) k2_wtile(const __grid_constant__ K2Maps maps,
                                                          const __grid_constant__ StepParams<R> p, K2Args q,
                                                          RowPtrs<R> dst) {
  constexpr int C = kRowBytes / sizeof(R);
  typedef Geom<R, C> G;
  constexpr uint32_t kArrayBytes = 32 * kRowBytes;                      // one array of one warp tile: 2 KB
  constexpr uint32_t kWarpBytes = (kNumIn + (DIRECT ? 0 : 3)) * kArrayBytes;

  __shared__ __align__(8) uint64_t mbars[NW];
  extern __shared__ uint8_t smem_raw[];
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const uint32_t base = smem_u32(smem_raw);
  const uint32_t sin = base + ((1024u - (base & 1023u)) & 1023u) + warp * kWarpBytes;
  const uint32_t sout = sin + kNumIn * kArrayBytes;
  uint64_t *mbar = &mbars[warp];

  // (g, ti, first row) of a tile; 32-bit arithmetic: this sits on the serial path between two tiles
  auto locate = [&](uint32_t tile, uint32_t &g, uint32_t &ti, int &row0) {
    g = tile / q.tiles_per_grid;
    ti = tile - g * q.tiles_per_grid;
    row0 = (int)(ti * q.rows_out) - q.HR;
  };
  auto issue_loads = [&](uint32_t g, int row0) {   // lane 0
    mbar_expect_tx(mbar, (uint32_t)kNumIn * kArrayBytes);
#pragma unroll
    for (int a = 0; a < kNumIn; ++a) tma_load_3d(sin + a * kArrayBytes, &maps.ld[a], mbar, 0, row0, (int)g);
  };
  auto row_flag = [&](int row0) -> uint32_t {
    const int64_t rowg = (int64_t)row0 + lane;
    return (rowg >= 0 && rowg < q.nrows) ? p.rowflag[rowg] : 0u;
  };

  if (lane == 0) {
    mbar_init(mbar, 1);
    fence_barrier_init();
  }
  __syncwarp();
  const uint32_t stride = gridDim.x * NW;
  // the warps of a CTA work on consecutive tiles, so that the tiles in flight at any time are neighbours
  // in memory and the halo rows two tiles share are served by L2
  // (a problem smaller than one wave is latency bound: there one warp per SM beats twelve warps sharing an SM)
  uint32_t tile = q.tile_first + (q.spread ? warp * gridDim.x + blockIdx.x : blockIdx.x * NW + warp);
  uint32_t g = 0, ti = 0, flag = 0;
  int row0 = 0;
  if (tile < q.total_tiles) {
    locate(tile, g, ti, row0);
    if (lane == 0) issue_loads(g, row0);
    flag = row_flag(row0);
  }
  uint32_t phase = 0;

  const int r_out = lane - q.HR;
  const bool owner = r_out >= 0 && r_out < q.rows_out;
  uint32_t off_in[G::NCH], off_out[G::NCH];
#pragma unroll
  for (int j = 0; j < G::NCH; ++j) {
    off_in[j] = swz_off(lane, j);
    off_out[j] = swz_off(owner ? r_out : 0, j);
  }

  for (; tile < q.total_tiles; tile += stride) {
    const int64_t rowg = (int64_t)row0 + lane;       // this lane's row in grid g
    const uint32_t g_cur = g, ti_cur = ti;

    mbar_wait(mbar, phase);
    phase ^= 1u;

    R E[C], H[C], J[C];
    CoefRegs<R, C> cf;
    tile_to_regs<R, C>(sin, off_in, kArrayBytes, E, H, J, cf);
    const bool special = __any_sync(0xffffffffu, flag != 0u);   // also: every lane has left the input stage
    const uint32_t myflag = flag;
    flag = 0u;
    if (tile + stride < q.total_tiles) {             // next tile: loads and flags fly behind the steps below
      locate(tile + stride, g, ti, row0);
      if (lane == 0) issue_loads(g, row0);
      flag = row_flag(row0);
    }
    if (!DIRECT && lane == 0) tma_wait_read0();      // previous tile's stores have drained the output stage

    if (special)
      warp_time_loop<true, PML, R, C>(E, H, J, cf, p, myflag, rowg * C, g_cur, owner, q.T);
    else
      warp_time_loop<false, false, R, C>(E, H, J, cf, p, 0u, 0, g_cur, false, q.T);

    if constexpr (DIRECT) {
      if (owner && rowg < q.nrows) {
        const int64_t first = ((int64_t)g_cur * q.nrows + rowg) * C;
        store_nodes_global<R, C>(dst.E, first, E);
        store_nodes_global<R, C>(dst.H, first, H);
        store_nodes_global<R, C>(dst.J, first, J);
      }
    } else {
      __syncwarp();                                    // orders lane 0's tma_wait_read0 before the writes below
      if (owner) regs_to_tile<R, C>(sout, off_out, kArrayBytes, E, H, J);
      fence_proxy_async_smem();
      __syncwarp();
      if (lane == 0) {
        const int row_out0 = (int)(ti_cur * q.rows_out);
#pragma unroll
        for (int a = 0; a < 3; ++a) tma_store_3d(&maps.st[a], sout + a * kArrayBytes, 0, row_out0, (int)g_cur);
        tma_commit();
      }
    }
  }
  if (!DIRECT && lane == 0) tma_wait0();
}

// ------------------------------------------------------------------------------------ launchers
// Every stencil kernel exists twice: PML = false (first-order Mur ends; exactly the code without any trace of the
// absorbing layer) and PML = true (rketd_set_boundary: layer pre-step of H, conductor behind the layer).
template <typename R>
static cudaError_t launch_k1_t(const Layout &L, FieldPtrs src, FieldPtrs dst, void *const coef[kNumCoef],
                               const StepCommon &sc, cudaStream_t st) {
  const int64_t total = L.nrows * L.nbatch;
  const int64_t blocks = (total + 127) / 128;
  if (sc.npml > 0)
    k1_step<R, true><<<(unsigned)blocks, 128, 0, st>>>(rp<R>(src), rp<R>(dst), cpz<R>(coef), make_params<R>(sc), L.nrows, total);
  else
    k1_step<R, false><<<(unsigned)blocks, 128, 0, st>>>(rp<R>(src), rp<R>(dst), cpz<R>(coef), make_params<R>(sc), L.nrows, total);
  return cudaGetLastError();
}
cudaError_t launch_k1(int dtype, const Layout &L, FieldPtrs src, FieldPtrs dst, void *const coef[kNumCoef],
                      const StepCommon &sc, cudaStream_t st) {
  return dtype == 0 ? launch_k1_t<double>(L, src, dst, coef, sc, st) : launch_k1_t<float>(L, src, dst, coef, sc, st);
}

// K3 variants.  variant 0: a thread owns a whole 64-B row (ROWS = NT); coefficients in registers
// up to 256 rows, in shared memory at 512 rows.  variant 1: a thread owns half a row (twice the
// warps per grid, half the registers per thread); up to 256 rows.  variant 2: whole rows with the
// coefficients in shared memory at every size (fewer registers: more CTAs per SM); 64 rows and up.
int k3_threads_for_rows(int, int64_t nrows, int variant) {
  const int opts[] = {32, 64, 128, 256, 512};
  for (int o : opts)
    if (nrows <= o) {
      if (variant == 1) return 0;      // (half-row threads: removed, slower at every size measured)
      if (variant == 2) return o >= 64 ? o : 0;
      return o;
    }
  return 0;
}

template <typename R, int C, int NT, bool CSM, int MINB, bool PML>
static cudaError_t launch_k3_p(const Layout &L, FieldPtrs f, void *const coef[kNumCoef], const StepCommon &sc,
                               int64_t nsteps, const K3Map &map, cudaStream_t st) {
  auto kern = k3_resident<R, C, NT, CSM, MINB, PML>;
  const size_t smem = CSM ? (size_t)kNumCoef * (NT / Geom<R, C>::TPR) * kRowBytes + 1024 : 0;
  if (smem > 48 * 1024) {
    cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
  }
  kern<<<(unsigned)L.nbatch, NT, smem, st>>>(rp<R>(f), cpz<R>(coef), make_params<R>(sc), L.nrows, nsteps, map);
  return cudaGetLastError();
}
template <typename R, int C, int NT, bool CSM, int MINB>
static cudaError_t launch_k3_v(const Layout &L, FieldPtrs f, void *const coef[kNumCoef], const StepCommon &sc,
                               int64_t nsteps, const K3Map &map, cudaStream_t st) {
  return sc.npml > 0 ? launch_k3_p<R, C, NT, CSM, MINB, true>(L, f, coef, sc, nsteps, map, st)
                     : launch_k3_p<R, C, NT, CSM, MINB, false>(L, f, coef, sc, nsteps, map, st);
}
template <typename R>
static cudaError_t launch_k3_t(const Layout &L, FieldPtrs f, void *const coef[kNumCoef], const StepCommon &sc,
                               int64_t nsteps, int NT, int variant, const K3Map &map, cudaStream_t st) {
  constexpr int CF = kRowBytes / sizeof(R);
  if (variant == 0) switch (NT) {
    case 32: return launch_k3_v<R, CF, 32, false, 8>(L, f, coef, sc, nsteps, map, st);
    case 64: return launch_k3_v<R, CF, 64, false, 6>(L, f, coef, sc, nsteps, map, st);
    case 128: return launch_k3_v<R, CF, 128, false, 3>(L, f, coef, sc, nsteps, map, st);
    case 256: return launch_k3_v<R, CF, 256, false, 1>(L, f, coef, sc, nsteps, map, st);
    case 512: return launch_k3_v<R, CF, 512, true, 1>(L, f, coef, sc, nsteps, map, st);
  }
  else if (variant == 2) switch (NT) {   // whole rows, coefficients in shared memory (warps of uniform rows: registers)
    case 64: return launch_k3_v<R, CF, 64, true, 8>(L, f, coef, sc, nsteps, map, st);
    case 128: return launch_k3_v<R, CF, 128, true, 4>(L, f, coef, sc, nsteps, map, st);
    case 256: return launch_k3_v<R, CF, 256, true, 2>(L, f, coef, sc, nsteps, map, st);
    case 512: return launch_k3_v<R, CF, 512, true, 1>(L, f, coef, sc, nsteps, map, st);
  }
  return cudaErrorInvalidValue;
}
// tiles -> hardware warps: heaviest tiles first, each to the scheduler (warp index mod 4) with the least work so far
static K3Map k3_balance(int NW, const uint8_t *tile_flags, bool balance) {
  K3Map m;
  for (int i = 0; i < 16; ++i) m.tile[i] = (uint8_t)i;
  if (!balance || !tile_flags || NW < 2) return m;
  const int ncls = NW < 4 ? NW : 4, per = NW / ncls;
  double w[16], load[4] = {0, 0, 0, 0};
  int used[4] = {0, 0, 0, 0}, order[16];
  for (int t = 0; t < NW; ++t) {
    const bool mur = tile_flags[t] & (F_MURL | F_MURR), sp = tile_flags[t] & (F_SRC | F_PROBE);
    w[t] = (tile_flags[t] & F_PML) ? 2.5 : (mur && sp) ? 2.2 : sp ? 1.6 : mur ? 1.5 : 1.0;   // issued work / a plain warp's (from config-5 runs with and without source and probes)
    order[t] = t;
  }
  std::stable_sort(order, order + NW, [&](int a, int b) { return w[a] > w[b]; });
  for (int o = 0; o < NW; ++o) {
    int best = -1;
    for (int c = 0; c < ncls; ++c)
      if (used[c] < per && (best < 0 || load[c] < load[best])) best = c;
    m.tile[best + ncls * used[best]] = (uint8_t)order[o];
    load[best] += w[order[o]];
    ++used[best];
  }
  return m;
}
cudaError_t launch_k3(int dtype, const Layout &L, FieldPtrs f, void *const coef[kNumCoef], const StepCommon &sc,
                      int64_t nsteps, int NT, int variant, cudaStream_t st, const uint8_t *tile_flags, bool balance) {
  const K3Map map = k3_balance(NT / 32, tile_flags, balance);
  return dtype == 0 ? launch_k3_t<double>(L, f, coef, sc, nsteps, NT, variant, map, st)
                    : launch_k3_t<float>(L, f, coef, sc, nsteps, NT, variant, map, st);
}

// K2 variants (numbers kept from round 1; 1, 3, 4, 5, 7 were slower everywhere measured and are gone):
//   0: CTA tile, full row, 128 threads, 2 CTAs/SM     2: CTA tile, full row, 256 threads, 1 CTA/SM
//      (one block barrier per step: structurally different cross-checks of the default)
//   6: warp tiles, 12 warps, 1 CTA/SM, 256-bit global stores (default)
int k2_tile_rows(int variant) { const int r[] = {128, 0, 256, 0, 0, 0, 32, 0}; return (variant >= 0 && variant < kK2Variants) ? r[variant] : 0; }
int k2_tiles_per_cta(int variant) { const int t[] = {1, 0, 1, 0, 0, 0, 12, 0}; return (variant >= 0 && variant < kK2Variants) ? t[variant] : 0; }
size_t k2_smem_bytes(int variant) {
  const int arrays = variant >= 6 ? kNumIn : kNumIn + 3;
  return (size_t)arrays * k2_tile_rows(variant) * k2_tiles_per_cta(variant) * kRowBytes + 1024;
}

template <typename R, int V> struct K2Variant;
template <typename R> struct K2Variant<R, 0> { static constexpr int C = kRowBytes / sizeof(R), NT = 128, MINB = 2; };
template <typename R> struct K2Variant<R, 2> { static constexpr int C = kRowBytes / sizeof(R), NT = 256, MINB = 1; };

template <typename K, typename KP>
static cudaError_t k2_configure_k(K kern, KP kern_pml, int variant, int threads, int *ctas) {
  cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)k2_smem_bytes(variant));
  if (e != cudaSuccess) return e;
  e = cudaFuncSetAttribute(kern_pml, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)k2_smem_bytes(variant));
  if (e != cudaSuccess) return e;
  return cudaOccupancyMaxActiveBlocksPerMultiprocessor(ctas, kern, threads, k2_smem_bytes(variant));
}
template <typename R, int V>
static cudaError_t k2_configure_v(int *ctas) {
  typedef K2Variant<R, V> KV;
  return k2_configure_k(k2_tblock<R, KV::C, KV::NT, KV::MINB, false>, k2_tblock<R, KV::C, KV::NT, KV::MINB, true>, V, KV::NT, ctas);
}
template <typename R>
static cudaError_t k2_configure_t(int variant, int *ctas) {
  switch (variant) {
    case 0: return k2_configure_v<R, 0>(ctas);
    case 2: return k2_configure_v<R, 2>(ctas);
    case 6: return k2_configure_k(k2_wtile<R, 12, 1, true, false>, k2_wtile<R, 12, 1, true, true>, 6, 384, ctas);
  }
  return cudaErrorInvalidValue;
}
cudaError_t k2_configure(int dtype, int variant, int *ctas) {
  return dtype == 0 ? k2_configure_t<double>(variant, ctas) : k2_configure_t<float>(variant, ctas);
}

template <typename R, int V>
static cudaError_t launch_k2_v(const K2Plan &plan, int src_buf, const StepParams<R> &sp, const K2Args &q, cudaStream_t st) {
  typedef K2Variant<R, V> KV;
  if (sp.npml > 0)
    k2_tblock<R, KV::C, KV::NT, KV::MINB, true><<<plan.grid, KV::NT, plan.smem_bytes, st>>>(plan.maps[src_buf], sp, q);
  else
    k2_tblock<R, KV::C, KV::NT, KV::MINB, false><<<plan.grid, KV::NT, plan.smem_bytes, st>>>(plan.maps[src_buf], sp, q);
  return cudaGetLastError();
}
template <typename R, int NW, int MINB, bool DIRECT>
static void launch_k2_w(const K2Plan &plan, const K2Maps &m, const StepParams<R> &sp, const K2Args &q, RowPtrs<R> dst,
                        cudaStream_t st) {
  if (sp.npml > 0) k2_wtile<R, NW, MINB, DIRECT, true><<<plan.grid, NW * 32, plan.smem_bytes, st>>>(m, sp, q, dst);
  else k2_wtile<R, NW, MINB, DIRECT, false><<<plan.grid, NW * 32, plan.smem_bytes, st>>>(m, sp, q, dst);
}
template <typename R>
static cudaError_t launch_k2_t(const Layout &L, const K2Plan &plan_all, int src_buf, FieldPtrs dst, const StepCommon &sc,
                               int steps, int64_t tile_begin, int64_t tile_end, cudaStream_t st) {
  K2Args q;
  K2Plan plan = plan_all;
  q.T = steps; q.HR = plan.HR; q.rows_out = plan.rows_out;
  q.tiles_per_grid = (uint32_t)plan.tiles_per_grid; q.total_tiles = (uint32_t)plan.total_tiles; q.nrows = L.nrows;
  q.spread = plan.spread;
  q.tile_first = 0;
  if (tile_end >= 0) {     // a range of tiles: the grid shrinks with it
    if (tile_begin < 0 || tile_end > plan.total_tiles || tile_begin >= tile_end) return cudaErrorInvalidValue;
    q.tile_first = (uint32_t)tile_begin; q.total_tiles = (uint32_t)tile_end;
    const int tpc = k2_tiles_per_cta(plan.variant);
    const int64_t n = tile_end - tile_begin;
    if (plan.spread) plan.grid = (int)std::min<int64_t>(n, plan.grid);
    else plan.grid = (int)std::min<int64_t>((n + tpc - 1) / tpc, plan.grid);
  }
  const StepParams<R> sp = make_params<R>(sc);
  const K2Maps &m = plan.maps[src_buf];
  switch (plan.variant) {
    case 0: return launch_k2_v<R, 0>(plan, src_buf, sp, q, st);
    case 2: return launch_k2_v<R, 2>(plan, src_buf, sp, q, st);
    case 6: launch_k2_w<R, 12, 1, true>(plan, m, sp, q, rp<R>(dst), st); break;
    default: return cudaErrorInvalidValue;
  }
  return cudaGetLastError();
}
cudaError_t launch_k2(int dtype, const Layout &L, const K2Plan &plan, int src_buf, FieldPtrs dst, const StepCommon &sc,
                      int steps, cudaStream_t st, int64_t tile_begin, int64_t tile_end) {
  return dtype == 0 ? launch_k2_t<double>(L, plan, src_buf, dst, sc, steps, tile_begin, tile_end, st)
                    : launch_k2_t<float>(L, plan, src_buf, dst, sc, steps, tile_begin, tile_end, st);
}

}  // namespace rketd
