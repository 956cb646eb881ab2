// rketd_kernels.cu — the three stencil kernels of librketd (sm_100a) and their launchers.
//
//   K1  k1_step      one fused H/E/J step per launch; a thread owns one 64-B row; halos from
//                    global memory; ping-pong buffers.  HBM-bound baseline and cross-check
//                    (this is the paper's H-kernel + E-kernel pair, fused).
//   K2  k2_tblock    temporal blocking: a persistent CTA stages a tile (NT rows, halo included)
//                    of all nine arrays into shared memory with 3-D tiled TMA loads (hardware
//                    64-B swizzle -> conflict-free 128-bit reads), moves it into registers,
//                    advances T steps exchanging halos by warp shuffles (+ one shared-memory
//                    slot per warp edge and one barrier per step), and writes the valid
//                    interior back with TMA stores.  Every HBM byte serves T steps.  The next
//                    tile's TMA loads are in flight while the current tile computes.
//   K3  k3_resident  one CTA per grid keeps the whole grid on chip (fields in registers,
//                    coefficients in registers or shared memory) for ALL steps of the run and
//                    streams probe samples out; the batched variant of the north_star.
//
// Mur boundaries, the soft source and probe recording are folded into the rows that hold
// those nodes (rowflag) inside the same kernels — see step_fields in rketd_device.cuh.
#include "rketd_device.cuh"
#include "rketd_internal.h"

namespace rketd {

template <typename R> struct RowPtrs { R *E, *H, *J; };
template <typename R> struct CoefPtrs { const R *c[6]; };

// a thread's C nodes <-> global memory (first node at physical index `first`, 16-B aligned)
template <typename R, int C>
__device__ __forceinline__ void load_nodes_global(const R *base, int64_t first, R (&out)[C]) {
  typedef typename Arith<R>::Vec Vec;
  const Vec *p = reinterpret_cast<const Vec *>(base + first);
#pragma unroll
  for (int j = 0; j < Geom<R, C>::NCH; ++j) vec_to_regs<R, C>(p[j], out, j);
}
template <typename R, int C>
__device__ __forceinline__ void store_nodes_global(R *base, int64_t first, const R (&in)[C]) {
  typedef typename Arith<R>::Vec Vec;
  Vec *p = reinterpret_cast<Vec *>(base + first);
#pragma unroll
  for (int j = 0; j < Geom<R, C>::NCH; ++j) p[j] = regs_to_vec<R, C>(in, j);
}

// ------------------------------------------------------------------------------------ K1
template <typename R>
__global__ void __launch_bounds__(128) k1_step(RowPtrs<R> src, RowPtrs<R> dst, CoefPtrs<R> cp,
                                               const __grid_constant__ StepParams<R> p, int64_t nrows,
                                               int64_t total_rows) {
  constexpr int C = kRowBytes / sizeof(R);
  const int64_t r = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (r >= total_rows) return;
  const int64_t g = r / nrows, row = r - g * nrows;
  R E[C], En[C], H[C], J[C], t[C];
  CoefRegs<R, C> cf;
  load_nodes_global<R, C>(src.E, r * C, E);
  load_nodes_global<R, C>(src.H, r * C, H);
  load_nodes_global<R, C>(src.J, r * C, J);
#pragma unroll
  for (int a = 0; a < 6; ++a) load_nodes_global<R, C>(cp.c[a], r * C, cf.c[a]);
  const R El = row > 0 ? src.E[r * C - 1] : R(0);
  const R Hl = row > 0 ? src.H[r * C - 1] : R(0);
  const R Er = row < nrows - 1 ? src.E[(r + 1) * C] : R(0);
  const uint32_t flag = p.rowflag[row];
  step_fields<true, R, C>(E, En, H, J, t, cf, El, Hl, Er, p.nchh, p, flag, row * C, g, p.n0, true);
  step_current<R, C>(J, En, t, cf);
  store_nodes_global<R, C>(dst.E, r * C, En);
  store_nodes_global<R, C>(dst.H, r * C, H);
  store_nodes_global<R, C>(dst.J, r * C, J);
}

// The time loop shared by K2 and K3: nsteps leapfrog steps of this thread's nodes, halos
// exchanged inside the CTA.  One __syncthreads per step, placed after phase 2.  The loop is
// unrolled by two so that E ping-pongs between two register arrays without copies.
template <bool SPECIAL, typename R, int C, int NW, typename CF>
__device__ __forceinline__ void time_loop(R (&E)[C], R (&H)[C], R (&J)[C], const CF &cf, HaloSlots<R, NW> &hs,
                                          const StepParams<R> &p, uint32_t flag, int64_t k0, int64_t g, bool owner,
                                          int64_t nsteps, int warp, int lane) {
  const R nchh = pin_register(p.nchh);
  int64_t nloc = p.n0;
  R El, Hl, Er;
  send_halo<R, C, NW>(E, H, hs, 0, warp, lane, El, Hl, Er);
  __syncthreads();
  recv_halo<R, NW>(hs, 0, warp, lane, El, Hl, Er);
  R Eb[C];
  auto one_step = [&](const R (&Ein)[C], R (&Eout)[C], int par) {
    R t[C];
    step_fields<SPECIAL, R, C>(Ein, Eout, H, J, t, cf, El, Hl, Er, nchh, p, flag, k0, g, nloc, owner);
    send_halo<R, C, NW>(Eout, H, hs, par, warp, lane, El, Hl, Er);     // for the next step
    step_current<R, C>(J, Eout, t, cf);
    __syncthreads();
    recv_halo<R, NW>(hs, par, warp, lane, El, Hl, Er);
    if (SPECIAL) ++nloc;
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
}

// ------------------------------------------------------------------------------------ K3
// One CTA per grid; NT threads x C nodes cover the grid (NT * C >= physical nodes per grid).
template <typename R, int C, int NT, bool CSM, int MINB>
__global__ void __launch_bounds__(NT, MINB) k3_resident(RowPtrs<R> f, CoefPtrs<R> cp,
                                                        const __grid_constant__ StepParams<R> p, int64_t nrows,
                                                        int64_t nsteps) {
  typedef Geom<R, C> G;
  constexpr int NW = NT / 32;
  constexpr int ROWS = NT / G::TPR;
  typedef typename Arith<R>::Vec Vec;
  __shared__ HaloSlots<R, NW> hs;
  extern __shared__ uint8_t smem_raw[];

  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int64_t g = blockIdx.x;
  const int row = tid / G::TPR;
  const bool valid = row < nrows;
  const int64_t k0 = (int64_t)tid * C;                       // physical in-grid index of the first node
  const int64_t first = g * nrows * G::CR + k0;
  hs.clear(tid);

  R E[C], H[C], J[C];
#pragma unroll
  for (int i = 0; i < C; ++i) { E[i] = R(0); H[i] = R(0); J[i] = R(0); }
  if (valid) {
    load_nodes_global<R, C>(f.E, first, E);
    load_nodes_global<R, C>(f.H, first, H);
    load_nodes_global<R, C>(f.J, first, J);
  }
  const uint32_t flag = valid ? p.rowflag[row] : 0u;
  __syncthreads();

  if constexpr (CSM) {
    uint8_t *sm = reinterpret_cast<uint8_t *>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~uintptr_t(1023));
    CoefSmem<R, C, ROWS> cf;
    cf.init(sm, tid);
    // each thread stages its own coefficient chunks (only it reads them back: no barrier needed)
    auto stage = [&](auto ac) {
      constexpr int a = decltype(ac)::value;
#pragma unroll
      for (int j = 0; j < G::NCH; ++j) {
        R z[G::V] = {};
        Vec v = vec_pack(z);
        if (valid) v = reinterpret_cast<const Vec *>(cp.c[a] + first)[j];
        cf.template store_chunk<a>(j, v);
      }
    };
    stage(std::integral_constant<int, 0>{}); stage(std::integral_constant<int, 1>{});
    stage(std::integral_constant<int, 2>{}); stage(std::integral_constant<int, 3>{});
    stage(std::integral_constant<int, 4>{}); stage(std::integral_constant<int, 5>{});
    time_loop<true, R, C, NW>(E, H, J, cf, hs, p, flag, k0, g, true, nsteps, warp, lane);
  } else {
    CoefRegs<R, C> cf;
#pragma unroll
    for (int a = 0; a < 6; ++a) {
#pragma unroll
      for (int i = 0; i < C; ++i) cf.c[a][i] = R(0);
      if (valid) load_nodes_global<R, C>(cp.c[a], first, cf.c[a]);
    }
    time_loop<true, R, C, NW>(E, H, J, cf, hs, p, flag, k0, g, true, nsteps, warp, lane);
  }

  if (valid) {
    store_nodes_global<R, C>(f.E, first, E);
    store_nodes_global<R, C>(f.H, first, H);
    store_nodes_global<R, C>(f.J, first, J);
  }
}

// ------------------------------------------------------------------------------------ K2
struct K2Args {
  int T;                  // steps this pass
  int HR;                 // halo rows
  int rows_out;           // ROWS - 2 HR
  int64_t tiles_per_grid, total_tiles, nrows;
};

// Persistent CTAs; tile = ROWS = NT / TPR rows of 64 B (halo of HR rows on each side included).
template <typename R, int C, int NT, int MINB>
__global__ void __launch_bounds__(NT, MINB) k2_tblock(const __grid_constant__ K2Maps maps,
                                                      const __grid_constant__ StepParams<R> p, K2Args q) {
  typedef Geom<R, C> G;
  constexpr int NW = NT / 32;
  constexpr int ROWS = NT / G::TPR;
  constexpr uint32_t kArrayBytes = ROWS * kRowBytes;
  typedef typename Arith<R>::Vec Vec;

  __shared__ HaloSlots<R, NW> hs;
  __shared__ __align__(8) uint64_t mbar;
  extern __shared__ uint8_t smem_raw[];
  uint8_t *sin = reinterpret_cast<uint8_t *>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~uintptr_t(1023));
  uint8_t *sout = sin + 9 * kArrayBytes;

  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int row = tid / G::TPR, sub = tid % G::TPR;

  auto issue_loads = [&](int64_t tile) {   // one elected thread
    const int64_t g = tile / q.tiles_per_grid, ti = tile - g * q.tiles_per_grid;
    const int row0 = (int)(ti * q.rows_out - q.HR);
    mbar_expect_tx(&mbar, 9u * kArrayBytes);
#pragma unroll 1
    for (int a = 0; a < 9; ++a) tma_load_3d(sin + a * kArrayBytes, &maps.ld[a], &mbar, 0, row0, (int)g);
  };

  hs.clear(tid);
  if (tid == 0) {
    mbar_init(&mbar, 1);
    fence_barrier_init();
  }
  __syncthreads();
  int64_t tile = blockIdx.x;
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
    const int64_t g = tile / q.tiles_per_grid, ti = tile - g * q.tiles_per_grid;
    const int64_t rowg = ti * q.rows_out - q.HR + row;     // this thread's row in the grid

    mbar_wait(&mbar, phase);
    phase ^= 1u;

    R E[C], H[C], J[C];
    CoefRegs<R, C> cf;
#pragma unroll
    for (int j = 0; j < G::NCH; ++j) {
      const uint8_t *my = sin + off_in[j];
      vec_to_regs<R, C>(*reinterpret_cast<const Vec *>(my + 0 * kArrayBytes), E, j);
      vec_to_regs<R, C>(*reinterpret_cast<const Vec *>(my + 1 * kArrayBytes), H, j);
      vec_to_regs<R, C>(*reinterpret_cast<const Vec *>(my + 2 * kArrayBytes), J, j);
#pragma unroll
      for (int a = 0; a < 6; ++a)
        vec_to_regs<R, C>(*reinterpret_cast<const Vec *>(my + (3 + a) * kArrayBytes), cf.c[a], j);
    }
    const uint32_t flag = (rowg >= 0 && rowg < q.nrows) ? p.rowflag[rowg] : 0u;
    const bool special = __syncthreads_or(flag != 0u);   // barrier: everyone has left the input stage
    if (tid == 0) {
      const int64_t next = tile + gridDim.x;
      if (next < q.total_tiles) issue_loads(next);   // overlaps with the T steps below
      tma_wait_read0();                    // previous tile's stores have drained the output stage
    }

    if (special)   // tile holds a boundary, source or probe row (a handful of tiles per grid)
      time_loop<true, R, C, NW>(E, H, J, cf, hs, p, flag, rowg * G::CR + sub * C, g, owner, q.T, warp, lane);
    else
      time_loop<false, R, C, NW>(E, H, J, cf, hs, p, 0u, 0, g, false, q.T, warp, lane);

    // (the barriers of the time loop order tma_wait_read0 before the writes below)
    if (owner) {
#pragma unroll
      for (int j = 0; j < G::NCH; ++j) {
        uint8_t *my = sout + off_out[j];
        *reinterpret_cast<Vec *>(my + 0 * kArrayBytes) = regs_to_vec<R, C>(E, j);
        *reinterpret_cast<Vec *>(my + 1 * kArrayBytes) = regs_to_vec<R, C>(H, j);
        *reinterpret_cast<Vec *>(my + 2 * kArrayBytes) = regs_to_vec<R, C>(J, j);
      }
    }
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

// ------------------------------------------------------------------------------------ K2, warp tiles
// Same temporal blocking, but every WARP owns an independent tile of 32 rows (halo included),
// its own shared-memory stage and its own mbarrier: halos travel by warp shuffles only, there is
// no block barrier and no shared-memory exchange in the time loop.  Lanes 0 and 31 receive their
// own values from the shuffles at the tile edge, which is fine: those nodes are in the halo that
// is thrown away.  The price is a smaller tile (more redundant halo work per tile).
template <bool SPECIAL, typename R, int C, typename CF>
__device__ __forceinline__ void warp_time_loop(R (&E)[C], R (&H)[C], R (&J)[C], const CF &cf, const StepParams<R> &p,
                                               uint32_t flag, int64_t k0, int64_t g, bool owner, int nsteps) {
  const R nchh = pin_register(p.nchh);
  int64_t nloc = p.n0;
  R El = __shfl_up_sync(0xffffffffu, E[C - 1], 1);
  R Hl = __shfl_up_sync(0xffffffffu, H[C - 1], 1);
  R Er = __shfl_down_sync(0xffffffffu, E[0], 1);
  R Eb[C];
  auto one_step = [&](const R (&Ein)[C], R (&Eout)[C]) {
    R t[C];
    step_fields<SPECIAL, R, C>(Ein, Eout, H, J, t, cf, El, Hl, Er, nchh, p, flag, k0, g, nloc, owner);
    El = __shfl_up_sync(0xffffffffu, Eout[C - 1], 1);
    Hl = __shfl_up_sync(0xffffffffu, H[C - 1], 1);
    Er = __shfl_down_sync(0xffffffffu, Eout[0], 1);
    step_current<R, C>(J, Eout, t, cf);
    if (SPECIAL) ++nloc;
  };
  int left = nsteps;
  for (; left >= 2; left -= 2) {
    one_step(E, Eb);
    one_step(Eb, E);
  }
  if (left) {
    one_step(E, Eb);
#pragma unroll
    for (int i = 0; i < C; ++i) E[i] = Eb[i];
  }
}

template <typename R, int NW, int MINB>
__global__ void __launch_bounds__(NW * 32, MINB) k2_wtile(const __grid_constant__ K2Maps maps,
                                                          const __grid_constant__ StepParams<R> p, K2Args q) {
  constexpr int C = kRowBytes / sizeof(R);
  typedef Geom<R, C> G;
  constexpr uint32_t kArrayBytes = 32 * kRowBytes;      // one array of one warp tile: 2 KB
  constexpr uint32_t kWarpBytes = 12 * kArrayBytes;     // 9 input + 3 output arrays
  typedef typename Arith<R>::Vec Vec;

  __shared__ __align__(8) uint64_t mbars[NW];
  extern __shared__ uint8_t smem_raw[];
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  uint8_t *sin = reinterpret_cast<uint8_t *>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~uintptr_t(1023)) +
                 warp * kWarpBytes;
  uint8_t *sout = sin + 9 * kArrayBytes;
  uint64_t *mbar = &mbars[warp];

  auto issue_loads = [&](int64_t tile) {   // lane 0
    const int64_t g = tile / q.tiles_per_grid, ti = tile - g * q.tiles_per_grid;
    const int row0 = (int)(ti * q.rows_out - q.HR);
    mbar_expect_tx(mbar, 9u * kArrayBytes);
#pragma unroll 1
    for (int a = 0; a < 9; ++a) tma_load_3d(sin + a * kArrayBytes, &maps.ld[a], mbar, 0, row0, (int)g);
  };

  if (lane == 0) {
    mbar_init(mbar, 1);
    fence_barrier_init();
  }
  __syncwarp();
  const int64_t stride = (int64_t)gridDim.x * NW;
  int64_t tile = (int64_t)blockIdx.x * NW + warp;
  if (lane == 0 && tile < q.total_tiles) issue_loads(tile);
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
    const int64_t g = tile / q.tiles_per_grid, ti = tile - g * q.tiles_per_grid;
    const int64_t rowg = ti * q.rows_out - q.HR + lane;

    mbar_wait(mbar, phase);
    phase ^= 1u;

    R E[C], H[C], J[C];
    CoefRegs<R, C> cf;
#pragma unroll
    for (int j = 0; j < G::NCH; ++j) {
      const uint8_t *my = sin + off_in[j];
      vec_to_regs<R, C>(*reinterpret_cast<const Vec *>(my + 0 * kArrayBytes), E, j);
      vec_to_regs<R, C>(*reinterpret_cast<const Vec *>(my + 1 * kArrayBytes), H, j);
      vec_to_regs<R, C>(*reinterpret_cast<const Vec *>(my + 2 * kArrayBytes), J, j);
#pragma unroll
      for (int a = 0; a < 6; ++a)
        vec_to_regs<R, C>(*reinterpret_cast<const Vec *>(my + (3 + a) * kArrayBytes), cf.c[a], j);
    }
    const uint32_t flag = (rowg >= 0 && rowg < q.nrows) ? p.rowflag[rowg] : 0u;
    const bool special = __any_sync(0xffffffffu, flag != 0u);   // also: every lane has left the input stage
    if (lane == 0) {
      const int64_t next = tile + stride;
      if (next < q.total_tiles) issue_loads(next);   // overlaps with the T steps below
      tma_wait_read0();                              // previous tile's stores have drained the output stage
    }

    if (special)
      warp_time_loop<true, R, C>(E, H, J, cf, p, flag, rowg * C, g, owner, q.T);
    else
      warp_time_loop<false, R, C>(E, H, J, cf, p, 0u, 0, g, false, q.T);

    __syncwarp();                                    // orders lane 0's tma_wait_read0 before the writes below
    if (owner) {
#pragma unroll
      for (int j = 0; j < G::NCH; ++j) {
        uint8_t *my = sout + off_out[j];
        *reinterpret_cast<Vec *>(my + 0 * kArrayBytes) = regs_to_vec<R, C>(E, j);
        *reinterpret_cast<Vec *>(my + 1 * kArrayBytes) = regs_to_vec<R, C>(H, j);
        *reinterpret_cast<Vec *>(my + 2 * kArrayBytes) = regs_to_vec<R, C>(J, j);
      }
    }
    fence_proxy_async_smem();
    __syncwarp();
    if (lane == 0) {
      const int row_out0 = (int)(ti * q.rows_out);
#pragma unroll 1
      for (int a = 0; a < 3; ++a) tma_store_3d(&maps.st[a], sout + a * kArrayBytes, 0, row_out0, (int)g);
      tma_commit();
    }
  }
  if (lane == 0) tma_wait0();
}

// ------------------------------------------------------------------------------------ launchers
template <typename R>
static StepParams<R> make_params(const StepCommon &sc) {
  StepParams<R> p;
  p.nchh = (R)sc.nchh;
  p.mur_m = (R)sc.mur_m;
  p.cellL = sc.cellL; p.cellR = sc.cellR; p.cellS = sc.cellS;
  p.nprobes = sc.nprobes;
  p.rec_stride = sc.rec_stride; p.n0 = sc.n0;
  p.src_tab = (const R *)sc.src_tab;
  p.rec = (R *)sc.rec;
  p.rowflag = sc.rowflag;
  for (int i = 0; i < kMaxProbes; ++i) p.probe_cell[i] = sc.probe_cell[i];
  return p;
}
template <typename R> static RowPtrs<R> rp(FieldPtrs f) { return RowPtrs<R>{(R *)f.E, (R *)f.H, (R *)f.J}; }
template <typename R> static CoefPtrs<R> cpz(void *const coef[6]) {
  CoefPtrs<R> c;
  for (int a = 0; a < 6; ++a) c.c[a] = (const R *)coef[a];
  return c;
}

template <typename R>
static cudaError_t launch_k1_t(const Layout &L, FieldPtrs src, FieldPtrs dst, void *const coef[6],
                               const StepCommon &sc, cudaStream_t st) {
  const int64_t total = L.nrows * L.nbatch;
  const int64_t blocks = (total + 127) / 128;
  k1_step<R><<<(unsigned)blocks, 128, 0, st>>>(rp<R>(src), rp<R>(dst), cpz<R>(coef), make_params<R>(sc), L.nrows, total);
  return cudaGetLastError();
}
cudaError_t launch_k1(int dtype, const Layout &L, FieldPtrs src, FieldPtrs dst, void *const coef[6],
                      const StepCommon &sc, cudaStream_t st) {
  return dtype == 0 ? launch_k1_t<double>(L, src, dst, coef, sc, st) : launch_k1_t<float>(L, src, dst, coef, sc, st);
}

// K3 variants.  variant 0: a thread owns a whole 64-B row (ROWS = NT); coefficients in registers
// up to 256 rows, in shared memory at 512 rows.  variant 1: a thread owns half a row (twice the
// warps per grid, half the registers per thread); up to 256 rows.
int k3_threads_for_rows(int, int64_t nrows, int variant) {
  const int opts[] = {32, 64, 128, 256, 512};
  for (int o : opts)
    if (nrows <= o) {
      if (variant == 1) return o <= 256 ? 2 * o : 0;
      return o;
    }
  return 0;
}

template <typename R, int C, int NT, bool CSM, int MINB>
static cudaError_t launch_k3_v(const Layout &L, FieldPtrs f, void *const coef[6], const StepCommon &sc,
                               int64_t nsteps, cudaStream_t st) {
  auto kern = k3_resident<R, C, NT, CSM, MINB>;
  const size_t smem = CSM ? (size_t)6 * (NT / Geom<R, C>::TPR) * kRowBytes + 1024 : 0;
  if (smem > 48 * 1024) {
    cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
  }
  kern<<<(unsigned)L.nbatch, NT, smem, st>>>(rp<R>(f), cpz<R>(coef), make_params<R>(sc), L.nrows, nsteps);
  return cudaGetLastError();
}
template <typename R>
static cudaError_t launch_k3_t(const Layout &L, FieldPtrs f, void *const coef[6], const StepCommon &sc,
                               int64_t nsteps, int NT, int variant, cudaStream_t st) {
  constexpr int CF = kRowBytes / sizeof(R), CH = CF / 2;
  if (variant == 0) switch (NT) {
    case 32: return launch_k3_v<R, CF, 32, false, 8>(L, f, coef, sc, nsteps, st);
    case 64: return launch_k3_v<R, CF, 64, false, 4>(L, f, coef, sc, nsteps, st);
    case 128: return launch_k3_v<R, CF, 128, false, 2>(L, f, coef, sc, nsteps, st);
    case 256: return launch_k3_v<R, CF, 256, false, 1>(L, f, coef, sc, nsteps, st);
    case 512: return launch_k3_v<R, CF, 512, true, 1>(L, f, coef, sc, nsteps, st);
  }
  else switch (NT) {
    case 64: return launch_k3_v<R, CH, 64, false, 8>(L, f, coef, sc, nsteps, st);
    case 128: return launch_k3_v<R, CH, 128, false, 4>(L, f, coef, sc, nsteps, st);
    case 256: return launch_k3_v<R, CH, 256, false, 2>(L, f, coef, sc, nsteps, st);
    case 512: return launch_k3_v<R, CH, 512, false, 1>(L, f, coef, sc, nsteps, st);
  }
  return cudaErrorInvalidValue;
}
cudaError_t launch_k3(int dtype, const Layout &L, FieldPtrs f, void *const coef[6], const StepCommon &sc,
                      int64_t nsteps, int NT, int variant, cudaStream_t st) {
  return dtype == 0 ? launch_k3_t<double>(L, f, coef, sc, nsteps, NT, variant, st)
                    : launch_k3_t<float>(L, f, coef, sc, nsteps, NT, variant, st);
}

// K2 variants: {nodes per thread, threads per CTA, CTAs per SM aimed at}
//   0: full row, 128 threads, 2 CTAs/SM     1: half row, 256 threads, 2 CTAs/SM
//   2: full row, 256 threads, 1 CTA/SM      3: half row, 512 threads, 1 CTA/SM
//   4: warp tiles (32 rows per warp), 8 warps, 1 CTA/SM      5: warp tiles, 4 warps, 2 CTAs/SM
int k2_tile_rows(int variant) { const int r[] = {128, 128, 256, 256, 32, 32}; return (variant >= 0 && variant < 6) ? r[variant] : 0; }
int k2_tiles_per_cta(int variant) { return variant == 4 ? 8 : variant == 5 ? 4 : 1; }
size_t k2_smem_bytes(int variant) {
  return (size_t)12 * k2_tile_rows(variant) * k2_tiles_per_cta(variant) * kRowBytes + 1024;
}

template <typename R, int V> struct K2Variant;
template <typename R> struct K2Variant<R, 0> { static constexpr int C = kRowBytes / sizeof(R), NT = 128, MINB = 2; };
template <typename R> struct K2Variant<R, 1> { static constexpr int C = kRowBytes / sizeof(R) / 2, NT = 256, MINB = 2; };
template <typename R> struct K2Variant<R, 2> { static constexpr int C = kRowBytes / sizeof(R), NT = 256, MINB = 1; };
template <typename R> struct K2Variant<R, 3> { static constexpr int C = kRowBytes / sizeof(R) / 2, NT = 512, MINB = 1; };

template <typename K>
static cudaError_t k2_configure_k(K kern, int variant, int threads, int *ctas) {
  cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)k2_smem_bytes(variant));
  if (e != cudaSuccess) return e;
  return cudaOccupancyMaxActiveBlocksPerMultiprocessor(ctas, kern, threads, k2_smem_bytes(variant));
}
template <typename R, int V>
static cudaError_t k2_configure_v(int *ctas) {
  typedef K2Variant<R, V> KV;
  return k2_configure_k(k2_tblock<R, KV::C, KV::NT, KV::MINB>, V, KV::NT, ctas);
}
template <typename R>
static cudaError_t k2_configure_t(int variant, int *ctas) {
  switch (variant) {
    case 0: return k2_configure_v<R, 0>(ctas);
    case 1: return k2_configure_v<R, 1>(ctas);
    case 2: return k2_configure_v<R, 2>(ctas);
    case 3: return k2_configure_v<R, 3>(ctas);
    case 4: return k2_configure_k(k2_wtile<R, 8, 1>, 4, 256, ctas);
    case 5: return k2_configure_k(k2_wtile<R, 4, 2>, 5, 128, ctas);
  }
  return cudaErrorInvalidValue;
}
cudaError_t k2_configure(int dtype, int variant, int *ctas) {
  return dtype == 0 ? k2_configure_t<double>(variant, ctas) : k2_configure_t<float>(variant, ctas);
}

template <typename R, int V>
static cudaError_t launch_k2_v(const Layout &L, const K2Plan &plan, int src_buf, const StepCommon &sc, int steps,
                               cudaStream_t st) {
  typedef K2Variant<R, V> KV;
  K2Args q;
  q.T = steps; q.HR = plan.HR; q.rows_out = plan.rows_out;
  q.tiles_per_grid = plan.tiles_per_grid; q.total_tiles = plan.total_tiles; q.nrows = L.nrows;
  k2_tblock<R, KV::C, KV::NT, KV::MINB><<<plan.grid, KV::NT, plan.smem_bytes, st>>>(plan.maps[src_buf],
                                                                                   make_params<R>(sc), q);
  return cudaGetLastError();
}
template <typename R>
static cudaError_t launch_k2_t(const Layout &L, const K2Plan &plan, int src_buf, const StepCommon &sc, int steps,
                               cudaStream_t st) {
  switch (plan.variant) {
    case 0: return launch_k2_v<R, 0>(L, plan, src_buf, sc, steps, st);
    case 1: return launch_k2_v<R, 1>(L, plan, src_buf, sc, steps, st);
    case 2: return launch_k2_v<R, 2>(L, plan, src_buf, sc, steps, st);
    case 3: return launch_k2_v<R, 3>(L, plan, src_buf, sc, steps, st);
    case 4:
    case 5: {
      K2Args q;
      q.T = steps; q.HR = plan.HR; q.rows_out = plan.rows_out;
      q.tiles_per_grid = plan.tiles_per_grid; q.total_tiles = plan.total_tiles; q.nrows = L.nrows;
      if (plan.variant == 4)
        k2_wtile<R, 8, 1><<<plan.grid, 256, plan.smem_bytes, st>>>(plan.maps[src_buf], make_params<R>(sc), q);
      else
        k2_wtile<R, 4, 2><<<plan.grid, 128, plan.smem_bytes, st>>>(plan.maps[src_buf], make_params<R>(sc), q);
      return cudaGetLastError();
    }
  }
  return cudaErrorInvalidValue;
}
cudaError_t launch_k2(int dtype, const Layout &L, const K2Plan &plan, int src_buf, const StepCommon &sc, int steps,
                      cudaStream_t st) {
  return dtype == 0 ? launch_k2_t<double>(L, plan, src_buf, sc, steps, st)
                    : launch_k2_t<float>(L, plan, src_buf, sc, steps, st);
}

}  // namespace rketd
