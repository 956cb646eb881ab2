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
// those nodes (rowflag) inside the same kernels — see leapfrog_row in rketd_device.cuh.
#include "rketd_device.cuh"
#include "rketd_internal.h"

namespace rketd {

template <typename R> struct RowPtrs { R *E, *H, *J; };
template <typename R> struct CoefPtrs { const R *c[6]; };

template <typename R, int C>
__device__ __forceinline__ void load_row_global(const R *base, int64_t row, R (&out)[C]) {
  typedef typename Arith<R>::Vec Vec;
  constexpr int V = 16 / sizeof(R);
  const Vec *p = reinterpret_cast<const Vec *>(base + row * C);
#pragma unroll
  for (int j = 0; j < C / V; ++j) vec_to_regs<R, C>(p[j], out, j);
}
template <typename R, int C>
__device__ __forceinline__ void store_row_global(R *base, int64_t row, const R (&in)[C]) {
  typedef typename Arith<R>::Vec Vec;
  constexpr int V = 16 / sizeof(R);
  Vec *p = reinterpret_cast<Vec *>(base + row * C);
#pragma unroll
  for (int j = 0; j < C / V; ++j) p[j] = regs_to_vec(in, j);
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
  R E[C], H[C], J[C];
  CoefRegs<R, C> cf;
  load_row_global<R, C>(src.E, r, E);
  load_row_global<R, C>(src.H, r, H);
  load_row_global<R, C>(src.J, r, J);
#pragma unroll
  for (int a = 0; a < 6; ++a) load_row_global<R, C>(cp.c[a], r, cf.c[a]);
  const R El = row > 0 ? src.E[r * C - 1] : R(0);
  const R Hl = row > 0 ? src.H[r * C - 1] : R(0);
  const R Er = row < nrows - 1 ? src.E[(r + 1) * C] : R(0);
  const uint32_t flag = p.rowflag[row];
  leapfrog_row<R, C>(E, H, J, cf, El, Hl, Er, p, flag, row * C, g, p.n0, true);
  store_row_global<R, C>(dst.E, r, E);
  store_row_global<R, C>(dst.H, r, H);
  store_row_global<R, C>(dst.J, r, J);
}

// ------------------------------------------------------------------------------------ K3
template <typename R, int NT, bool CSM, int MINB>
__global__ void __launch_bounds__(NT, MINB) k3_resident(RowPtrs<R> f, CoefPtrs<R> cp,
                                                        const __grid_constant__ StepParams<R> p, int64_t nrows,
                                                        int64_t nsteps) {
  constexpr int C = kRowBytes / sizeof(R);
  constexpr int V = 16 / sizeof(R);
  constexpr int NW = NT / 32;
  typedef typename Arith<R>::Vec Vec;
  __shared__ HaloSlots<R, NW> hs;
  extern __shared__ uint8_t smem_raw[];

  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int64_t g = blockIdx.x;
  const bool valid = tid < nrows;
  const int64_t r = g * nrows + tid;

  R E[C], H[C], J[C];
#pragma unroll
  for (int i = 0; i < C; ++i) { E[i] = R(0); H[i] = R(0); J[i] = R(0); }
  if (valid) {
    load_row_global<R, C>(f.E, r, E);
    load_row_global<R, C>(f.H, r, H);
    load_row_global<R, C>(f.J, r, J);
  }
  const uint32_t flag = valid ? p.rowflag[tid] : 0u;
  const int64_t k0 = (int64_t)tid * C;

  auto time_loop = [&](const auto &cf) {
    for (int64_t n = 0; n < nsteps; ++n) {
      R El, Hl, Er;
      exchange_halo<R, C, NW>(E, H, hs, (int)(n & 1), warp, lane, El, Hl, Er);
      leapfrog_row<R, C>(E, H, J, cf, El, Hl, Er, p, flag, k0, g, p.n0 + n, true);
    }
  };

  if constexpr (CSM) {
    uint8_t *sm = reinterpret_cast<uint8_t *>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~uintptr_t(1023));
    CoefSmem<R, C, NT> cf;
    cf.init(sm, tid);
    // each thread stages its own coefficient rows (only it reads them back: no barrier needed)
    auto stage = [&](auto ac) {
      constexpr int a = decltype(ac)::value;
#pragma unroll
      for (int j = 0; j < C / V; ++j) {
        Vec v;
        if (valid) v = reinterpret_cast<const Vec *>(cp.c[a] + r * C)[j];
        else { R z[C] = {}; v = regs_to_vec(z, 0); }
        cf.template store_chunk<a>(j, v);
      }
    };
    stage(std::integral_constant<int, 0>{}); stage(std::integral_constant<int, 1>{});
    stage(std::integral_constant<int, 2>{}); stage(std::integral_constant<int, 3>{});
    stage(std::integral_constant<int, 4>{}); stage(std::integral_constant<int, 5>{});
    time_loop(cf);
  } else {
    CoefRegs<R, C> cf;
#pragma unroll
    for (int a = 0; a < 6; ++a) {
#pragma unroll
      for (int i = 0; i < C; ++i) cf.c[a][i] = R(0);
      if (valid) load_row_global<R, C>(cp.c[a], r, cf.c[a]);
    }
    time_loop(cf);
  }

  if (valid) {
    store_row_global<R, C>(f.E, r, E);
    store_row_global<R, C>(f.H, r, H);
    store_row_global<R, C>(f.J, r, J);
  }
}

// ------------------------------------------------------------------------------------ K2
struct K2Args {
  int T;                  // steps this pass
  int HR;                 // halo rows
  int rows_out;           // NT - 2 HR
  int64_t tiles_per_grid, total_tiles, nrows;
};

template <typename R, int NT, int MINB>
__global__ void __launch_bounds__(NT, MINB) k2_tblock(const __grid_constant__ K2Maps maps,
                                                      const __grid_constant__ StepParams<R> p, K2Args q) {
  constexpr int C = kRowBytes / sizeof(R);
  constexpr int V = 16 / sizeof(R);
  constexpr int NCH = C / V;
  constexpr int NW = NT / 32;
  constexpr uint32_t kArrayBytes = NT * kRowBytes;
  typedef typename Arith<R>::Vec Vec;

  __shared__ HaloSlots<R, NW> hs;
  __shared__ __align__(8) uint64_t mbar;
  extern __shared__ uint8_t smem_raw[];
  uint8_t *sin = reinterpret_cast<uint8_t *>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~uintptr_t(1023));
  uint8_t *sout = sin + 9 * kArrayBytes;

  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;

  auto issue_loads = [&](int64_t tile) {   // one elected thread
    const int64_t g = tile / q.tiles_per_grid, ti = tile - g * q.tiles_per_grid;
    const int row0 = (int)(ti * q.rows_out - q.HR);
    mbar_expect_tx(&mbar, 9u * kArrayBytes);
#pragma unroll 1
    for (int a = 0; a < 9; ++a) tma_load_3d(sin + a * kArrayBytes, &maps.ld[a], &mbar, 0, row0, (int)g);
  };

  if (tid == 0) {
    mbar_init(&mbar, 1);
    fence_barrier_init();
  }
  __syncthreads();
  int64_t tile = blockIdx.x;
  if (tid == 0 && tile < q.total_tiles) issue_loads(tile);
  uint32_t phase = 0;

  const uint32_t sw_in = (tid >> 1) & 3;
  const int r_out = tid - q.HR;
  const bool owner = r_out >= 0 && r_out < q.rows_out;
  const uint32_t sw_out = (r_out >> 1) & 3;

  for (; tile < q.total_tiles; tile += gridDim.x) {
    const int64_t g = tile / q.tiles_per_grid, ti = tile - g * q.tiles_per_grid;
    const int64_t rowg = ti * q.rows_out - q.HR + tid;     // this thread's row in the grid

    mbar_wait(&mbar, phase);
    phase ^= 1u;

    R E[C], H[C], J[C];
    CoefRegs<R, C> cf;
    {
      const uint8_t *my = sin + tid * kRowBytes;
#pragma unroll
      for (int j = 0; j < NCH; ++j) {
        const uint32_t o = (j ^ sw_in) << 4;
        vec_to_regs<R, C>(*reinterpret_cast<const Vec *>(my + 0 * kArrayBytes + o), E, j);
        vec_to_regs<R, C>(*reinterpret_cast<const Vec *>(my + 1 * kArrayBytes + o), H, j);
        vec_to_regs<R, C>(*reinterpret_cast<const Vec *>(my + 2 * kArrayBytes + o), J, j);
#pragma unroll
        for (int a = 0; a < 6; ++a)
          vec_to_regs<R, C>(*reinterpret_cast<const Vec *>(my + (3 + a) * kArrayBytes + o), cf.c[a], j);
      }
    }
    const uint32_t flag = (rowg >= 0 && rowg < q.nrows) ? p.rowflag[rowg] : 0u;
    __syncthreads();                       // everyone has left the input stage
    if (tid == 0) {
      const int64_t next = tile + gridDim.x;
      if (next < q.total_tiles) issue_loads(next);   // overlaps with the T steps below
      tma_wait_read0();                    // previous tile's stores have drained the output stage
    }

    const int64_t k0 = rowg * C;
    for (int s = 0; s < q.T; ++s) {
      R El, Hl, Er;
      exchange_halo<R, C, NW>(E, H, hs, s & 1, warp, lane, El, Hl, Er);
      leapfrog_row<R, C>(E, H, J, cf, El, Hl, Er, p, flag, k0, g, p.n0 + s, owner);
    }
    // (the barrier inside the first exchange orders tma_wait_read0 before the writes below)
    if (owner) {
      uint8_t *my = sout + r_out * kRowBytes;
#pragma unroll
      for (int j = 0; j < NCH; ++j) {
        const uint32_t o = (j ^ sw_out) << 4;
        *reinterpret_cast<Vec *>(my + 0 * kArrayBytes + o) = regs_to_vec(E, j);
        *reinterpret_cast<Vec *>(my + 1 * kArrayBytes + o) = regs_to_vec(H, j);
        *reinterpret_cast<Vec *>(my + 2 * kArrayBytes + o) = regs_to_vec(J, j);
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

// K3 variants: NT rows per grid; coefficients in registers up to NT = 256, in shared memory at 512.
int k3_threads_for_rows(int, int64_t nrows) {
  const int opts[] = {32, 64, 128, 256, 512};
  for (int o : opts)
    if (nrows <= o) return o;
  return 0;
}
size_t k3_smem_bytes(int, int NT) { return NT == 512 ? (size_t)6 * NT * kRowBytes + 1024 : 0; }

template <typename R, int NT, bool CSM, int MINB>
static cudaError_t launch_k3_v(const Layout &L, FieldPtrs f, void *const coef[6], const StepCommon &sc,
                               int64_t nsteps, cudaStream_t st) {
  auto kern = k3_resident<R, NT, CSM, MINB>;
  const size_t smem = CSM ? (size_t)6 * NT * kRowBytes + 1024 : 0;
  if (smem > 48 * 1024) {
    cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
  }
  kern<<<(unsigned)L.nbatch, NT, smem, st>>>(rp<R>(f), cpz<R>(coef), make_params<R>(sc), L.nrows, nsteps);
  return cudaGetLastError();
}
template <typename R>
static cudaError_t launch_k3_t(const Layout &L, FieldPtrs f, void *const coef[6], const StepCommon &sc,
                               int64_t nsteps, int NT, cudaStream_t st) {
  switch (NT) {
    case 32: return launch_k3_v<R, 32, false, 8>(L, f, coef, sc, nsteps, st);
    case 64: return launch_k3_v<R, 64, false, 5>(L, f, coef, sc, nsteps, st);
    case 128: return launch_k3_v<R, 128, false, 2>(L, f, coef, sc, nsteps, st);
    case 256: return launch_k3_v<R, 256, false, 1>(L, f, coef, sc, nsteps, st);
    case 512: return launch_k3_v<R, 512, true, 1>(L, f, coef, sc, nsteps, st);
  }
  return cudaErrorInvalidValue;
}
cudaError_t launch_k3(int dtype, const Layout &L, FieldPtrs f, void *const coef[6], const StepCommon &sc,
                      int64_t nsteps, int NT, cudaStream_t st) {
  return dtype == 0 ? launch_k3_t<double>(L, f, coef, sc, nsteps, NT, st)
                    : launch_k3_t<float>(L, f, coef, sc, nsteps, NT, st);
}

// K2 variants
int k2_threads_options(int idx) { const int o[] = {128, 256}; return idx < 2 ? o[idx] : 0; }
size_t k2_smem_bytes(int NT) { return (size_t)12 * NT * kRowBytes + 1024; }

template <typename R, int NT, int MINB>
static cudaError_t k2_configure_v(int *ctas) {
  auto kern = k2_tblock<R, NT, MINB>;
  cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)k2_smem_bytes(NT));
  if (e != cudaSuccess) return e;
  return cudaOccupancyMaxActiveBlocksPerMultiprocessor(ctas, kern, NT, k2_smem_bytes(NT));
}
cudaError_t k2_configure(int dtype, int NT, int *ctas) {
  if (dtype == 0) return NT == 128 ? k2_configure_v<double, 128, 2>(ctas) : k2_configure_v<double, 256, 1>(ctas);
  return NT == 128 ? k2_configure_v<float, 128, 2>(ctas) : k2_configure_v<float, 256, 1>(ctas);
}

template <typename R, int NT, int MINB>
static cudaError_t launch_k2_v(const Layout &L, const K2Plan &plan, int src_buf, const StepCommon &sc, int steps,
                               cudaStream_t st) {
  K2Args q;
  q.T = steps; q.HR = plan.HR; q.rows_out = plan.rows_out;
  q.tiles_per_grid = plan.tiles_per_grid; q.total_tiles = plan.total_tiles; q.nrows = L.nrows;
  k2_tblock<R, NT, MINB><<<plan.grid, NT, plan.smem_bytes, st>>>(plan.maps[src_buf], make_params<R>(sc), q);
  return cudaGetLastError();
}
cudaError_t launch_k2(int dtype, const Layout &L, const K2Plan &plan, int src_buf, const StepCommon &sc, int steps,
                      cudaStream_t st) {
  if (dtype == 0)
    return plan.NT == 128 ? launch_k2_v<double, 128, 2>(L, plan, src_buf, sc, steps, st)
                          : launch_k2_v<double, 256, 1>(L, plan, src_buf, sc, steps, st);
  return plan.NT == 128 ? launch_k2_v<float, 128, 2>(L, plan, src_buf, sc, steps, st)
                        : launch_k2_v<float, 256, 1>(L, plan, src_buf, sc, steps, st);
}

}  // namespace rketd
