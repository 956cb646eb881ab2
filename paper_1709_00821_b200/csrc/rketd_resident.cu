// rketd_resident.cu — K3 `k3_wtile`: the resident kernel of librketd (north_star kernels (2) + (3) combined; SURVEY.md
// §3.2 "ONE persistent launch ... runs ALL nsteps on chip", H5 "warp-private trapezoids (no per-step __syncthreads)").
//
// A chunk = k whole grids of the batch (consecutive rows of the [nbatch][nrows][C] layout) is held in the registers of a
// cluster of NC CTAs x NW warps for the whole run: every warp owns a tile of 32 rows x 64 B (one row per lane; E, H, G
// and the four coefficients of its nodes), tiles overlap by 2 HR rows, HR = ceil(T / C).  A round is T leapfrog steps of
// the tile by warp_step (rketd_wtile.cuh: halos by two shuffles per step, no barrier, no shared memory) — the same
// instruction sequence as K1 and K2, so the three agree bit for bit.  Garbage enters a tile from its two ends one node
// per step and the halo absorbs it; after the round every warp publishes the 2 HR outermost rows it OWNS into its
// neighbours' halo slots (shared memory of the neighbour's CTA: plain stores inside a CTA, st.shared::cluster over
// DSMEM across CTAs), ONE barrier (bar.sync, or the cluster barrier), and the halo lanes reload.  A barrier is paid once
// per T steps instead of once per step (profiles/r01_ncu_k3.md: `barrier` was the leading stall, 2.6-2.8 warps per issue).
// HBM is touched at the start, at the end and for probe samples.  Grids never interact inside a tile that spans two of
// them: the end nodes are rewritten by Mur / the conductor every step from their own grid's values, H behind the last
// node is forced to zero, and padding nodes carry zero coefficients (rketd_internal.h Layout).
#include <algorithm>

#include "rketd_wtile.cuh"

namespace rketd {

// "row" below = the C nodes one lane holds: a 64-B row of the layout, or half of one (HALF: twice the warps on a grid,
// half the dependent work per step — what a few grids, i.e. a chain of dependent steps, want)
struct K3WArgs {
  int T, HR, rows_out;          // steps per round, halo rows, 32 - 2 HR
  int cluster;                  // CTAs per chunk
  int chunk_rows;               // rows of a chunk = grids_per_chunk * nrows
  int tiles_per_chunk;          // ceil(chunk_rows / rows_out) <= cluster * warps per CTA
  int64_t nrows;                // rows per grid
  int64_t total_rows;           // nbatch * nrows
  int64_t nsteps;
};

__device__ __forceinline__ uint32_t cluster_ctarank() {
  uint32_t r;
  asm volatile("mov.u32 %0, %%cluster_ctarank;" : "=r"(r));
  return r;
}
__device__ __forceinline__ uint32_t map_to_cta(uint32_t local_smem_addr, uint32_t rank) {
  uint32_t a;
  asm volatile("mapa.shared::cluster.u32 %0, %1, %2;" : "=r"(a) : "r"(local_smem_addr), "r"(rank));
  return a;
}
__device__ __forceinline__ void st_cluster128(uint32_t a, const double2 &v) {
  asm volatile("st.shared::cluster.v2.f64 [%0], {%1, %2};" ::"r"(a), "d"(v.x), "d"(v.y) : "memory");
}
__device__ __forceinline__ void st_cluster128(uint32_t a, const float4 &v) {
  asm volatile("st.shared::cluster.v4.f32 [%0], {%1, %2, %3, %4};" ::"r"(a), "f"(v.x), "f"(v.y), "f"(v.z), "f"(v.w) : "memory");
}
__device__ __forceinline__ void cluster_barrier() {
  asm volatile("barrier.cluster.arrive.release.aligned;\n\tbarrier.cluster.wait.acquire.aligned;" ::: "memory");
}

#ifdef RKETD_K3W_TRACE
__device__ long long g_k3w_trace[16 * 12 * 8 * 6];
#define K3W_STAMP(k) do { if (lane == 0 && rnd >= 100 && rnd < 108) g_k3w_trace[((blockIdx.x * 12 + warp) * 8 + (rnd - 100)) * 6 + (k)] = clock64(); } while (0)
#else
#define K3W_STAMP(k) do { } while (0)
#endif

// halo slots of one CTA: [parity 2][warp][side 2][row HR][array 3][64 B]; side 0 = the tile's lanes 0..HR-1
constexpr int kMaxHR = 4;
__host__ __device__ constexpr uint32_t slot_bytes_per_warp() { return 2u * kMaxHR * 3u * kRowBytes; }

// LEAN: E in place and coefficients from four registers or the warp's shared-memory rows (warp_step_lean): 168
// registers, twelve warps per SM instead of eight.  The host picks it unless a layer is live or one lane records more than two probes.
template <typename R, bool CLUSTER, bool PML, bool LEAN, bool HALF = false>
__global__ void __launch_bounds__(LEAN ? 384 : 256, 1) k3_wtile(RowPtrs<R> f, CoefPtrs<R> cp, const __grid_constant__ StepParams<R> p,
                                                               const K3WArgs q) {
  static_assert(!HALF || (!LEAN && !PML), "half rows: plain instantiation only");
  constexpr int C = (int)(kRowBytes / sizeof(R)) / (HALF ? 2 : 1);
  typedef Geom<R, C> G;
  typedef typename Arith<R>::Vec Vec;
  extern __shared__ __align__(16) uint8_t slots_raw[];
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, nw = blockDim.x >> 5;
  const uint32_t rank = CLUSTER ? cluster_ctarank() : 0u;
  const int64_t chunk = CLUSTER ? (int64_t)(blockIdx.x / q.cluster) : (int64_t)blockIdx.x;
  const int tile = (int)rank * nw + warp;
  const bool active = tile < q.tiles_per_chunk;
  const uint32_t slots = smem_u32(slots_raw);
  const uint32_t par_bytes = (uint32_t)nw * slot_bytes_per_warp();

  // this lane's row
  const int r = tile * q.rows_out - q.HR + lane;                        // row within the chunk
  const int64_t rowc = chunk * q.chunk_rows + r;                        // row within the batch
  const bool valid = active && r >= 0 && r < q.chunk_rows && rowc < q.total_rows;
  const int64_t g = valid ? rowc / q.nrows : 0;
  const int64_t rowg = valid ? rowc - g * q.nrows : 0;
  const bool owner = valid && lane >= q.HR && lane < 32 - q.HR;

  R E[C], H[C], J[C];
  typename std::conditional<LEAN, int, CoefRegs<R, C>>::type cf_regs;      // (LEAN keeps no per-node coefficient registers)
  CoefUniform<R, C> cu;
  CoefWarpSmem<R, C> cs;
  bool warp_uniform = false;
#pragma unroll
  for (int i = 0; i < C; ++i) { E[i] = R(0); H[i] = R(0); J[i] = R(0); }
  uint32_t flag = 0u;
  if (valid) {
    const int64_t first = rowc * C;
    load_nodes_global<R, C>(f.E, first, E);
    load_nodes_global<R, C>(f.H, first, H);
    load_nodes_global<R, C>(f.J, first, J);
    flag = p.rowflag[HALF ? rowg >> 1 : rowg];
  }
  if constexpr (LEAN) {
    // coefficients: each lane stages its row of the four arrays in the warp's shared-memory area (only this warp reads
    // it back) and notes whether its nodes all carry one set; a warp of such lanes then runs from four registers
    const uint32_t cbase = slots + 2u * par_bytes + (uint32_t)nw * SourceRound<R>::kBytesPerWarp;
    cs.base = ((cbase + 1023u) & ~1023u) + (uint32_t)warp * (kNumCoef * 32u * kRowBytes);
    cs.lane = lane;
    bool uni = true;
#pragma unroll
    for (int a = 0; a < kNumCoef; ++a) {
      R c[C];
#pragma unroll
      for (int i = 0; i < C; ++i) c[i] = R(0);
      if (valid) load_nodes_global<R, C>(cp.c[a], rowc * C, c);
      cu.v[a] = c[0];
#pragma unroll
      for (int i = 1; i < C; ++i) uni = uni && (c[i] == c[0]);
#pragma unroll
      for (int j = 0; j < G::NCH; ++j) sts128(cs.base + a * (32 * kRowBytes) + swz_off(lane, j), regs_to_vec<R, C>(c, j));
    }
    warp_uniform = __all_sync(0xffffffffu, uni);
    __syncwarp();
  } else {
#pragma unroll
    for (int a = 0; a < kNumCoef; ++a) {
#pragma unroll
      for (int i = 0; i < C; ++i) cf_regs.c[a][i] = R(0);
      if (valid) load_nodes_global<R, C>(cp.c[a], rowc * C, cf_regs.c[a]);
    }
  }
  const bool special = __any_sync(0xffffffffu, flag != 0u);
  const SpecialIdx sx = special ? make_special<R, C, PML>(p, flag, rowg * C, g, owner) : SpecialIdx();
  const WarpSpecial ws = special ? make_warp_special<R, C, PML>(p, sx) : WarpSpecial();
  SourceRound<R> src;           // the round's source samples in the warp's strip behind the halo slots
  src.start(p, special && __any_sync(0xffffffffu, (flag & F_SRC) != 0u), p.n0, lane, q.T,
            slots + 2u * par_bytes + (uint32_t)warp * SourceRound<R>::kBytesPerWarp);

  // where this lane's row goes after a round: lanes HR..2HR-1 are the right halo of tile-1, lanes 32-2HR..32-HR-1 the left
  // halo of tile+1; and where its own halo row arrives
  const bool send_left = active && lane >= q.HR && lane < 2 * q.HR && tile > 0;
  const bool send_right = active && lane >= 32 - 2 * q.HR && lane < 32 - q.HR && tile + 1 < q.tiles_per_chunk;
  const bool recv_left = active && lane < q.HR && tile > 0;
  const bool recv_right = active && lane >= 32 - q.HR && tile + 1 < q.tiles_per_chunk;
  uint32_t send_addr = 0u, recv_addr = 0u;
  if (send_left || send_right) {
    const int dt = send_left ? tile - 1 : tile + 1;                    // destination tile
    const int dw = dt % nw, dr = dt / nw;
    const int side = send_left ? 1 : 0, hrow = send_left ? lane - q.HR : lane - (32 - 2 * q.HR);
    const uint32_t local = slots + (uint32_t)dw * slot_bytes_per_warp() + (uint32_t)(side * kMaxHR + hrow) * 3u * kRowBytes;
    send_addr = CLUSTER ? map_to_cta(local, (uint32_t)dr) : local;
  }
  if (recv_left || recv_right) {
    const int side = recv_left ? 0 : 1, hrow = recv_left ? lane : lane - (32 - q.HR);
    recv_addr = slots + (uint32_t)warp * slot_bytes_per_warp() + (uint32_t)(side * kMaxHR + hrow) * 3u * kRowBytes;
  }
  if constexpr (CLUSTER) cluster_barrier();       // every CTA of the cluster is resident before the first remote store

  uint32_t par = 0u;
  [[maybe_unused]] int rnd = -1;
  for (int64_t n = 0; n < q.nsteps; n += q.T) {
    const int Tr = (int)(q.nsteps - n < q.T ? q.nsteps - n : q.T);
    ++rnd;
    K3W_STAMP(0);
    if (n > 0) src.next_round(p, p.n0 + n, lane);
    if (active) {
      if constexpr (LEAN) {
        if (warp_uniform) warp_round_lean<R, C>(E, H, J, cu, p, sx, ws, src, p.n0 + n, Tr);
        else warp_round_lean<R, C>(E, H, J, cs, p, sx, ws, src, p.n0 + n, Tr);
      } else {
        warp_round<PML, R, C>(E, H, J, cf_regs, p, sx, ws, src, p.n0 + n, Tr);
      }
    }
    K3W_STAMP(1);
    if (n + Tr >= q.nsteps) break;
    // halo refresh: double-buffered by round parity, so one barrier per round is enough (a warp can overwrite buffer
    // `par` again only after the NEXT barrier, which every reader of this round's data has passed its reads to reach)
    if (send_left || send_right) {
      const uint32_t a = send_addr + par * par_bytes;
#pragma unroll
      for (int j = 0; j < G::NCH; ++j) {
        const Vec ve = regs_to_vec<R, C>(E, j), vh = regs_to_vec<R, C>(H, j), vg = regs_to_vec<R, C>(J, j);
        if constexpr (CLUSTER) {
          st_cluster128(a + 0 * kRowBytes + j * 16, ve); st_cluster128(a + 1 * kRowBytes + j * 16, vh); st_cluster128(a + 2 * kRowBytes + j * 16, vg);
        } else {
          sts128(a + 0 * kRowBytes + j * 16, ve); sts128(a + 1 * kRowBytes + j * 16, vh); sts128(a + 2 * kRowBytes + j * 16, vg);
        }
      }
    }
    K3W_STAMP(2);
    if constexpr (CLUSTER) cluster_barrier(); else cta_barrier();
    K3W_STAMP(3);
    if (recv_left || recv_right) {
      const uint32_t a = recv_addr + par * par_bytes;
#pragma unroll
      for (int j = 0; j < G::NCH; ++j) {
        Vec v;
        lds128(a + 0 * kRowBytes + j * 16, v); vec_to_regs<R, C>(v, E, j);
        lds128(a + 1 * kRowBytes + j * 16, v); vec_to_regs<R, C>(v, H, j);
        lds128(a + 2 * kRowBytes + j * 16, v); vec_to_regs<R, C>(v, J, j);
      }
    }
    par ^= 1u;
    K3W_STAMP(4);
  }

  if (owner) {
    const int64_t first = rowc * C;
    store_nodes_global<R, C>(f.E, first, E);
    store_nodes_global<R, C>(f.H, first, H);
    store_nodes_global<R, C>(f.J, first, J);
  }
  if constexpr (CLUSTER) cluster_barrier();       // no CTA leaves while a neighbour may still store into its slots
}

// ------------------------------------------------------------------------------------ plan + launch
// Tiles needed by `grids` whole grids at halo HR; the two ends of a chunk need no halo but tiles are laid out uniformly
// (tile i = rows i RO - HR .. i RO - HR + 31), so the count is ceil(rows / RO).
static int tiles_for(int64_t rows, int RO) { return (int)((rows + RO - 1) / RO); }

// fewer warp tiles in the whole batch than four per SM: latency, not throughput, decides
bool k3w_few_grids(const Layout &L, int sms) { return L.nbatch * ((L.nrows + 29) / 30) < (int64_t)sms * 4; }

bool k3w_plan(const Layout &L, int depth, int sms, int64_t want_nw, int64_t want_nc, int64_t want_k, bool lean, bool half, K3WPlan *out) {
  K3WPlan P;
  if (half && lean) return false;
  P.lean = lean;
  P.half = half;
  const int Cl = half ? L.C / 2 : L.C;                 // nodes per lane
  const int64_t nrows = half ? 2 * L.nrows : L.nrows;   // lane rows per grid
  // default depth: one halo row (8 steps per round in fp64, 16 in fp32) when many grids keep the SMs busy; two halo
  // rows when a few grids are a chain of dependent rounds, where halving the number of barriers pays for the wider
  // halo (config 1: 1.55 against 1.76 ms)
  const bool few = k3w_few_grids(L, sms);
  P.T = depth > 0 ? depth : (few ? 2 * L.C : L.C);
  P.HR = (P.T + Cl - 1) / Cl;
  if (P.HR > kMaxHR) return false;
  P.rows_out = 32 - 2 * P.HR;
  // 8 warps per CTA: the feature variants of the time loop need up to 242 registers, and a scheduler's 16 K registers
  // then hold two warps (12 warps would need <= 168 and spill); 4 warps per SM already saturate the FP64 pipe with this
  // instruction mix (profiles/r02_peaks.md).  16 = largest (non-portable) cluster.
  const int maxw = lean ? 12 : 8, maxc = 16;       // (the lean instantiation: 168 registers, three warps per scheduler)
  if (nrows > (int64_t)maxw * maxc * P.rows_out) return false;
  const int w1 = tiles_for(nrows, P.rows_out);       // tiles of one grid
  int k = 1, nc = 1, nw = w1;
  if (want_nw > 0 || want_nc > 0 || want_k > 0) {      // explicit (rketd_set_plan)
    k = (int)std::max<int64_t>(1, want_k);
    const int w = tiles_for(k * nrows, P.rows_out);
    nw = (int)want_nw;
    nc = want_nc > 0 ? (int)want_nc : (nw > 0 ? (w + nw - 1) / nw : (w + maxw - 1) / maxw);
    if (nw <= 0) nw = (w + nc - 1) / nc;
    if (nw > maxw || nc > maxc || (int64_t)nw * nc < w || k > L.nbatch) return false;
  } else if (few) {
    // few grids: the run is a chain of dependent steps.  One warp per scheduler at most, the rest of the
    // grid on other SMs of a cluster: a step then costs one warp's latency, not a queue of warps
    nw = std::min(w1, 4);
    nc = (w1 + nw - 1) / nw;
    if (nc > maxc) nc = maxc;
    nw = (w1 + nc - 1) / nc;
  } else {
    // many grids: throughput.  Score of a packing = rows that are real work / rows the warps hold, times how evenly
    // the warps load the four schedulers of an SM (the busiest one sets the pace: nw / (4 ceil(nw / 4))); a cluster
    // pays a little for its wider barrier.  k whole grids per chunk, up to 4 CTAs per chunk.
    double best = -1.0;
    for (int c = 1; c <= 4; ++c)
      for (int kk = 1; kk <= 256 && kk <= L.nbatch; ++kk) {
        const int w = tiles_for(kk * nrows, P.rows_out);
        const int n = (w + c - 1) / c;
        if (n > maxw) break;
        if (c > 1 && w <= (c - 1) * maxw) continue;          // fits a smaller cluster
        const int cap = lean ? 12 : 8;                        // warps an SM holds at this kernel's register count
        const double score = (double)(kk * nrows) / (32.0 * n * c) * ((double)((cap / n) * n) / cap) * (c > 1 ? 0.97 : 1.0);
        if (score > best + 1e-9) { best = score; k = kk; nc = c; nw = n; }
      }
    if (best < 0.0) {                                    // a grid needs more than 4 SMs: warps spread evenly over a cluster
      nc = (w1 + maxw - 1) / maxw;
      nw = (w1 + nc - 1) / nc;
    }
  }
  if (nw > maxw || nc > maxc || nw < 1 || nc < 1) return false;
  P.k = k; P.nc = nc; P.nw = nw;
  P.chunk_rows = k * nrows;
  if (P.chunk_rows > 0x7fffff00LL) return false;
  P.tiles_per_chunk = tiles_for(P.chunk_rows, P.rows_out);
  P.nchunks = (L.nbatch + k - 1) / k;
  P.smem_bytes = 2u * (uint32_t)nw * slot_bytes_per_warp() + (uint32_t)nw * 64u * (uint32_t)sizeof(double) +      // halo slots, source strips
                 (lean ? 1024u + (uint32_t)nw * kNumCoef * 32u * kRowBytes : 0u);
  *out = P;
  return true;
}

template <typename R, bool CLUSTER, bool PML, bool LEAN, bool HALF = false>
static cudaError_t launch_k3w_k(const Layout &L, const K3WPlan &P, FieldPtrs f, void *const coef[kNumCoef], const StepCommon &sc,
                                int64_t nsteps, cudaStream_t st) {
  auto kern = k3_wtile<R, CLUSTER, PML, LEAN, HALF>;
  if (P.smem_bytes > 48 * 1024) {
    cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)P.smem_bytes);
    if (e != cudaSuccess) return e;
  }
  K3WArgs q;
  q.T = P.T; q.HR = P.HR; q.rows_out = P.rows_out; q.cluster = P.nc; q.chunk_rows = (int)P.chunk_rows;
  q.tiles_per_chunk = P.tiles_per_chunk; q.nrows = (HALF ? 2 : 1) * L.nrows; q.total_rows = q.nrows * L.nbatch; q.nsteps = nsteps;
  cudaLaunchConfig_t cfg = {};
  cfg.gridDim = dim3((unsigned)(P.nchunks * P.nc));
  cfg.blockDim = dim3((unsigned)P.nw * 32);
  cfg.dynamicSmemBytes = P.smem_bytes;
  cfg.stream = st;
  cudaLaunchAttribute attr[1];
  if (CLUSTER) {
    if (P.nc > 8) {
      cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeNonPortableClusterSizeAllowed, 1);
      if (e != cudaSuccess) return e;
    }
    attr[0].id = cudaLaunchAttributeClusterDimension;
    attr[0].val.clusterDim.x = (unsigned)P.nc; attr[0].val.clusterDim.y = 1; attr[0].val.clusterDim.z = 1;
    cfg.attrs = attr; cfg.numAttrs = 1;
  }
  return cudaLaunchKernelEx(&cfg, kern, rp<R>(f), cpz<R>(coef), make_params<R>(sc), q);
}
template <typename R>
static cudaError_t launch_k3w_t(const Layout &L, const K3WPlan &P, FieldPtrs f, void *const coef[kNumCoef], const StepCommon &sc,
                                int64_t nsteps, cudaStream_t st) {
  const bool pml = sc.npml > 0;
  if (P.half) {                                  // (clusters only: one instantiation per type; a cluster of one CTA is fine)
    if (pml || P.lean) return cudaErrorInvalidValue;
    return launch_k3w_k<R, true, false, false, true>(L, P, f, coef, sc, nsteps, st);
  }
  if (P.lean && !pml)
    return P.nc > 1 ? launch_k3w_k<R, true, false, true>(L, P, f, coef, sc, nsteps, st) : launch_k3w_k<R, false, false, true>(L, P, f, coef, sc, nsteps, st);
  if (P.nc > 1) return pml ? launch_k3w_k<R, true, true, false>(L, P, f, coef, sc, nsteps, st) : launch_k3w_k<R, true, false, false>(L, P, f, coef, sc, nsteps, st);
  return pml ? launch_k3w_k<R, false, true, false>(L, P, f, coef, sc, nsteps, st) : launch_k3w_k<R, false, false, false>(L, P, f, coef, sc, nsteps, st);
}
cudaError_t launch_k3w(int dtype, const Layout &L, const K3WPlan &P, FieldPtrs f, void *const coef[kNumCoefArrays], const StepCommon &sc,
                       int64_t nsteps, cudaStream_t st) {
  return dtype == 0 ? launch_k3w_t<double>(L, P, f, coef, sc, nsteps, st) : launch_k3w_t<float>(L, P, f, coef, sc, nsteps, st);
}

// can a cluster of P.nc CTAs of this kernel be co-scheduled at all on this device?
template <typename R>
static cudaError_t k3w_max_clusters_t(const K3WPlan &P, int *nclusters) {
  auto kern = P.half ? k3_wtile<R, true, false, false, true> : P.lean ? k3_wtile<R, true, false, true> : k3_wtile<R, true, false, false>;
  if (P.smem_bytes > 48 * 1024) {
    cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)P.smem_bytes);
    if (e != cudaSuccess) return e;
  }
  if (P.nc > 8) {
    cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeNonPortableClusterSizeAllowed, 1);
    if (e != cudaSuccess) return e;
  }
  cudaLaunchConfig_t cfg = {};
  cfg.gridDim = dim3((unsigned)P.nc);
  cfg.blockDim = dim3((unsigned)P.nw * 32);
  cfg.dynamicSmemBytes = P.smem_bytes;
  cudaLaunchAttribute attr[1];
  attr[0].id = cudaLaunchAttributeClusterDimension;
  attr[0].val.clusterDim.x = (unsigned)P.nc; attr[0].val.clusterDim.y = 1; attr[0].val.clusterDim.z = 1;
  cfg.attrs = attr; cfg.numAttrs = 1;
  return cudaOccupancyMaxActiveClusters(nclusters, kern, &cfg);
}
cudaError_t k3w_max_clusters(int dtype, const K3WPlan &P, int *nclusters) {
  return dtype == 0 ? k3w_max_clusters_t<double>(P, nclusters) : k3w_max_clusters_t<float>(P, nclusters);
}

}  // namespace rketd

#ifdef RKETD_K3W_TRACE
extern "C" int rketd_debug_k3w_trace(long long *out, int n) {
  return (int)cudaMemcpyFromSymbol(out, rketd::g_k3w_trace, sizeof(long long) * n);
}
#endif
