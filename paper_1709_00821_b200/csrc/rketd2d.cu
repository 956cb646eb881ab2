// rketd2d.cu — the 2-D TMz generalisation of the RKETD-FDTD leapfrog (include/rketd2d.h; SURVEY.md §8(f) NEXT-3,
// PAPER.md:164): C ABI, setup kernels and the two stencil kernels
//   k1_2d   one fused H/E/J launch per time step (HBM-bound baseline and cross-check),
//   k2_2d   temporal blocking by streaming: a CTA owns a strip of columns, rows enter one per iteration and pass
//           through T pipeline stages held in registers, so every HBM byte serves T steps.
// Both run the same sequence of correctly rounded operations per node (struct Ops) and agree bit for bit.
//
// The form computed (the 2-D twin of rketd_device.cuh's 7-operation form).  With the six coefficients of SURVEY a0
// (Ez' = ca Ez - cj Jz + cex dHy - cey dHx,  Jz' = ka Jz + kb Ez + kc Ez') and G := cj Jz - (cj kc) Ez, exactly:
//   Hx'[j][i] = fma(-chy, Ez[j+1][i], fma(chy, Ez[j][i], Hx[j][i]))                         eq. (14), y axis
//   Hy'[j][i] = fma(+chx, Ez[j][i+1] - Ez[j][i], Hy[j][i])                                   eq. (14), x axis
//   Ez'[j][i] = fma(A, Ez[j+1][i], B),   A = ce r chy,                                       eq. (12)+(11)
//               B = fma(ce, fma(-r, fma(chy, Ez[j][i], Hx[j][i]) - Hx'[j-1][i], Hy'[j][i] - Hy'[j][i-1]), fma(P, Ez, -G))
//   G'[j][i]  = fma(ka, G, Q Ez)                                                            eq. (11)
// P = ca - cj kc, ce = cex, r = dx/dy (cey = cex r), Q = ka cj kc + cj kb: 13 FP instructions and 4 per-node
// coefficients per node and step.  Ez' is written as "gain x the row above + rest" (the same real number as
// fma(ce, fma(-r, Hx'[j] - Hx'[j-1], dHy), fma(P, Ez, -G))): in the streaming kernel the row above is the only operand
// that arrives late, so the dependent chain from one pipeline stage to the next is a single fma.
#include <algorithm>
#include <cmath>
#include <cstdio>
#include <cstring>
#include <string>
#include <vector>

#include "../../include/rketd2d.h"
#include "rketd_coef.cuh"
#include "rketd_device.cuh"
#include "rketd_internal.h"

using rketd::Arith;
using rketd::kC0;
using rketd::kEps0;
using rketd::kMu0;

namespace {

constexpr int kMaxProbes2 = 64;
constexpr int kMaxT = 16;
// threads per CTA of the streaming kernel = columns of a strip, one per thread; as many as the registers of a depth allow
template <typename R, int T> struct StripThreads { static constexpr int value = 256; };
template <> struct StripThreads<float, 8> { static constexpr int value = 384; };   // 136 registers: 12 warps (394 against 338 Gcell/s with 8)
constexpr int kPF = 3;         // rows in flight (cp.async) ahead of the row entering the pipeline
constexpr int kK1Rows = 4;     // rows a K1 thread walks

enum : uint8_t { RF_SPECIAL = 1, RF_PROBE = 2 };

template <typename R>
struct P2 {
  int nx, ny;
  int64_t pitch;
  R chx, nchy, chy, nr, c2;    // dt/(mu0 dx), -dt/(mu0 dy), +dt/(mu0 dy), -(dx/dy), (dx/dy) dt/(mu0 dy)
  R mx, my;                    // first-order Mur (S-1)/(S+1) per axis
  int bc;
  int src_i, src_j;            // -1: none
  int nprobes;
  int probe_i[kMaxProbes2], probe_j[kMaxProbes2];
  R *rec;                      // [nprobes][rec_stride]
  int64_t rec_stride, n0;      // samples per probe in rec; local index of the first step of this launch
  R src[kMaxT];                // source sample of each level of this launch (a4)
  const uint8_t *rowflag;      // [ny] RF_* bits
  // streaming plan
  int HP, Wv, nstrips, nsegs, Sy, dlast;
};

template <typename R>
struct Arrays {
  const R *E, *Hx, *Hy, *G, *cP, *cce, *cka, *cQ;
  R *E2, *Hx2, *Hy2, *G2;
};

// The per-node operations, shared by both kernels.
template <typename R>
struct Ops {
  typedef Arith<R> A;
  // Hx' = (Hx + chy E) - chy E_up: the part without the row above first (chy_j = 0 on the padding row ny-1)
  static __device__ __forceinline__ R hx_part(R chy_j, R e, R hx) { return A::fma(chy_j, e, hx); }
  static __device__ __forceinline__ R hx_new(R nchy_j, R e_up, R hxq) { return A::fma(nchy_j, e_up, hxq); }
  static __device__ __forceinline__ R hy_new(R chx_i, R e, R e_rt, R hy) { return A::fma(chx_i, A::sub(e_rt, e), hy); }
  // Ez' = gain * E_up + rest
  static __device__ __forceinline__ R e_gain(R ce, R c2_j) { return A::mul(ce, c2_j); }
  static __device__ __forceinline__ R e_rest(R P, R ce, R nr, R e, R g, R hyn, R hyn_l, R hxq, R hxn_d) {
    const R t = A::fma(nr, A::sub(hxq, hxn_d), A::sub(hyn, hyn_l));
    return A::fma(ce, t, A::fma(P, e, -g));
  }
  static __device__ __forceinline__ R e_new(R gain, R e_up, R rest) { return A::fma(gain, e_up, rest); }
  static __device__ __forceinline__ R g_new(R ka, R Q, R g, R e) { return A::fma(ka, g, A::mul(Q, e)); }
  // first-order Mur along the inward normal: E'[edge] = Eold[in] + m (E'[in] - Eold[edge])
  static __device__ __forceinline__ R mur(R m, R eold_in, R enew_in, R eold_self) {
    return A::fma(m, A::sub(enew_in, eold_self), eold_in);
  }
};

// ------------------------------------------------------------------------------------------------ K1
// Interior formula of Ez' at node (i, j), everything read from global memory (neighbours outside the grid count as 0);
// also returns the node's own new Hx, Hy.
template <typename R>
__device__ __forceinline__ R interior_e(const P2<R> &p, const Arrays<R> &a, int i, int j, R &hxn, R &hyn) {
  typedef Ops<R> O;
  const int64_t idx = (int64_t)j * p.pitch + i;
  const R e = a.E[idx];
  const R e_rt = (i + 1 < p.nx) ? a.E[idx + 1] : R(0);
  const R e_up = (j + 1 < p.ny) ? a.E[idx + p.pitch] : R(0);
  const R chx_i = (i <= p.nx - 2) ? p.chx : R(0);
  const bool yin = (j <= p.ny - 2);
  const R hxq = O::hx_part(yin ? p.chy : R(0), e, a.Hx[idx]);
  hxn = O::hx_new(yin ? p.nchy : R(0), e_up, hxq);
  hyn = O::hy_new(chx_i, e, e_rt, a.Hy[idx]);
  R hyn_l = R(0), hxn_d = R(0);
  if (i >= 1) hyn_l = O::hy_new(p.chx, a.E[idx - 1], e, a.Hy[idx - 1]);
  if (j >= 1) hxn_d = O::hx_new(p.nchy, e, O::hx_part(p.chy, a.E[idx - p.pitch], a.Hx[idx - p.pitch]));
  const R ce = a.cce[idx];
  const R rest = O::e_rest(a.cP[idx], ce, p.nr, e, a.G[idx], hyn, hyn_l, hxq, hxn_d);
  return O::e_new(O::e_gain(ce, yin ? p.c2 : R(0)), e_up, rest);
}

template <typename R>
__global__ void __launch_bounds__(128) k1_2d(const P2<R> p, const Arrays<R> a) {
  typedef Ops<R> O;
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= p.nx) return;
  const int j0 = blockIdx.y * kK1Rows, j1 = min(p.ny, j0 + kK1Rows);
  const bool xe = (i == 0 || i == p.nx - 1);
  for (int j = j0; j < j1; ++j) {
    const int64_t idx = (int64_t)j * p.pitch + i;
    const bool ye = (j == 0 || j == p.ny - 1);
    R hxn, hyn;
    R en = interior_e(p, a, i, j, hxn, hyn);
    const R e = a.E[idx];
    if (xe && ye) {
      en = R(0);
    } else if (xe || ye) {
      if (p.bc == RKETD2D_BC_MUR) {
        const int ii = xe ? (i == 0 ? 1 : p.nx - 2) : i, jj = ye ? (j == 0 ? 1 : p.ny - 2) : j;
        R d1, d2;
        const R en_in = interior_e(p, a, ii, jj, d1, d2);
        en = O::mur(xe ? p.mx : p.my, a.E[(int64_t)jj * p.pitch + ii], en_in, e);
      } else {
        en = R(0);
      }
    }
    if (i == p.src_i && j == p.src_j) en = Arith<R>::add(en, p.src[0]);
    a.Hx2[idx] = hxn;
    a.Hy2[idx] = hyn;
    a.G2[idx] = O::g_new(a.cka[idx], a.cQ[idx], a.G[idx], e);
    a.E2[idx] = en;
    if (p.rowflag[j] & RF_PROBE)
      for (int q = 0; q < p.nprobes; ++q)
        if (p.probe_i[q] == i && p.probe_j[q] == j) p.rec[(int64_t)q * p.rec_stride + p.n0] = en;
  }
}

// ------------------------------------------------------------------------------------------------ K1 with the paper's layer
// Berenger's split-field layer on the four sides, a conductor behind it (rketd2d_set_boundary_pml; PAPER.md:93, :123;
// reading in DESIGN.md §15 = the 1-D reading of §12 per axis).  Per-axis tables over the whole axis (1 / the plain
// coefficient outside the layers): H is damped everywhere by its table, Ez = Ezx + Ezy on layer nodes, the plasma update
// in the (P, G) form elsewhere.  One launch per step, like k1_2d.
template <typename R>
struct PmlTabs {
  const R *hax, *hbx, *eax, *ebx;      // [nx]: Hy' = hax Hy + hbx dEz/di;  Ezx' = eax Ezx + ebx dHy/di
  const R *hay, *hby, *eay, *eby;      // [ny]: Hx' = hay Hx - hby dEz/dj;  Ezy' = eay Ezy - eby dHx/dj
  const R *Ezx, *Ezy;
  R *Ezx2, *Ezy2;
  int npml;
};
template <typename R>
__device__ __forceinline__ R pml_hx(const P2<R> &p, const Arrays<R> &a, const PmlTabs<R> &t, int i, int j) {
  typedef Arith<R> A;
  if (j < 0 || j > p.ny - 2) return R(0);
  const int64_t k = (int64_t)j * p.pitch + i;
  return A::fma(-t.hby[j], A::sub(a.E[k + p.pitch], a.E[k]), A::mul(t.hay[j], a.Hx[k]));
}
template <typename R>
__device__ __forceinline__ R pml_hy(const P2<R> &p, const Arrays<R> &a, const PmlTabs<R> &t, int i, int j) {
  typedef Arith<R> A;
  if (i < 0 || i > p.nx - 2) return R(0);
  const int64_t k = (int64_t)j * p.pitch + i;
  return A::fma(t.hbx[i], A::sub(a.E[k + 1], a.E[k]), A::mul(t.hax[i], a.Hy[k]));
}
template <typename R>
__global__ void __launch_bounds__(128) k1_2d_pml(const P2<R> p, const Arrays<R> a, const PmlTabs<R> t) {
  typedef Arith<R> A;
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= p.nx) return;
  const int j0 = blockIdx.y * kK1Rows, j1 = min(p.ny, j0 + kK1Rows);
  for (int j = j0; j < j1; ++j) {
    const int64_t k = (int64_t)j * p.pitch + i;
    const R e = a.E[k];
    const R hxn = pml_hx(p, a, t, i, j), hyn = pml_hy(p, a, t, i, j);
    const bool edge = i == 0 || i == p.nx - 1 || j == 0 || j == p.ny - 1;
    const bool layer = i < t.npml || i > p.nx - 1 - t.npml || j < t.npml || j > p.ny - 1 - t.npml;
    R en = R(0), exn = R(0), eyn = R(0), gn = R(0);
    if (!edge) {
      const R dhy = A::sub(hyn, pml_hy(p, a, t, i - 1, j)), dhx = A::sub(hxn, pml_hx(p, a, t, i, j - 1));
      if (layer) {
        exn = A::fma(t.ebx[i], dhy, A::mul(t.eax[i], t.Ezx[k]));
        eyn = A::fma(-t.eby[j], dhx, A::mul(t.eay[j], t.Ezy[k]));
        en = A::add(exn, eyn);
      } else {
        en = A::fma(a.cce[k], A::fma(p.nr, dhx, dhy), A::fma(a.cP[k], e, -a.G[k]));
        gn = A::fma(a.cka[k], a.G[k], A::mul(a.cQ[k], e));
      }
    }
    if (i == p.src_i && j == p.src_j) { en = A::add(en, p.src[0]); exn = A::add(exn, p.src[0]); }
    a.Hx2[k] = hxn; a.Hy2[k] = hyn; a.G2[k] = gn; a.E2[k] = en;
    t.Ezx2[k] = exn; t.Ezy2[k] = eyn;
    if (p.rowflag[j] & RF_PROBE)
      for (int q = 0; q < p.nprobes; ++q)
        if (p.probe_i[q] == i && p.probe_j[q] == j) p.rec[(int64_t)q * p.rec_stride + p.n0] = en;
  }
}

// ------------------------------------------------------------------------------------------------ K2
template <typename R>
__device__ __forceinline__ void cp_async_val(R *smem_dst, const R *gsrc, bool valid) {
  const unsigned sa = (unsigned)__cvta_generic_to_shared(smem_dst);
  const int sz = valid ? (int)sizeof(R) : 0;          // 0 source bytes: the destination is zero-filled
  asm volatile("cp.async.ca.shared.global [%0], [%1], %2, %3;\n" ::"r"(sa), "l"(gsrc), "n"((int)sizeof(R)), "r"(sz) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;\n" ::: "memory"); }
template <int N>
__device__ __forceinline__ void cp_async_wait() { asm volatile("cp.async.wait_group %0;\n" ::"n"(N) : "memory"); }

template <typename R>
__device__ __forceinline__ R shfl_down1(R v) { return __shfl_down_sync(0xffffffffu, v, 1); }
template <typename R>
__device__ __forceinline__ R shfl_up1(R v) { return __shfl_up_sync(0xffffffffu, v, 1); }

// 2 x R as one shared-memory access (16 B fp64, 8 B fp32)
__device__ __forceinline__ void ld_pair(const double *q, double &x, double &y) { const double2 v = *reinterpret_cast<const double2 *>(q); x = v.x; y = v.y; }
__device__ __forceinline__ void ld_pair(const float *q, float &x, float &y) { const float2 v = *reinterpret_cast<const float2 *>(q); x = v.x; y = v.y; }
__device__ __forceinline__ void st_pair(double *q, double x, double y) { *reinterpret_cast<double2 *>(q) = make_double2(x, y); }
__device__ __forceinline__ void st_pair(float *q, float x, float y) { *reinterpret_cast<float2 *>(q) = make_float2(x, y); }

// predicated shared stores (no branch, no reconvergence point around the warp-edge posts of every iteration)
__device__ __forceinline__ void st_pair_if(bool pred, uint32_t a, double x, double y) {
  asm volatile("{\n.reg .pred q;\nsetp.ne.u32 q, %0, 0;\n@q st.shared.v2.f64 [%1], {%2, %3};\n}" ::"r"((uint32_t)pred), "r"(a), "d"(x), "d"(y) : "memory");
}
__device__ __forceinline__ void st_pair_if(bool pred, uint32_t a, float x, float y) {
  asm volatile("{\n.reg .pred q;\nsetp.ne.u32 q, %0, 0;\n@q st.shared.v2.f32 [%1], {%2, %3};\n}" ::"r"((uint32_t)pred), "r"(a), "f"(x), "f"(y) : "memory");
}

__device__ __forceinline__ void lds_if_lane31(int lane, uint32_t a, double &v) {
  asm volatile("{\n.reg .pred q;\nsetp.eq.u32 q, %1, 31;\n@q ld.shared.f64 %0, [%2];\n}" : "+d"(v) : "r"(lane), "r"(a) : "memory");
}
__device__ __forceinline__ void lds_if_lane31(int lane, uint32_t a, float &v) {
  asm volatile("{\n.reg .pred q;\nsetp.eq.u32 q, %1, 31;\n@q ld.shared.f32 %0, [%2];\n}" : "+f"(v) : "r"(lane), "r"(a) : "memory");
}

// Rows of the eight input arrays arrive as 2-D tiled TMA boxes {strip columns, 1 row} (cp.async.bulk.tensor.2d, SASS UTMALDG):
// one elected thread issues them, completion on the ring slot's mbarrier; columns and rows outside the grid are zero-filled
// by the hardware (the tensor map's extent is nx x ny), which is what the strip halo at the grid's edges needs.
struct Maps2D { CUtensorMap m[8]; };      // Ez, Hx, Hy, G of the source buffer, then P, ce, ka, Q
__device__ __forceinline__ void tma_load_2d(uint32_t dst, const void *tmap, uint64_t *bar, int c0, int c1) {
  asm volatile("cp.async.bulk.tensor.2d.shared::cluster.global.tile.mbarrier::complete_tx::bytes [%0], [%1, {%3, %4}], [%2];"
               ::"r"(dst), "l"(tmap), "r"(rketd::smem_u32(bar)), "r"(c0), "r"(c1) : "memory");
}
template <int NT> struct TmaBox { static constexpr int W = NT <= 256 ? NT : NT / 2, N = NT / W; };   // box width <= 256 elements

constexpr int kRing = kPF + 1;      // entry ring, 8 arrays per row (Ez, Hx, Hy, G, P, ce, ka, Q): one slot more than the rows in
                                    // flight, so that a slot is refilled two iterations after it was read (a barrier lies between)
template <typename R, int T>
struct K2Shape {
  static constexpr int NT = StripThreads<R, T>::value;
  static constexpr size_t smem = sizeof(R) * ((size_t)kRing * 8 * NT + (size_t)2 * T * 4 * (NT / 32 + 2) + (size_t)T * NT);
};

// Per-thread constants of a job of the streaming kernel.
template <typename R>
struct JobCtx {
  int i, lane, warp, y_out0, y_out1;
  bool own_col, xl, xr, xin, src_col, is_mur;
  R chx_i, chx_im1;
};

// What a thread keeps per pipeline stage: E, Hx, Hy, G and the four coefficients of the row the stage holds (the
// coefficients travel down the pipeline with their row: registers only change names, nothing is copied or re-read).
template <typename R, int T>
struct Held {
  R e[T], hx[T], hy[T], g[T], cP[T], cce[T], cka[T], cQ[T];
  R hxp_last;          // new Hx of the row before the one the LAST stage holds (for s < T-1 that value is hx[s+1])
};

// The T pipeline stages of one iteration (row Y has just entered as (ein, hxin, hyin, gin)): reads the held rows `h`,
// leaves the rows held in the next iteration in `n` (two sets used alternately, so that no register is copied).
//   SPECIAL = false: none of the rows held by the stages is row 0, 1, ny-2, ny-1, the source row or a probe row.
//                    Everything that does not need the row above is computed for all stages first (shuffles, new Hy,
//                    new G, gain and rest of Ez'); what is left is one fma per stage along the pipeline.
//   SPECIAL = true:  stage by stage, with the y edges, the source and the probes; `xsb` (shared memory, [T][NT]) keeps
//                    one spare value per stage across iterations: the old E of the row before (needed on row 1 for the
//                    Mur value of row 0) or, on row ny-1, the edge value computed one iteration earlier.
//   XEDGE:           this warp holds column 0 or nx-1 (first-order Mur / conductor on the x edges).
template <typename R, int T, bool SPECIAL, bool XEDGE>
__device__ __forceinline__ void run_stages(const P2<R> &p, const Arrays<R> &a, const JobCtx<R> &c, const int Y, const uint32_t fq,
                                           R *xbuf, R *xsb, Held<R, T> &h, Held<R, T> &n,
                                           R &ein, R &hxin, R &hyin, R &gin, R &cPin, R &ccein, R &ckain, R &cQin) {
  typedef Ops<R> O;
  constexpr int NT = StripThreads<R, T>::value;
  constexpr int XS = NT / 32 + 2;     // exchange slots per stage: one per warp plus a zero slot at each end
  const int tid = c.warp * 32 + c.lane;
  R gain[T], rest[T], hxq[T], hyn[T], gn[T];
  if (!SPECIAL) {
#pragma unroll
    for (int s = 0; s < T; ++s) {        // everything that needs old values only
      const R cP = h.cP[s], cce = h.cce[s], cka = h.cka[s], cQ = h.cQ[s];
      const R es = h.e[s];
      // neighbours across the warp edge come from the exchange buffer (slots of the strip's outer neighbours hold zeros);
      // branch-free, so that the whole path stays one block the compiler can interleave
      const R *xl_ = xbuf + (s * XS + c.warp) * 4;           // slot of warp - 1: {E, Hy of its lane 31}
      R e31, hy31;
      ld_pair(xl_, e31, hy31);
      R e_rt = shfl_down1(es);
      lds_if_lane31(c.lane, rketd::smem_u32(xl_ + 2 * 4 + 2), e_rt);      // slot of warp + 1: E of its lane 0 (lane 31 only)
      hyn[s] = O::hy_new(c.chx_i, es, e_rt, h.hy[s]);
      const R hyn_edge = O::hy_new(c.chx_im1, e31, es, hy31);
      R hyn_l = shfl_up1(hyn[s]);
      hyn_l = (c.lane == 0) ? hyn_edge : hyn_l;
      // rows outside the grid hold zeros, so chy is right for them too (row ny-1, where it is not, is a special row)
      hxq[s] = O::hx_part(p.chy, es, h.hx[s]);
      const R hxp = (s + 1 < T) ? h.hx[s + 1 < T ? s + 1 : s] : h.hxp_last;
      rest[s] = O::e_rest(cP, cce, p.nr, es, h.g[s], hyn[s], hyn_l, hxq[s], hxp);
      gain[s] = O::e_gain(cce, p.c2);
      gn[s] = O::g_new(cka, cQ, h.g[s], es);
    }
#pragma unroll
    for (int s = 0; s < T; ++s) {        // along the pipeline: one fma per stage on the critical path
      const int y = Y - 1 - s;
      R en = O::e_new(gain[s], ein, rest[s]);
      const R hxn = O::hx_new(p.nchy, ein, hxq[s]);
      if (XEDGE) {                       // x edges of the rows 1..ny-2
        const R es = h.e[s];
        const R e_rt = shfl_down1(es), e_lf = shfl_up1(es), en_rt = shfl_down1(en), en_lf = shfl_up1(en);
        if (y >= 1 && y <= p.ny - 2) {
          if (c.xl) en = c.is_mur ? O::mur(p.mx, e_rt, en_rt, es) : R(0);
          if (c.xr) en = c.is_mur ? O::mur(p.mx, e_lf, en_lf, es) : R(0);
        }
      }
      if (s == T - 1) n.hxp_last = hxn;
      n.e[s] = ein; n.hx[s] = hxin; n.hy[s] = hyin; n.g[s] = gin;
      n.cP[s] = cPin; n.cce[s] = ccein; n.cka[s] = ckain; n.cQ[s] = cQin;
      ein = en; hxin = hxn; hyin = hyn[s]; gin = gn[s];
      cPin = h.cP[s]; ccein = h.cce[s]; ckain = h.cka[s]; cQin = h.cQ[s];
    }
    return;
  }
#pragma unroll
  for (int s = 0; s < T; ++s) {
    const int y = Y - 1 - s;
    const R cP = h.cP[s], cce = h.cce[s], cka = h.cka[s], cQ = h.cQ[s];
    const bool yin = (y >= 0 && y <= p.ny - 2);
    const R es = h.e[s];
    const R *xl_ = xbuf + (s * XS + c.warp) * 4;
    R e31, hy31;
    ld_pair(xl_, e31, hy31);
    const R e0r = xl_[2 * 4 + 2];
    R e_rt = shfl_down1(es);
    e_rt = (c.lane == 31) ? e0r : e_rt;
    const R hyn_s = O::hy_new(c.chx_i, es, e_rt, h.hy[s]);
    const R hyn_edge = O::hy_new(c.chx_im1, e31, es, hy31);
    R hyn_l = shfl_up1(hyn_s);
    hyn_l = (c.lane == 0) ? hyn_edge : hyn_l;
    const R hxq_s = O::hx_part(yin ? p.chy : R(0), es, h.hx[s]);
    const R hxn = O::hx_new(yin ? p.nchy : R(0), ein, hxq_s);
    const R hxp = (s + 1 < T) ? h.hx[s + 1 < T ? s + 1 : s] : h.hxp_last;
    R en = O::e_new(O::e_gain(cce, yin ? p.c2 : R(0)), ein, O::e_rest(cP, cce, p.nr, es, h.g[s], hyn_s, hyn_l, hxq_s, hxp));
    const R gn_s = O::g_new(cka, cQ, h.g[s], es);
    R xs_new = es;
    {                                    // x edges of the rows 1..ny-2 (every warp takes the shuffles here)
      const R en_rt = shfl_down1(en), en_lf = shfl_up1(en), e_lf = shfl_up1(es);
      if (y >= 1 && y <= p.ny - 2) {
        if (c.xl) en = c.is_mur ? O::mur(p.mx, e_rt, en_rt, es) : R(0);
        if (c.xr) en = c.is_mur ? O::mur(p.mx, e_lf, en_lf, es) : R(0);
      }
    }
    if ((fq >> (s + 1)) & 1u) {          // CTA-uniform
      const bool own = c.own_col && y >= c.y_out0 && y < c.y_out1;
      const R xs = xsb[s * NT + tid];
      if (y == p.ny - 1) en = xs;        // computed one iteration ago from rows ny-2 (new) and ny-1 (old)
      if (y == 0) en = R(0);             // set one iteration later, when E'[1] exists
      if (y == p.ny - 2) xs_new = (c.xin && c.is_mur) ? O::mur(p.my, es, en, ein) : R(0);
      if (y == 1) {                      // row 0 at level s+1: stage s+1 holds it by now (or it has been stored)
        R e0 = (c.xin && c.is_mur) ? O::mur(p.my, es, en, xs) : R(0);
        if (p.src_j == 0 && c.src_col) e0 = Arith<R>::add(e0, p.src[s]);
        if (c.own_col && c.y_out0 == 0 && (p.rowflag[0] & RF_PROBE))
          for (int q = 0; q < p.nprobes; ++q)
            if (p.probe_j[q] == 0 && p.probe_i[q] == c.i) p.rec[(int64_t)q * p.rec_stride + p.n0 + s] = e0;
        if (s + 1 < T) {
          h.e[s + 1 < T ? s + 1 : s] = e0;
          if (c.lane == 0) xbuf[((s + 1) * XS + c.warp + 1) * 4 + 2] = e0;
          if (c.lane == 31) xbuf[((s + 1) * XS + c.warp + 1) * 4 + 0] = e0;
          __syncthreads();
        } else if (c.own_col && c.y_out0 == 0) {
          a.E2[c.i] = e0;
        }
      }
      if (y == p.src_j && c.src_col && y != 0) en = Arith<R>::add(en, p.src[s]);
      if (own && y != 0 && (p.rowflag[y] & RF_PROBE))
        for (int q = 0; q < p.nprobes; ++q)
          if (p.probe_j[q] == y && p.probe_i[q] == c.i) p.rec[(int64_t)q * p.rec_stride + p.n0 + s] = en;
    }
    xsb[s * NT + tid] = xs_new;
    if (s == T - 1) n.hxp_last = hxn;
    n.e[s] = ein; n.hx[s] = hxin; n.hy[s] = hyin; n.g[s] = gin;
    n.cP[s] = cPin; n.cce[s] = ccein; n.cka[s] = ckain; n.cQ[s] = cQin;
    ein = en; hxin = hxn; hyin = hyn_s; gin = gn_s;
    cPin = cP; ccein = cce; ckain = cka; cQin = cQ;
  }
}

// Streaming temporal blocking.  Job = (strip of NT columns, halo HP (+ dlast) on each side) x (segment of Sy rows, T
// halo rows on each side).  Iteration `it` lets row Y = ya + it enter; stage s (s = 0..T-1) then holds row Y-1-s at
// level s (E, G at step n0+s, H half a step earlier) in registers, receives row Y-s at level s from stage s-1 (from
// shared memory for s = 0), and produces level s+1 of its held row, which is what stage s+1 receives.  The last stage
// writes row Y-T at level T to the other field buffer.  Per stage a thread keeps E, Hx, Hy, G of the held row and one
// spare value for the y edges; the four coefficients of a row wait in a shared-memory ring (written once by cp.async,
// read by each stage in turn; every thread touches its own column only).  Between lanes new Hy and old E travel by
// shuffle; between warps old E and old Hy of the warp-edge columns are posted to shared memory at the end of an
// iteration (one CTA barrier per row).
template <typename R, int T>
__global__ void __launch_bounds__(StripThreads<R, T>::value, 1) k2_2d(const P2<R> p, const Arrays<R> a, const __grid_constant__ Maps2D maps) {
  constexpr int NT = StripThreads<R, T>::value;
  constexpr int NW = NT / 32;
  constexpr int FR = kRing;
  constexpr int XS = NW + 2;
  constexpr int XB = T * XS * 4;                              // one exchange buffer: [T][XS]{E31, Hy31, E0, -}, end slots zero
  extern __shared__ __align__(128) uint8_t smem_raw[];
  __shared__ __align__(8) uint64_t ring_bar[kRing];           // one mbarrier per ring slot
  R *fring = reinterpret_cast<R *>(smem_raw);                 // [FR][8][NT]
  R *xch = fring + FR * 8 * NT;                              // [2][XB]
  R *xsb = xch + 2 * XB;                                      // [T][NT]
  const uint32_t xch_addr = rketd::smem_u32(xch);
  const int tid = threadIdx.x;
  JobCtx<R> c;
  c.lane = tid & 31; c.warp = tid >> 5;
  c.is_mur = (p.bc == RKETD2D_BC_MUR);

  for (int q = tid; q < 2 * XB; q += NT) xch[q] = R(0);
  if (tid == 0) {
#pragma unroll
    for (int r = 0; r < FR; ++r) rketd::mbar_init(&ring_bar[r], 8);      // eight issuing lanes, one per array
    rketd::fence_barrier_init();
  }
  uint32_t rows_issued = 0, rows_taken = 0;                   // running counts over all jobs of this CTA: slot = count % FR,
                                                              // mbarrier phase parity = (count / FR) & 1
  const int njobs = p.nstrips * p.nsegs;
  for (int job = blockIdx.x; job < njobs; job += gridDim.x) {
    const int strip = job % p.nstrips, seg = job / p.nstrips;
    const int x0 = strip * p.Wv - p.HP - (strip == p.nstrips - 1 ? p.dlast : 0);
    const int i = x0 + tid;
    c.i = i;
    const bool incol = (i >= 0 && i < p.nx);
    c.own_col = incol && i >= strip * p.Wv && i < (strip + 1) * p.Wv;
    c.y_out0 = seg * p.Sy; c.y_out1 = min(p.ny, c.y_out0 + p.Sy);
    const int ya = c.y_out0 - T;
    const int niter = (c.y_out1 - c.y_out0) + 2 * T;          // rows ya .. y_out1-1+T enter
    c.chx_i = (i >= 0 && i <= p.nx - 2) ? p.chx : R(0);
    c.chx_im1 = (i >= 1 && i <= p.nx - 1 && c.warp > 0) ? p.chx : R(0);
    c.xl = (i == 0); c.xr = (i == p.nx - 1); c.xin = (i >= 1 && i <= p.nx - 2);
    const bool xw = __any_sync(0xffffffffu, c.xl || c.xr);
    c.src_col = (i == p.src_i);

    Held<R, T> hA, hB;
#pragma unroll
    for (int s = 0; s < T; ++s) hA.e[s] = hA.hx[s] = hA.hy[s] = hA.g[s] = hA.cP[s] = hA.cce[s] = hA.cka[s] = hA.cQ[s] = R(0);
    hA.hxp_last = R(0);
    uint32_t fq = 0;

    __syncthreads();                       // xch zeroed / the previous job is done with it

    const int nrows_job = (niter + 1) & ~1;                   // rows that enter (the iteration count is rounded up to even)
    // lane 0 of warp `arr` (arr = 0..7) brings in array `arr` of a row: eight lanes share the issue work
    const bool issuer = c.lane == 0 && c.warp < 8;
    auto issue_row = [&](int ridx) {       // ridx = row index relative to ya; issuing lanes only
      if (ridx >= nrows_job) return;
      const uint32_t slot = rows_issued % FR;
      ++rows_issued;
      rketd::mbar_expect_tx(&ring_bar[slot], (uint32_t)(NT * sizeof(R)));
      const uint32_t dst = rketd::smem_u32(fring + slot * 8 * NT + c.warp * NT);
#pragma unroll
      for (int h = 0; h < TmaBox<NT>::N; ++h)
        tma_load_2d(dst + (uint32_t)(h * TmaBox<NT>::W * sizeof(R)), &maps.m[c.warp], &ring_bar[slot], x0 + h * TmaBox<NT>::W, ya + ridx);
    };
    if (issuer) {
#pragma unroll
      for (int r = 0; r < kPF; ++r) issue_row(r);
    }

    constexpr uint32_t kHeldMask = ((1u << T) - 1u) << 1;     // bits of the rows the T stages hold
    // flag byte of the row entering next: loaded one iteration ahead and left untouched until then (no instruction waits on the load)
    uint32_t raw_next = p.rowflag[min(max(ya, 0), p.ny - 1)];

    auto iteration = [&](const int it, Held<R, T> &h, Held<R, T> &n) {
      const int Y = ya + it;
      const bool special = ((fq << 1) & kHeldMask) != 0;       // the flag of row Y is not among the held rows yet
      fq = (fq << 1) | ((Y >= 0 && Y < p.ny) ? (raw_next & (uint32_t)RF_SPECIAL) : 0u);
      raw_next = p.rowflag[min(max(Y + 1, 0), p.ny - 1)];
      __syncthreads();                     // the warp-edge values posted at the end of the previous iteration; and every
                                           // thread has read the ring slot of the previous iteration, which is refilled now
      if (issuer) issue_row(it + kPF);
      const uint32_t slot = rows_taken % FR;
      rketd::mbar_wait(&ring_bar[slot], (rows_taken / FR) & 1u);
      ++rows_taken;
      const R *fs = fring + slot * 8 * NT + tid;
      R ein = fs[0], hxin = fs[NT], hyin = fs[2 * NT], gin = fs[3 * NT];
      R cPin = fs[4 * NT], ccein = fs[5 * NT], ckain = fs[6 * NT], cQin = fs[7 * NT];
      R *xbuf = xch + ((it + 1) & 1) * XB;                     // read buffer of this iteration
      if (special)
        run_stages<R, T, true, true>(p, a, c, Y, fq, xbuf, xsb, h, n, ein, hxin, hyin, gin, cPin, ccein, ckain, cQin);
      else if (xw)
        run_stages<R, T, false, true>(p, a, c, Y, fq, xbuf, xsb, h, n, ein, hxin, hyin, gin, cPin, ccein, ckain, cQin);
      else
        run_stages<R, T, false, false>(p, a, c, Y, fq, xbuf, xsb, h, n, ein, hxin, hyin, gin, cPin, ccein, ckain, cQin);
      {                                    // (ein, hxin, hyin, gin) is now row Y-T at level T
        const int y = Y - T;
        if (c.own_col && y >= c.y_out0 && y < c.y_out1) {
          const int64_t idx = (int64_t)y * p.pitch + i;
          a.E2[idx] = ein; a.Hx2[idx] = hxin; a.Hy2[idx] = hyin; a.G2[idx] = gin;
        }
      }
      // warp-edge values for the next iteration: lane 31 posts {E, Hy}, lane 0 posts E, as predicated stores
      const uint32_t xpa = xch_addr + (uint32_t)(((it & 1) * XB + (c.warp + 1) * 4) * (int)sizeof(R));
      const bool l31 = c.lane == 31, l0 = c.lane == 0;
#pragma unroll
      for (int s = 0; s < T; ++s) {
        st_pair_if(l31, xpa + (uint32_t)(s * XS * 4 * (int)sizeof(R)), n.e[s], n.hy[s]);
        rketd::sts_if(l0, xpa + (uint32_t)((s * XS * 4 + 2) * (int)sizeof(R)), n.e[s]);
      }
    };

    // two register sets used alternately; an odd count runs one more iteration on a zero row, which stores nothing
    for (int it = 0; it < niter; it += 2) {
      iteration(it, hA, hB);
      iteration(it + 1, hB, hA);
    }
    __syncthreads();                       // every issued row of the job has been taken (nrows_job of each)
    for (int q = tid; q < 2 * XB; q += NT) xch[q] = R(0);
  }
}

// ------------------------------------------------------------------------------------------------ setup kernels
// media -> pitch layout (fp64) + the four kernel coefficients; padding columns get zeros
template <typename R>
__global__ void coef2d_kernel(int nx, int ny, int64_t pitch, const double *__restrict__ wp, const double *__restrict__ nu,
                              double dx, double dt, double eps0, double *wp_p, double *nu_p, R *cP, R *cce, R *cka, R *cQ,
                              int *bad, int npml) {
  const int64_t idx = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (idx >= pitch * ny) return;
  const int64_t j = idx / pitch, i = idx - j * pitch;
  double vP = 0, vce = 0, vka = 0, vQ = 0, w = 0, v = 0;
  if (i < nx) {
    w = wp[j * nx + i];
    v = nu[j * nx + i];
    if (!(w >= 0.0) || !(v >= 0.0) || isinf(w) || isinf(v)) atomicOr(bad, 1);
    if (npml > 0 && (i < npml || i > nx - 1 - npml || j < npml || j > ny - 1 - npml)) { w = 0.0; v = 0.0; }   // layer nodes are vacuum
    const rketd::Six s = rketd::six_coefficients(w, v, dx, dt, eps0, 0);
    const double kcp = __dmul_rn(s.cj, s.kc), kbp = __dmul_rn(s.cj, s.kb);
    vP = __dsub_rn(s.ca, kcp);
    vce = s.ch;
    vka = s.ka;
    vQ = __dadd_rn(__dmul_rn(s.ka, kcp), kbp);
  }
  wp_p[idx] = w; nu_p[idx] = v;
  cP[idx] = (R)vP; cce[idx] = (R)vce; cka[idx] = (R)vka; cQ[idx] = (R)vQ;
}

// G = cj J - cj kc E (in place on the array holding J), fp64 arithmetic, one rounding to R
template <typename R>
__global__ void j_to_g_kernel(int nx, int ny, int64_t pitch, const double *__restrict__ wp_p, const double *__restrict__ nu_p,
                              double dx, double dt, double eps0, const R *__restrict__ E, R *JG) {
  const int64_t idx = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (idx >= pitch * ny) return;
  const int64_t i = idx % pitch;
  double G = 0.0;
  if (i < nx) {
    const rketd::Six s = rketd::six_coefficients(wp_p[idx], nu_p[idx], dx, dt, eps0, 0);
    G = __fma_rn(-__dmul_rn(s.cj, s.kc), (double)E[idx], __dmul_rn(s.cj, (double)JG[idx]));
  }
  JG[idx] = (R)G;
}
// J = (G + cj kc E)/cj
template <typename R>
__global__ void g_to_j_kernel(int nx, int ny, int64_t pitch, const double *__restrict__ wp_p, const double *__restrict__ nu_p,
                              double dx, double dt, double eps0, const R *__restrict__ E, const R *__restrict__ G, R *J) {
  const int64_t idx = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (idx >= pitch * ny) return;
  const int64_t i = idx % pitch;
  double v = 0.0;
  if (i < nx) {
    const rketd::Six s = rketd::six_coefficients(wp_p[idx], nu_p[idx], dx, dt, eps0, 0);
    v = __ddiv_rn(__fma_rn(__dmul_rn(s.cj, s.kc), (double)E[idx], (double)G[idx]), s.cj);
  }
  J[idx] = (R)v;
}
template <typename R>
__global__ void unpack2d_kernel(int nx, int ny, int64_t pitch, const R *c0, const R *c1, const R *c2, const R *c3, double *out) {
  const int64_t idx = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  const int64_t n = (int64_t)nx * ny;
  if (idx >= n) return;
  const int64_t j = idx / nx, i = idx - j * nx, src = j * pitch + i;
  out[idx] = (double)c0[src]; out[n + idx] = (double)c1[src]; out[2 * n + idx] = (double)c2[src]; out[3 * n + idx] = (double)c3[src];
}

std::string g_create_error2;

struct Chunk2 { void *buf; int64_t nsteps; };

struct Plan2 { int HP, Wv, nstrips, nsegs, Sy, dlast; };

}  // namespace

struct rketd2d_sim {
  int nx = 0, ny = 0, dtype = 0, esize = 8;
  int64_t pitch = 0;
  double dx = 0, dy = 0, dt = 0;
  cudaStream_t stream = nullptr;
  void *fld[2][4] = {{nullptr, nullptr, nullptr, nullptr}, {nullptr, nullptr, nullptr, nullptr}};   // E, Hx, Hy, G
  int cur = 0;
  void *coef[4] = {nullptr, nullptr, nullptr, nullptr};                                              // P, ce, ka, Q
  double *wp_p = nullptr, *nu_p = nullptr;
  uint8_t *rowflag = nullptr;
  int *d_bad = nullptr;
  bool flags_dirty = true, have_media = false, fields_zero = true, third_is_J = false;
  int bc = RKETD2D_BC_MUR, bc_next = RKETD2D_BC_MUR;
  // the paper's layer (rketd2d_set_boundary_pml): requested parameters; `pml_live` = the live coefficients were derived
  // with it (layer nodes vacuum); split parts Ezx, Ezy (ping-pong) and the eight per-axis tables, allocated on first use
  int pml_npml = 0, pml_live = 0;
  double pml_m = 3.0, pml_R0 = 1e-6;
  void *split[2][2] = {{nullptr, nullptr}, {nullptr, nullptr}};
  void *tabs = nullptr;
  int src_kind = RKETD_SRC_NONE;
  std::vector<double> src_params;
  int src_i = -1, src_j = -1;
  std::vector<int> probe_i, probe_j;
  std::vector<Chunk2> chunks;
  int64_t nsamples = 0, step = 0;
  int plan_kernel = RKETD2D_KERNEL_AUTO, plan_depth = 0;
  int num_sms = 148;
  int64_t ctr_launches = 0, ctr_step_launches = 0, ctr_kernel_used = 0, ctr_depth_used = 0, ctr_strip = 0, ctr_halo = 0,
          ctr_seg = 0, state_bytes = 0;
  std::string err;
};

namespace {

int fail2(rketd2d_sim *s, int code, const std::string &msg) {
  if (s) s->err = msg; else g_create_error2 = msg;
  return code;
}
#define CU_TRY2(s, expr)                                                                         \
  do {                                                                                           \
    cudaError_t e__ = (expr);                                                                    \
    if (e__ != cudaSuccess)                                                                      \
      return fail2(s, e__ == cudaErrorMemoryAllocation ? RKETD_ENOMEM : RKETD_ECUDA,             \
                   std::string(#expr) + ": " + cudaGetErrorString(e__));                         \
  } while (0)

size_t arr_bytes2(const rketd2d_sim *s) { return (size_t)s->pitch * s->ny * s->esize; }
unsigned blocks_for(int64_t n) { return (unsigned)((n + 255) / 256); }

cudaError_t copy_in2(const rketd2d_sim *s, void *dst, const void *src, size_t es) {
  return cudaMemcpy2DAsync(dst, (size_t)s->pitch * es, src, (size_t)s->nx * es, (size_t)s->nx * es, (size_t)s->ny,
                           cudaMemcpyDefault, s->stream);
}
cudaError_t copy_out2(const rketd2d_sim *s, void *dst, const void *src, size_t es) {
  return cudaMemcpy2DAsync(dst, (size_t)s->nx * es, src, (size_t)s->pitch * es, (size_t)s->nx * es, (size_t)s->ny,
                           cudaMemcpyDefault, s->stream);
}

void discard_records2(rketd2d_sim *s) {
  for (auto &c : s->chunks) cudaFree(c.buf);
  s->chunks.clear();
  s->nsamples = 0;
}

double source_sample2(const rketd2d_sim *s, int64_t step_index) {
  if (s->src_kind == RKETD_SRC_GAUSS_DERIV) {
    const double tau = s->src_params[0], t0 = s->src_params[1], A = s->src_params[2];
    const double t = double(step_index + 1) * s->dt;
    const double u = (t - t0) / tau;
    return A * u * std::exp(0.5 - 0.5 * u * u);
  }
  if (s->src_kind == RKETD_SRC_TABLE)
    return (step_index >= 0 && step_index < (int64_t)s->src_params.size()) ? s->src_params[(size_t)step_index] : 0.0;
  return 0.0;
}

int build_rowflags(rketd2d_sim *s) {
  std::vector<uint8_t> rf((size_t)s->ny, 0);
  rf[0] |= RF_SPECIAL; rf[1] |= RF_SPECIAL; rf[(size_t)s->ny - 2] |= RF_SPECIAL; rf[(size_t)s->ny - 1] |= RF_SPECIAL;
  if (s->src_kind != RKETD_SRC_NONE && s->src_j >= 0) {
    rf[(size_t)s->src_j] |= RF_SPECIAL;
    if (s->src_j == 0) rf[1] |= RF_SPECIAL;
  }
  for (size_t q = 0; q < s->probe_j.size(); ++q) rf[(size_t)s->probe_j[q]] |= RF_SPECIAL | RF_PROBE;
  CU_TRY2(s, cudaMemcpyAsync(s->rowflag, rf.data(), rf.size(), cudaMemcpyHostToDevice, s->stream));
  CU_TRY2(s, cudaStreamSynchronize(s->stream));      // rf is a local
  s->flags_dirty = false;
  return RKETD_OK;
}

typedef CUresult (*EncodeTiled2)(CUtensorMap *, CUtensorMapDataType, cuuint32_t, void *, const cuuint64_t *, const cuuint64_t *,
                                 const cuuint32_t *, const cuuint32_t *, CUtensorMapInterleave, CUtensorMapSwizzle,
                                 CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
// 2-D views {nx, ny} (row pitch = s->pitch elements) of the eight arrays the streaming kernel reads from the current
// buffer, box {boxw, 1}, no swizzle; out-of-range elements read as zero
int build_maps2d(rketd2d_sim *s, int boxw, Maps2D *out) {
  static EncodeTiled2 enc = nullptr;
  if (!enc) {
    void *fn = nullptr;
    cudaDriverEntryPointQueryResult q;
    if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &q) != cudaSuccess || q != cudaDriverEntryPointSuccess)
      return fail2(s, RKETD_ECUDA, "cuTensorMapEncodeTiled not available from the driver");
    enc = (EncodeTiled2)fn;
  }
  void *base[8] = {s->fld[s->cur][0], s->fld[s->cur][1], s->fld[s->cur][2], s->fld[s->cur][3], s->coef[0], s->coef[1], s->coef[2], s->coef[3]};
  for (int a = 0; a < 8; ++a) {
    cuuint64_t dims[2] = {(cuuint64_t)s->nx, (cuuint64_t)s->ny};
    cuuint64_t strides[1] = {(cuuint64_t)s->pitch * (cuuint64_t)s->esize};
    cuuint32_t box[2] = {(cuuint32_t)boxw, 1u}, estr[2] = {1u, 1u};
    const CUresult r = enc(&out->m[a], s->esize == 8 ? CU_TENSOR_MAP_DATA_TYPE_FLOAT64 : CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 2, base[a], dims,
                           strides, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
                           CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    if (r != CUDA_SUCCESS) return fail2(s, RKETD_ECUDA, "cuTensorMapEncodeTiled failed: " + std::to_string((int)r));
  }
  return RKETD_OK;
}

// strips and segments of the streaming kernel for depth T
Plan2 make_plan(const rketd2d_sim *s, int T, int NT) {
  Plan2 pl;
  pl.HP = std::max(8, (T + 7) / 8 * 8);
  pl.Wv = NT - 2 * pl.HP;
  while ((s->nx % pl.Wv) == 1 && pl.Wv > 16) pl.Wv -= 8;      // the last strip owns at least two columns (x Mur)
  pl.nstrips = (s->nx + pl.Wv - 1) / pl.Wv;
  const int x0_last = (pl.nstrips - 1) * pl.Wv - pl.HP;
  pl.dlast = (((s->nx - 1 - x0_last) % 32) == 0) ? 8 : 0;      // column nx-1 must not be lane 0 of its warp
  // segments: fewest iterations per SM, whole waves; first and last segment own at least two rows
  double best = 1e300;
  pl.nsegs = 1; pl.Sy = s->ny;
  const int max_segs = std::max(1, std::min(s->ny / 2, 4096));
  for (int ns = 1; ns <= max_segs; ++ns) {
    const int Sy = (s->ny + ns - 1) / ns;
    const int nsr = (s->ny + Sy - 1) / Sy;
    if (Sy < 2 || s->ny - (nsr - 1) * Sy < 2) continue;
    const int64_t jobs = (int64_t)pl.nstrips * nsr;
    const double cost = (double)((jobs + s->num_sms - 1) / s->num_sms) * (Sy + 2 * T + 8);
    if (cost < best - 1e-9) { best = cost; pl.nsegs = nsr; pl.Sy = Sy; }
  }
  return pl;
}

template <typename R>
void fill_params(const rketd2d_sim *s, P2<R> &p, void *rec, int64_t rec_stride, int64_t n0, int nlev) {
  p.nx = s->nx; p.ny = s->ny; p.pitch = s->pitch;
  p.chx = (R)(s->dt / (kMu0 * s->dx));
  p.nchy = (R)(-(s->dt / (kMu0 * s->dy)));
  p.chy = -p.nchy;
  p.nr = (R)(-(s->dx / s->dy));
  p.c2 = (R)((s->dx / s->dy) * (s->dt / (kMu0 * s->dy)));
  const double Sx = kC0 * s->dt / s->dx, Sy = kC0 * s->dt / s->dy;
  p.mx = (R)((Sx - 1.0) / (Sx + 1.0));
  p.my = (R)((Sy - 1.0) / (Sy + 1.0));
  p.bc = s->bc;
  const bool has_src = s->src_kind != RKETD_SRC_NONE;
  p.src_i = has_src ? s->src_i : -1;
  p.src_j = has_src ? s->src_j : -1;
  p.nprobes = (int)s->probe_i.size();
  for (int q = 0; q < p.nprobes; ++q) { p.probe_i[q] = s->probe_i[(size_t)q]; p.probe_j[q] = s->probe_j[(size_t)q]; }
  p.rec = (R *)rec; p.rec_stride = rec_stride; p.n0 = n0;
  for (int l = 0; l < kMaxT; ++l) p.src[l] = (l < nlev && has_src) ? (R)source_sample2(s, s->step + l) : R(0);
  p.rowflag = s->rowflag;
  p.HP = p.Wv = p.nstrips = p.nsegs = p.Sy = p.dlast = 0;
}

template <typename R>
Arrays<R> arrays_of(const rketd2d_sim *s) {
  Arrays<R> a;
  const int c = s->cur, d = 1 - s->cur;
  a.E = (const R *)s->fld[c][0]; a.Hx = (const R *)s->fld[c][1]; a.Hy = (const R *)s->fld[c][2]; a.G = (const R *)s->fld[c][3];
  a.cP = (const R *)s->coef[0]; a.cce = (const R *)s->coef[1]; a.cka = (const R *)s->coef[2]; a.cQ = (const R *)s->coef[3];
  a.E2 = (R *)s->fld[d][0]; a.Hx2 = (R *)s->fld[d][1]; a.Hy2 = (R *)s->fld[d][2]; a.G2 = (R *)s->fld[d][3];
  return a;
}

template <typename R, int T>
cudaError_t launch_k2_T(rketd2d_sim *s, P2<R> &p) {
  constexpr int NT = StripThreads<R, T>::value;
  const Plan2 pl = make_plan(s, T, NT);
  p.HP = pl.HP; p.Wv = pl.Wv; p.nstrips = pl.nstrips; p.nsegs = pl.nsegs; p.Sy = pl.Sy; p.dlast = pl.dlast;
  if (T == s->ctr_depth_used || s->ctr_strip == 0) { s->ctr_strip = NT; s->ctr_halo = pl.HP; s->ctr_seg = pl.Sy; }   // the main passes, not a remainder pass
  constexpr size_t smem = K2Shape<R, T>::smem;
  static unsigned long long configured = 0ull;      // bit = device id: the attribute is per device and context
  int dev = 0;
  cudaGetDevice(&dev);
  if (dev >= 64 || !((configured >> dev) & 1ull)) {
    cudaError_t e = cudaFuncSetAttribute(k2_2d<R, T>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    if (dev < 64) configured |= 1ull << dev;
  }
  const int grid = pl.nstrips * pl.nsegs;
  Maps2D maps;
  { const int rc = build_maps2d(s, TmaBox<NT>::W, &maps); if (rc) return cudaErrorInvalidValue; }
  k2_2d<R, T><<<grid, NT, smem, s->stream>>>(p, arrays_of<R>(s), maps);
  return cudaGetLastError();
}

template <typename R>
cudaError_t launch_k2(rketd2d_sim *s, P2<R> &p, int T) {
  switch (T) {
    case 1: return launch_k2_T<R, 1>(s, p);
    case 2: return launch_k2_T<R, 2>(s, p);
    case 4: return launch_k2_T<R, 4>(s, p);
    case 6: return launch_k2_T<R, 6>(s, p);
    case 8: return launch_k2_T<R, 8>(s, p);
    case 16: if (sizeof(R) == 4) return launch_k2_T<float, 16>(s, reinterpret_cast<P2<float> &>(p)); break;
  }
  return cudaErrorInvalidValue;
}

template <typename R>
int run_typed(rketd2d_sim *s, int64_t nsteps, void *rec) {
  const bool pml = s->bc == RKETD2D_BC_PML;
  const bool stream_kernel = s->plan_kernel != RKETD2D_KERNEL_STEP && !pml;      // the layer runs in the one-step kernel
  const int Tdef = s->plan_depth > 0 ? s->plan_depth : 8;
  s->ctr_kernel_used = stream_kernel ? RKETD2D_KERNEL_STREAM : RKETD2D_KERNEL_STEP;
  s->ctr_depth_used = stream_kernel ? Tdef : 1;
  int64_t done = 0;
  while (done < nsteps) {
    int T = 1;
    if (stream_kernel) {
      const int depths[6] = {16, 8, 6, 4, 2, 1};       // the chosen depth, then what fits the remainder
      for (int q = 0; q < 6; ++q) {
        T = depths[q];
        if (T <= Tdef && (int64_t)T <= nsteps - done && (T != 6 || Tdef == 6)) break;
      }
    }
    P2<R> p;
    fill_params<R>(s, p, rec, nsteps, done, T);
    if (stream_kernel) {
      CU_TRY2(s, launch_k2<R>(s, p, T));
    } else {
      dim3 grid((unsigned)((s->nx + 127) / 128), (unsigned)((s->ny + kK1Rows - 1) / kK1Rows));
      if (pml) {
        PmlTabs<R> t;
        const R *tb = (const R *)s->tabs;
        t.hax = tb; t.hbx = tb + s->nx; t.eax = tb + 2 * s->nx; t.ebx = tb + 3 * s->nx;
        const R *ty = tb + 4 * (int64_t)s->nx;
        t.hay = ty; t.hby = ty + s->ny; t.eay = ty + 2 * s->ny; t.eby = ty + 3 * s->ny;
        t.Ezx = (const R *)s->split[s->cur][0]; t.Ezy = (const R *)s->split[s->cur][1];
        t.Ezx2 = (R *)s->split[1 - s->cur][0]; t.Ezy2 = (R *)s->split[1 - s->cur][1];
        t.npml = s->pml_live;
        k1_2d_pml<R><<<grid, 128, 0, s->stream>>>(p, arrays_of<R>(s), t);
      } else {
        k1_2d<R><<<grid, 128, 0, s->stream>>>(p, arrays_of<R>(s));
      }
      CU_TRY2(s, cudaGetLastError());
    }
    s->cur = 1 - s->cur;
    s->step += T;
    done += T;
    s->ctr_launches++; s->ctr_step_launches++;
  }
  return RKETD_OK;
}

// the array holding G (or J before the first media) <-> J
template <typename R>
int convert_current(rketd2d_sim *s, bool to_G, void *dstJ) {
  const int64_t n = s->pitch * s->ny;
  if (to_G)
    j_to_g_kernel<R><<<blocks_for(n), 256, 0, s->stream>>>(s->nx, s->ny, s->pitch, s->wp_p, s->nu_p, s->dx, s->dt, kEps0,
                                                           (const R *)s->fld[s->cur][0], (R *)s->fld[s->cur][3]);
  else
    g_to_j_kernel<R><<<blocks_for(n), 256, 0, s->stream>>>(s->nx, s->ny, s->pitch, s->wp_p, s->nu_p, s->dx, s->dt, kEps0,
                                                           (const R *)s->fld[s->cur][0], (const R *)s->fld[s->cur][3], (R *)dstJ);
  CU_TRY2(s, cudaGetLastError());
  s->ctr_launches++;
  return RKETD_OK;
}
int convert_current_any(rketd2d_sim *s, bool to_G, void *dstJ) {
  return s->dtype == RKETD_F64 ? convert_current<double>(s, to_G, dstJ) : convert_current<float>(s, to_G, dstJ);
}

// split parts (allocated once) and the eight per-axis tables of the layer, in the handle's dtype:
// tabs = [hax, hbx, eax, ebx](nx each) then [hay, hby, eay, eby](ny each); 1 / the plain coefficient outside the layers
int prepare_pml(rketd2d_sim *s, int npml) {
  for (int b = 0; b < 2; ++b)
    for (int c = 0; c < 2; ++c)
      if (!s->split[b][c]) {
        CU_TRY2(s, cudaMalloc(&s->split[b][c], arr_bytes2(s)));
        CU_TRY2(s, cudaMemsetAsync(s->split[b][c], 0, arr_bytes2(s), s->stream));
        s->state_bytes += (int64_t)arr_bytes2(s);
      }
  const size_t nt = (size_t)4 * s->nx + (size_t)4 * s->ny;
  if (!s->tabs) CU_TRY2(s, cudaMalloc(&s->tabs, nt * s->esize));
  std::vector<double> t(nt);
  auto fill = [&](double *base, int N, double d) {
    double *ha = base, *hb = base + N, *ea = base + 2 * N, *eb = base + 3 * N;
    for (int k = 0; k < N; ++k) { ha[k] = 1.0; hb[k] = s->dt / (kMu0 * d); ea[k] = 1.0; eb[k] = s->dt / (kEps0 * d); }
    const double smax = -(s->pml_m + 1.0) * kEps0 * kC0 * std::log(s->pml_R0) / (2.0 * (double)npml * d);
    for (int j = 0; j < npml; ++j) {
      const double se = smax * std::pow((double)(npml - j) / npml, s->pml_m) * s->dt / (2.0 * kEps0);
      const double sh = smax * std::pow(((double)(npml - j) - 0.5) / npml, s->pml_m) * s->dt / (2.0 * kEps0);
      ea[j] = ea[N - 1 - j] = (1.0 - se) / (1.0 + se);
      eb[j] = eb[N - 1 - j] = (s->dt / (kEps0 * d)) / (1.0 + se);
      ha[j] = ha[N - 2 - j] = (1.0 - sh) / (1.0 + sh);
      hb[j] = hb[N - 2 - j] = (s->dt / (kMu0 * d)) / (1.0 + sh);
    }
  };
  fill(t.data(), s->nx, s->dx);
  fill(t.data() + 4 * (size_t)s->nx, s->ny, s->dy);
  if (s->dtype == RKETD_F64) {
    CU_TRY2(s, cudaMemcpyAsync(s->tabs, t.data(), nt * 8, cudaMemcpyHostToDevice, s->stream));
  } else {
    std::vector<float> tf(t.begin(), t.end());
    CU_TRY2(s, cudaMemcpyAsync(s->tabs, tf.data(), nt * 4, cudaMemcpyHostToDevice, s->stream));
  }
  CU_TRY2(s, cudaStreamSynchronize(s->stream));      // t is a local
  return RKETD_OK;
}

}  // namespace

extern "C" {

int rketd2d_create(rketd2d_sim **out, int64_t nx, int64_t ny, double dx, double dy, double dt, int dtype, void *cuda_stream) {
  if (!out) return fail2(nullptr, RKETD_EINVAL, "out is NULL");
  *out = nullptr;
  if (nx < 3 || ny < 3 || nx > (1 << 30) || ny > (1 << 30)) return fail2(nullptr, RKETD_EINVAL, "nx, ny must be in 3..2^30");
  if (!(dx > 0) || !(dy > 0) || !(dt > 0)) return fail2(nullptr, RKETD_EINVAL, "dx, dy, dt must be positive");
  if (kC0 * dt * std::sqrt(1.0 / (dx * dx) + 1.0 / (dy * dy)) > 1.0 + 1e-12)
    return fail2(nullptr, RKETD_EINVAL, "c dt sqrt(1/dx^2 + 1/dy^2) > 1: unstable");
  if (dtype != RKETD_F64 && dtype != RKETD_F32) return fail2(nullptr, RKETD_EINVAL, "unknown dtype");
  int ndev = 0;
  if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev < 1) {
    cudaGetLastError();
    return fail2(nullptr, RKETD_ECUDA, "no usable CUDA device; librketd has no CPU fallback");
  }
  rketd2d_sim *s = new rketd2d_sim();
  s->nx = (int)nx; s->ny = (int)ny; s->dx = dx; s->dy = dy; s->dt = dt; s->dtype = dtype;
  s->esize = dtype == RKETD_F64 ? 8 : 4;
  s->pitch = (nx + 31) / 32 * 32;
  s->stream = (cudaStream_t)cuda_stream;
  int dev = 0;
  cudaGetDevice(&dev);
  cudaDeviceGetAttribute(&s->num_sms, cudaDevAttrMultiProcessorCount, dev);
  const size_t ab = arr_bytes2(s);
  auto alloc = [&](void **p, size_t bytes) {
    cudaError_t e = cudaMalloc(p, bytes);
    if (e == cudaSuccess) { e = cudaMemsetAsync(*p, 0, bytes, s->stream); s->state_bytes += (int64_t)bytes; }
    return e;
  };
  cudaError_t e = cudaSuccess;
  for (int b = 0; b < 2 && e == cudaSuccess; ++b)
    for (int f = 0; f < 4 && e == cudaSuccess; ++f) e = alloc(&s->fld[b][f], ab);
  for (int c = 0; c < 4 && e == cudaSuccess; ++c) e = alloc(&s->coef[c], ab);
  if (e == cudaSuccess) e = alloc((void **)&s->wp_p, (size_t)s->pitch * s->ny * 8);
  if (e == cudaSuccess) e = alloc((void **)&s->nu_p, (size_t)s->pitch * s->ny * 8);
  if (e == cudaSuccess) e = alloc((void **)&s->rowflag, (size_t)s->ny);
  if (e == cudaSuccess) e = alloc((void **)&s->d_bad, sizeof(int));
  if (e != cudaSuccess) {
    const int code = e == cudaErrorMemoryAllocation ? RKETD_ENOMEM : RKETD_ECUDA;
    const std::string msg = std::string("device allocation: ") + cudaGetErrorString(e);
    cudaGetLastError();
    rketd2d_destroy(s);
    return fail2(nullptr, code, msg);
  }
  *out = s;
  return RKETD_OK;
}

int rketd2d_set_media(rketd2d_sim *s, const double *wp, const double *nu) {
  if (!s) return RKETD_EINVAL;
  if (!wp || !nu) return fail2(s, RKETD_EINVAL, "wp and nu must not be NULL");
  const int64_t n = s->pitch * s->ny, nu_n = (int64_t)s->nx * s->ny;
  double *d_wp = nullptr, *d_nu = nullptr;      // user layout on the device
  CU_TRY2(s, cudaMalloc((void **)&d_wp, (size_t)nu_n * 8));
  cudaError_t e = cudaMalloc((void **)&d_nu, (size_t)nu_n * 8);
  if (e != cudaSuccess) { cudaFree(d_wp); CU_TRY2(s, e); }
  e = cudaMemcpyAsync(d_wp, wp, (size_t)nu_n * 8, cudaMemcpyDefault, s->stream);
  if (e == cudaSuccess) e = cudaMemcpyAsync(d_nu, nu, (size_t)nu_n * 8, cudaMemcpyDefault, s->stream);
  // read-only validation first: a rejected call leaves coefficients, media and fields exactly as they were
  int bad = 0;
  if (e == cudaSuccess) e = cudaMemsetAsync(s->d_bad, 0, sizeof(int), s->stream);
  if (e == cudaSuccess) e = rketd::launch_validate_media(d_wp, d_nu, nu_n, s->d_bad, s->stream);
  if (e == cudaSuccess) { s->ctr_launches++; e = cudaMemcpyAsync(&bad, s->d_bad, sizeof(int), cudaMemcpyDeviceToHost, s->stream); }
  if (e == cudaSuccess) e = cudaStreamSynchronize(s->stream);
  if (e != cudaSuccess || bad) {
    cudaFree(d_wp); cudaFree(d_nu);
    CU_TRY2(s, e);
    return fail2(s, RKETD_EINVAL, "wp and nu must be finite and non-negative");
  }
  // live fields under the old media: back to J first (in place), and third_is_J says so at once, so that a CUDA
  // failure further down leaves array and flag in agreement
  const bool live = s->have_media && !s->fields_zero && !s->third_is_J;
  if (live) {
    const int rc = convert_current_any(s, false, s->fld[s->cur][3]);
    if (rc) { cudaFree(d_wp); cudaFree(d_nu); return rc; }
    s->third_is_J = true;
  }
  const int npml_new = s->pml_npml;
  if (npml_new > 0) {                              // the paper's layer: split parts and per-axis tables
    const int rc = prepare_pml(s, npml_new);
    if (rc) { cudaFree(d_wp); cudaFree(d_nu); return rc; }
  }
  s->have_media = false;      // until the new coefficients are in place
  if (s->dtype == RKETD_F64)
    coef2d_kernel<double><<<blocks_for(n), 256, 0, s->stream>>>(s->nx, s->ny, s->pitch, d_wp, d_nu, s->dx, s->dt, kEps0, s->wp_p,
                                                                s->nu_p, (double *)s->coef[0], (double *)s->coef[1],
                                                                (double *)s->coef[2], (double *)s->coef[3], s->d_bad, npml_new);
  else
    coef2d_kernel<float><<<blocks_for(n), 256, 0, s->stream>>>(s->nx, s->ny, s->pitch, d_wp, d_nu, s->dx, s->dt, kEps0, s->wp_p,
                                                               s->nu_p, (float *)s->coef[0], (float *)s->coef[1],
                                                               (float *)s->coef[2], (float *)s->coef[3], s->d_bad, npml_new);
  e = cudaGetLastError();
  s->ctr_launches++;
  if (e == cudaSuccess) e = cudaStreamSynchronize(s->stream);
  cudaFree(d_wp); cudaFree(d_nu);
  CU_TRY2(s, e);
  s->have_media = true;
  if (npml_new > 0 && s->pml_live == 0) {          // entering the layer with live fields: Ez starts as its x part
    CU_TRY2(s, cudaMemcpyAsync(s->split[s->cur][0], s->fld[s->cur][0], arr_bytes2(s), cudaMemcpyDeviceToDevice, s->stream));
    CU_TRY2(s, cudaMemsetAsync(s->split[s->cur][1], 0, arr_bytes2(s), s->stream));
  }
  s->pml_live = npml_new;
  s->bc = npml_new > 0 ? RKETD2D_BC_PML : s->bc_next;
  if (s->third_is_J) { const int rc = convert_current_any(s, true, nullptr); if (rc) return rc; }
  s->third_is_J = false;
  CU_TRY2(s, cudaStreamSynchronize(s->stream));
  return RKETD_OK;
}

int rketd2d_set_boundary(rketd2d_sim *s, int kind) {
  if (!s) return RKETD_EINVAL;
  if (kind != RKETD2D_BC_MUR && kind != RKETD2D_BC_PEC) return fail2(s, RKETD_EINVAL, "unknown boundary kind (the layer: rketd2d_set_boundary_pml)");
  if (s->pml_live > 0) { s->pml_npml = 0; s->bc_next = kind; return RKETD_OK; }      // leaves the layer at the next rketd2d_set_media
  s->pml_npml = 0;
  s->bc = s->bc_next = kind;
  return RKETD_OK;
}

int rketd2d_set_boundary_pml(rketd2d_sim *s, int npml, double grading, double R0) {
  if (!s) return RKETD_EINVAL;
  if (npml < 1 || npml > 64 || 2 * (int64_t)npml + 1 > s->nx || 2 * (int64_t)npml + 1 > s->ny || !(R0 > 0.0) || R0 > 1.0 || !(grading >= 0.0))
    return fail2(s, RKETD_EINVAL, "need 1 <= npml <= 64, 2 npml + 1 <= nx, ny, 0 < R0 <= 1, grading >= 0");
  s->pml_npml = npml; s->pml_m = grading; s->pml_R0 = R0;
  return RKETD_OK;
}

int rketd2d_set_source(rketd2d_sim *s, int kind, const double *params, int64_t nparams, int64_t i, int64_t j) {
  if (!s) return RKETD_EINVAL;
  if (kind == RKETD_SRC_NONE) { s->src_kind = kind; s->src_i = s->src_j = -1; s->flags_dirty = true; return RKETD_OK; }
  if (kind != RKETD_SRC_GAUSS_DERIV && kind != RKETD_SRC_TABLE) return fail2(s, RKETD_EINVAL, "unknown source kind");
  if (i < 0 || i >= s->nx || j < 0 || j >= s->ny) return fail2(s, RKETD_EINVAL, "source node outside the grid");
  if (kind == RKETD_SRC_GAUSS_DERIV && (nparams != 3 || !params || !(params[0] > 0)))
    return fail2(s, RKETD_EINVAL, "GAUSS_DERIV needs params = {tau > 0, t0, amplitude}");
  if (kind == RKETD_SRC_TABLE && (nparams < 0 || (nparams > 0 && !params))) return fail2(s, RKETD_EINVAL, "bad table");
  s->src_kind = kind;
  s->src_params.assign(params, params + nparams);
  s->src_i = (int)i; s->src_j = (int)j;
  s->flags_dirty = true;
  return RKETD_OK;
}

int rketd2d_set_probes(rketd2d_sim *s, const int64_t *ij, int nprobes) {
  if (!s) return RKETD_EINVAL;
  if (nprobes < 0 || nprobes > kMaxProbes2 || (nprobes > 0 && !ij)) return fail2(s, RKETD_EINVAL, "0..64 probes");
  for (int q = 0; q < nprobes; ++q)
    if (ij[2 * q] < 0 || ij[2 * q] >= s->nx || ij[2 * q + 1] < 0 || ij[2 * q + 1] >= s->ny)
      return fail2(s, RKETD_EINVAL, "probe node outside the grid");
  CU_TRY2(s, cudaStreamSynchronize(s->stream));
  discard_records2(s);
  s->probe_i.clear(); s->probe_j.clear();
  for (int q = 0; q < nprobes; ++q) { s->probe_i.push_back((int)ij[2 * q]); s->probe_j.push_back((int)ij[2 * q + 1]); }
  s->flags_dirty = true;
  return RKETD_OK;
}

int rketd2d_set_fields(rketd2d_sim *s, const void *Ez, const void *Hx, const void *Hy, const void *Jz) {
  if (!s) return RKETD_EINVAL;
  const void *src[4] = {Ez, Hx, Hy, Jz};
  for (int f = 0; f < 4; ++f) {
    if (src[f]) CU_TRY2(s, copy_in2(s, s->fld[s->cur][f], src[f], (size_t)s->esize));
    else CU_TRY2(s, cudaMemsetAsync(s->fld[s->cur][f], 0, arr_bytes2(s), s->stream));
  }
  s->fields_zero = !Ez && !Hx && !Hy && !Jz;
  if (s->split[0][0]) {                            // the layer's split parts restart from Ezx = Ez, Ezy = 0
    CU_TRY2(s, cudaMemcpyAsync(s->split[s->cur][0], s->fld[s->cur][0], arr_bytes2(s), cudaMemcpyDeviceToDevice, s->stream));
    CU_TRY2(s, cudaMemsetAsync(s->split[s->cur][1], 0, arr_bytes2(s), s->stream));
  }
  if (s->have_media) { const int rc = convert_current_any(s, true, nullptr); if (rc) return rc; s->third_is_J = false; }
  else s->third_is_J = true;
  CU_TRY2(s, cudaStreamSynchronize(s->stream));
  return RKETD_OK;
}

int rketd2d_get_fields(rketd2d_sim *s, void *Ez, void *Hx, void *Hy, void *Jz) {
  if (!s) return RKETD_EINVAL;
  void *dst[3] = {Ez, Hx, Hy};
  for (int f = 0; f < 3; ++f)
    if (dst[f]) CU_TRY2(s, copy_out2(s, dst[f], s->fld[s->cur][f], (size_t)s->esize));
  if (Jz) {
    const void *srcJ = s->fld[s->cur][3];
    if (s->have_media && !s->third_is_J) {       // the other buffer's G array is scratch between runs
      const int rc = convert_current_any(s, false, s->fld[1 - s->cur][3]);
      if (rc) return rc;
      srcJ = s->fld[1 - s->cur][3];
    }
    CU_TRY2(s, copy_out2(s, Jz, srcJ, (size_t)s->esize));
  }
  CU_TRY2(s, cudaStreamSynchronize(s->stream));
  return RKETD_OK;
}

int rketd2d_reset(rketd2d_sim *s) {
  if (!s) return RKETD_EINVAL;
  CU_TRY2(s, cudaStreamSynchronize(s->stream));
  for (int f = 0; f < 4; ++f) CU_TRY2(s, cudaMemsetAsync(s->fld[s->cur][f], 0, arr_bytes2(s), s->stream));
  for (int c = 0; c < 2; ++c)
    if (s->split[s->cur][c]) CU_TRY2(s, cudaMemsetAsync(s->split[s->cur][c], 0, arr_bytes2(s), s->stream));
  discard_records2(s);
  s->step = 0;
  s->fields_zero = true;
  s->third_is_J = false;
  return RKETD_OK;
}

int rketd2d_discard_records(rketd2d_sim *s) {
  if (!s) return RKETD_EINVAL;
  CU_TRY2(s, cudaStreamSynchronize(s->stream));
  discard_records2(s);
  return RKETD_OK;
}

int rketd2d_set_plan(rketd2d_sim *s, int kernel, int depth) {
  if (!s) return RKETD_EINVAL;
  if (kernel < RKETD2D_KERNEL_AUTO || kernel > RKETD2D_KERNEL_STREAM) return fail2(s, RKETD_EINVAL, "unknown kernel");
  if (depth != 0 && depth != 1 && depth != 2 && depth != 4 && depth != 6 && depth != 8 && depth != 16)
    return fail2(s, RKETD_EINVAL, "depth must be 0, 1, 2, 4, 6, 8 or 16");
  if (depth == 16 && s->dtype == RKETD_F64) return fail2(s, RKETD_EINVAL, "depth 16 is for fp32 (registers and shared memory)");
  s->plan_kernel = kernel;
  s->plan_depth = depth;
  return RKETD_OK;
}

int rketd2d_run(rketd2d_sim *s, int64_t nsteps) {
  if (!s) return RKETD_EINVAL;
  if (nsteps < 0) return fail2(s, RKETD_EINVAL, "nsteps < 0");
  if (!s->have_media) return fail2(s, RKETD_ESTATE, "rketd2d_run before rketd2d_set_media");
  if (nsteps == 0) return RKETD_OK;
  if (s->flags_dirty) { const int rc = build_rowflags(s); if (rc) return rc; }
  void *rec = nullptr;
  if (!s->probe_i.empty()) {
    CU_TRY2(s, cudaMalloc(&rec, (size_t)s->probe_i.size() * (size_t)nsteps * s->esize));
  }
  s->fields_zero = false;
  const int rc = s->dtype == RKETD_F64 ? run_typed<double>(s, nsteps, rec) : run_typed<float>(s, nsteps, rec);
  if (rc) {               // a failed run records nothing: the chunk list and nsamples stay in step
    if (rec) { cudaStreamSynchronize(s->stream); cudaFree(rec); cudaGetLastError(); }
    return rc;
  }
  if (rec) s->chunks.push_back({rec, nsteps});
  s->nsamples += s->probe_i.empty() ? 0 : nsteps;
  return RKETD_OK;
}

int rketd2d_read_probes(rketd2d_sim *s, void *out, int64_t out_bytes, int64_t *nsamples) {
  if (!s) return RKETD_EINVAL;
  CU_TRY2(s, cudaStreamSynchronize(s->stream));
  if (nsamples) *nsamples = s->nsamples;
  if (!out) return RKETD_OK;
  const int64_t np = (int64_t)s->probe_i.size();
  if (out_bytes < np * s->nsamples * s->esize) return fail2(s, RKETD_EINVAL, "out_bytes too small");
  int64_t off = 0;
  for (auto &c : s->chunks) {
    CU_TRY2(s, cudaMemcpy2DAsync((char *)out + off * s->esize, (size_t)s->nsamples * s->esize, c.buf, (size_t)c.nsteps * s->esize,
                                 (size_t)c.nsteps * s->esize, (size_t)np, cudaMemcpyDefault, s->stream));
    off += c.nsteps;
  }
  CU_TRY2(s, cudaStreamSynchronize(s->stream));
  return RKETD_OK;
}

int rketd2d_get_kernel_coefficients(rketd2d_sim *s, double *out, double *globals) {
  if (!s) return RKETD_EINVAL;
  if (!s->have_media) return fail2(s, RKETD_ESTATE, "no media yet");
  if (globals) {
    const double Sx = kC0 * s->dt / s->dx, Sy = kC0 * s->dt / s->dy;
    globals[0] = s->dt / (kMu0 * s->dx); globals[1] = s->dt / (kMu0 * s->dy);
    globals[2] = (Sx - 1.0) / (Sx + 1.0); globals[3] = (Sy - 1.0) / (Sy + 1.0);
  }
  if (!out) return RKETD_OK;
  const int64_t n = (int64_t)s->nx * s->ny;
  double *d = nullptr;
  CU_TRY2(s, cudaMalloc((void **)&d, (size_t)n * 4 * 8));
  if (s->dtype == RKETD_F64)
    unpack2d_kernel<double><<<blocks_for(n), 256, 0, s->stream>>>(s->nx, s->ny, s->pitch, (double *)s->coef[0], (double *)s->coef[1],
                                                                  (double *)s->coef[2], (double *)s->coef[3], d);
  else
    unpack2d_kernel<float><<<blocks_for(n), 256, 0, s->stream>>>(s->nx, s->ny, s->pitch, (float *)s->coef[0], (float *)s->coef[1],
                                                                 (float *)s->coef[2], (float *)s->coef[3], d);
  cudaError_t e = cudaGetLastError();
  if (e == cudaSuccess) e = cudaMemcpyAsync(out, d, (size_t)n * 4 * 8, cudaMemcpyDefault, s->stream);
  if (e == cudaSuccess) e = cudaStreamSynchronize(s->stream);
  cudaFree(d);
  CU_TRY2(s, e);
  s->ctr_launches++;
  return RKETD_OK;
}

int64_t rketd2d_get_counter(const rketd2d_sim *s, int which) {
  if (!s) return -1;
  switch (which) {
    case RKETD2D_CTR_LAUNCHES: return s->ctr_launches;
    case RKETD2D_CTR_STEP_LAUNCHES: return s->ctr_step_launches;
    case RKETD2D_CTR_KERNEL_USED: return s->ctr_kernel_used;
    case RKETD2D_CTR_DEPTH_USED: return s->ctr_depth_used;
    case RKETD2D_CTR_STEPS_DONE: return s->step;
    case RKETD2D_CTR_STRIP_COLS: return s->ctr_strip;
    case RKETD2D_CTR_HALO_COLS: return s->ctr_halo;
    case RKETD2D_CTR_SEG_ROWS: return s->ctr_seg;
    case RKETD2D_CTR_STATE_BYTES: return s->state_bytes;
  }
  return -1;
}

void rketd2d_destroy(rketd2d_sim *s) {
  if (!s) return;
  cudaStreamSynchronize(s->stream);
  for (int b = 0; b < 2; ++b)
    for (int f = 0; f < 4; ++f) cudaFree(s->fld[b][f]);
  for (int c = 0; c < 4; ++c) cudaFree(s->coef[c]);
  cudaFree(s->wp_p); cudaFree(s->nu_p); cudaFree(s->rowflag); cudaFree(s->d_bad);
  for (int b = 0; b < 2; ++b)
    for (int c = 0; c < 2; ++c) cudaFree(s->split[b][c]);
  cudaFree(s->tabs);
  for (auto &c : s->chunks) cudaFree(c.buf);
  cudaGetLastError();
  delete s;
}

const char *rketd2d_last_error(const rketd2d_sim *s) { return s ? s->err.c_str() : g_create_error2.c_str(); }

}  // extern "C"
