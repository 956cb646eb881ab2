// rketd_wtile.cuh — the register-resident warp tile shared by the temporal-blocking kernel K2 (k2_wtile,
// rketd_kernels.cu) and the resident kernel K3 (k3_wtile, rketd_resident.cu): a warp owns 32 rows x 64 B of every
// array, one row per lane, and advances them with halos travelling by warp shuffles only.  Also the small host-side
// helpers both launcher files use.
#pragma once
#include "rketd_device.cuh"
#include "rketd_internal.h"

namespace rketd {

template <typename R> struct RowPtrs { R *E, *H, *J; };
template <typename R> struct CoefPtrs { const R *c[kNumCoef]; };

// One leapfrog step of a warp tile.  Only NEW values travel: H'[C-1] goes up one lane as soon as it
// exists (the left neighbour's H' that E'[0] needs), E'[0] goes down one lane at the end (the E[C] the
// next step's H'[C-1] needs).  Two 64-bit shuffles per step and no redundant arithmetic.  Lanes 0 and 31
// receive their own values at the tile edge, which is fine: those nodes are in the halo that is thrown
// away (garbage moves inwards one node per step; the halo is >= T nodes wide).
// MASK: SF_* features of the tile (0: none; SF_SLOW: step_special's per-lane chains — absorbing layer, or more than
// two probes in one lane).
template <int MASK, bool PML, typename R, int C>
__device__ __forceinline__ void warp_step(const R (&E)[C], R (&En)[C], R (&H)[C], R (&G)[C], const CoefRegs<R, C> &cf,
                                          R &Er, R nchh, const StepParams<R> &p, const SpecialIdx &sx, const WarpSpecial &ws,
                                          int64_t nloc, R src_now) {
  typedef Arith<R> A;
  // Issue cost of an FP64 instruction on sm_100 = max(2, distinct 64-bit register operands) cycles per scheduler
  // (measured: profiles/r02_peaks.md): the two FMAs that multiply E[i] sit next to each other so that the
  // second one finds E[i] in the operand-reuse cache, and nchh comes from the constant bank.
  if constexpr (MASK == SF_SLOW && PML) {
    if (sx.pml_mask) pml_pre<R, C>(E, Er, H, p, sx);                           // absorbing-layer H nodes, on old E
  }
  H[C - 1] = A::fma(nchh, A::sub(Er, E[C - 1]), H[C - 1]);                    // a1, last node first
  const R Hl = __shfl_up_sync(0xffffffffu, H[C - 1], 1);
#pragma unroll
  for (int i = 0; i < C - 1; ++i) H[i] = A::fma(nchh, A::sub(E[i + 1], E[i]), H[i]);
#pragma unroll
  for (int i = C - 1; i >= 0; --i) {
    const R w = A::mul(cf.c[COEF_Q][i], E[i]);
    const R t = A::fma(cf.c[COEF_P][i], E[i], -G[i]);
    G[i] = A::fma(cf.c[COEF_KA][i], G[i], w);                                 // a5 (old E, old G)
    En[i] = A::fma(-cf.c[COEF_CH][i], A::sub(H[i], i ? H[i - 1] : Hl), t);    // a2
  }
  if constexpr (MASK == SF_SLOW) {                                             // a3, a4, a6
    if (sx.any) step_special<R, C, PML>(E, En, H, p, sx, nloc, src_now);
  } else if constexpr (MASK != 0) {
    special_select<MASK, R, C>(E, En, p, sx, ws, nloc, src_now);
  }
  Er = __shfl_down_sync(0xffffffffu, En[0], 1);
}

template <int MASK, bool PML, typename R, int C, typename SRCT>
__device__ __forceinline__ void warp_steps(R (&E)[C], R (&H)[C], R (&G)[C], const CoefRegs<R, C> &cf, const StepParams<R> &p,
                                           const SpecialIdx &sx, const WarpSpecial &ws, SRCT &src, int64_t nloc,
                                           int nsteps) {
  constexpr bool SRC = MASK == SF_SLOW || (MASK & SF_SRC) != 0;
  const R nchh = p.nchh;       // stays a constant-bank operand of the FMAs (one register read less each)
  const int lane = threadIdx.x & 31;
  R Er = __shfl_down_sync(0xffffffffu, E[0], 1);
  R Eb[C];
  int left = nsteps;
  for (; left >= 2; left -= 2) {
    R s0 = R(0), s1 = R(0);
    if constexpr (MASK == SF_SLOW) { s0 = src.sample(p, nloc, lane); s1 = src.sample(p, nloc + 1, lane); }
    else if constexpr (SRC) src.sample2(p, nloc, lane, s0, s1);
    warp_step<MASK, PML, R, C>(E, Eb, H, G, cf, Er, nchh, p, sx, ws, nloc, s0);
    warp_step<MASK, PML, R, C>(Eb, E, H, G, cf, Er, nchh, p, sx, ws, nloc + 1, s1);
    nloc += 2;
  }
  if (left) {
    const R s0 = SRC ? src.sample(p, nloc, lane) : R(0);
    warp_step<MASK, PML, R, C>(E, Eb, H, G, cf, Er, nchh, p, sx, ws, nloc, s0);
#pragma unroll
    for (int i = 0; i < C; ++i) E[i] = Eb[i];
  }
  if constexpr (MASK != 0 && MASK != SF_SLOW) zero_padding_H<R, C>(H, ws);
}

// T steps of one staged tile of K2 (k2_wtile): special indices and the source stream are set up per tile.  K2 meets a
// special tile once in thousands, so it keeps step_special's per-lane chains (SF_SLOW) and, with them, the register
// budget of its 12-warp CTAs: the select instantiations cost it spills and 10 % on config 4 (measured).
template <bool SPECIAL, bool PML, typename R, int C>
__device__ __forceinline__ void warp_time_loop(R (&E)[C], R (&H)[C], R (&G)[C], const CoefRegs<R, C> &cf,
                                               const StepParams<R> &p, uint32_t flag, int64_t k0, int64_t g, bool owner,
                                               int nsteps) {
  constexpr int MASK = SPECIAL ? SF_SLOW : 0;
  const R nchh = p.nchh;       // stays a constant-bank operand of the FMAs (one register read less each)
  int64_t nloc = p.n0;
  R Er = __shfl_down_sync(0xffffffffu, E[0], 1);
  R Eb[C];
  const int lane = threadIdx.x & 31;
  SourceStream<R> src;
  src.start(p, SPECIAL && __any_sync(0xffffffffu, (flag & F_SRC) != 0u), nloc, lane);
  const SpecialIdx sx = SPECIAL ? make_special<R, C, PML>(p, flag, k0, g, owner) : SpecialIdx();
  const WarpSpecial ws;
  int left = nsteps;
  for (; left >= 2; left -= 2) {
    const R s0 = SPECIAL ? src.sample(p, nloc, lane) : R(0);
    warp_step<MASK, PML, R, C>(E, Eb, H, G, cf, Er, nchh, p, sx, ws, nloc, s0);
    const R s1 = SPECIAL ? src.sample(p, nloc + 1, lane) : R(0);
    warp_step<MASK, PML, R, C>(Eb, E, H, G, cf, Er, nchh, p, sx, ws, nloc + 1, s1);
    nloc += 2;
  }
  if (left) {
    const R s0 = SPECIAL ? src.sample(p, nloc, lane) : R(0);
    warp_step<MASK, PML, R, C>(E, Eb, H, G, cf, Er, nchh, p, sx, ws, nloc, s0);
#pragma unroll
    for (int i = 0; i < C; ++i) E[i] = Eb[i];
  }
}

// T steps of a warp tile between two halo refreshes of the resident kernel: the step counter, the special indices
// and the source stream belong to the caller and live across rounds (restarting the stream would put two global
// loads on the critical path of every round).  One instantiation per feature set, chosen here once per round.
template <bool PML, typename R, int C, typename SRCT>
__device__ __forceinline__ void warp_round(R (&E)[C], R (&H)[C], R (&G)[C], const CoefRegs<R, C> &cf, const StepParams<R> &p,
                                           const SpecialIdx &sx, const WarpSpecial &ws, SRCT &src, int64_t nloc,
                                           int nsteps) {
#define RKETD_ROUND_CASE(M) case M: warp_steps<M, false, R, C>(E, H, G, cf, p, sx, ws, src, nloc, nsteps); break;
  constexpr int kFastAll = SF_MURR | SF_SRC | SF_PROBE;
  if (PML || ws.mask == SF_SLOW) {
    warp_steps<SF_SLOW, PML, R, C>(E, H, G, cf, p, sx, ws, src, nloc, nsteps);
  } else if (C >= 8 && ws.mask != 0 && ws.fast == kFastAll) {
    // every feature at a fixed local index (special_select, SF_FAST): one candidate per feature, so two instantiations
    // (with and without the source stream) serve all fifteen feature sets.  Not for half rows of fp64 (C = 4): there the
    // exact feature set with its three or four candidates is shorter than all four features with one each (config 1:
    // 0.76 against 0.82 ms)
    if (ws.mask & SF_SRC) warp_steps<SF_FAST | 15, false, R, C>(E, H, G, cf, p, sx, ws, src, nloc, nsteps);
    else warp_steps<SF_FAST | 11, false, R, C>(E, H, G, cf, p, sx, ws, src, nloc, nsteps);
  } else {
    switch (ws.mask) {
      RKETD_ROUND_CASE(0) RKETD_ROUND_CASE(1) RKETD_ROUND_CASE(2) RKETD_ROUND_CASE(3) RKETD_ROUND_CASE(4) RKETD_ROUND_CASE(5)
      RKETD_ROUND_CASE(6) RKETD_ROUND_CASE(7) RKETD_ROUND_CASE(8) RKETD_ROUND_CASE(9) RKETD_ROUND_CASE(10) RKETD_ROUND_CASE(11)
      RKETD_ROUND_CASE(12) RKETD_ROUND_CASE(13) RKETD_ROUND_CASE(14) RKETD_ROUND_CASE(15)
      default: break;
    }
  }
#undef RKETD_ROUND_CASE
}

// ---- the lean warp tile of the resident kernel: E advanced IN PLACE (no second E buffer) and the coefficients taken
// from a source CF instead of 4 C registers per lane — four registers when the lane's nodes all carry one coefficient
// set (piecewise-constant media: every lane that does not straddle an interface; CoefUniform), the warp's own swizzled
// shared-memory rows otherwise (CoefWarpSmem).  About 100 registers instead of 232: three to four chunks share an SM
// and fill each other's barrier waits.  Same operations per node, same order of the special nodes, same bits.
template <typename R, int C>
struct CoefWarpSmem {
  static constexpr int V = 16 / sizeof(R);
  uint32_t base;              // shared address of this lane's row in array 0: warp area + swizzle applied per chunk
  int lane;
  template <int a>
  __device__ __forceinline__ void chunk(int j, R (&out)[V]) const {
    typename Arith<R>::Vec v;
    lds128(base + a * (32 * kRowBytes) + swz_off(lane, j), v);
    vec_unpack(v, out);
  }
};

// One step, in place.  Ascending node order: E'[i] needs the old E[i] only (through t and the current update), the Mur
// candidate of node i needs the NEW E[i-1] and the OLD E[i-1], E[i] — one rolling temporary.
template <int MASK, typename R, int C, typename CF>
__device__ __forceinline__ void warp_step_lean(R (&E)[C], R (&H)[C], R (&G)[C], const CF &cf, R &Er, R nchh,
                                               const StepParams<R> &p, const SpecialIdx &sx, const WarpSpecial &ws,
                                               int64_t nloc, R src_now) {
  typedef Arith<R> A;
  constexpr int V = 16 / sizeof(R);
  H[C - 1] = A::fma(nchh, A::sub(Er, E[C - 1]), H[C - 1]);                    // a1, last node first
  const R Hl = __shfl_up_sync(0xffffffffu, H[C - 1], 1);
#pragma unroll
  for (int i = 0; i < C - 1; ++i) H[i] = A::fma(nchh, A::sub(E[i + 1], E[i]), H[i]);
  const R e0 = E[0], e1 = E[1], e2 = E[2];                                    // old values Mur at node 0 needs
  R prev_old = R(0);
#pragma unroll
  for (int j = 0; j < C / V; ++j) {
    R cP[V], cch[V], cka[V], cQ[V];
    cf.template chunk<COEF_P>(j, cP); cf.template chunk<COEF_CH>(j, cch);
    cf.template chunk<COEF_KA>(j, cka); cf.template chunk<COEF_Q>(j, cQ);
#pragma unroll
    for (int u = 0; u < V; ++u) {
      const int i = j * V + u;
      const R eo = E[i];
      const R w = A::mul(cQ[u], eo);
      const R t = A::fma(cP[u], eo, -G[i]);
      G[i] = A::fma(cka[u], G[i], w);                                         // a5 (old E, old G)
      R en = A::fma(-cch[u], A::sub(H[i], i ? H[i - 1] : Hl), t);             // a2
      if constexpr ((MASK & SF_MURR) != 0) {
        if (i >= 1) {
          const R cand = A::fma(p.mur_m, A::sub(E[i - 1], eo), prev_old);     // E[i-1] is already the new interior value
          en = ((ws.mR >> i) & 1u) ? cand : en;
        }
        prev_old = eo;
      }
      E[i] = en;
    }
  }
  if constexpr ((MASK & SF_MURL) != 0) {
    const R c0 = A::fma(p.mur_m, A::sub(E[1], e0), e1);
    const R c1 = A::fma(p.mur_m, A::sub(E[2], e1), e2);
    E[0] = ws.mL0 ? c0 : E[0];
    E[1] = ws.mL1 ? c1 : E[1];
  }
  if constexpr ((MASK & SF_SRC) != 0) {
#pragma unroll
    for (int i = 0; i < C; ++i) {
      const R sum = A::add(E[i], src_now);
      E[i] = ((ws.mS >> i) & 1u) ? sum : E[i];
    }
  }
  if constexpr ((MASK & SF_PROBE) != 0) {
    const R v0 = select_node<R, C>(E, sx.pi0), v1 = select_node<R, C>(E, sx.pi1);
    stg_if(ws.l_p0, p.rec + (sx.pr0 + nloc), v0);
    stg_if(ws.l_p1, p.rec + (sx.pr1 + nloc), v1);
  }
  Er = __shfl_down_sync(0xffffffffu, E[0], 1);
}

template <int MASK, typename R, int C, typename CF, typename SRCT>
__device__ __forceinline__ void warp_steps_lean(R (&E)[C], R (&H)[C], R (&G)[C], const CF &cf, const StepParams<R> &p,
                                                const SpecialIdx &sx, const WarpSpecial &ws, SRCT &src,
                                                int64_t nloc, int nsteps) {
  const R nchh = p.nchh;
  const int lane = threadIdx.x & 31;
  R Er = __shfl_down_sync(0xffffffffu, E[0], 1);
  int left = nsteps;
  for (; left >= 2; left -= 2) {
    R s0 = R(0), s1 = R(0);
    if constexpr ((MASK & SF_SRC) != 0) src.sample2(p, nloc, lane, s0, s1);
    warp_step_lean<MASK, R, C>(E, H, G, cf, Er, nchh, p, sx, ws, nloc, s0);
    warp_step_lean<MASK, R, C>(E, H, G, cf, Er, nchh, p, sx, ws, nloc + 1, s1);
    nloc += 2;
  }
  if (left) {
    const R s0 = (MASK & SF_SRC) != 0 ? src.sample(p, nloc, lane) : R(0);
    warp_step_lean<MASK, R, C>(E, H, G, cf, Er, nchh, p, sx, ws, nloc, s0);
  }
  if constexpr (MASK != 0) zero_padding_H<R, C>(H, ws);
}

template <typename R, int C, typename CF, typename SRCT>
__device__ __forceinline__ void warp_round_lean(R (&E)[C], R (&H)[C], R (&G)[C], const CF &cf, const StepParams<R> &p,
                                                const SpecialIdx &sx, const WarpSpecial &ws, SRCT &src,
                                                int64_t nloc, int nsteps) {
#define RKETD_LEAN_CASE(M) case M: warp_steps_lean<M, R, C>(E, H, G, cf, p, sx, ws, src, nloc, nsteps); break;
  switch (ws.mask) {
    RKETD_LEAN_CASE(0) RKETD_LEAN_CASE(1) RKETD_LEAN_CASE(2) RKETD_LEAN_CASE(3) RKETD_LEAN_CASE(4) RKETD_LEAN_CASE(5)
    RKETD_LEAN_CASE(6) RKETD_LEAN_CASE(7) RKETD_LEAN_CASE(8) RKETD_LEAN_CASE(9) RKETD_LEAN_CASE(10) RKETD_LEAN_CASE(11)
    RKETD_LEAN_CASE(12) RKETD_LEAN_CASE(13) RKETD_LEAN_CASE(14) RKETD_LEAN_CASE(15)
    default: break;
  }
#undef RKETD_LEAN_CASE
}

// ---- host side
template <typename R>
inline StepParams<R> make_params(const StepCommon &sc) {
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
  p.npml = sc.npml;
  for (int j = 0; j < kMaxPml; ++j) { p.pml_ha[j] = (R)sc.pml_ha[j]; p.pml_hd[j] = (R)sc.pml_hd[j]; }
  return p;
}
template <typename R> inline RowPtrs<R> rp(FieldPtrs f) { return RowPtrs<R>{(R *)f.E, (R *)f.H, (R *)f.J}; }
template <typename R> inline CoefPtrs<R> cpz(void *const coef[kNumCoef]) {
  CoefPtrs<R> c;
  for (int a = 0; a < kNumCoef; ++a) c.c[a] = (const R *)coef[a];
  return c;
}


}  // namespace rketd
