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

// ---- Mur, source and probes of a warp tile without divergence.
// Every grid has the same layout, so the LOCAL index (0..C-1, inside its 64-B row) of node 0, node ncells-1 and the
// source node is a launch-wide constant that comes straight from kernel parameters: a switch on it is a uniform branch
// (no reconvergence stack), and which LANE holds the node is a predicate that turns the update into a select.  Probe
// nodes differ from lane to lane; their value is picked by a select tree and written by one predicated store.
// step_special (rketd_device.cuh) does the same with per-lane else-if chains: in a warp whose lanes take different
// chains every step costs ~1000 cycles of branch latency (profiles/r02_ncu_k3_wtile.md), which is what one warp tile
// in three pays in the batched configs, and every warp of the chunk waits for it at the next halo refresh.
struct WarpSpecial {
  bool w_murL = false, w_murR = false, w_src = false, w_probe = false, w_probe2 = false, w_slow = false;   // some lane of the warp ...
  bool l_murL = false, l_murR = false, l_src = false, l_p0 = false, l_p1 = false;                           // this lane ...
  int iL = 0, iR = 1, iS = 0;         // launch-wide local indices
};

template <typename R, int C, bool PML>
__device__ __forceinline__ WarpSpecial make_warp_special(const StepParams<R> &p, const SpecialIdx &sx) {
  WarpSpecial ws;
  constexpr unsigned full = 0xffffffffu;
  ws.iL = (int)(p.cellL % C); ws.iR = (int)(p.cellR % C); ws.iS = p.cellS >= 0 ? (int)(p.cellS % C) : 0;
  ws.l_murL = sx.iL >= 0; ws.l_murR = sx.iR >= 0; ws.l_src = sx.iS >= 0;
  ws.l_p0 = sx.np >= 1 && sx.np <= 2; ws.l_p1 = sx.np == 2;
  ws.w_murL = __any_sync(full, ws.l_murL); ws.w_murR = __any_sync(full, ws.l_murR); ws.w_src = __any_sync(full, ws.l_src);
  ws.w_probe = __any_sync(full, ws.l_p0); ws.w_probe2 = __any_sync(full, ws.l_p1);
  // more than two probes among one lane's nodes, or an absorbing layer: the general per-lane path
  ws.w_slow = PML || __any_sync(full, sx.np == 3);
  return ws;
}

// f(integral_constant<int, i>) for i == idx, idx warp-uniform: a switch (jump table or uniform branches)
template <int C, typename F>
__device__ __forceinline__ void uniform_switch(int idx, F &&f) {
  switch (idx) {
    case 0: f(std::integral_constant<int, 0>{}); break;
    case 1: f(std::integral_constant<int, 1>{}); break;
    case 2: f(std::integral_constant<int, 2 % C>{}); break;
    case 3: f(std::integral_constant<int, 3 % C>{}); break;
    case 4: f(std::integral_constant<int, 4 % C>{}); break;
    case 5: f(std::integral_constant<int, 5 % C>{}); break;
    case 6: f(std::integral_constant<int, 6 % C>{}); break;
    case 7: f(std::integral_constant<int, 7 % C>{}); break;
    case 8: f(std::integral_constant<int, 8 % C>{}); break;
    case 9: f(std::integral_constant<int, 9 % C>{}); break;
    case 10: f(std::integral_constant<int, 10 % C>{}); break;
    case 11: f(std::integral_constant<int, 11 % C>{}); break;
    case 12: f(std::integral_constant<int, 12 % C>{}); break;
    case 13: f(std::integral_constant<int, 13 % C>{}); break;
    case 14: f(std::integral_constant<int, 14 % C>{}); break;
    case 15: f(std::integral_constant<int, 15 % C>{}); break;
    default: break;
  }
}

// value of v[idx], idx per lane: a select tree (no branch, no local memory)
template <typename R, int C>
__device__ __forceinline__ R select_node(const R (&v)[C], int idx) {
  R t[C];
#pragma unroll
  for (int i = 0; i < C; ++i) t[i] = v[i];
#pragma unroll
  for (int w = 1; w < C; w <<= 1)
#pragma unroll
    for (int i = 0; i + w < C; i += 2 * w) t[i] = (idx & w) ? t[i + w] : t[i];
  return t[0];
}

// a3, a4, a6 for the lanes of a warp tile (same order and the same arithmetic as step_special; Mur ends only)
template <typename R, int C>
__device__ __forceinline__ void special_uniform(const R (&E)[C], R (&En)[C], R (&H)[C], const StepParams<R> &p,
                                                const SpecialIdx &sx, const WarpSpecial &ws, int64_t nloc, R src_now) {
  typedef Arith<R> A;
  if (ws.w_murL) {      // node 0 sits at local index 0 or 1 (Layout: off), node 1 in the same row
    if (ws.iL == 0) {
      const R cand = A::fma(p.mur_m, A::sub(En[1], E[0]), E[1]);
      En[0] = ws.l_murL ? cand : En[0];
    } else {
      const R cand = A::fma(p.mur_m, A::sub(En[2], E[1]), E[2]);
      En[1] = ws.l_murL ? cand : En[1];
      H[0] = ws.l_murL ? R(0) : H[0];                                   // padding left of node 0
    }
  }
  if (ws.w_murR) {      // node ncells-1 at local index iR >= 1, node ncells-2 in the same row
    uniform_switch<C>(ws.iR, [&](auto ic) {
      constexpr int i = decltype(ic)::value;
      if constexpr (i >= 1) {
        const R cand = A::fma(p.mur_m, A::sub(En[i - 1], E[i]), E[i - 1]);
        En[i] = ws.l_murR ? cand : En[i];
#pragma unroll
        for (int j = i; j < C; ++j) H[j] = ws.l_murR ? R(0) : H[j];     // H[ncells-1] and padding
      }
    });
  }
  if (ws.w_src) {
    uniform_switch<C>(ws.iS, [&](auto ic) {
      constexpr int i = decltype(ic)::value;
      const R sum = A::add(En[i], src_now);
      En[i] = ws.l_src ? sum : En[i];
    });
  }
  if (ws.w_probe) {
    const R v = select_node<R, C>(En, sx.pi0);
    if (ws.l_p0) p.rec[sx.pr0 + nloc] = v;
    if (ws.w_probe2) {
      const R v1 = select_node<R, C>(En, sx.pi1);
      if (ws.l_p1) p.rec[sx.pr1 + nloc] = v1;
    }
  }
}

// One leapfrog step of a warp tile.  Only NEW values travel: H'[C-1] goes up one lane as soon as it
// exists (the left neighbour's H' that E'[0] needs), E'[0] goes down one lane at the end (the E[C] the
// next step's H'[C-1] needs).  Two 64-bit shuffles per step and no redundant arithmetic.  Lanes 0 and 31
// receive their own values at the tile edge, which is fine: those nodes are in the halo that is thrown
// away (garbage moves inwards one node per step; the halo is >= T nodes wide).
// SLOW: the special lanes take step_special's per-lane chains (absorbing layer, or more than two probes in one lane)
template <bool SPECIAL, bool PML, bool SLOW, typename R, int C>
__device__ __forceinline__ void warp_step(const R (&E)[C], R (&En)[C], R (&H)[C], R (&G)[C], const CoefRegs<R, C> &cf,
                                          R &Er, R nchh, const StepParams<R> &p, const SpecialIdx &sx, const WarpSpecial &ws,
                                          int64_t nloc, R src_now) {
  typedef Arith<R> A;
  // Issue cost of an FP64 instruction on sm_100 = max(2, distinct 64-bit register operands) cycles per
  // scheduler (measured): the two FMAs that multiply E[i] sit next to each other so that the
  // second one finds E[i] in the operand-reuse cache, and nchh comes from the constant bank.
  if constexpr (SPECIAL && PML) {
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
  if constexpr (SPECIAL) {                                                     // a3, a4, a6
    if constexpr (PML || SLOW) { if (sx.any) step_special<R, C, PML>(E, En, H, p, sx, nloc, src_now); }
    else special_uniform<R, C>(E, En, H, p, sx, ws, nloc, src_now);
  }
  Er = __shfl_down_sync(0xffffffffu, En[0], 1);
}

template <bool SPECIAL, bool PML, bool SLOW, typename R, int C>
__device__ __forceinline__ void warp_steps(R (&E)[C], R (&H)[C], R (&G)[C], const CoefRegs<R, C> &cf, const StepParams<R> &p,
                                           const SpecialIdx &sx, const WarpSpecial &ws, SourceStream<R> &src, int64_t nloc,
                                           int nsteps) {
  const R nchh = p.nchh;       // stays a constant-bank operand of the FMAs (one register read less each)
  const int lane = threadIdx.x & 31;
  R Er = __shfl_down_sync(0xffffffffu, E[0], 1);
  R Eb[C];
  int left = nsteps;
  for (; left >= 2; left -= 2) {
    const R s0 = SPECIAL ? src.sample(p, nloc, lane) : R(0);
    warp_step<SPECIAL, PML, SLOW, R, C>(E, Eb, H, G, cf, Er, nchh, p, sx, ws, nloc, s0);
    const R s1 = SPECIAL ? src.sample(p, nloc + 1, lane) : R(0);
    warp_step<SPECIAL, PML, SLOW, R, C>(Eb, E, H, G, cf, Er, nchh, p, sx, ws, nloc + 1, s1);
    nloc += 2;
  }
  if (left) {
    const R s0 = SPECIAL ? src.sample(p, nloc, lane) : R(0);
    warp_step<SPECIAL, PML, SLOW, R, C>(E, Eb, H, G, cf, Er, nchh, p, sx, ws, nloc, s0);
#pragma unroll
    for (int i = 0; i < C; ++i) E[i] = Eb[i];
  }
}

// T steps of one staged tile of K2 (k2_wtile): special indices and the source stream are set up per tile
template <bool SPECIAL, bool PML, typename R, int C>
__device__ __forceinline__ void warp_time_loop(R (&E)[C], R (&H)[C], R (&G)[C], const CoefRegs<R, C> &cf,
                                               const StepParams<R> &p, uint32_t flag, int64_t k0, int64_t g, bool owner,
                                               int nsteps) {
  const int lane = threadIdx.x & 31;
  SourceStream<R> src;
  src.start(p, SPECIAL && __any_sync(0xffffffffu, (flag & F_SRC) != 0u), p.n0, lane);
  const SpecialIdx sx = SPECIAL ? make_special<R, C, PML>(p, flag, k0, g, owner) : SpecialIdx();
  const WarpSpecial ws = SPECIAL ? make_warp_special<R, C, PML>(p, sx) : WarpSpecial();
  if constexpr (SPECIAL && !PML) {
    if (ws.w_slow) { warp_steps<true, false, true, R, C>(E, H, G, cf, p, sx, ws, src, p.n0, nsteps); return; }
  }
  warp_steps<SPECIAL, PML, false, R, C>(E, H, G, cf, p, sx, ws, src, p.n0, nsteps);
}

// T steps of a warp tile between two halo refreshes of the resident kernel: the step counter, the special indices
// and the source stream belong to the caller and live across rounds (restarting the stream would put two global
// loads on the critical path of every round).
template <bool SPECIAL, bool PML, typename R, int C>
__device__ __forceinline__ void warp_round(R (&E)[C], R (&H)[C], R (&G)[C], const CoefRegs<R, C> &cf, const StepParams<R> &p,
                                           const SpecialIdx &sx, const WarpSpecial &ws, SourceStream<R> &src, int64_t nloc,
                                           int nsteps) {
  if constexpr (SPECIAL && !PML) {
    if (ws.w_slow) { warp_steps<true, false, true, R, C>(E, H, G, cf, p, sx, ws, src, nloc, nsteps); return; }
  }
  warp_steps<SPECIAL, PML, false, R, C>(E, H, G, cf, p, sx, ws, src, nloc, nsteps);
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
