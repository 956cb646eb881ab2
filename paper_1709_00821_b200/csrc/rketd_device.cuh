// rketd_device.cuh — device-side building blocks shared by the stencil kernels (K1 one step per
// launch, K2 temporal blocking, K3 grid resident).  All of them advance a thread's C consecutive
// nodes with the SAME sequence of correctly rounded operations (explicit fma/mul/sub intrinsics, so
// the compiler cannot contract or reassociate differently per kernel): K1, K2 and K3 agree bit for
// bit on the same input, which tests/test_gpu_parity.py checks.
//
// The recurrence (eqs. (14), (12)+(11), (11)) in the form the
// kernels run it.  With the six coefficients of row a0 (E' = ca E - cj J - ch dH; J' = ka J + kb E + kc E')
// define the scaled, shifted current  G := cj J - (cj kc) E.  Then, exactly:
//   H'[k] = fma(-chh, E[k+1] - E[k], H[k])                                  2 flop-instr   eq. (14)
//   E'[k] = fma(-ch, H'[k] - H'[k-1], fma(P, E[k], -G[k])),  P = ca - cj kc  3              eq. (12)+(11)
//   G'[k] = fma(ka, G[k], Q * E[k]),                         Q = ka cj kc + cj kb   2       eq. (11)
// G' needs only OLD values, so Mur, the source and the probes (which change E') do not touch it, and
// J is recovered on read-out as J = (G + cj kc E)/cj.  7 instructions and 4 per-node coefficients
// (P, ch, ka, Q) per node and step instead of 9 and 6.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include <type_traits>

namespace rketd {

constexpr int kRowBytes = 64;       // one thread owns 64 B (or 32 B) of every array
constexpr int kMaxProbes = 64;
constexpr int kNumCoef = 4;         // P, ch, ka, Q
enum { COEF_P = 0, COEF_CH = 1, COEF_KA = 2, COEF_Q = 3 };

enum : uint32_t { F_MURL = 1u, F_MURR = 2u, F_SRC = 4u, F_PROBE = 8u, F_PML = 16u };
constexpr int kMaxPml = 32;         // deepest absorbing layer, in nodes

template <typename R> struct Arith;
template <> struct Arith<double> {
  typedef double2 Vec;                         // 16 B
  static __device__ __forceinline__ double mul(double a, double b) { return __dmul_rn(a, b); }
  static __device__ __forceinline__ double sub(double a, double b) { return __dsub_rn(a, b); }
  static __device__ __forceinline__ double add(double a, double b) { return __dadd_rn(a, b); }
  static __device__ __forceinline__ double fma(double a, double b, double c) { return __fma_rn(a, b, c); }
};
template <> struct Arith<float> {
  typedef float4 Vec;
  static __device__ __forceinline__ float mul(float a, float b) { return __fmul_rn(a, b); }
  static __device__ __forceinline__ float sub(float a, float b) { return __fsub_rn(a, b); }
  static __device__ __forceinline__ float add(float a, float b) { return __fadd_rn(a, b); }
  static __device__ __forceinline__ float fma(float a, float b, float c) { return __fmaf_rn(a, b, c); }
};

// Everything a step needs besides the fields and coefficients.  Cell indices are
// PHYSICAL in-grid indices (node index + layout offset, see rketd_internal.h).
template <typename R>
struct StepParams {
  R nchh;                    // -dt/(mu0 dz)                     eq. (14)
  R mur_m;                   // (S-1)/(S+1), S = c dt/dz
  int64_t cellL, cellR;      // physical index of node 0 and node ncells-1
  int64_t cellS;             // physical index of the source node, -1 if none
  int nprobes;
  int64_t rec_stride;        // samples per (grid, probe) in rec (= steps of this rketd_run call)
  int64_t n0;                // local step index (within this call) of the first step of this launch
  const R *src_tab;          // [rec_stride] source sample per local step (a4), or nullptr
  R *rec;                    // [nbatch][nprobes][rec_stride] (a6), or nullptr
  const uint8_t *rowflag;    // [nrows] F_* bits per row
  int64_t probe_cell[kMaxProbes];
  // PML (rketd_set_boundary): npml = 0 means first-order Mur ends.  H node j nodes from an outer
  // end updates as H' = ha[j] H + (nchh/(1+s_j)) dE; the kernels apply it as a pre-step H <- ha[j] H + hd[j] dE,
  // hd[j] = nchh/(1+s_j) - nchh, followed by the ordinary update H <- H + nchh dE.
  int npml;
  R pml_ha[kMaxPml], pml_hd[kMaxPml];
};

// 16-B vector <-> scalars
__device__ __forceinline__ void vec_unpack(const double2 &v, double (&o)[2]) { o[0] = v.x; o[1] = v.y; }
__device__ __forceinline__ void vec_unpack(const float4 &v, float (&o)[4]) { o[0] = v.x; o[1] = v.y; o[2] = v.z; o[3] = v.w; }
__device__ __forceinline__ double2 vec_pack(const double (&o)[2]) { return make_double2(o[0], o[1]); }
__device__ __forceinline__ float4 vec_pack(const float (&o)[4]) { return make_float4(o[0], o[1], o[2], o[3]); }

// chunk j (16 B) of a thread's C values
template <typename R, int C>
__device__ __forceinline__ void vec_to_regs(const typename Arith<R>::Vec &v, R (&r)[C], int j) {
  constexpr int V = 16 / sizeof(R);
  R o[V];
  vec_unpack(v, o);
#pragma unroll
  for (int u = 0; u < V; ++u) r[j * V + u] = o[u];
}
template <typename R, int C>
__device__ __forceinline__ typename Arith<R>::Vec regs_to_vec(const R (&r)[C], int j) {
  constexpr int V = 16 / sizeof(R);
  R o[V];
#pragma unroll
  for (int u = 0; u < V; ++u) o[u] = r[j * V + u];
  return vec_pack(o);
}

// keep a loop-invariant kernel parameter in a vector register: a value that went through a
// shuffle cannot be re-read from the constant bank by ptxas inside the time loop, where the
// load latency would sit on the critical path
template <typename R> __device__ __forceinline__ R pin_register(R x) { return __shfl_sync(0xffffffffu, x, 0); }

// Geometry of the register tiling: a thread owns C consecutive nodes (32 or 64 B) of every
// array; a 64-B row of the HBM layout is shared by TPR = 1 or 2 threads.
template <typename R, int C>
struct Geom {
  static constexpr int V = 16 / sizeof(R);          // nodes per 16-B chunk
  static constexpr int NCH = C / V;                 // chunks per thread
  static constexpr int CR = kRowBytes / sizeof(R);  // nodes per row
  static constexpr int TPR = CR / C;                // threads per row
  static_assert(C % V == 0 && CR % C == 0 && (TPR == 1 || TPR == 2), "bad cells per thread");
};

// Swizzled shared-memory offset of chunk j (0..3) of row `row` in an array of 64-B rows whose base
// is 512-B aligned: CU_TENSOR_MAP_SWIZZLE_64B = XOR of address bits [4:5] with bits [7:8].  With it
// a warp's 128-bit accesses (thread stride 32 or 64 B) cover all 32 banks.
__device__ __forceinline__ uint32_t swz_off(int row, int j) { return row * kRowBytes + ((j ^ ((row >> 1) & 3)) << 4); }

// ---- shared-memory access by 32-bit shared address (LDS.128 / STS.128, never generic LD/ST)
__device__ __forceinline__ uint32_t smem_u32(const void *p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void lds128(uint32_t a, double2 &v) {
  asm volatile("ld.shared.v2.f64 {%0, %1}, [%2];" : "=d"(v.x), "=d"(v.y) : "r"(a));
}
__device__ __forceinline__ void lds128(uint32_t a, float4 &v) {
  asm volatile("ld.shared.v4.f32 {%0, %1, %2, %3}, [%4];" : "=f"(v.x), "=f"(v.y), "=f"(v.z), "=f"(v.w) : "r"(a));
}
__device__ __forceinline__ void sts128(uint32_t a, const double2 &v) {
  asm volatile("st.shared.v2.f64 [%0], {%1, %2};" ::"r"(a), "d"(v.x), "d"(v.y) : "memory");
}
__device__ __forceinline__ void sts128(uint32_t a, const float4 &v) {
  asm volatile("st.shared.v4.f32 [%0], {%1, %2, %3, %4};" ::"r"(a), "f"(v.x), "f"(v.y), "f"(v.z), "f"(v.w) : "memory");
}

// ---- 256-bit global access (sm_100: LDG.E.ENL2.256 / STG.E.ENL2.256): a thread's 64-B row in two
// instructions, every store a full 32-B sector.  p must be 32-B aligned.
__device__ __forceinline__ void ldg256(const double *p, double (&o)[4]) {
  asm volatile("ld.global.v4.f64 {%0, %1, %2, %3}, [%4];" : "=d"(o[0]), "=d"(o[1]), "=d"(o[2]), "=d"(o[3]) : "l"(p));
}
__device__ __forceinline__ void ldg256(const float *p, float (&o)[8]) {
  asm volatile("ld.global.v8.f32 {%0, %1, %2, %3, %4, %5, %6, %7}, [%8];"
               : "=f"(o[0]), "=f"(o[1]), "=f"(o[2]), "=f"(o[3]), "=f"(o[4]), "=f"(o[5]), "=f"(o[6]), "=f"(o[7]) : "l"(p));
}
__device__ __forceinline__ void stg256(double *p, const double (&o)[4]) {
  asm volatile("st.global.v4.f64 [%0], {%1, %2, %3, %4};" ::"l"(p), "d"(o[0]), "d"(o[1]), "d"(o[2]), "d"(o[3]) : "memory");
}
__device__ __forceinline__ void stg256(float *p, const float (&o)[8]) {
  asm volatile("st.global.v8.f32 [%0], {%1, %2, %3, %4, %5, %6, %7, %8};"
               ::"l"(p), "f"(o[0]), "f"(o[1]), "f"(o[2]), "f"(o[3]), "f"(o[4]), "f"(o[5]), "f"(o[6]), "f"(o[7]) : "memory");
}
// store v to p when pred holds, as one predicated instruction (no branch, no reconvergence point)
__device__ __forceinline__ void stg_if(bool pred, double *p, double v) {
  asm volatile("{\n.reg .pred q;\nsetp.ne.u32 q, %0, 0;\n@q st.global.f64 [%1], %2;\n}" ::"r"((uint32_t)pred), "l"(p), "d"(v) : "memory");
}
__device__ __forceinline__ void stg_if(bool pred, float *p, float v) {
  asm volatile("{\n.reg .pred q;\nsetp.ne.u32 q, %0, 0;\n@q st.global.f32 [%1], %2;\n}" ::"r"((uint32_t)pred), "l"(p), "f"(v) : "memory");
}
// a thread's C nodes (32 or 64 B, 32-B aligned) <-> global memory
template <typename R, int C>
__device__ __forceinline__ void load_nodes_global(const R *base, int64_t first, R (&out)[C]) {
  constexpr int W = 32 / sizeof(R);
  static_assert(C % W == 0, "a thread owns a multiple of 32 B");
#pragma unroll
  for (int j = 0; j < C / W; ++j) {
    R o[W];
    ldg256(base + first + j * W, o);
#pragma unroll
    for (int u = 0; u < W; ++u) out[j * W + u] = o[u];
  }
}
template <typename R, int C>
__device__ __forceinline__ void store_nodes_global(R *base, int64_t first, const R (&in)[C]) {
  constexpr int W = 32 / sizeof(R);
#pragma unroll
  for (int j = 0; j < C / W; ++j) {
    R o[W];
#pragma unroll
    for (int u = 0; u < W; ++u) o[u] = in[j * W + u];
    stg256(base + first + j * W, o);
  }
}

// Coefficients of a thread's nodes held in registers: c[a][i], a = COEF_*.
template <typename R, int C>
struct CoefRegs {
  static constexpr int V = 16 / sizeof(R);
  R c[kNumCoef][C];
  template <int a>
  __device__ __forceinline__ void chunk(int j, R (&out)[V]) const {
#pragma unroll
    for (int u = 0; u < V; ++u) out[u] = c[a][j * V + u];
  }
};

// Coefficients of a thread whose C nodes all carry the same four values (piecewise-constant media: every row that
// does not straddle a media interface): one register per array.
template <typename R, int C>
struct CoefUniform {
  static constexpr int V = 16 / sizeof(R);
  R v[kNumCoef];
  template <int a>
  __device__ __forceinline__ void chunk(int, R (&out)[V]) const {
#pragma unroll
    for (int u = 0; u < V; ++u) out[u] = v[a];
  }
};

// Block barrier by PTX: warps of one CTA may reach it from different instantiations of the time loop (K3 picks the
// coefficient source per warp); bar.sync counts arriving warps, not program counters.
__device__ __forceinline__ void cta_barrier() { asm volatile("bar.sync 0;" ::: "memory"); }

// Coefficients held in shared memory: kNumCoef arrays of ROWS swizzled 64-B rows.
template <typename R, int C, int ROWS>
struct CoefSmem {
  static constexpr int V = 16 / sizeof(R);
  uint32_t chunk_addr[C / V];     // shared address of the thread's chunk j in array 0
  __device__ __forceinline__ void init(uint32_t array0, int tid) {
    const int row = tid / Geom<R, C>::TPR, sub = tid % Geom<R, C>::TPR;
#pragma unroll
    for (int j = 0; j < C / V; ++j) chunk_addr[j] = array0 + swz_off(row, sub * (C / V) + j);
  }
  template <int a>
  __device__ __forceinline__ void chunk(int j, R (&out)[V]) const {
    typename Arith<R>::Vec v;
    lds128(chunk_addr[j] + a * (ROWS * kRowBytes), v);
    vec_unpack(v, out);
  }
  template <int a>
  __device__ __forceinline__ void store_chunk(int j, const typename Arith<R>::Vec &v) const {
    sts128(chunk_addr[j] + a * (ROWS * kRowBytes), v);
  }
};

// ---- source samples (a4) without a global load on the time loop's critical path: a warp that holds the
// source node keeps 32 consecutive samples of the table in one register per lane (lane i <-> step base + i), with
// the next 32 already in flight, and picks the sample of the current step by shuffle.  Every call is warp-uniform.
template <typename R>
struct SourceStream {
  R cur, nxt;
  int64_t base;
  bool on;
  __device__ __forceinline__ R fetch(const StepParams<R> &p, int64_t idx) const {
    return (p.src_tab != nullptr && idx < p.rec_stride) ? p.src_tab[idx] : R(0);
  }
  // on: some lane of this warp holds the source node (warp-uniform)
  __device__ __forceinline__ void start(const StepParams<R> &p, bool warp_has_source, int64_t n0, int lane) {
    on = warp_has_source;
    base = n0;
    cur = R(0);
    nxt = R(0);
    if (on) {
      cur = fetch(p, base + lane);
      nxt = fetch(p, base + 32 + lane);
    }
  }
  // samples of steps nloc and nloc + 1 with one check per pair (the stream is on)
  __device__ __forceinline__ void sample2(const StepParams<R> &p, int64_t nloc, int lane, R &s0, R &s1) {
    const int j = (int)(nloc - base);
    if (j >= 31) {            // the pair touches the next 32 samples: once in 16 pairs
      s0 = sample(p, nloc, lane);
      s1 = sample(p, nloc + 1, lane);
    } else {
      s0 = __shfl_sync(0xffffffffu, cur, j);
      s1 = __shfl_sync(0xffffffffu, cur, j + 1);
    }
  }
  __device__ __forceinline__ R sample(const StepParams<R> &p, int64_t nloc, int lane) {
    if (!on) return R(0);
    if (nloc - base >= 32) {
      cur = nxt;
      base += 32;
      nxt = fetch(p, base + 32 + lane);
    }
    return __shfl_sync(0xffffffffu, cur, (int)(nloc - base));
  }
};

// The same samples for the resident warp tiles (k3_wtile), one round of T <= 64 steps at a time: the samples of the round
// sit in the warp's own shared-memory strip (one LDS per step, no shuffle with a computed lane, no branch); the next
// round's are fetched into a register pair while this round steps, so no global load is ever waited for.
__device__ __forceinline__ void lds_scalar(uint32_t a, double &v) { asm volatile("ld.shared.f64 %0, [%1];" : "=d"(v) : "r"(a)); }
__device__ __forceinline__ void lds_scalar(uint32_t a, float &v) { asm volatile("ld.shared.f32 %0, [%1];" : "=f"(v) : "r"(a)); }
__device__ __forceinline__ void sts_scalar(uint32_t a, double v) { asm volatile("st.shared.f64 [%0], %1;" ::"r"(a), "d"(v) : "memory"); }
__device__ __forceinline__ void sts_scalar(uint32_t a, float v) { asm volatile("st.shared.f32 [%0], %1;" ::"r"(a), "f"(v) : "memory"); }
template <typename R>
struct SourceRound {
  static constexpr uint32_t kBytesPerWarp = 64u * sizeof(double);
  uint32_t strip = 0;           // shared address of the warp's strip (64 samples)
  int64_t round0 = 0;           // step index of the strip's first sample
  R nxt0 = R(0), nxt1 = R(0);   // samples lane, lane + 32 of the next round
  bool on = false;
  int T = 0;
  __device__ __forceinline__ R fetch(const StepParams<R> &p, int64_t idx) const {
    return (p.src_tab != nullptr && idx < p.rec_stride) ? p.src_tab[idx] : R(0);
  }
  __device__ __forceinline__ void publish(int lane) {
    sts_scalar(strip + (uint32_t)lane * (uint32_t)sizeof(R), nxt0);
    sts_scalar(strip + (uint32_t)(lane + 32) * (uint32_t)sizeof(R), nxt1);
    __syncwarp();
  }
  // on: some lane of this warp holds the source node (warp-uniform); steps_per_round <= 64
  __device__ __forceinline__ void start(const StepParams<R> &p, bool warp_has_source, int64_t n0, int lane, int steps_per_round, uint32_t strip_addr) {
    on = warp_has_source; T = steps_per_round; strip = strip_addr; round0 = n0;
    if (on) {
      nxt0 = fetch(p, n0 + lane); nxt1 = fetch(p, n0 + 32 + lane);
      publish(lane);
      nxt0 = fetch(p, n0 + T + lane); nxt1 = fetch(p, n0 + T + 32 + lane);
    }
  }
  // before the round that starts at step n (not the first one)
  __device__ __forceinline__ void next_round(const StepParams<R> &p, int64_t n, int lane) {
    if (on) {
      __syncwarp();
      round0 = n;
      publish(lane);
      nxt0 = fetch(p, n + T + lane); nxt1 = fetch(p, n + T + 32 + lane);
    }
  }
  __device__ __forceinline__ R sample(const StepParams<R> &, int64_t nloc, int) const {
    R v = R(0);
    if (on) lds_scalar(strip + (uint32_t)(nloc - round0) * (uint32_t)sizeof(R), v);
    return v;
  }
  __device__ __forceinline__ void sample2(const StepParams<R> &, int64_t nloc, int, R &s0, R &s1) const {
    s0 = R(0); s1 = R(0);
    if (on) {
      const uint32_t a = strip + (uint32_t)(nloc - round0) * (uint32_t)sizeof(R);
      lds_scalar(a, s0); lds_scalar(a + (uint32_t)sizeof(R), s1);
    }
  }
};

// ---- Mur (a3), soft source (a4), probe record (a6) and padding hygiene for the threads whose nodes include a
// boundary, the source or a probe.  These threads run alone in their warp (divergent), so what counts is the
// number of instructions on that path: everything that does not change from step to step is worked out once
// per tile (SpecialIdx, 32-bit local indices) and the time loop only dispatches on small integers.
struct SpecialIdx {
  int iL = -1, iR = -1, iS = -1;   // local index (0..C-1) of node 0 / node ncells-1 / the source node, or -1
  int np = 0;                      // probes among this thread's nodes that it records: 0, 1, 2; 3 = more (generic loop)
  int pi0 = -1, pi1 = -1;          // local indices of the first two
  int64_t pr0 = 0, pr1 = 0;        // their record offsets (grid * nprobes + q) * rec_stride; np == 3: k0 and grid
  // absorbing layer, packed into two registers: pml_mask bit i (left layer) / bit 16+i (right layer): local node i is
  // an H node of that layer; pml_j = (jL0 + 64) | (jR0 + 64) << 8 | (jN + 1) << 16, where the layer index of local
  // node i is jL0 + i (left) or jR0 - i (right) and jN is that of the node left of the thread's nodes (-1: none)
  uint32_t pml_mask = 0, pml_j = 0;
  __device__ __forceinline__ int jL0() const { return (int)(pml_j & 255u) - 64; }
  __device__ __forceinline__ int jR0() const { return (int)((pml_j >> 8) & 255u) - 64; }
  __device__ __forceinline__ int jN() const { return (int)((pml_j >> 16) & 255u) - 1; }
  bool any = false;
};

// k0: physical in-grid index of the thread's first node; g: grid; owner: this thread records the probes among
// its nodes (halo threads of a K2 tile do not).
template <typename R, int C, bool PML>
__device__ __forceinline__ SpecialIdx make_special(const StepParams<R> &p, uint32_t flag, int64_t k0, int64_t g, bool owner) {
  SpecialIdx sx;
  if (!flag) return sx;
  if (flag & F_MURL) { const int64_t d = p.cellL - k0; if (d >= 0 && d < C) sx.iL = (int)d; }
  if (flag & F_MURR) { const int64_t d = p.cellR - k0; if (d >= 0 && d < C) sx.iR = (int)d; }
  if (flag & F_SRC)  { const int64_t d = p.cellS - k0; if (d >= 0 && d < C) sx.iS = (int)d; }
  if ((flag & F_PROBE) && owner && p.rec) {
    for (int q = 0; q < p.nprobes; ++q) {
      const int64_t d = p.probe_cell[q] - k0;
      if (d >= 0 && d < C) {
        const int64_t off = (g * p.nprobes + q) * p.rec_stride;
        if (sx.np == 0) { sx.pi0 = (int)d; sx.pr0 = off; }
        else if (sx.np == 1) { sx.pi1 = (int)d; sx.pr1 = off; }
        sx.np = sx.np < 3 ? sx.np + 1 : 3;
      }
    }
  }
  if (sx.np == 3) { sx.pr0 = k0; sx.pr1 = g; }
  if constexpr (PML) if ((flag & F_PML) && p.npml > 0) {
    const int64_t jl = k0 - p.cellL, jr = p.cellR - 1 - k0;      // H node k0+i: jl + i from the left end, jr - i from the right
    uint32_t mL = 0, mR = 0;
#pragma unroll
    for (int i = 0; i < C; ++i) {
      if (jl + i >= 0 && jl + i < p.npml) mL |= 1u << i;
      if (jr - i >= 0 && jr - i < p.npml) mR |= 1u << i;
    }
    int jn = -1;
    if (jl - 1 >= 0 && jl - 1 < p.npml) jn = (int)(jl - 1);
    else if (jr + 1 >= 0 && jr + 1 < p.npml) jn = (int)(jr + 1);
    sx.pml_mask = mL | (mR << 16);
    sx.pml_j = (uint32_t)((mL ? (int)jl : 0) + 64) | ((uint32_t)((mR ? (int)jr : 0) + 64) << 8) | ((uint32_t)(jn + 1) << 16);
  }
  sx.any = (PML && (sx.pml_mask != 0u || sx.jN() >= 0)) || sx.iL >= 0 || sx.iR >= 0 || sx.iS >= 0 || sx.np > 0;
  return sx;
}

// f(integral_constant<int, i>) for the i in [I, C) that equals idx: an else-if chain over compile-time indices,
// so that register arrays are indexed statically and the chain stops at the hit
template <int I, int C, typename F>
__device__ __forceinline__ void at_index(int idx, F &&f) {
  if constexpr (I < C) {
    if (idx == I) f(std::integral_constant<int, I>{});
    else at_index<I + 1, C>(idx, f);
  }
}

// Pre-step of the H nodes inside an absorbing layer (see StepParams): runs BEFORE the ordinary H update, on old E.
// Er: old E of the node right of the thread's nodes.
template <typename R, int C>
__device__ __forceinline__ void pml_pre(const R (&E)[C], R Er, R (&H)[C], const StepParams<R> &p, const SpecialIdx &sx) {
  typedef Arith<R> A;
#pragma unroll
  for (int i = 0; i < C; ++i) {
    const bool l = (sx.pml_mask >> i) & 1u, r = (sx.pml_mask >> (16 + i)) & 1u;
    if (l || r) {
      const int j = l ? sx.jL0() + i : sx.jR0() - i;
      const R dE = A::sub(i + 1 < C ? E[i + 1] : Er, E[i]);
      H[i] = A::fma(p.pml_ha[j], H[i], A::mul(p.pml_hd[j], dE));
    }
  }
}

// E: old values, En: new values (modified), H: new values (padding zeroed).
template <typename R, int C, bool PML>
__device__ __forceinline__ void step_special(const R (&E)[C], R (&En)[C], R (&H)[C], const StepParams<R> &p,
                                             const SpecialIdx &sx, int64_t nloc, R src_now) {
  typedef Arith<R> A;
  constexpr bool pec = PML;       // a conductor behind the absorbing layer instead of Mur
  if (sx.iL >= 0) {   // a3, left end.  The layout puts node 0 at local index 0 or 1, node 1 in the same thread.
    if (sx.iL == 0) En[0] = pec ? R(0) : A::fma(p.mur_m, A::sub(En[1], E[0]), E[1]);
    else { En[1] = pec ? R(0) : A::fma(p.mur_m, A::sub(En[2], E[1]), E[2]); H[0] = R(0); }      // H[0]: padding left of node 0
  }
  if (sx.iR >= 0) {   // a3, right end.  Node ncells-2 is held by the same thread.
    at_index<1, C>(sx.iR, [&](auto ic) {
      constexpr int i = decltype(ic)::value;
      En[i] = pec ? R(0) : A::fma(p.mur_m, A::sub(En[i - 1], E[i]), E[i - 1]);
#pragma unroll
      for (int j = i; j < C; ++j) H[j] = R(0);                                     // H[ncells-1] and padding
    });
  }
  if (sx.iS >= 0)     // a4: soft source (sample of this step, streamed by SourceStream)
    at_index<0, C>(sx.iS, [&](auto ic) { En[decltype(ic)::value] = A::add(En[decltype(ic)::value], src_now); });
  if (sx.np > 0) {    // a6: probe record
    if (sx.np <= 2) {
      at_index<0, C>(sx.pi0, [&](auto ic) { p.rec[sx.pr0 + nloc] = En[decltype(ic)::value]; });
      if (sx.np == 2) at_index<0, C>(sx.pi1, [&](auto ic) { p.rec[sx.pr1 + nloc] = En[decltype(ic)::value]; });
    } else {          // more than two probes in one thread's nodes: generic loop
      for (int q = 0; q < p.nprobes; ++q) {
        const int64_t d = p.probe_cell[q] - sx.pr0;
        if (d >= 0 && d < C)
          at_index<0, C>((int)d, [&](auto ic) { p.rec[(sx.pr1 * p.nprobes + q) * p.rec_stride + nloc] = En[decltype(ic)::value]; });
      }
    }
  }
}

// ---- Mur, source and probes without a branch in the time loop (warp tiles of K2 / K3, and the threads of k3_resident).
// step_special (rketd_device.cuh) dispatches per lane with else-if chains.  In a warp tile whose lanes take different
// chains that costs 700-1000 cycles of branch latency per step (measured, profiles/r02_ncu_k3_wtile.md), which is what
// one warp tile in three pays in the batched configs while every other warp of the chunk waits for it at the next halo
// refresh.  Here the features a warp tile has (SF_* bits, warp-uniform) are a TEMPLATE parameter, chosen once per
// round, and inside the step every feature is straight-line code: the candidate value is computed for each local
// index it could apply to and a per-lane bit mask turns it into a select.  Same arithmetic, same order (Mur left, Mur
// right, source, probes) and the same bits as step_special.  H behind the last node and left of node 0 is zeroed once
// at the end (zero_padding_H) instead of every step: those values feed only nodes that Mur rewrites or whose
// coefficients are zero.
enum : int { SF_MURL = 1, SF_MURR = 2, SF_SRC = 4, SF_PROBE = 8, SF_SLOW = 16,
              SF_FAST = 32 };   // with feature bits: every feature of the warp sits at a fixed local index (WarpSpecial::fast)

struct WarpSpecial {
  int mask = 0;                       // SF_* of the warp tile (warp-uniform)
  bool mL0 = false, mL1 = false;      // this lane holds node 0 at local index 0 / 1
  uint32_t mR = 0, mS = 0;            // bit i: this lane's local node i is node ncells-1 / the source node
  uint32_t mHz = 0;                   // bit i: H of local node i is padding (behind node ncells-1, or left of node 0)
  bool l_p0 = false, l_p1 = false;    // this lane records one / two probes
  bool two_probes = false;            // some lane of the warp records two (warp-uniform)
  int fast = 0;                       // SF_* bits (warp-uniform): the feature sits at the one local index a lane can name
                                      // without a search — node ncells-1 last in its lane, the source / every probe first
};

template <typename R, int C, bool PML>
__device__ __forceinline__ WarpSpecial make_warp_special(const StepParams<R> &p, const SpecialIdx &sx) {
  WarpSpecial ws;
  constexpr unsigned full = 0xffffffffu;
  ws.mL0 = sx.iL == 0; ws.mL1 = sx.iL == 1;
  ws.mR = sx.iR >= 0 ? 1u << sx.iR : 0u;
  ws.mS = sx.iS >= 0 ? 1u << sx.iS : 0u;
  ws.mHz = (sx.iR >= 0 ? (0xffffffffu << sx.iR) & ((1u << C) - 1u) : 0u) | (sx.iL == 1 ? 1u : 0u);
  ws.l_p0 = sx.np >= 1 && sx.np <= 2; ws.l_p1 = sx.np == 2;
  ws.two_probes = __any_sync(full, ws.l_p1);
  ws.fast = (__any_sync(full, sx.iR >= 0 && sx.iR != C - 1) ? 0 : SF_MURR) | (__any_sync(full, sx.iS > 0) ? 0 : SF_SRC) |
            ((ws.two_probes || __any_sync(full, ws.l_p0 && sx.pi0 != 0)) ? 0 : SF_PROBE);
  ws.mask = (__any_sync(full, sx.iL >= 0) ? SF_MURL : 0) | (__any_sync(full, sx.iR >= 0) ? SF_MURR : 0) |
            (__any_sync(full, sx.iS >= 0) ? SF_SRC : 0) | (__any_sync(full, ws.l_p0) ? SF_PROBE : 0);
  // an absorbing layer, or more than two probes among one lane's nodes: the general per-lane path
  if (PML || __any_sync(full, sx.np == 3) || __any_sync(full, sx.pml_mask != 0u)) ws.mask = SF_SLOW;
  return ws;
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

// a3, a4, a6 for the lanes of a warp tile with the features MASK (first-order Mur ends only)
// GUARD (k3_resident, whose instantiations group the features: Mur, source/probe, all): each feature's block sits behind a
// warp-uniform branch on the warp's own features, so that e.g. the warp with node 0 and the source does not pay for the
// C - 1 candidates of the right end.
template <int MASK, typename R, int C, bool GUARD = false>
__device__ __forceinline__ void special_select(const R (&E)[C], R (&En)[C], const StepParams<R> &p, const SpecialIdx &sx,
                                               const WarpSpecial &ws, int64_t nloc, R src_now) {
  typedef Arith<R> A;
  if constexpr ((MASK & SF_FAST) != 0) {
    // Every feature at a fixed local index (node ncells-1 last in its lane, the source and every probe first, at most one
    // probe per lane): one candidate each, turned into a select by the lane's own bits; no branch and no search.  This is
    // every BASELINE config (grid lengths, source and probe cells are multiples of the row).  Same expressions on the same
    // operands as below, in the same order.
    if constexpr ((MASK & SF_MURL) != 0) {
      const R c0 = A::fma(p.mur_m, A::sub(En[1], E[0]), E[1]);
      const R c1 = A::fma(p.mur_m, A::sub(En[2], E[1]), E[2]);
      En[0] = ws.mL0 ? c0 : En[0];
      En[1] = ws.mL1 ? c1 : En[1];
    }
    if constexpr ((MASK & SF_MURR) != 0) {
      const R cand = A::fma(p.mur_m, A::sub(En[C - 2], E[C - 1]), E[C - 2]);
      En[C - 1] = ((ws.mR >> (C - 1)) & 1u) ? cand : En[C - 1];
    }
    if constexpr ((MASK & SF_SRC) != 0) {
      const R sum = A::add(En[0], src_now);
      En[0] = (ws.mS & 1u) ? sum : En[0];
    }
    if constexpr ((MASK & SF_PROBE) != 0) stg_if(ws.l_p0, p.rec + (sx.pr0 + nloc), En[0]);
    return;
  }
  if constexpr ((MASK & SF_MURL) != 0) {      // node 0 sits at local index 0 or 1 (Layout: off), node 1 in the same row
    const R c0 = A::fma(p.mur_m, A::sub(En[1], E[0]), E[1]);
    const R c1 = A::fma(p.mur_m, A::sub(En[2], E[1]), E[2]);
    En[0] = ws.mL0 ? c0 : En[0];
    En[1] = ws.mL1 ? c1 : En[1];
  }
  if constexpr ((MASK & SF_MURR) != 0) {      // node ncells-1 at local index >= 1, node ncells-2 in the same row
    // (descending, so that every candidate sees the interior value of its inward neighbour; one bit of mR is set at most)
    // GUARD: grids whose length is a multiple of the row (every BASELINE config) hold node ncells-1 last in its lane: one
    // candidate instead of C - 1 (the same expression on the same operands: the same bits)
    if (GUARD && (ws.mask & SF_MURR) && (ws.fast & SF_MURR)) {
      const R cand = A::fma(p.mur_m, A::sub(En[C - 2], E[C - 1]), E[C - 2]);
      En[C - 1] = ((ws.mR >> (C - 1)) & 1u) ? cand : En[C - 1];
    } else if (!GUARD || (ws.mask & SF_MURR)) {
#pragma unroll
      for (int i = C - 1; i >= 1; --i) {
        const R cand = A::fma(p.mur_m, A::sub(En[i - 1], E[i]), E[i - 1]);
        En[i] = ((ws.mR >> i) & 1u) ? cand : En[i];
      }
    }
  }
  if constexpr ((MASK & SF_SRC) != 0) {
    if (GUARD && (ws.mask & SF_SRC) && (ws.fast & SF_SRC)) {      // the source node is the first of its lane
      const R sum = A::add(En[0], src_now);
      En[0] = (ws.mS & 1u) ? sum : En[0];
    } else if (!GUARD || (ws.mask & SF_SRC)) {
#pragma unroll
      for (int i = 0; i < C; ++i) {
        const R sum = A::add(En[i], src_now);
        En[i] = ((ws.mS >> i) & 1u) ? sum : En[i];
      }
    }
  }
  if constexpr ((MASK & SF_PROBE) != 0) {      // up to two probes among a lane's nodes; predicated stores, no branch
    if constexpr (!GUARD) {
      const R v0 = select_node<R, C>(En, sx.pi0), v1 = select_node<R, C>(En, sx.pi1);
      stg_if(ws.l_p0, p.rec + (sx.pr0 + nloc), v0);
      stg_if(ws.l_p1, p.rec + (sx.pr1 + nloc), v1);
    } else if ((ws.mask & SF_PROBE) && (ws.fast & SF_PROBE)) {      // every probe of the warp is the first node of its lane
      stg_if(ws.l_p0, p.rec + (sx.pr0 + nloc), En[0]);
    } else if (ws.mask & SF_PROBE) {
      const R v0 = select_node<R, C>(En, sx.pi0);
      stg_if(ws.l_p0, p.rec + (sx.pr0 + nloc), v0);
      if (ws.two_probes) {
        const R v1 = select_node<R, C>(En, sx.pi1);
        stg_if(ws.l_p1, p.rec + (sx.pr1 + nloc), v1);
      }
    }
  }
}

// H of padding nodes (behind node ncells-1, left of node 0): reported as zero; called once after the time loop
template <typename R, int C>
__device__ __forceinline__ void zero_padding_H(R (&H)[C], const WarpSpecial &ws) {
#pragma unroll
  for (int i = 0; i < C; ++i) H[i] = ((ws.mHz >> i) & 1u) ? R(0) : H[i];
}

// ---- one leapfrog step of a thread's C nodes, halos given as OLD values (K1, K3, CTA-tile K2):
// El, Hl: old E and H of the node left of the thread's nodes; Er: old E of the node to the right.
// The left neighbour's new H is recomputed here from old values (same expression, same bits as the
// neighbour's own), so that one exchange of old values per step is enough.
// MASK: SF_* features of the warp (0: none, the boundary/source/probe handling is compiled out; SF_SLOW: step_special's
// per-lane chains; else the select arithmetic of special_select, H padding zeroed by the caller after the time loop).
template <int MASK, bool PML, typename R, int C, typename CF, bool GUARD = false>
__device__ __forceinline__ void step_fields(const R (&E)[C], R (&En)[C], R (&H)[C], const R (&G)[C], const CF &cf, R El,
                                            R Hl, R Er, R nchh, const StepParams<R> &p, const SpecialIdx &sx,
                                            const WarpSpecial &ws, int64_t nloc, R src_now) {
  typedef Arith<R> A;
  constexpr int V = 16 / sizeof(R);
  R Hl_old = Hl;
  if constexpr (MASK == SF_SLOW && PML) {
    if (sx.pml_mask) pml_pre<R, C>(E, Er, H, p, sx);
    // the left neighbour's new H is recomputed below from old values: a layer node needs the same pre-step first
    const int jn = sx.jN();
    if (jn >= 0) Hl_old = A::fma(p.pml_ha[jn], Hl, A::mul(p.pml_hd[jn], A::sub(E[0], El)));
  }
  // a1: H update, eq. (14)
  const R Hl_new = A::fma(nchh, A::sub(E[0], El), Hl_old);
#pragma unroll
  for (int i = 0; i < C; ++i) H[i] = A::fma(nchh, A::sub(i + 1 < C ? E[i + 1] : Er, E[i]), H[i]);
  // a2: E update, eq. (12) with (11) substituted, in the (P, G) form
#pragma unroll
  for (int j = 0; j < C / V; ++j) {
    R cp[V], ch[V];
    cf.template chunk<COEF_P>(j, cp);
    cf.template chunk<COEF_CH>(j, ch);
#pragma unroll
    for (int u = 0; u < V; ++u) {
      const int i = j * V + u;
      En[i] = A::fma(-ch[u], A::sub(H[i], i ? H[i - 1] : Hl_new), A::fma(cp[u], E[i], -G[i]));
    }
  }
  if constexpr (MASK == SF_SLOW) {
    if (sx.any) step_special<R, C, PML>(E, En, H, p, sx, nloc, src_now);
  } else if constexpr (MASK != 0) {
    special_select<MASK, R, C, GUARD>(E, En, p, sx, ws, nloc, src_now);
  }
}

// a5 — eq. (11) in the G form: G' = ka G + Q E with the OLD E (independent of E').
template <typename R, int C, typename CF>
__device__ __forceinline__ void step_current(R (&G)[C], const R (&E)[C], const CF &cf) {
  typedef Arith<R> A;
  constexpr int V = 16 / sizeof(R);
#pragma unroll
  for (int j = 0; j < C / V; ++j) {
    R ka[V], cq[V];
    cf.template chunk<COEF_KA>(j, ka);
    cf.template chunk<COEF_Q>(j, cq);
#pragma unroll
    for (int u = 0; u < V; ++u) G[j * V + u] = A::fma(ka[u], G[j * V + u], A::mul(cq[u], E[j * V + u]));
  }
}

// ---- halo exchange inside a CTA: shuffles inside a warp, shared-memory slots between warps
// (index warp+1; slots 0 and NW+1 stay zero = the outside of the tile), double-buffered by step
// parity so that one __syncthreads per step is enough.  send_halo is called as soon as a step's
// E', H' exist; the G update, the barrier and recv_halo come after, off the critical path.
template <typename R, int NW>
struct HaloSlots {
  R e_first[2][NW + 2], e_last[2][NW + 2], h_last[2][NW + 2];
  __device__ __forceinline__ void clear(int tid) {
    if (tid < 2) {
      e_first[tid][0] = e_first[tid][NW + 1] = R(0);
      e_last[tid][0] = e_last[tid][NW + 1] = R(0);
      h_last[tid][0] = h_last[tid][NW + 1] = R(0);
    }
  }
};

template <typename R, int C, int NW>
__device__ __forceinline__ void send_halo(const R (&E)[C], const R (&H)[C], HaloSlots<R, NW> &hs, int par, int warp,
                                          int lane, R &El, R &Hl, R &Er) {
  El = __shfl_up_sync(0xffffffffu, E[C - 1], 1);
  Hl = __shfl_up_sync(0xffffffffu, H[C - 1], 1);
  Er = __shfl_down_sync(0xffffffffu, E[0], 1);
  if (lane == 0) hs.e_first[par][warp + 1] = E[0];
  if (lane == 31) hs.e_last[par][warp + 1] = E[C - 1];
  if (lane == 31) hs.h_last[par][warp + 1] = H[C - 1];
}
template <typename R, int NW>
__device__ __forceinline__ void recv_halo(const HaloSlots<R, NW> &hs, int par, int warp, int lane, R &El, R &Hl,
                                          R &Er) {
  const R a = hs.e_last[par][warp], b = hs.h_last[par][warp], c = hs.e_first[par][warp + 2];
  El = lane == 0 ? a : El;
  Hl = lane == 0 ? b : Hl;
  Er = lane == 31 ? c : Er;
}

__device__ __forceinline__ void sts_if(bool pred, uint32_t a, double v) {
  asm volatile("{\n.reg .pred p;\nsetp.ne.u32 p, %0, 0;\n@p st.shared.f64 [%1], %2;\n}\n" ::"r"((uint32_t)pred), "r"(a), "d"(v) : "memory");
}
__device__ __forceinline__ void sts_if(bool pred, uint32_t a, float v) {
  asm volatile("{\n.reg .pred p;\nsetp.ne.u32 p, %0, 0;\n@p st.shared.f32 [%1], %2;\n}\n" ::"r"((uint32_t)pred), "r"(a), "f"(v) : "memory");
}
__device__ __forceinline__ void halo_post(int lane, uint32_t a0, double e0, uint32_t a1, double e31, uint32_t a2, double h31) {
  asm volatile("{\n.reg .pred p0, p31;\nsetp.eq.u32 p0, %0, 0;\nsetp.eq.u32 p31, %0, 31;\n"
               "@p0 st.shared.f64 [%1], %2;\n@p31 st.shared.f64 [%3], %4;\n@p31 st.shared.f64 [%5], %6;\n}\n"
               ::"r"(lane), "r"(a0), "d"(e0), "r"(a1), "d"(e31), "r"(a2), "d"(h31) : "memory");
}
// fp32 keeps three separate predicated stores and select-after-load (measured: the fused blocks cost it 6-8 %, while fp64
// gains 6 % on config 3)
__device__ __forceinline__ void halo_post(int lane, uint32_t a0, float e0, uint32_t a1, float e31, uint32_t a2, float h31) {
  sts_if(lane == 0, a0, e0);
  sts_if(lane == 31, a1, e31);
  sts_if(lane == 31, a2, h31);
}
__device__ __forceinline__ void halo_fetch(int lane, uint32_t a0, double &el, uint32_t a1, double &hl, uint32_t a2, double &er) {
  asm volatile("{\n.reg .pred p0, p31;\nsetp.eq.u32 p0, %3, 0;\nsetp.eq.u32 p31, %3, 31;\n"
               "@p0 ld.shared.f64 %0, [%4];\n@p0 ld.shared.f64 %1, [%5];\n@p31 ld.shared.f64 %2, [%6];\n}\n"
               : "+d"(el), "+d"(hl), "+d"(er) : "r"(lane), "r"(a0), "r"(a1), "r"(a2) : "memory");
}
__device__ __forceinline__ void halo_fetch(int lane, uint32_t a0, float &el, uint32_t a1, float &hl, uint32_t a2, float &er) {
  float a, b, c;
  lds_scalar(a0, a);
  lds_scalar(a1, b);
  lds_scalar(a2, c);
  el = lane == 0 ? a : el;
  hl = lane == 0 ? b : hl;
  er = lane == 31 ? c : er;
}
// The same exchange through a 32-bit shared-space address held in a register (wa = address of HaloSlots + warp * sizeof(R),
// taken once before the time loop).  Through the struct reference the compiler rebuilds the generic address of the slots at
// every access (S2UR SR_CgaCtaId + ULEA, 25 cycles of latency three times per step: 8 % of all stall samples of config 5
// fp32, profiles/r02_ncu_k3.md).
template <typename R, int NW>
__device__ __forceinline__ constexpr uint32_t halo_off(int array, int par, int w) {
  return (uint32_t)(((array * 2 + par) * (NW + 2) + w) * (int)sizeof(R));
}
template <typename R, int C, int NW>
__device__ __forceinline__ void send_halo_a(const R (&E)[C], const R (&H)[C], uint32_t wa, int par, int lane, R &El, R &Hl,
                                            R &Er) {
  El = __shfl_up_sync(0xffffffffu, E[C - 1], 1);
  Hl = __shfl_up_sync(0xffffffffu, H[C - 1], 1);
  Er = __shfl_down_sync(0xffffffffu, E[0], 1);
  // predicated stores: no branch in the step; the two lane tests sit inside the block (one setp each)
  halo_post(lane, wa + halo_off<R, NW>(0, par, 1), E[0], wa + halo_off<R, NW>(1, par, 1), E[C - 1],
            wa + halo_off<R, NW>(2, par, 1), H[C - 1]);
}
template <typename R, int NW>
__device__ __forceinline__ void recv_halo_a(uint32_t wa, int par, int lane, R &El, R &Hl, R &Er) {
  // predicated loads straight into the registers the shuffles filled: lane 0 / lane 31 take the neighbour warp's values,
  // every other lane keeps its own (no select behind the load)
  halo_fetch(lane, wa + halo_off<R, NW>(1, par, 0), El, wa + halo_off<R, NW>(2, par, 0), Hl, wa + halo_off<R, NW>(0, par, 2), Er);
}

// ---- PTX wrappers: mbarrier, TMA (cp.async.bulk.tensor)
__device__ __forceinline__ void mbar_init(uint64_t *bar, uint32_t count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count));
}
__device__ __forceinline__ void mbar_expect_tx(uint64_t *bar, uint32_t bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t *bar, uint32_t parity) {
  uint32_t done;
  do {
    asm volatile(
        "{\n.reg .pred p;\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n"
        "selp.u32 %0, 1, 0, p;\n}\n"
        : "=r"(done) : "r"(smem_u32(bar)), "r"(parity) : "memory");
  } while (!done);
}
__device__ __forceinline__ void fence_barrier_init() { asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory"); }
__device__ __forceinline__ void fence_proxy_async_smem() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }

// 3-D tiled TMA load global -> shared, completion on an mbarrier (SASS: UTMALDG)
__device__ __forceinline__ void tma_load_3d(uint32_t dst, const void *tmap, uint64_t *bar, int c0, int c1, int c2) {
  asm volatile(
      "cp.async.bulk.tensor.3d.shared::cluster.global.tile.mbarrier::complete_tx::bytes [%0], [%1, {%3, %4, %5}], [%2];"
      ::"r"(dst), "l"(tmap), "r"(smem_u32(bar)), "r"(c0), "r"(c1), "r"(c2) : "memory");
}
// 3-D tiled TMA store shared -> global (SASS: UTMASTG)
__device__ __forceinline__ void tma_store_3d(const void *tmap, uint32_t src, int c0, int c1, int c2) {
  asm volatile("cp.async.bulk.tensor.3d.global.shared::cta.tile.bulk_group [%0, {%2, %3, %4}], [%1];"
               ::"l"(tmap), "r"(src), "r"(c0), "r"(c1), "r"(c2) : "memory");
}
__device__ __forceinline__ void tma_commit() { asm volatile("cp.async.bulk.commit_group;" ::: "memory"); }
__device__ __forceinline__ void tma_wait_read0() { asm volatile("cp.async.bulk.wait_group.read 0;" ::: "memory"); }
__device__ __forceinline__ void tma_wait0() { asm volatile("cp.async.bulk.wait_group 0;" ::: "memory"); }
__device__ __forceinline__ void prefetch_tmap(const void *tmap) {
  asm volatile("prefetch.tensormap [%0];" ::"l"(tmap) : "memory");
}

}  // namespace rketd
