// rketd_device.cuh — device-side building blocks shared by the three stencil kernels
// (K1 one step per launch, K2 temporal blocking, K3 grid resident).  All three advance
// a "row" (64 bytes = C consecutive nodes held in one thread's registers) with the SAME
// sequence of correctly rounded operations (explicit fma/mul/sub intrinsics, so the
// compiler cannot contract or reassociate differently per kernel): K1, K2 and K3 agree
// bit for bit on the same input, which tests/test_gpu_parity.py checks.
//
// Per node and step (eqs. (14), (12)+(11), (11)):
//   H'[k] = fma(-chh, E[k+1] - E[k], H[k])                                  2 flop-instr
//   E'[k] = fma(-ch, H'[k] - H'[k-1], fma(-cj, J[k], ca * E[k]))            4
//   J'[k] = fma(kc, E'[k], fma(kb, E[k], ka * J[k]))                        3
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace rketd {

constexpr int kRowBytes = 64;       // one thread owns 64 B of every array
constexpr int kMaxProbes = 64;

enum : uint32_t { F_MURL = 1u, F_MURR = 2u, F_SRC = 4u, F_PROBE = 8u };

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
};

// Unpack / pack a 64-B row between C scalars and 16-B vectors.
template <typename R, int C>
__device__ __forceinline__ void vec_to_regs(const typename Arith<R>::Vec &v, R (&r)[C], int j);
template <>
__device__ __forceinline__ void vec_to_regs<double, 8>(const double2 &v, double (&r)[8], int j) {
  r[2 * j] = v.x; r[2 * j + 1] = v.y;
}
template <>
__device__ __forceinline__ void vec_to_regs<float, 16>(const float4 &v, float (&r)[16], int j) {
  r[4 * j] = v.x; r[4 * j + 1] = v.y; r[4 * j + 2] = v.z; r[4 * j + 3] = v.w;
}
__device__ __forceinline__ double2 regs_to_vec(const double (&r)[8], int j) { return make_double2(r[2 * j], r[2 * j + 1]); }
__device__ __forceinline__ float4 regs_to_vec(const float (&r)[16], int j) {
  return make_float4(r[4 * j], r[4 * j + 1], r[4 * j + 2], r[4 * j + 3]);
}

__device__ __forceinline__ void vec_unpack(const double2 &v, double (&o)[2]) { o[0] = v.x; o[1] = v.y; }
__device__ __forceinline__ void vec_unpack(const float4 &v, float (&o)[4]) { o[0] = v.x; o[1] = v.y; o[2] = v.z; o[3] = v.w; }

// Coefficients of one row held in registers.  chunk<a>(j, out) hands out the V = 16/sizeof(R)
// values of array a (0..5 = ca, cj, ch, ka, kb, kc) for nodes j*V .. j*V+V-1 of the row.
template <typename R, int C>
struct CoefRegs {
  static constexpr int V = 16 / sizeof(R);
  R c[6][C];
  template <int a>
  __device__ __forceinline__ void chunk(int j, R (&out)[V]) const {
#pragma unroll
    for (int u = 0; u < V; ++u) out[u] = c[a][j * V + u];
  }
};

// Coefficients of one row held in shared memory: six arrays of NT 64-B rows; the 16-B chunks
// of a row are XOR-swizzled with (row>>1)&3 so that a warp's 128-bit accesses cover all banks.
template <typename R, int C, int NT>
struct CoefSmem {
  static constexpr int V = 16 / sizeof(R);
  const uint8_t *chunk_ptr[C / V];     // address of chunk j of this thread's row in array 0
  __device__ __forceinline__ void init(const uint8_t *array0, int row) {
    const uint32_t sw = (row >> 1) & 3;
#pragma unroll
    for (int j = 0; j < C / V; ++j) chunk_ptr[j] = array0 + row * kRowBytes + ((j ^ sw) << 4);
  }
  template <int a>
  __device__ __forceinline__ void chunk(int j, R (&out)[V]) const {
    typedef typename Arith<R>::Vec Vec;
    vec_unpack(*reinterpret_cast<const Vec *>(chunk_ptr[j] + a * (NT * kRowBytes)), out);
  }
  template <int a>
  __device__ __forceinline__ void store_chunk(int j, const typename Arith<R>::Vec &v) const {
    typedef typename Arith<R>::Vec Vec;
    *reinterpret_cast<Vec *>(const_cast<uint8_t *>(chunk_ptr[j]) + a * (NT * kRowBytes)) = v;
  }
};

// One leapfrog step of one row.  El, Hl: E and H (both OLD) of the node left of the row;
// Er: old E of the node right of the row.  k0: physical in-grid index of the row's first
// node; g: grid; nloc: local step index; owner: this thread records probes in its row.
template <typename R, int C, typename CF>
__device__ __forceinline__ void leapfrog_row(R (&E)[C], R (&H)[C], R (&J)[C], const CF &cf, R El, R Hl, R Er,
                                             const StepParams<R> &p, uint32_t flag, int64_t k0, int64_t g,
                                             int64_t nloc, bool owner) {
  typedef Arith<R> A;
  // a1: H update, eq. (14).  The left neighbour's new H is recomputed here from old values
  // so that one exchange of old values per step is enough.
  const R Hl_new = A::fma(p.nchh, A::sub(E[0], El), Hl);
#pragma unroll
  for (int i = 0; i < C; ++i) H[i] = A::fma(p.nchh, A::sub(i + 1 < C ? E[i + 1] : Er, E[i]), H[i]);
  // a2: E update, eq. (12) with (11) substituted
  R En[C];
  constexpr int V = 16 / sizeof(R);
#pragma unroll
  for (int j = 0; j < C / V; ++j) {
    R ca[V], cj[V], ch[V];
    cf.template chunk<0>(j, ca);
    cf.template chunk<1>(j, cj);
    cf.template chunk<2>(j, ch);
#pragma unroll
    for (int u = 0; u < V; ++u) {
      const int i = j * V + u;
      En[i] = A::fma(-ch[u], A::sub(H[i], i ? H[i - 1] : Hl_new), A::fma(-cj[u], J[i], A::mul(ca[u], E[i])));
    }
  }
  if (flag) {   // rows that hold a boundary node, the source node or a probe (rare)
    if (flag & F_MURL) {   // a3, left end.  The layout guarantees node 1 is in the same row.
#pragma unroll
      for (int i = 0; i < C - 1; ++i)
        if (k0 + i == p.cellL) En[i] = A::fma(p.mur_m, A::sub(En[i + 1], E[i]), E[i + 1]);
#pragma unroll
      for (int i = 0; i < C; ++i)
        if (k0 + i < p.cellL) H[i] = R(0);      // padding left of node 0
    }
    if (flag & F_MURR) {   // a3, right end.  Node ncells-2 is in the same row.
#pragma unroll
      for (int i = 1; i < C; ++i)
        if (k0 + i == p.cellR) En[i] = A::fma(p.mur_m, A::sub(En[i - 1], E[i]), E[i - 1]);
#pragma unroll
      for (int i = 0; i < C; ++i)
        if (k0 + i >= p.cellR) H[i] = R(0);     // H[ncells-1] and padding
    }
    if (flag & F_SRC) {    // a4: soft source
      const R s = p.src_tab[nloc];
#pragma unroll
      for (int i = 0; i < C; ++i)
        if (k0 + i == p.cellS) En[i] = A::add(En[i], s);
    }
    if ((flag & F_PROBE) && owner && p.rec) {   // a6: probe record
      for (int q = 0; q < p.nprobes; ++q) {
        const int64_t d = p.probe_cell[q] - k0;
        if (d >= 0 && d < C) {
          R v = En[0];
#pragma unroll
          for (int i = 1; i < C; ++i)
            if (d == i) v = En[i];
          p.rec[(g * p.nprobes + q) * p.rec_stride + nloc] = v;
        }
      }
    }
  }
  // a5: J update, eq. (11), with the final E'
#pragma unroll
  for (int j = 0; j < C / V; ++j) {
    R ka[V], kb[V], kc[V];
    cf.template chunk<3>(j, ka);
    cf.template chunk<4>(j, kb);
    cf.template chunk<5>(j, kc);
#pragma unroll
    for (int u = 0; u < V; ++u) {
      const int i = j * V + u;
      J[i] = A::fma(kc[u], En[i], A::fma(kb[u], E[i], A::mul(ka[u], J[i])));
      E[i] = En[i];
    }
  }
}

// ---- halo exchange inside a CTA: shuffles inside a warp, shared-memory slots between warps.
// One __syncthreads per step: slots are double-buffered by step parity.
template <typename R, int NW>
struct HaloSlots {
  R e_first[2][NW], e_last[2][NW], h_last[2][NW];
};

template <typename R, int C, int NW>
__device__ __forceinline__ void exchange_halo(const R (&E)[C], const R (&H)[C], HaloSlots<R, NW> &hs, int par,
                                              int warp, int lane, R &El, R &Hl, R &Er) {
  if (NW > 1) {
    if (lane == 0) hs.e_first[par][warp] = E[0];
    if (lane == 31) { hs.e_last[par][warp] = E[C - 1]; hs.h_last[par][warp] = H[C - 1]; }
    __syncthreads();
  }
  El = __shfl_up_sync(0xffffffffu, E[C - 1], 1);
  Hl = __shfl_up_sync(0xffffffffu, H[C - 1], 1);
  Er = __shfl_down_sync(0xffffffffu, E[0], 1);
  if (lane == 0) {
    const bool has = NW > 1 && warp > 0;
    El = has ? hs.e_last[par][has ? warp - 1 : 0] : R(0);
    Hl = has ? hs.h_last[par][has ? warp - 1 : 0] : R(0);
  }
  if (lane == 31) {
    const bool has = NW > 1 && warp < NW - 1;
    Er = has ? hs.e_first[par][has ? warp + 1 : 0] : R(0);
  }
}

// ---- PTX wrappers: shared-memory 128-bit access, mbarrier, TMA (cp.async.bulk.tensor)
__device__ __forceinline__ uint32_t smem_u32(const void *p) { return (uint32_t)__cvta_generic_to_shared(p); }

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
__device__ __forceinline__ void tma_load_3d(void *dst, const void *tmap, uint64_t *bar, int c0, int c1, int c2) {
  asm volatile(
      "cp.async.bulk.tensor.3d.shared::cluster.global.tile.mbarrier::complete_tx::bytes [%0], [%1, {%3, %4, %5}], [%2];"
      ::"r"(smem_u32(dst)), "l"(tmap), "r"(smem_u32(bar)), "r"(c0), "r"(c1), "r"(c2) : "memory");
}
// 3-D tiled TMA store shared -> global (SASS: UTMASTG)
__device__ __forceinline__ void tma_store_3d(const void *tmap, const void *src, int c0, int c1, int c2) {
  asm volatile("cp.async.bulk.tensor.3d.global.shared::cta.tile.bulk_group [%0, {%2, %3, %4}], [%1];"
               ::"l"(tmap), "r"(smem_u32(src)), "r"(c0), "r"(c1), "r"(c2) : "memory");
}
__device__ __forceinline__ void tma_commit() { asm volatile("cp.async.bulk.commit_group;" ::: "memory"); }
__device__ __forceinline__ void tma_wait_read0() { asm volatile("cp.async.bulk.wait_group.read 0;" ::: "memory"); }
__device__ __forceinline__ void tma_wait0() { asm volatile("cp.async.bulk.wait_group 0;" ::: "memory"); }

}  // namespace rketd
