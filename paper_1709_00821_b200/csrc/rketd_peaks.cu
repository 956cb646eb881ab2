// rketd_peaks.cu — microbenchmarks behind the "alu" roofline of bench.py ("builder must microbenchmark
// DFMA and shared-memory peaks and use the measured values").  rketd_measure_peak (include/rketd.h) runs one of them on
// the current device and reports thread-instructions (or shared-memory bytes) per second, per clock and SM, and the SM
// clock the run held (clock64 against globaltimer).  Nothing here is on the hot path.
//
//   DFMA / FFMA forms: 8 independent accumulator chains per thread, 32 warps per SM, inline PTX so that the number of
//   DISTINCT register source operands of every instruction is what the form says:
//     1 reg   fma a, a, a, a            2 regs  fma a, a, b, a            3 regs  fma a, b, c, a
//     2 regs + constant bank            fma a, b, c[param], a   (the form of the H update: nchh is a kernel parameter)
//   stencil mix: the 7-instruction node update of rketd_device.cuh (H 2, E 3, G 2) on a lane's 64-B row held in
//     registers, neighbours inside the lane, no shuffles, no memory: the issue ceiling of the real instruction mix at
//     the occupancy of the warp-tile kernels (12 warps per SM).
//   LDS.128: every thread reads 16 B per instruction from a conflict-free shared-memory tile.
//   latencies (cycles per operation in out[1]): a chain of dependent DFMAs, a chain of 64-bit shuffles, one leapfrog
//     step of a warp tile (warp_step of rketd_wtile.cuh, no special lanes) with one warp per scheduler, bar.sync of
//     256 threads, the cluster barrier of 8 CTAs x 128 threads.
#include <cuda_runtime.h>
#include <stdint.h>

#include "../../include/rketd.h"
#include "rketd_device.cuh"
#include "rketd_wtile.cuh"

namespace rketd {
namespace {

struct Stamp { unsigned long long clk0, clk1, ns0, ns1; };

__device__ __forceinline__ unsigned long long globaltimer_ns() {
  unsigned long long t;
  asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t));
  return t;
}
// Block 0 times itself: earliest start and latest end over ALL its warps (the scheduler favours the oldest warps, so one
// warp's own span would overstate the rate), clock64 (same SM) against globaltimer.
__device__ __forceinline__ void stamp_begin(Stamp *st) {
  if (blockIdx.x == 0 && (threadIdx.x & 31) == 0) {
    atomicMin(&st->ns0, globaltimer_ns());
    atomicMin(&st->clk0, (unsigned long long)clock64());
  }
}
__device__ __forceinline__ void stamp_end(Stamp *st) {
  if (blockIdx.x == 0 && (threadIdx.x & 31) == 0) {
    atomicMax(&st->clk1, (unsigned long long)clock64());
    atomicMax(&st->ns1, globaltimer_ns());
  }
}

constexpr int kChains = 8, kUnroll = 8;

// FORM: 1, 2, 3 = distinct register sources; 4 = two registers + constant bank
template <int FORM>
__global__ void __launch_bounds__(1024) dfma_kernel(const double *in, double *out, int iters, double k, Stamp *st) {
  double a[kChains], b[kChains], c[kChains];
#pragma unroll
  for (int i = 0; i < kChains; ++i) { a[i] = in[i]; b[i] = in[kChains + i]; c[i] = in[2 * kChains + i]; }
  stamp_begin(st);
  for (int it = 0; it < iters; ++it) {
#pragma unroll
    for (int u = 0; u < kUnroll; ++u)
#pragma unroll
      for (int i = 0; i < kChains; ++i) {
        if (FORM == 1) asm volatile("fma.rn.f64 %0, %0, %0, %0;" : "+d"(a[i]));
        if (FORM == 2) asm volatile("fma.rn.f64 %0, %0, %1, %0;" : "+d"(a[i]) : "d"(b[i]));
        if (FORM == 3) asm volatile("fma.rn.f64 %0, %1, %2, %0;" : "+d"(a[i]) : "d"(b[i]), "d"(c[i]));
        if (FORM == 4) asm volatile("fma.rn.f64 %0, %1, %2, %0;" : "+d"(a[i]) : "d"(b[i]), "d"(k));
      }
  }
  stamp_end(st);
  double s = 0;
#pragma unroll
  for (int i = 0; i < kChains; ++i) s += a[i];
  if (s == 123.456) out[0] = s;
}
template <int FORM>
__global__ void __launch_bounds__(1024) ffma_kernel(const float *in, float *out, int iters, float k, Stamp *st) {
  float a[kChains], b[kChains], c[kChains];
#pragma unroll
  for (int i = 0; i < kChains; ++i) { a[i] = in[i]; b[i] = in[kChains + i]; c[i] = in[2 * kChains + i]; }
  stamp_begin(st);
  for (int it = 0; it < iters; ++it) {
#pragma unroll
    for (int u = 0; u < kUnroll; ++u)
#pragma unroll
      for (int i = 0; i < kChains; ++i) {
        if (FORM == 1) asm volatile("fma.rn.f32 %0, %0, %0, %0;" : "+f"(a[i]));
        if (FORM == 2) asm volatile("fma.rn.f32 %0, %0, %1, %0;" : "+f"(a[i]) : "f"(b[i]));
        if (FORM == 3) asm volatile("fma.rn.f32 %0, %1, %2, %0;" : "+f"(a[i]) : "f"(b[i]), "f"(c[i]));
        if (FORM == 4) asm volatile("fma.rn.f32 %0, %1, %2, %0;" : "+f"(a[i]) : "f"(b[i]), "f"(k));
      }
  }
  stamp_end(st);
  float s = 0;
#pragma unroll
  for (int i = 0; i < kChains; ++i) s += a[i];
  if (s == 123.456f) out[0] = s;
}

// the node update of the stencil kernels (warp_step in rketd_kernels.cu) without its two shuffles
template <typename R>
__global__ void __launch_bounds__(384, 1) mix_kernel(const R *in, R *out, int iters, R nchh, Stamp *st) {
  typedef Arith<R> A;
  constexpr int C = kRowBytes / sizeof(R);
  R E[C], Eb[C], H[C], G[C], cP[C], cch[C], cka[C], cQ[C];
#pragma unroll
  for (int i = 0; i < C; ++i) {
    E[i] = in[i]; H[i] = in[C + i]; G[i] = in[2 * C + i];
    cP[i] = in[3 * C + i]; cch[i] = in[4 * C + i]; cka[i] = in[5 * C + i]; cQ[i] = in[6 * C + i];
  }
  auto step = [&](const R (&Ei)[C], R (&Eo)[C]) {
    H[C - 1] = A::fma(nchh, A::sub(Ei[0], Ei[C - 1]), H[C - 1]);
#pragma unroll
    for (int i = 0; i < C - 1; ++i) H[i] = A::fma(nchh, A::sub(Ei[i + 1], Ei[i]), H[i]);
#pragma unroll
    for (int i = C - 1; i >= 0; --i) {
      const R w = A::mul(cQ[i], Ei[i]);
      const R t = A::fma(cP[i], Ei[i], -G[i]);
      G[i] = A::fma(cka[i], G[i], w);
      Eo[i] = A::fma(-cch[i], A::sub(H[i], H[i ? i - 1 : C - 1]), t);
    }
  };
  stamp_begin(st);
  for (int it = 0; it < iters; ++it) {
    step(E, Eb);
    step(Eb, E);
  }
  stamp_end(st);
  R s = 0;
#pragma unroll
  for (int i = 0; i < C; ++i) s += E[i] + H[i] + G[i];
  if (s == R(123.456)) out[0] = s;
}

__global__ void __launch_bounds__(1024) lds_kernel(float *out, int iters, Stamp *st) {
  extern __shared__ float4 tile[];
  for (int i = threadIdx.x; i < 2048; i += blockDim.x) tile[i] = make_float4((float)i, 1.f, 2.f, 3.f);
  __syncthreads();
  const uint32_t base = smem_u32(tile);
  float4 acc = make_float4(0.f, 0.f, 0.f, 0.f);
  uint32_t off = threadIdx.x * 16u;                            // lane stride 16 B: conflict-free, 512 B per warp instruction
  stamp_begin(st);
  for (int it = 0; it < iters; ++it) {
#pragma unroll
    for (int u = 0; u < 8; ++u) {                              // eight different addresses per iteration
      float4 v;
      lds128(base + ((off + u * 4096u) & 32767u), v);
      acc.x += v.x; acc.y += v.y; acc.z += v.z; acc.w += v.w;
    }
    off += 16u;
  }
  stamp_end(st);
  if (acc.x + acc.y + acc.z + acc.w == 123.456f) out[0] = acc.x;
}

__global__ void lat_dfma_kernel(double *io, int iters, Stamp *st) {
  double a = io[0], b = io[1], c = io[2];
  stamp_begin(st);
  for (int i = 0; i < iters; ++i) {
#pragma unroll
    for (int u = 0; u < 16; ++u) asm volatile("fma.rn.f64 %0, %0, %1, %2;" : "+d"(a) : "d"(b), "d"(c));
  }
  stamp_end(st);
  if (a == 123.456) io[3] = a;
}
__global__ void lat_shfl_kernel(double *io, int iters, Stamp *st) {
  double a = io[threadIdx.x & 3];
  stamp_begin(st);
  for (int i = 0; i < iters; ++i) {
#pragma unroll
    for (int u = 0; u < 16; ++u) a = __shfl_up_sync(0xffffffffu, a, 1);
  }
  stamp_end(st);
  if (a == 123.456) io[3] = a;
}
template <typename R>
__global__ void __launch_bounds__(128, 1) lat_step_kernel(const R *in, R *out, int nsteps, const __grid_constant__ StepParams<R> p, Stamp *st) {
  constexpr int C = kRowBytes / sizeof(R);
  R E[C], H[C], G[C];
  CoefRegs<R, C> cf;
#pragma unroll
  for (int i = 0; i < C; ++i) {
    E[i] = in[i]; H[i] = in[C + i]; G[i] = in[2 * C + i];
#pragma unroll
    for (int a = 0; a < kNumCoef; ++a) cf.c[a][i] = in[(3 + a) * C + i];
  }
  SourceStream<R> src;
  stamp_begin(st);
  warp_steps<0, false, R, C>(E, H, G, cf, p, SpecialIdx(), WarpSpecial(), src, 0, nsteps);
  stamp_end(st);
  R s = 0;
#pragma unroll
  for (int i = 0; i < C; ++i) s += E[i] + H[i] + G[i];
  if (s == R(123.456)) out[0] = s;
}
__global__ void lat_bar_kernel(int iters, Stamp *st) {
  stamp_begin(st);
  for (int i = 0; i < iters; ++i) {
#pragma unroll
    for (int u = 0; u < 16; ++u) asm volatile("bar.sync 0;" ::: "memory");
  }
  stamp_end(st);
}
__global__ void lat_cluster_kernel(int iters, Stamp *st) {
  stamp_begin(st);
  for (int i = 0; i < iters; ++i) {
#pragma unroll
    for (int u = 0; u < 16; ++u)
      asm volatile("barrier.cluster.arrive.release.aligned;\n\tbarrier.cluster.wait.acquire.aligned;" ::: "memory");
  }
  stamp_end(st);
}

}  // namespace
}  // namespace rketd

using namespace rketd;

extern "C" int rketd_measure_peak(int what, int iters, double *out, void *cuda_stream) {
  if (!out || iters < 1 || what < 0 || what > RKETD_LAT_CLUSTER_BARRIER) return RKETD_EINVAL;
  int dev = 0, sms = 0;
  if (cudaGetDevice(&dev) != cudaSuccess || cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess) {
    cudaGetLastError();
    return RKETD_ECUDA;
  }
  cudaStream_t st = (cudaStream_t)cuda_stream;
  void *buf = nullptr;
  Stamp *stamp = nullptr;
  if (cudaMalloc(&buf, 4096) != cudaSuccess || cudaMalloc((void **)&stamp, sizeof(Stamp)) != cudaSuccess) {
    if (buf) cudaFree(buf);
    cudaGetLastError();
    return RKETD_ENOMEM;
  }
  // inputs: small non-trivial values; products stay finite for any iteration count (|b|, |c| << 1)
  double hd[256];
  float hf[256];
  for (int i = 0; i < 256; ++i) { hd[i] = 1e-3 * (double)((i * 37) % 101 - 50) * 1e-2; hf[i] = (float)hd[i]; }
  const bool f32 = (what >= RKETD_PEAK_FFMA_1REG && what <= RKETD_PEAK_FFMA_2REG_CONST) || what == RKETD_PEAK_MIX_F32 || what == RKETD_LAT_STEP_F32;
  cudaMemcpyAsync(buf, f32 ? (const void *)hf : (const void *)hd, f32 ? sizeof(hf) : sizeof(hd), cudaMemcpyHostToDevice, st);
  double per_thread = 0.0;          // thread-instructions (or bytes) per thread
  int threads = 1024, blocks = sms;
  const Stamp stamp0 = {~0ull, 0ull, ~0ull, 0ull};
  for (int rep = 0; rep < 2; ++rep) {          // first pass warms up (clocks, instruction cache)
    cudaMemcpyAsync(stamp, &stamp0, sizeof(Stamp), cudaMemcpyHostToDevice, st);
    switch (what) {
      case RKETD_PEAK_DFMA_1REG: dfma_kernel<1><<<blocks, threads, 0, st>>>((double *)buf, (double *)buf + 300, iters, 1e-9, stamp); break;
      case RKETD_PEAK_DFMA_2REG: dfma_kernel<2><<<blocks, threads, 0, st>>>((double *)buf, (double *)buf + 300, iters, 1e-9, stamp); break;
      case RKETD_PEAK_DFMA_3REG: dfma_kernel<3><<<blocks, threads, 0, st>>>((double *)buf, (double *)buf + 300, iters, 1e-9, stamp); break;
      case RKETD_PEAK_DFMA_2REG_CONST: dfma_kernel<4><<<blocks, threads, 0, st>>>((double *)buf, (double *)buf + 300, iters, 1e-9, stamp); break;
      case RKETD_PEAK_FFMA_1REG: ffma_kernel<1><<<blocks, threads, 0, st>>>((float *)buf, (float *)buf + 300, iters, 1e-6f, stamp); break;
      case RKETD_PEAK_FFMA_2REG: ffma_kernel<2><<<blocks, threads, 0, st>>>((float *)buf, (float *)buf + 300, iters, 1e-6f, stamp); break;
      case RKETD_PEAK_FFMA_3REG: ffma_kernel<3><<<blocks, threads, 0, st>>>((float *)buf, (float *)buf + 300, iters, 1e-6f, stamp); break;
      case RKETD_PEAK_FFMA_2REG_CONST: ffma_kernel<4><<<blocks, threads, 0, st>>>((float *)buf, (float *)buf + 300, iters, 1e-6f, stamp); break;
      case RKETD_PEAK_MIX_F64: threads = 384; mix_kernel<double><<<blocks, threads, 0, st>>>((double *)buf, (double *)buf + 300, iters, -1e-3, stamp); break;
      case RKETD_PEAK_MIX_F32: threads = 384; mix_kernel<float><<<blocks, threads, 0, st>>>((float *)buf, (float *)buf + 300, iters, -1e-3f, stamp); break;
      case RKETD_PEAK_LDS128: lds_kernel<<<blocks, threads, 32768, st>>>((float *)buf + 300, iters, stamp); break;
      case RKETD_LAT_DFMA: lat_dfma_kernel<<<1, 32, 0, st>>>((double *)buf, iters, stamp); break;
      case RKETD_LAT_SHFL64: lat_shfl_kernel<<<1, 32, 0, st>>>((double *)buf, iters, stamp); break;
      case RKETD_LAT_STEP_F64: {
        StepParams<double> sp = {}; sp.nchh = -1e-3;
        lat_step_kernel<double><<<blocks, 128, 0, st>>>((double *)buf, (double *)buf + 300, 16 * iters, sp, stamp);
      } break;
      case RKETD_LAT_STEP_F32: {
        StepParams<float> sp = {}; sp.nchh = -1e-3f;
        lat_step_kernel<float><<<blocks, 128, 0, st>>>((float *)buf, (float *)buf + 300, 16 * iters, sp, stamp);
      } break;
      case RKETD_LAT_BAR_SYNC: lat_bar_kernel<<<1, 256, 0, st>>>(iters, stamp); break;
      case RKETD_LAT_CLUSTER_BARRIER: {
        cudaLaunchConfig_t cfg = {};
        cfg.gridDim = dim3(8); cfg.blockDim = dim3(128); cfg.stream = st;
        cudaLaunchAttribute attr[1];
        attr[0].id = cudaLaunchAttributeClusterDimension;
        attr[0].val.clusterDim.x = 8; attr[0].val.clusterDim.y = 1; attr[0].val.clusterDim.z = 1;
        cfg.attrs = attr; cfg.numAttrs = 1;
        cudaLaunchKernelEx(&cfg, lat_cluster_kernel, iters, stamp);
      } break;
    }
  }
  if (what <= RKETD_PEAK_FFMA_2REG_CONST) per_thread = (double)iters * kUnroll * kChains;
  else if (what == RKETD_PEAK_MIX_F64) per_thread = (double)iters * 2 * 7 * 8;
  else if (what == RKETD_PEAK_MIX_F32) per_thread = (double)iters * 2 * 7 * 16;
  else per_thread = (double)iters * 8 * 16;      // bytes
  Stamp h;
  cudaError_t e = cudaGetLastError();
  if (e == cudaSuccess) e = cudaMemcpyAsync(&h, stamp, sizeof(h), cudaMemcpyDeviceToHost, st);
  if (e == cudaSuccess) e = cudaStreamSynchronize(st);
  cudaFree(buf);
  cudaFree(stamp);
  if (e != cudaSuccess) { cudaGetLastError(); return RKETD_ECUDA; }
  // block 0's own clock and wall time: every block does the same work at the same time (one block per SM)
  const double cycles = (double)(h.clk1 - h.clk0), ns = (double)(h.ns1 - h.ns0);
  out[0] = per_thread * threads * blocks / ns;          // G thread-instructions/s (or GB/s), whole device
  out[1] = per_thread * threads / cycles;               // thread-instructions (or bytes) per clock and SM
  out[2] = 1e3 * cycles / ns;                           // SM clock held during the run, MHz
  out[3] = (double)sms;
  if (what >= RKETD_LAT_DFMA) {                          // latencies: per operation instead of per clock
    const double ops = 16.0 * iters;
    out[0] = ns / ops;                                   // ns per operation
    out[1] = cycles / ops;                               // cycles per operation
  }
  return RKETD_OK;
}
