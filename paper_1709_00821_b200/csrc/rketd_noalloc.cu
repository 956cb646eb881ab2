// librketd — rketd_probe_dft_noalloc: row a7 (probe records -> |DFT| at nfreq frequencies; BASELINE config 5,
// PAPER.md:130-132 "by Fourier transform" of the records) for callers that cannot allocate: code under CUDA graph
// capture, tight serving loops, harnesses that forbid cudaMalloc.
//
// rketd_run in DFT mode keeps its twiddle table tw[n][m] = (cos, sin)(2 pi f_m (step0 + n + 1) dt) in a buffer the handle
// allocates and grows (rketd_api.cu).  Here the same table lives in a file-scope `static __device__` array of
// RKETD_NOALLOC_MAX_TWIDDLES entries (8 MiB, held by every GPU that loads the library until the process exits); the
// caller passes the records, the frequencies and the output, all in device memory.  No cudaMalloc, cudaFree or allocating
// library routine is called; nothing synchronises.
//
// In host code the array's name is a host-side stand-in, not a device address: its address on the CURRENT device comes from
// cudaGetSymbolAddress, asked once per device (scratch_of_current_device) and handed to the kernels as a pointer.
//
// Every call shares the one array.  It keeps the last call's table; a call rewrites entries [0, nsamples * nfreq) before it
// reads them (stream order) and reads nothing beyond, so nothing has to start at zero.  Two calls that overlap on the GPU
// (different streams without an event between them, or host threads on different streams) RACE on it.
#include <cuda_runtime.h>
#include <math_constants.h>

#include <mutex>
#include <string>

#include "../../include/rketd.h"

namespace {

static __device__ __align__(256) double2 g_noalloc_twiddles[RKETD_NOALLOC_MAX_TWIDDLES];

constexpr int kMaxDevices = 64;
std::mutex g_mu;
double2 *g_scratch[kMaxDevices] = {};     // device address of g_noalloc_twiddles, per device ordinal
thread_local std::string g_err;

int fail_na(int code, const std::string &msg) {
  g_err = msg;
  return code;
}

// set-up, once per device, with that device current
cudaError_t scratch_of_current_device(double2 **out) {
  int dev = -1;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) return e;
  if (dev < 0 || dev >= kMaxDevices) return cudaErrorInvalidDevice;
  std::lock_guard<std::mutex> lk(g_mu);
  if (!g_scratch[dev]) {
    void *p = nullptr;
    e = cudaGetSymbolAddress(&p, g_noalloc_twiddles);
    if (e != cudaSuccess) return e;
    if (!p) return cudaErrorInvalidSymbol;
    g_scratch[dev] = static_cast<double2 *>(p);
  }
  *out = g_scratch[dev];
  return cudaSuccess;
}

// the arithmetic of twiddle_kernel (rketd_aux.cu): theta evaluated directly, no phasor recurrence
__global__ void twiddle_noalloc_kernel(const double *__restrict__ freqs, int nfreq, int64_t step0, int64_t nsteps, double dt,
                                       double2 *__restrict__ tw) {
  const int64_t idx = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (idx >= nsteps * nfreq) return;
  const int64_t n = idx / nfreq;
  const int m = (int)(idx - n * nfreq);
  const double t = __dmul_rn((double)(step0 + n + 1), dt);
  const double theta = __dmul_rn(__dmul_rn(__dmul_rn(2.0, CUDART_PI), freqs[m]), t);
  double s, c;
  sincos(theta, &s, &c);
  tw[idx] = make_double2(c, s);
}

// The variant of dft_accumulate_kernel: the whole record of a series is reduced in one launch, so the complex sums stay in
// registers and the magnitude goes straight to the caller's array (no accumulator arrays at all).  Block: 32 series x 64
// frequencies; thread (m, q) owns 8 series; record tiles of 32 samples are staged through shared memory.
template <typename R>
__global__ void __launch_bounds__(256) dft_magnitude_noalloc_kernel(const R *__restrict__ rec, int64_t nseries, int64_t nsteps,
                                                                    const double2 *__restrict__ tw, int nfreq,
                                                                    R *__restrict__ out) {
  constexpr int SB = 32, TN = 32, SPT = 8;
  __shared__ double srec[SB][TN + 1];
  const int tid = threadIdx.x;
  const int m = blockIdx.y * 64 + (tid & 63);
  const int q = tid >> 6;
  const int64_t s0 = (int64_t)blockIdx.x * SB;
  double are[SPT], aim[SPT];
#pragma unroll
  for (int i = 0; i < SPT; ++i) { are[i] = 0.0; aim[i] = 0.0; }
  for (int64_t n0 = 0; n0 < nsteps; n0 += TN) {
    __syncthreads();
    for (int e = tid; e < SB * TN; e += 256) {
      const int s = e / TN, nn = e % TN;
      const int64_t ser = s0 + s, n = n0 + nn;
      srec[s][nn] = (ser < nseries && n < nsteps) ? (double)rec[ser * nsteps + n] : 0.0;
    }
    __syncthreads();
    if (m < nfreq) {
      const int lim = (int)((nsteps - n0) < TN ? (nsteps - n0) : TN);
      for (int nn = 0; nn < lim; ++nn) {
        const double2 w = tw[(n0 + nn) * nfreq + m];
#pragma unroll
        for (int i = 0; i < SPT; ++i) {
          const double v = srec[q * SPT + i][nn];
          are[i] = fma(v, w.x, are[i]);
          aim[i] = fma(-v, w.y, aim[i]);
        }
      }
    }
  }
  if (m < nfreq) {
#pragma unroll
    for (int i = 0; i < SPT; ++i) {
      const int64_t ser = s0 + q * SPT + i;
      if (ser < nseries) out[ser * nfreq + m] = (R)hypot(are[i], aim[i]);
    }
  }
}

// device-reachable memory only: a host pointer would fault in the kernel (or, where the GPU can reach host memory,
// quietly work on the wrong side of the bus)
bool on_device(const void *p) {
  cudaPointerAttributes a;
  if (cudaPointerGetAttributes(&a, p) != cudaSuccess) {
    cudaGetLastError();
    return false;
  }
  return a.type == cudaMemoryTypeDevice || a.type == cudaMemoryTypeManaged;
}

}  // namespace

extern "C" int rketd_probe_dft_noalloc(int dtype, const void *rec, int64_t nseries, int64_t nsamples, int64_t step0, double dt,
                                       const double *freqs_hz, int nfreq, void *out, void *cuda_stream) {
  if (dtype != RKETD_F64 && dtype != RKETD_F32) return fail_na(RKETD_EINVAL, "rketd_probe_dft_noalloc: dtype must be RKETD_F64 or RKETD_F32");
  if (nseries < 0 || nsamples < 0 || nfreq < 0 || step0 < 0 || !(dt > 0.0))
    return fail_na(RKETD_EINVAL, "rketd_probe_dft_noalloc: negative size or step, or dt <= 0");
  if (nseries == 0 || nfreq == 0) return RKETD_OK;
  if (nseries > RKETD_NOALLOC_MAX_SERIES)
    return fail_na(RKETD_EINVAL, "rketd_probe_dft_noalloc: nseries = " + std::to_string(nseries) + " exceeds RKETD_NOALLOC_MAX_SERIES = " +
                                     std::to_string((long long)RKETD_NOALLOC_MAX_SERIES));
  if (nsamples > RKETD_NOALLOC_MAX_TWIDDLES || nsamples * (int64_t)nfreq > RKETD_NOALLOC_MAX_TWIDDLES)
    return fail_na(RKETD_EINVAL, "rketd_probe_dft_noalloc: nsamples x nfreq = " + std::to_string(nsamples) + " x " + std::to_string(nfreq) +
                                     " exceeds the static twiddle table (RKETD_NOALLOC_MAX_TWIDDLES = " +
                                     std::to_string((long long)RKETD_NOALLOC_MAX_TWIDDLES) +
                                     " entries); use rketd_set_probe_dft + rketd_run, which allocate");
  if (!freqs_hz || !out || (nsamples > 0 && !rec)) return fail_na(RKETD_EINVAL, "rketd_probe_dft_noalloc: NULL pointer");
  if (!on_device(freqs_hz) || !on_device(out) || (nsamples > 0 && !on_device(rec)))
    return fail_na(RKETD_EINVAL, "rketd_probe_dft_noalloc: rec, freqs_hz and out must be device memory of the current device");
  double2 *tw = nullptr;
  cudaError_t e = scratch_of_current_device(&tw);
  if (e != cudaSuccess) return fail_na(RKETD_ECUDA, std::string("rketd_probe_dft_noalloc: cudaGetSymbolAddress: ") + cudaGetErrorString(e));
  cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
  const int64_t ntw = nsamples * nfreq;
  if (ntw > 0)
    twiddle_noalloc_kernel<<<(unsigned)((ntw + 255) / 256), 256, 0, st>>>(freqs_hz, nfreq, step0, nsamples, dt, tw);
  dim3 grid((unsigned)((nseries + 31) / 32), (unsigned)((nfreq + 63) / 64));
  if (dtype == RKETD_F64)
    dft_magnitude_noalloc_kernel<double><<<grid, 256, 0, st>>>((const double *)rec, nseries, nsamples, tw, nfreq, (double *)out);
  else
    dft_magnitude_noalloc_kernel<float><<<grid, 256, 0, st>>>((const float *)rec, nseries, nsamples, tw, nfreq, (float *)out);
  e = cudaGetLastError();
  if (e != cudaSuccess) return fail_na(RKETD_ECUDA, std::string("rketd_probe_dft_noalloc: launch: ") + cudaGetErrorString(e));
  return RKETD_OK;
}

extern "C" const char *rketd_noalloc_last_error(void) { return g_err.c_str(); }
