// rketd_aux.cu — setup and post-processing kernels of librketd:
//   coefficient precompute (eqs. (11), (13) PAPER.md:68, :79),
//   coefficient read-back, the J <-> G change of variable at the boundary, DFT twiddles / accumulation / magnitude (row a7, BASELINE config 5).
#include <math_constants.h>

#include <algorithm>

#include "rketd_coef.cuh"
#include "rketd_internal.h"

namespace rketd {

const double kC0 = 299792458.0;
static const double kPiH = 3.14159265358979323846;
const double kMu0 = 4.0 * kPiH * 1e-7;
const double kEps0 = 1.0 / (kMu0 * kC0 * kC0);

// ---------------------------------------------------------------------------- a0 (phi-functions and the six coefficients: rketd_coef.cuh)
// index of E node k inside an absorbing layer (distance in nodes from the outer end), or -1
__device__ __forceinline__ int pml_index(const PmlE &pml, int64_t k, int64_t ncells) {
  if (pml.npml <= 0) return -1;
  if (k < pml.npml) return (int)k;
  if (k > ncells - 1 - pml.npml) return (int)(ncells - 1 - k);
  return -1;
}
// layer nodes are vacuum with an electric conductivity (media there are ignored): E' = a E - b dH, J = 0
__device__ __forceinline__ Six pml_six(const PmlE &pml, int j) {
  Six s;
  s.ca = pml.a[j]; s.cj = 0.0; s.ch = pml.b[j]; s.ka = 1.0; s.kb = 0.0; s.kc = 0.0;
  return s;
}

// read-only check of user media (finite, non-negative): rketd_set_media / rketd2d_set_media run it BEFORE anything of
// the handle changes, so that a rejected call leaves coefficients and fields untouched
__global__ void validate_media_kernel(const double *__restrict__ wp, const double *__restrict__ nu, int64_t n, int *bad) {
  int flag = 0;
  for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (int64_t)gridDim.x * blockDim.x) {
    const double w = wp[i], v = nu[i];
    if (!(w >= 0.0) || !(v >= 0.0) || isinf(w) || isinf(v)) flag = 1;
  }
  if (flag) atomicOr(bad, 1);
}
cudaError_t launch_validate_media(const double *wp, const double *nu, int64_t n, int *d_bad, cudaStream_t st) {
  const unsigned blocks = (unsigned)std::min<int64_t>((n + 255) / 256, 148 * 16);
  validate_media_kernel<<<blocks, 256, 0, st>>>(wp, nu, n, d_bad);
  return cudaGetLastError();
}

// a0: pads the media into the physical layout and derives the four per-node coefficients the stencil
// kernels use (rketd_device.cuh): P = ca - cj kc, ch, ka, Q = ka (cj kc) + cj kb; padding nodes get zeros.
template <typename R>
__global__ void coefficients_kernel(Layout L, const double *__restrict__ wp, const double *__restrict__ nu,
                                    double dz, double dt, double eps0, int scheme, PmlE pml, double *wp_p, double *nu_p, R *cP, R *cch, R *cka,
                                    R *cQ, int *bad) {
  const int64_t idx = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (idx >= L.gstride * L.nbatch) return;
  const int64_t g = idx / L.gstride, kp = idx - g * L.gstride, k = kp - L.off;
  double vP = 0, vch = 0, vka = 0, vQ = 0, w = 0, v = 0;     // padding nodes: all zero
  if (k >= 0 && k < L.ncells) {
    w = wp[g * L.ncells + k];
    v = nu[g * L.ncells + k];
    if (!(w >= 0.0) || !(v >= 0.0) || isinf(w) || isinf(v)) atomicOr(bad, 1);
    const int jp = pml_index(pml, k, L.ncells);
    const Six s = jp >= 0 ? pml_six(pml, jp) : six_coefficients(w, v, dz, dt, eps0, scheme);
    const double kcp = __dmul_rn(s.cj, s.kc), kbp = __dmul_rn(s.cj, s.kb);
    vP = __dsub_rn(s.ca, kcp);
    vch = s.ch;
    vka = s.ka;
    vQ = __dadd_rn(__dmul_rn(s.ka, kcp), kbp);
  }
  wp_p[idx] = w; nu_p[idx] = v;
  cP[idx] = (R)vP; cch[idx] = (R)vch; cka[idx] = (R)vka; cQ[idx] = (R)vQ;
}

cudaError_t launch_coefficients(int dtype, const Layout &L, const double *wp, const double *nu, double dz,
                                double dt, int scheme, const PmlE &pml, double *wp_p, double *nu_p, void *const coef[kNumCoefArrays],
                                int *d_bad, cudaStream_t st) {
  const int64_t total = L.gstride * L.nbatch;
  const unsigned blocks = (unsigned)((total + 255) / 256);
  if (dtype == 0)
    coefficients_kernel<double><<<blocks, 256, 0, st>>>(L, wp, nu, dz, dt, kEps0, scheme, pml, wp_p, nu_p, (double *)coef[0],
                                                        (double *)coef[1], (double *)coef[2], (double *)coef[3], d_bad);
  else
    coefficients_kernel<float><<<blocks, 256, 0, st>>>(L, wp, nu, dz, dt, kEps0, scheme, pml, wp_p, nu_p, (float *)coef[0],
                                                       (float *)coef[1], (float *)coef[2], (float *)coef[3], d_bad);
  return cudaGetLastError();
}

// rketd_run_from_host, one piece of a single line (nbatch = 1): the physical nodes [i0, i1).  The media of the piece
// were copied straight into wp_p / nu_p (for one grid the padded layout is the user's shifted by L.off) and E0 into E.
// Same arithmetic as coefficients_kernel and current_to_G_kernel with J = 0, so the job is bit-identical to
// rketd_set_media + rketd_set_fields(E0, NULL, NULL).
template <typename R>
__global__ void stage_piece_kernel(Layout L, int64_t i0, int64_t i1, double dz, double dt, double eps0, int scheme, PmlE pml,
                                   double *wp_p, double *nu_p, R *cP, R *cch, R *cka, R *cQ, const R *E, R *G, int *bad) {
  const int64_t idx = i0 + (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (idx >= i1) return;
  const int64_t k = idx - L.off;
  double vP = 0, vch = 0, vka = 0, vQ = 0, vG = 0;
  if (k >= 0 && k < L.ncells) {
    const double w = wp_p[idx], v = nu_p[idx];
    if (!(w >= 0.0) || !(v >= 0.0) || isinf(w) || isinf(v)) atomicOr(bad, 1);
    const int jp = pml_index(pml, k, L.ncells);
    const Six s = jp >= 0 ? pml_six(pml, jp) : six_coefficients(w, v, dz, dt, eps0, scheme);
    const double kcp = __dmul_rn(s.cj, s.kc), kbp = __dmul_rn(s.cj, s.kb);
    vP = __dsub_rn(s.ca, kcp);
    vch = s.ch;
    vka = s.ka;
    vQ = __dadd_rn(__dmul_rn(s.ka, kcp), kbp);
    if (jp < 0) vG = __fma_rn(-kcp, (double)E[idx], __dmul_rn(s.cj, 0.0));
  } else {
    wp_p[idx] = 0.0; nu_p[idx] = 0.0;
  }
  cP[idx] = (R)vP; cch[idx] = (R)vch; cka[idx] = (R)vka; cQ[idx] = (R)vQ;
  G[idx] = (R)vG;
}
cudaError_t launch_stage_piece(int dtype, const Layout &L, int64_t i0, int64_t i1, double dz, double dt, int scheme, const PmlE &pml,
                               double *wp_p, double *nu_p, void *const coef[kNumCoefArrays], const void *E, void *G, int *d_bad,
                               cudaStream_t st) {
  if (i1 <= i0) return cudaSuccess;
  const unsigned blocks = (unsigned)((i1 - i0 + 255) / 256);
  if (dtype == 0)
    stage_piece_kernel<double><<<blocks, 256, 0, st>>>(L, i0, i1, dz, dt, kEps0, scheme, pml, wp_p, nu_p, (double *)coef[0], (double *)coef[1],
                                                       (double *)coef[2], (double *)coef[3], (const double *)E, (double *)G, d_bad);
  else
    stage_piece_kernel<float><<<blocks, 256, 0, st>>>(L, i0, i1, dz, dt, kEps0, scheme, pml, wp_p, nu_p, (float *)coef[0], (float *)coef[1],
                                                      (float *)coef[2], (float *)coef[3], (const float *)E, (float *)G, d_bad);
  return cudaGetLastError();
}

__global__ void six_coefficients_kernel(Layout L, const double *__restrict__ wp_p, const double *__restrict__ nu_p,
                                        double dz, double dt, double eps0, int scheme, PmlE pml, double *out) {
  const int64_t idx = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  const int64_t n = L.ncells * L.nbatch;
  if (idx >= n) return;
  const int64_t g = idx / L.ncells, k = idx - g * L.ncells, src = g * L.gstride + L.off + k;
  const int jp = pml_index(pml, k, L.ncells);
  const Six s = jp >= 0 ? pml_six(pml, jp) : six_coefficients(wp_p[src], nu_p[src], dz, dt, eps0, scheme);
  out[0 * n + idx] = s.ca; out[1 * n + idx] = s.cj; out[2 * n + idx] = s.ch;
  out[3 * n + idx] = s.ka; out[4 * n + idx] = s.kb; out[5 * n + idx] = s.kc;
}
cudaError_t launch_six_coefficients(const Layout &L, const double *wp_p, const double *nu_p, double dz, double dt,
                                    int scheme, const PmlE &pml, double *out, cudaStream_t st) {
  const int64_t n = L.ncells * L.nbatch;
  six_coefficients_kernel<<<(unsigned)((n + 255) / 256), 256, 0, st>>>(L, wp_p, nu_p, dz, dt, kEps0, scheme, pml, out);
  return cudaGetLastError();
}

template <typename R>
__global__ void unpack_coefficients_kernel(Layout L, const R *c0, const R *c1, const R *c2, const R *c3, double *out) {
  const int64_t idx = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  const int64_t n = L.ncells * L.nbatch;
  if (idx >= n) return;
  const int64_t g = idx / L.ncells, k = idx - g * L.ncells, src = g * L.gstride + L.off + k;
  out[0 * n + idx] = (double)c0[src]; out[1 * n + idx] = (double)c1[src];
  out[2 * n + idx] = (double)c2[src]; out[3 * n + idx] = (double)c3[src];
}
cudaError_t launch_unpack_coefficients(int dtype, const Layout &L, void *const c[kNumCoefArrays], double *out,
                                       cudaStream_t st) {
  const int64_t n = L.ncells * L.nbatch;
  const unsigned blocks = (unsigned)((n + 255) / 256);
  if (dtype == 0)
    unpack_coefficients_kernel<double><<<blocks, 256, 0, st>>>(L, (double *)c[0], (double *)c[1], (double *)c[2],
                                                               (double *)c[3], out);
  else
    unpack_coefficients_kernel<float><<<blocks, 256, 0, st>>>(L, (float *)c[0], (float *)c[1], (float *)c[2],
                                                              (float *)c[3], out);
  return cudaGetLastError();
}

// ---------------------------------------------------------------------------- J <-> G
// The kernels carry G = cj J - (cj kc) E instead of J (rketd_device.cuh).  Both conversions run in
// fp64 and round once to the storage type.  Padding nodes: G = 0.
template <typename R>
__global__ void current_to_G_kernel(Layout L, const double *__restrict__ wp_p, const double *__restrict__ nu_p, double dz,
                                    double dt, double eps0, int scheme, PmlE pml, const R *__restrict__ E, R *JG) {
  const int64_t idx = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (idx >= L.gstride * L.nbatch) return;
  const int64_t kp = idx % L.gstride, k = kp - L.off;
  double G = 0.0;
  if (k >= 0 && k < L.ncells && pml_index(pml, k, L.ncells) < 0) {     // layer nodes carry no current: G = 0
    const Six s = six_coefficients(wp_p[idx], nu_p[idx], dz, dt, eps0, scheme);
    G = __fma_rn(-__dmul_rn(s.cj, s.kc), (double)E[idx], __dmul_rn(s.cj, (double)JG[idx]));
  }
  JG[idx] = (R)G;
}
cudaError_t launch_current_to_G(int dtype, const Layout &L, const double *wp_p, const double *nu_p, double dz,
                                double dt, int scheme, const PmlE &pml, const void *E, void *JG, cudaStream_t st) {
  const int64_t total = L.gstride * L.nbatch;
  const unsigned blocks = (unsigned)((total + 255) / 256);
  if (dtype == 0) current_to_G_kernel<double><<<blocks, 256, 0, st>>>(L, wp_p, nu_p, dz, dt, kEps0, scheme, pml, (const double *)E, (double *)JG);
  else current_to_G_kernel<float><<<blocks, 256, 0, st>>>(L, wp_p, nu_p, dz, dt, kEps0, scheme, pml, (const float *)E, (float *)JG);
  return cudaGetLastError();
}

// J = (G + cj kc E)/cj, written in the user's [nbatch][ncells] layout
template <typename R>
__global__ void G_to_current_kernel(Layout L, const double *__restrict__ wp_p, const double *__restrict__ nu_p, double dz,
                                    double dt, double eps0, int scheme, PmlE pml, const R *__restrict__ E, const R *__restrict__ G, R *J_user) {
  const int64_t idx = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  const int64_t n = L.ncells * L.nbatch;
  if (idx >= n) return;
  const int64_t g = idx / L.ncells, k = idx - g * L.ncells, src = g * L.gstride + L.off + k;
  if (pml_index(pml, k, L.ncells) >= 0) { J_user[idx] = R(0); return; }     // layer nodes carry no current
  const Six s = six_coefficients(wp_p[src], nu_p[src], dz, dt, eps0, scheme);
  const double J = __ddiv_rn(__fma_rn(__dmul_rn(s.cj, s.kc), (double)E[src], (double)G[src]), s.cj);
  J_user[idx] = (R)J;
}
cudaError_t launch_G_to_current(int dtype, const Layout &L, const double *wp_p, const double *nu_p, double dz,
                                double dt, int scheme, const PmlE &pml, const void *E, const void *G, void *J_user, cudaStream_t st) {
  const int64_t n = L.ncells * L.nbatch;
  const unsigned blocks = (unsigned)((n + 255) / 256);
  if (dtype == 0)
    G_to_current_kernel<double><<<blocks, 256, 0, st>>>(L, wp_p, nu_p, dz, dt, kEps0, scheme, pml, (const double *)E, (const double *)G, (double *)J_user);
  else
    G_to_current_kernel<float><<<blocks, 256, 0, st>>>(L, wp_p, nu_p, dz, dt, kEps0, scheme, pml, (const float *)E, (const float *)G, (float *)J_user);
  return cudaGetLastError();
}

// ---------------------------------------------------------------------------- a7
// tw[n][m] = (cos theta, sin theta), theta = 2 pi f_m ((step0 + n + 1) dt), evaluated directly
// (no phasor recurrence).
__global__ void twiddle_kernel(const double *__restrict__ freqs, int nfreq, int64_t step0, int64_t nsteps, double dt,
                               double2 *tw) {
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
cudaError_t launch_twiddles(const double *d_freqs, int nfreq, int64_t step0, int64_t nsteps, double dt, double2 *tw,
                            cudaStream_t st) {
  const int64_t n = nsteps * nfreq;
  twiddle_kernel<<<(unsigned)((n + 255) / 256), 256, 0, st>>>(d_freqs, nfreq, step0, nsteps, dt, tw);
  return cudaGetLastError();
}

// X[s][m] += sum_n rec[s][n] (cos - j sin)(theta[n][m]).  Block: 32 series x 64 frequencies;
// thread (m, q) owns 8 series; record tiles of 32 steps are staged through shared memory.
template <typename R>
__global__ void __launch_bounds__(256) dft_accumulate_kernel(const R *__restrict__ rec, int64_t nseries, int64_t nsteps,
                                                             const double2 *__restrict__ tw, int nfreq, double *re,
                                                             double *im) {
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
      if (ser < nseries) {
        re[ser * nfreq + m] += are[i];
        im[ser * nfreq + m] += aim[i];
      }
    }
  }
}
cudaError_t launch_dft_accumulate(int dtype, const void *rec, int64_t nseries, int64_t nsteps, const double2 *tw,
                                  int nfreq, double *re, double *im, cudaStream_t st) {
  dim3 grid((unsigned)((nseries + 31) / 32), (unsigned)((nfreq + 63) / 64));
  if (dtype == 0)
    dft_accumulate_kernel<double><<<grid, 256, 0, st>>>((const double *)rec, nseries, nsteps, tw, nfreq, re, im);
  else
    dft_accumulate_kernel<float><<<grid, 256, 0, st>>>((const float *)rec, nseries, nsteps, tw, nfreq, re, im);
  return cudaGetLastError();
}

template <typename R>
__global__ void dft_magnitude_kernel(const double *re, const double *im, int64_t n, R *out) {
  const int64_t idx = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (idx < n) out[idx] = (R)hypot(re[idx], im[idx]);
}
cudaError_t launch_dft_magnitude(int dtype, const double *re, const double *im, int64_t n, void *out, cudaStream_t st) {
  const unsigned blocks = (unsigned)((n + 255) / 256);
  if (dtype == 0) dft_magnitude_kernel<double><<<blocks, 256, 0, st>>>(re, im, n, (double *)out);
  else dft_magnitude_kernel<float><<<blocks, 256, 0, st>>>(re, im, n, (float *)out);
  return cudaGetLastError();
}

// |R| = |X_slab - X_vac| / |X_vac| at probe pr, |T| = |X_slab| / |X_vac| at probe pt, per grid and frequency
// (reflection and transmission "by Fourier transform" of the records; the vacuum run gives the
// incident spectrum).  Complex differences and moduli in fp64.
__global__ void sweep_rt_kernel(const double *__restrict__ sre, const double *__restrict__ sim, const double *__restrict__ vre,
                                const double *__restrict__ vim, int64_t nbatch, int nprobes, int nfreq, int pr, int pt,
                                double *R, double *T) {
  const int64_t idx = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (idx >= nbatch * nfreq) return;
  const int64_t g = idx / nfreq;
  const int m = (int)(idx - g * nfreq);
  const int64_t ir = (g * nprobes + pr) * nfreq + m, it = (g * nprobes + pt) * nfreq + m;
  const int64_t vr = (int64_t)pr * nfreq + m, vt = (int64_t)pt * nfreq + m;      // vacuum: grid 0
  R[idx] = __ddiv_rn(hypot(__dsub_rn(sre[ir], vre[vr]), __dsub_rn(sim[ir], vim[vr])), hypot(vre[vr], vim[vr]));
  T[idx] = __ddiv_rn(hypot(sre[it], sim[it]), hypot(vre[vt], vim[vt]));
}
cudaError_t launch_sweep_rt(const double *sre, const double *sim, const double *vre, const double *vim, int64_t nbatch,
                            int nprobes, int nfreq, int pr, int pt, double *R, double *T, cudaStream_t st) {
  const int64_t n = nbatch * nfreq;
  sweep_rt_kernel<<<(unsigned)((n + 255) / 256), 256, 0, st>>>(sre, sim, vre, vim, nbatch, nprobes, nfreq, pr, pt, R, T);
  return cudaGetLastError();
}

}  // namespace rketd
