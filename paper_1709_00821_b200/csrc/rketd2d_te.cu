// rketd2d_te.cu — the 2-D TEz polarisation of the RKETD-FDTD leapfrog (include/rketd2d.h, second half; SURVEY.md §8(f)
// NEXT-3 "2-D TMz/TEz"; eqs. (1)-(3) PAPER.md:33-37 in the components Ex, Ey, Hz, Jx, Jy; J per component by eq. (11)
// PAPER.md:68, E per component by eq. (12), H by eq. (14) PAPER.md:84 along each axis).
//
// As in the 1-D and TMz kernels the current is carried as G = cj J - cj kc E per component, with the four per-cell
// arrays P = ca - cj kc, ce (= cex), ka, Q = ka cj kc + cj kb; cey = ce dx/dy.  Per cell and step:
//     Hz'       = fma(chy, Ex[j+1][i] - Ex[j][i], fma(-chx, Ey[j][i+1] - Ey[j][i], Hz))                      4 instr
//     Ex'[j][i] = fma(ce r,  Hz'[j][i] - Hz'[j-1][i], fma(P, Ex, -Gx))      r = dx/dy                        4
//     Ey'[j][i] = fma(-ce,   Hz'[j][i] - Hz'[j][i-1], fma(P, Ey, -Gy))                                       3
//     Gx' = fma(ka, Gx, Q Ex),   Gy' = fma(ka, Gy, Q Ey)                                                     4
// One kernel, k1_te: one fused launch per step, a thread walks four cells of a column, the neighbours' new Hz are
// recomputed from old values (L1/L2 hits), ping-pong buffers; HBM-bound: 14 arrays per step (read Ex, Ey, Hz, Gx, Gy,
// P, ce, ka, Q; write Ex, Ey, Hz, Gx, Gy).  Host side: handle, setup kernels, C ABI.
#include <algorithm>
#include <cmath>
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

constexpr int kMaxProbesTE = 64;
constexpr int kRowsPerThread = 4;

template <typename R>
struct PTE {
  int nx, ny;
  int64_t pitch;
  R nchx, chy, r;            // -dt/(mu0 dx), +dt/(mu0 dy), dx/dy
  R mx, my;                  // first-order Mur (S-1)/(S+1) per axis
  int bc;
  int src_i, src_j, src_c;   // src_i = -1: none
  R src;                     // source sample of this step
  int nprobes;
  int probe_i[kMaxProbesTE], probe_j[kMaxProbesTE], probe_c[kMaxProbesTE];
  R *rec;                    // [nprobes][rec_stride]
  int64_t rec_stride, n0;
  const uint8_t *rowflag;    // [ny]: 1 = the row holds a probe
};

template <typename R>
struct ArraysTE {
  const R *Ex, *Ey, *Hz, *Gx, *Gy, *cP, *cce, *cka, *cQ;
  R *Ex2, *Ey2, *Hz2, *Gx2, *Gy2;
};

// new Hz of cell (i, j) from old values; 0 on the padding row / column and outside the grid
template <typename R>
__device__ __forceinline__ R hz_new(const PTE<R> &p, const ArraysTE<R> &a, int i, int j) {
  typedef Arith<R> A;
  if (i < 0 || j < 0 || i > p.nx - 2 || j > p.ny - 2) return R(0);
  const int64_t k = (int64_t)j * p.pitch + i;
  const R dEy = A::sub(a.Ey[k + 1], a.Ey[k]);
  const R dEx = A::sub(a.Ex[k + p.pitch], a.Ex[k]);
  return A::fma(p.chy, dEx, A::fma(p.nchx, dEy, a.Hz[k]));
}
// interior formulas (callers check the index ranges): hz = new Hz of the cell itself
template <typename R>
__device__ __forceinline__ R ex_interior(const PTE<R> &p, const ArraysTE<R> &a, int i, int j, R hz) {
  typedef Arith<R> A;
  const int64_t k = (int64_t)j * p.pitch + i;
  const R hzd = hz_new(p, a, i, j - 1);
  return A::fma(A::mul(a.cce[k], p.r), A::sub(hz, hzd), A::fma(a.cP[k], a.Ex[k], -a.Gx[k]));
}
template <typename R>
__device__ __forceinline__ R ey_interior(const PTE<R> &p, const ArraysTE<R> &a, int i, int j, R hz) {
  typedef Arith<R> A;
  const int64_t k = (int64_t)j * p.pitch + i;
  const R hzl = hz_new(p, a, i - 1, j);
  return A::fma(-a.cce[k], A::sub(hz, hzl), A::fma(a.cP[k], a.Ey[k], -a.Gy[k]));
}

// ------------------------------------------------------------------------------------------------ k1_te
template <typename R>
__global__ void __launch_bounds__(128) k1_te(const PTE<R> p, const ArraysTE<R> a) {
  typedef Arith<R> A;
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= p.nx) return;
  const int j0 = blockIdx.y * kRowsPerThread, j1 = min(p.ny, j0 + kRowsPerThread);
  const bool mur = p.bc == RKETD2D_BC_MUR;
  for (int j = j0; j < j1; ++j) {
    const int64_t k = (int64_t)j * p.pitch + i;
    const R ex = a.Ex[k], ey = a.Ey[k];
    const R hz = hz_new(p, a, i, j);
    // Ex: interior rows 1..ny-2; rows 0 and ny-1 are tangential to the y edges; column nx-1 is padding
    R exn = R(0);
    if (i <= p.nx - 2) {
      if (j >= 1 && j <= p.ny - 2) {
        exn = ex_interior(p, a, i, j, hz);
      } else if (mur) {
        const int jj = j == 0 ? 1 : p.ny - 2;                    // the inward neighbour along the normal
        const R in_new = ex_interior(p, a, i, jj, hz_new(p, a, i, jj));
        exn = A::fma(p.my, A::sub(in_new, ex), a.Ex[(int64_t)jj * p.pitch + i]);
      }
    }
    // Ey: interior columns 1..nx-2; columns 0 and nx-1 are tangential to the x edges; row ny-1 is padding
    R eyn = R(0);
    if (j <= p.ny - 2) {
      if (i >= 1 && i <= p.nx - 2) {
        eyn = ey_interior(p, a, i, j, hz);
      } else if (mur) {
        const int ii = i == 0 ? 1 : p.nx - 2;
        const R in_new = ey_interior(p, a, ii, j, hz_new(p, a, ii, j));
        eyn = A::fma(p.mx, A::sub(in_new, ey), a.Ey[(int64_t)j * p.pitch + ii]);
      }
    }
    if (i == p.src_i && j == p.src_j) {
      if (p.src_c == RKETD2D_EX) exn = A::add(exn, p.src); else eyn = A::add(eyn, p.src);
    }
    const R ka = a.cka[k], q = a.cQ[k];
    a.Hz2[k] = hz;
    a.Gx2[k] = A::fma(ka, a.Gx[k], A::mul(q, ex));
    a.Gy2[k] = A::fma(ka, a.Gy[k], A::mul(q, ey));
    a.Ex2[k] = exn;
    a.Ey2[k] = eyn;
    if (p.rowflag[j])
      for (int q2 = 0; q2 < p.nprobes; ++q2)
        if (p.probe_i[q2] == i && p.probe_j[q2] == j)
          p.rec[(int64_t)q2 * p.rec_stride + p.n0] = p.probe_c[q2] == RKETD2D_EX ? exn : eyn;
  }
}

// ------------------------------------------------------------------------------------------------ setup kernels
// media -> pitch layout (fp64) + the four kernel coefficients; padding columns get zeros
template <typename R>
__global__ void coef_te_kernel(int nx, int ny, int64_t pitch, const double *__restrict__ wp, const double *__restrict__ nu,
                               double dx, double dt, double eps0, double *wp_p, double *nu_p, R *cP, R *cce, R *cka, R *cQ) {
  const int64_t idx = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (idx >= pitch * ny) return;
  const int64_t j = idx / pitch, i = idx - j * pitch;
  double vP = 0, vce = 0, vka = 0, vQ = 0, w = 0, v = 0;
  if (i < nx) {
    w = wp[j * nx + i];
    v = nu[j * nx + i];
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
// G = cj J - cj kc E (to_G) or J = (G + cj kc E)/cj, in place on the array holding J / G; fp64 arithmetic, one rounding
template <typename R>
__global__ void convert_te_kernel(int nx, int ny, int64_t pitch, const double *__restrict__ wp_p, const double *__restrict__ nu_p,
                                  double dx, double dt, double eps0, const R *__restrict__ E, R *JG, int to_G) {
  const int64_t idx = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (idx >= pitch * ny) return;
  const int64_t i = idx % pitch;
  double v = 0.0;
  if (i < nx) {
    const rketd::Six s = rketd::six_coefficients(wp_p[idx], nu_p[idx], dx, dt, eps0, 0);
    const double ckc = __dmul_rn(s.cj, s.kc);
    v = to_G ? __fma_rn(-ckc, (double)E[idx], __dmul_rn(s.cj, (double)JG[idx]))
             : __ddiv_rn(__fma_rn(ckc, (double)E[idx], (double)JG[idx]), s.cj);
  }
  JG[idx] = (R)v;
}

std::string g_create_error_te;
struct ChunkTE { void *buf; int64_t nsteps; };

}  // namespace

struct rketd2d_te_sim {
  int nx = 0, ny = 0, dtype = 0, esize = 8;
  int64_t pitch = 0;
  double dx = 0, dy = 0, dt = 0;
  cudaStream_t stream = nullptr;
  void *fld[2][5] = {};                // Ex, Ey, Hz, Gx, Gy (ping-pong)
  int cur = 0;
  void *coef[4] = {};                  // P, ce, ka, Q
  double *wp_p = nullptr, *nu_p = nullptr;
  uint8_t *rowflag = nullptr;
  int *d_bad = nullptr;
  bool flags_dirty = true, have_media = false, fields_zero = true, holds_J = false;   // holds_J: arrays 3, 4 hold J, not G
  int bc = RKETD2D_BC_MUR;
  int src_kind = RKETD_SRC_NONE, src_i = -1, src_j = -1, src_c = RKETD2D_EY;
  std::vector<double> src_params;
  std::vector<int> probe_i, probe_j, probe_c;
  std::vector<ChunkTE> chunks;
  int64_t nsamples = 0, step = 0, ctr_launches = 0, ctr_step_launches = 0, state_bytes = 0;
  std::string err;
};

namespace {

int fail_te(rketd2d_te_sim *s, int code, const std::string &msg) {
  if (s) s->err = msg; else g_create_error_te = msg;
  return code;
}
#define CU_TE(s, expr)                                                                            \
  do {                                                                                            \
    cudaError_t e__ = (expr);                                                                     \
    if (e__ != cudaSuccess)                                                                       \
      return fail_te(s, e__ == cudaErrorMemoryAllocation ? RKETD_ENOMEM : RKETD_ECUDA,            \
                     std::string(#expr) + ": " + cudaGetErrorString(e__));                        \
  } while (0)

size_t arr_bytes_te(const rketd2d_te_sim *s) { return (size_t)s->pitch * s->ny * s->esize; }
unsigned blocks_te(int64_t n) { return (unsigned)((n + 255) / 256); }

cudaError_t copy_in_te(const rketd2d_te_sim *s, void *dst, const void *src) {
  const size_t es = (size_t)s->esize;
  return cudaMemcpy2DAsync(dst, (size_t)s->pitch * es, src, (size_t)s->nx * es, (size_t)s->nx * es, (size_t)s->ny,
                           cudaMemcpyDefault, s->stream);
}
cudaError_t copy_out_te(const rketd2d_te_sim *s, void *dst, const void *src) {
  const size_t es = (size_t)s->esize;
  return cudaMemcpy2DAsync(dst, (size_t)s->nx * es, src, (size_t)s->pitch * es, (size_t)s->nx * es, (size_t)s->ny,
                           cudaMemcpyDefault, s->stream);
}
void discard_te(rketd2d_te_sim *s) {
  for (auto &c : s->chunks) cudaFree(c.buf);
  s->chunks.clear();
  s->nsamples = 0;
}
double source_te(const rketd2d_te_sim *s, int64_t step_index) {
  if (s->src_kind == RKETD_SRC_GAUSS_DERIV) {
    const double tau = s->src_params[0], t0 = s->src_params[1], A = s->src_params[2];
    const double u = (double(step_index + 1) * s->dt - t0) / tau;
    return A * u * std::exp(0.5 - 0.5 * u * u);
  }
  if (s->src_kind == RKETD_SRC_TABLE)
    return (step_index >= 0 && step_index < (int64_t)s->src_params.size()) ? s->src_params[(size_t)step_index] : 0.0;
  return 0.0;
}
// arrays 3, 4 of buffer `buf` between J and G (in place), against E in arrays 0, 1 of the CURRENT buffer
cudaError_t convert_te(rketd2d_te_sim *s, int buf, bool to_G) {
  const int64_t n = s->pitch * s->ny;
  for (int c = 0; c < 2; ++c) {
    if (s->dtype == RKETD_F64)
      convert_te_kernel<double><<<blocks_te(n), 256, 0, s->stream>>>(s->nx, s->ny, s->pitch, s->wp_p, s->nu_p, s->dx, s->dt, kEps0,
                                                                     (const double *)s->fld[s->cur][c], (double *)s->fld[buf][3 + c], to_G ? 1 : 0);
    else
      convert_te_kernel<float><<<blocks_te(n), 256, 0, s->stream>>>(s->nx, s->ny, s->pitch, s->wp_p, s->nu_p, s->dx, s->dt, kEps0,
                                                                    (const float *)s->fld[s->cur][c], (float *)s->fld[buf][3 + c], to_G ? 1 : 0);
    s->ctr_launches++;
  }
  return cudaGetLastError();
}

template <typename R>
int run_te(rketd2d_te_sim *s, int64_t nsteps, void *rec) {
  PTE<R> p;
  p.nx = s->nx; p.ny = s->ny; p.pitch = s->pitch;
  p.nchx = (R)(-(s->dt / (kMu0 * s->dx)));
  p.chy = (R)(s->dt / (kMu0 * s->dy));
  p.r = (R)(s->dx / s->dy);
  const double Sx = kC0 * s->dt / s->dx, Sy = kC0 * s->dt / s->dy;
  p.mx = (R)((Sx - 1.0) / (Sx + 1.0));
  p.my = (R)((Sy - 1.0) / (Sy + 1.0));
  p.bc = s->bc;
  const bool has_src = s->src_kind != RKETD_SRC_NONE;
  p.src_i = has_src ? s->src_i : -1; p.src_j = has_src ? s->src_j : -1; p.src_c = s->src_c;
  p.nprobes = (int)s->probe_i.size();
  for (int q = 0; q < p.nprobes; ++q) { p.probe_i[q] = s->probe_i[q]; p.probe_j[q] = s->probe_j[q]; p.probe_c[q] = s->probe_c[q]; }
  p.rec = (R *)rec; p.rec_stride = nsteps;
  p.rowflag = s->rowflag;
  const dim3 grid((unsigned)((s->nx + 127) / 128), (unsigned)((s->ny + kRowsPerThread - 1) / kRowsPerThread));
  for (int64_t n = 0; n < nsteps; ++n) {
    p.n0 = n;
    p.src = has_src ? (R)source_te(s, s->step) : R(0);
    ArraysTE<R> a;
    const int c = s->cur, d = 1 - s->cur;
    a.Ex = (const R *)s->fld[c][0]; a.Ey = (const R *)s->fld[c][1]; a.Hz = (const R *)s->fld[c][2];
    a.Gx = (const R *)s->fld[c][3]; a.Gy = (const R *)s->fld[c][4];
    a.cP = (const R *)s->coef[0]; a.cce = (const R *)s->coef[1]; a.cka = (const R *)s->coef[2]; a.cQ = (const R *)s->coef[3];
    a.Ex2 = (R *)s->fld[d][0]; a.Ey2 = (R *)s->fld[d][1]; a.Hz2 = (R *)s->fld[d][2]; a.Gx2 = (R *)s->fld[d][3]; a.Gy2 = (R *)s->fld[d][4];
    k1_te<R><<<grid, 128, 0, s->stream>>>(p, a);
    CU_TE(s, cudaGetLastError());
    s->cur = d;
    s->step++;
    s->ctr_launches++; s->ctr_step_launches++;
  }
  return RKETD_OK;
}

}  // namespace

extern "C" {

int rketd2d_te_create(rketd2d_te_sim **out, int64_t nx, int64_t ny, double dx, double dy, double dt, int dtype, void *cuda_stream) {
  if (!out) return fail_te(nullptr, RKETD_EINVAL, "out is NULL");
  *out = nullptr;
  if (nx < 3 || ny < 3 || nx > (1 << 30) || ny > (1 << 30)) return fail_te(nullptr, RKETD_EINVAL, "nx, ny must be in 3..2^30");
  if (!(dx > 0) || !(dy > 0) || !(dt > 0)) return fail_te(nullptr, RKETD_EINVAL, "dx, dy, dt must be positive");
  if (kC0 * dt * std::sqrt(1.0 / (dx * dx) + 1.0 / (dy * dy)) > 1.0 + 1e-12)
    return fail_te(nullptr, RKETD_EINVAL, "c dt sqrt(1/dx^2 + 1/dy^2) > 1: unstable");
  if (dtype != RKETD_F64 && dtype != RKETD_F32) return fail_te(nullptr, RKETD_EINVAL, "unknown dtype");
  int ndev = 0;
  if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev < 1) {
    cudaGetLastError();
    return fail_te(nullptr, RKETD_ECUDA, "no usable CUDA device; librketd has no CPU fallback");
  }
  rketd2d_te_sim *s = new rketd2d_te_sim();
  s->nx = (int)nx; s->ny = (int)ny; s->dx = dx; s->dy = dy; s->dt = dt; s->dtype = dtype;
  s->esize = dtype == RKETD_F64 ? 8 : 4;
  s->pitch = (nx + 31) / 32 * 32;
  s->stream = (cudaStream_t)cuda_stream;
  const size_t ab = arr_bytes_te(s);
  auto alloc = [&](void **p, size_t bytes) {
    cudaError_t e = cudaMalloc(p, bytes);
    if (e == cudaSuccess) { e = cudaMemsetAsync(*p, 0, bytes, s->stream); s->state_bytes += (int64_t)bytes; }
    return e;
  };
  cudaError_t e = cudaSuccess;
  for (int b = 0; b < 2 && e == cudaSuccess; ++b)
    for (int f = 0; f < 5 && e == cudaSuccess; ++f) e = alloc(&s->fld[b][f], ab);
  for (int c = 0; c < 4 && e == cudaSuccess; ++c) e = alloc(&s->coef[c], ab);
  if (e == cudaSuccess) e = alloc((void **)&s->wp_p, (size_t)s->pitch * s->ny * 8);
  if (e == cudaSuccess) e = alloc((void **)&s->nu_p, (size_t)s->pitch * s->ny * 8);
  if (e == cudaSuccess) e = alloc((void **)&s->rowflag, (size_t)s->ny);
  if (e == cudaSuccess) e = alloc((void **)&s->d_bad, sizeof(int));
  if (e != cudaSuccess) {
    const int code = e == cudaErrorMemoryAllocation ? RKETD_ENOMEM : RKETD_ECUDA;
    const std::string msg = std::string("device allocation: ") + cudaGetErrorString(e);
    cudaGetLastError();
    rketd2d_te_destroy(s);
    return fail_te(nullptr, code, msg);
  }
  *out = s;
  return RKETD_OK;
}

int rketd2d_te_set_media(rketd2d_te_sim *s, const double *wp, const double *nu) {
  if (!s) return RKETD_EINVAL;
  if (!wp || !nu) return fail_te(s, RKETD_EINVAL, "wp and nu must not be NULL");
  const int64_t n = s->pitch * s->ny, nn = (int64_t)s->nx * s->ny;
  double *d_wp = nullptr, *d_nu = nullptr;
  CU_TE(s, cudaMalloc((void **)&d_wp, (size_t)nn * 8));
  cudaError_t e = cudaMalloc((void **)&d_nu, (size_t)nn * 8);
  if (e != cudaSuccess) { cudaFree(d_wp); CU_TE(s, e); }
  int bad = 0;
  e = cudaMemcpyAsync(d_wp, wp, (size_t)nn * 8, cudaMemcpyDefault, s->stream);
  if (e == cudaSuccess) e = cudaMemcpyAsync(d_nu, nu, (size_t)nn * 8, cudaMemcpyDefault, s->stream);
  if (e == cudaSuccess) e = cudaMemsetAsync(s->d_bad, 0, sizeof(int), s->stream);
  if (e == cudaSuccess) e = rketd::launch_validate_media(d_wp, d_nu, nn, s->d_bad, s->stream);   // read-only, before anything changes
  if (e == cudaSuccess) e = cudaMemcpyAsync(&bad, s->d_bad, sizeof(int), cudaMemcpyDeviceToHost, s->stream);
  if (e == cudaSuccess) e = cudaStreamSynchronize(s->stream);
  if (e != cudaSuccess || bad) {
    cudaFree(d_wp); cudaFree(d_nu);
    CU_TE(s, e);
    return fail_te(s, RKETD_EINVAL, "wp and nu must be finite and non-negative");
  }
  s->ctr_launches++;
  if (s->have_media && !s->fields_zero && !s->holds_J) {      // live fields under the old media: back to J first
    e = convert_te(s, s->cur, false);
    if (e != cudaSuccess) { cudaFree(d_wp); cudaFree(d_nu); CU_TE(s, e); }
    s->holds_J = true;
  }
  s->have_media = false;
  if (s->dtype == RKETD_F64)
    coef_te_kernel<double><<<blocks_te(n), 256, 0, s->stream>>>(s->nx, s->ny, s->pitch, d_wp, d_nu, s->dx, s->dt, kEps0, s->wp_p, s->nu_p,
                                                                (double *)s->coef[0], (double *)s->coef[1], (double *)s->coef[2], (double *)s->coef[3]);
  else
    coef_te_kernel<float><<<blocks_te(n), 256, 0, s->stream>>>(s->nx, s->ny, s->pitch, d_wp, d_nu, s->dx, s->dt, kEps0, s->wp_p, s->nu_p,
                                                               (float *)s->coef[0], (float *)s->coef[1], (float *)s->coef[2], (float *)s->coef[3]);
  e = cudaGetLastError();
  s->ctr_launches++;
  if (e == cudaSuccess) e = cudaStreamSynchronize(s->stream);
  cudaFree(d_wp); cudaFree(d_nu);
  CU_TE(s, e);
  s->have_media = true;
  if (s->holds_J) { CU_TE(s, convert_te(s, s->cur, true)); s->holds_J = false; }
  CU_TE(s, cudaStreamSynchronize(s->stream));
  return RKETD_OK;
}

int rketd2d_te_set_boundary(rketd2d_te_sim *s, int kind) {
  if (!s) return RKETD_EINVAL;
  if (kind != RKETD2D_BC_MUR && kind != RKETD2D_BC_PEC) return fail_te(s, RKETD_EINVAL, "unknown boundary kind");
  s->bc = kind;
  return RKETD_OK;
}

int rketd2d_te_set_source(rketd2d_te_sim *s, int kind, const double *params, int64_t nparams, int64_t i, int64_t j, int component) {
  if (!s) return RKETD_EINVAL;
  if (kind == RKETD_SRC_NONE) { s->src_kind = kind; s->src_params.clear(); s->src_i = s->src_j = -1; return RKETD_OK; }
  if (kind != RKETD_SRC_GAUSS_DERIV && kind != RKETD_SRC_TABLE) return fail_te(s, RKETD_EINVAL, "unknown source kind");
  if (i < 0 || i >= s->nx || j < 0 || j >= s->ny) return fail_te(s, RKETD_EINVAL, "source cell outside the grid");
  if (component != RKETD2D_EX && component != RKETD2D_EY) return fail_te(s, RKETD_EINVAL, "component must be RKETD2D_EX or RKETD2D_EY");
  if (nparams < 0 || (nparams > 0 && !params)) return fail_te(s, RKETD_EINVAL, "bad params");
  if (kind == RKETD_SRC_GAUSS_DERIV && (nparams != 3 || !(params[0] > 0))) return fail_te(s, RKETD_EINVAL, "GAUSS_DERIV needs {tau > 0, t0, amplitude}");
  s->src_kind = kind;
  s->src_params.assign(params, params + nparams);
  s->src_i = (int)i; s->src_j = (int)j; s->src_c = component;
  return RKETD_OK;
}

int rketd2d_te_set_probes(rketd2d_te_sim *s, const int64_t *ijc, int nprobes) {
  if (!s) return RKETD_EINVAL;
  if (nprobes < 0 || nprobes > kMaxProbesTE || (nprobes > 0 && !ijc)) return fail_te(s, RKETD_EINVAL, "0..64 probes");
  for (int q = 0; q < nprobes; ++q)
    if (ijc[3 * q] < 0 || ijc[3 * q] >= s->nx || ijc[3 * q + 1] < 0 || ijc[3 * q + 1] >= s->ny || ijc[3 * q + 2] < 0 || ijc[3 * q + 2] > 1)
      return fail_te(s, RKETD_EINVAL, "probe outside the grid or bad component");
  CU_TE(s, cudaStreamSynchronize(s->stream));
  discard_te(s);
  s->probe_i.clear(); s->probe_j.clear(); s->probe_c.clear();
  for (int q = 0; q < nprobes; ++q) {
    s->probe_i.push_back((int)ijc[3 * q]); s->probe_j.push_back((int)ijc[3 * q + 1]); s->probe_c.push_back((int)ijc[3 * q + 2]);
  }
  s->flags_dirty = true;
  return RKETD_OK;
}

int rketd2d_te_set_fields(rketd2d_te_sim *s, const void *Ex, const void *Ey, const void *Hz, const void *Jx, const void *Jy) {
  if (!s) return RKETD_EINVAL;
  const void *src[5] = {Ex, Ey, Hz, Jx, Jy};
  for (int f = 0; f < 5; ++f) {
    CU_TE(s, cudaMemsetAsync(s->fld[s->cur][f], 0, arr_bytes_te(s), s->stream));
    if (src[f]) CU_TE(s, copy_in_te(s, s->fld[s->cur][f], src[f]));
  }
  s->fields_zero = !Ex && !Ey && !Hz && !Jx && !Jy;
  if (s->have_media) { CU_TE(s, convert_te(s, s->cur, true)); s->holds_J = false; }
  else s->holds_J = true;                      // converted by rketd2d_te_set_media
  CU_TE(s, cudaStreamSynchronize(s->stream));
  return RKETD_OK;
}

int rketd2d_te_get_fields(rketd2d_te_sim *s, void *Ex, void *Ey, void *Hz, void *Jx, void *Jy) {
  if (!s) return RKETD_EINVAL;
  void *dst[3] = {Ex, Ey, Hz};
  for (int f = 0; f < 3; ++f)
    if (dst[f]) CU_TE(s, copy_out_te(s, dst[f], s->fld[s->cur][f]));
  if (Jx || Jy) {
    int from = s->cur;
    if (s->have_media && !s->holds_J) {        // J = (G + cj kc E)/cj in the other buffer's G arrays (scratch between runs)
      from = 1 - s->cur;
      for (int c = 3; c < 5; ++c)
        CU_TE(s, cudaMemcpyAsync(s->fld[from][c], s->fld[s->cur][c], arr_bytes_te(s), cudaMemcpyDeviceToDevice, s->stream));
      CU_TE(s, convert_te(s, from, false));
    }
    if (Jx) CU_TE(s, copy_out_te(s, Jx, s->fld[from][3]));
    if (Jy) CU_TE(s, copy_out_te(s, Jy, s->fld[from][4]));
  }
  CU_TE(s, cudaStreamSynchronize(s->stream));
  return RKETD_OK;
}

int rketd2d_te_run(rketd2d_te_sim *s, int64_t nsteps) {
  if (!s) return RKETD_EINVAL;
  if (nsteps < 0) return fail_te(s, RKETD_EINVAL, "nsteps < 0");
  if (!s->have_media) return fail_te(s, RKETD_ESTATE, "rketd2d_te_run before rketd2d_te_set_media");
  if (nsteps == 0) return RKETD_OK;
  if (s->flags_dirty) {
    std::vector<uint8_t> rf((size_t)s->ny, 0);
    for (size_t q = 0; q < s->probe_j.size(); ++q) rf[(size_t)s->probe_j[q]] = 1;
    CU_TE(s, cudaMemcpyAsync(s->rowflag, rf.data(), rf.size(), cudaMemcpyHostToDevice, s->stream));
    CU_TE(s, cudaStreamSynchronize(s->stream));
    s->flags_dirty = false;
  }
  void *rec = nullptr;
  if (!s->probe_i.empty()) CU_TE(s, cudaMalloc(&rec, s->probe_i.size() * (size_t)nsteps * s->esize));
  s->fields_zero = false;
  const int rc = s->dtype == RKETD_F64 ? run_te<double>(s, nsteps, rec) : run_te<float>(s, nsteps, rec);
  if (rc) {
    if (rec) { cudaStreamSynchronize(s->stream); cudaFree(rec); cudaGetLastError(); }
    return rc;
  }
  if (rec) { s->chunks.push_back({rec, nsteps}); s->nsamples += nsteps; }
  return RKETD_OK;
}

int rketd2d_te_read_probes(rketd2d_te_sim *s, void *out, int64_t out_bytes, int64_t *nsamples) {
  if (!s) return RKETD_EINVAL;
  CU_TE(s, cudaStreamSynchronize(s->stream));
  if (nsamples) *nsamples = s->nsamples;
  if (!out) return RKETD_OK;
  const int64_t np = (int64_t)s->probe_i.size();
  if (out_bytes < np * s->nsamples * s->esize) return fail_te(s, RKETD_EINVAL, "out_bytes too small");
  int64_t off = 0;
  for (auto &c : s->chunks) {
    CU_TE(s, cudaMemcpy2DAsync((char *)out + off * s->esize, (size_t)s->nsamples * s->esize, c.buf, (size_t)c.nsteps * s->esize,
                               (size_t)c.nsteps * s->esize, (size_t)np, cudaMemcpyDefault, s->stream));
    off += c.nsteps;
  }
  CU_TE(s, cudaStreamSynchronize(s->stream));
  return RKETD_OK;
}

int64_t rketd2d_te_get_counter(const rketd2d_te_sim *s, int which) {
  if (!s) return -1;
  switch (which) {
    case RKETD2D_CTR_LAUNCHES: return s->ctr_launches;
    case RKETD2D_CTR_STEP_LAUNCHES: return s->ctr_step_launches;
    case RKETD2D_CTR_STEPS_DONE: return s->step;
    case RKETD2D_CTR_STATE_BYTES: return s->state_bytes;
  }
  return -1;
}

void rketd2d_te_destroy(rketd2d_te_sim *s) {
  if (!s) return;
  cudaStreamSynchronize(s->stream);
  for (int b = 0; b < 2; ++b)
    for (int f = 0; f < 5; ++f) cudaFree(s->fld[b][f]);
  for (int c = 0; c < 4; ++c) cudaFree(s->coef[c]);
  cudaFree(s->wp_p); cudaFree(s->nu_p); cudaFree(s->rowflag); cudaFree(s->d_bad);
  for (auto &c : s->chunks) cudaFree(c.buf);
  cudaGetLastError();
  delete s;
}

const char *rketd2d_te_last_error(const rketd2d_te_sim *s) { return s ? s->err.c_str() : g_create_error_te.c_str(); }

}  // extern "C"
