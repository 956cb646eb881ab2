// rketd_coef.cuh — coefficient precompute shared by the 1-D and 2-D setup kernels (
// eqs. (11), (13) PAPER.md:68, :79).  Device code only; included by rketd_aux.cu and rketd2d.cu.
#pragma once
#include <cuda_runtime.h>

namespace rketd {

// phi1(x) = (1 - e^-x)/x and phi2(x) = (e^-x - 1 + x)/x^2 are the two brackets of eq. (11)
// divided by dt; the printed forms are 0/0 at nu = 0 and lose all digits for
// small nu dt, so: expm1 for phi1, Taylor series for phi2 when |x| < 1/2.
// Explicit round-to-nearest intrinsics keep the compiler from fusing or reassociating.
__device__ __forceinline__ void phi_functions(double x, double &p1, double &p2) {
  p1 = (x == 0.0) ? 1.0 : __ddiv_rn(-expm1(-x), x);
  if (fabs(x) < 0.5) {
    double term = 0.5, sum = 0.5;
    for (int j = 1; j <= 40; ++j) {
      term = __ddiv_rn(__dmul_rn(term, -x), (double)(j + 2));
      const double next = __dadd_rn(sum, term);
      if (next == sum) break;
      sum = next;
    }
    p2 = sum;
  } else {
    p2 = __ddiv_rn(__dadd_rn(expm1(-x), x), __dmul_rn(x, x));
  }
}

// The six coefficients of SURVEY a0 for one node, in fp64 with explicit round-to-nearest operations.
struct Six { double ca, cj, ch, ka, kb, kc; };
// scheme 0: eq. (11) (second-order ETD, the paper's method).  scheme 1: eq. (9) PAPER.md:59 (first-order ETD, F held
// at F_n): J' = a J + b E put into eq. (12) gives D = 1, ca = 1 - wp^2 beta dt/2, kb = b, kc = 0.
__device__ __forceinline__ Six six_coefficients(double w, double v, double dz, double dt, double eps0, int scheme) {
  const double x = __dmul_rn(v, dt);
  const double a = exp(-x);
  double p1, p2;
  phi_functions(x, p1, p2);
  const double beta = __dmul_rn(dt, p1);              // (1 - a)/nu
  if (scheme == 1) {
    const double w2 = __dmul_rn(w, w);
    Six s;
    s.ca = __dsub_rn(1.0, __ddiv_rn(__dmul_rn(__dmul_rn(w2, beta), dt), 2.0));
    s.cj = __dmul_rn(__ddiv_rn(dt, __dmul_rn(2.0, eps0)), __dadd_rn(1.0, a));
    s.ch = __ddiv_rn(dt, __dmul_rn(eps0, dz));
    s.ka = a;
    s.kb = __dmul_rn(__dmul_rn(eps0, w2), beta);
    s.kc = 0.0;
    return s;
  }
  const double gamma = __dmul_rn(dt, p2);             // (a - 1 + nu dt)/(nu^2 dt)
  const double w2 = __dmul_rn(w, w);
  const double b = __dmul_rn(__dmul_rn(eps0, w2), beta);
  const double c = __dmul_rn(__dmul_rn(eps0, w2), gamma);
  const double D = __dadd_rn(1.0, __ddiv_rn(__dmul_rn(__dmul_rn(w2, gamma), dt), 2.0));
  Six s;
  s.ca = __dsub_rn(1.0, __ddiv_rn(__ddiv_rn(__dmul_rn(__dmul_rn(w2, beta), dt), 2.0), D));
  s.cj = __ddiv_rn(__dmul_rn(__ddiv_rn(dt, __dmul_rn(2.0, eps0)), __dadd_rn(1.0, a)), D);
  s.ch = __ddiv_rn(__ddiv_rn(dt, __dmul_rn(eps0, dz)), D);
  s.ka = a;
  s.kb = __dsub_rn(b, c);
  s.kc = c;
  return s;
}

}  // namespace rketd
