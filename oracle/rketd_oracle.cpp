// ============================================================================
// oracle/rketd_oracle.cpp  —  TEST INFRASTRUCTURE, NOT PRODUCT CODE.
//
// Plain, serial, fp64 restatement of the 1-D RKETD-FDTD leapfrog of
// arxiv 1709.00821 (§II, eqs. (11), (12), (14)), plus
// the parts BASELINE.json's north_star adds around it (Mur-1 ABC, soft source,
// probe records, probe DFT).  It follows SURVEY.md §8(c) S0-S6 step by step, in
// that order, with no blocking, fusion or reordering, so that it can be checked
// against the paper by eye.
//
// Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl
// reference legs may build, load or call this file.  It shares no code, header,
// table or helper with paper_1709_00821_b200/ (the CUDA path) and neither
// imports the other.  Build: g++ -O2 -ffp-contract=off [-fopenmp] -shared -fPIC.
// The OpenMP build is the same source; it parallelises the k loops of a single
// grid or the grid loop of a batch, has no reductions, and is therefore
// bit-identical to the serial build (pin P9).
//
// Parity pins (tests/test_oracle_pins.py): P1 Courant-1 translation, P2 eq.(12)
// residual with eq.(11) literal, P3 discrete energy, P4 RK4 brute force of
// eq.(6), P5 analytic slab R/T, P6 stability, P7 domain of dependence, P8 DFT,
// P9 OpenMP == serial, and the phi-functions against 50-digit arithmetic.
// The 2-D TMz generalisation at the end of the file has its own pins Q1-Q9
// (tests/test_oracle2d_pins.py), listed above it, and the 2-D TEz polarisation after it pins R1-R7
// (tests/test_oracle2d_te_pins.py).  Nothing in this file is "parity unpinned".
//
// Notation: N E-nodes k = 0..N-1; E[k] = Ex(k dz) at integer steps;
// H[k] = Hy((k+1/2) dz) at half steps, k = 0..N-2 (H[N-1] is padding, kept 0);
// J[k] = Jx(k dz) collocated with E in space and time (eq. (11)/(12) use J^n,
// J^{n+1}: PAPER.md:68, :74).  x = nu dt, a = exp(-x).
// ============================================================================
#include <cmath>
#include <cstdint>
#include <cstring>
#include <vector>

namespace {

// the paper gives no values; both sides hard-code SI values.
const double kC0 = 299792458.0;                 // m/s
const double kPi = 3.14159265358979323846;
const double kMu0 = 4.0 * kPi * 1e-7;           // H/m
const double kEps0 = 1.0 / (kMu0 * kC0 * kC0);  // F/m

// phi1(x) = (1 - e^-x)/x,  phi2(x) = (e^-x - 1 + x)/x^2   (the two brackets of
// eq. (11), divided by dt and by dt resp.).  The literal forms are
// 0/0 at x = 0 and lose digits for small x, hence expm1 / a series.
void phi(double x, double* phi1, double* phi2) {
  *phi1 = (x == 0.0) ? 1.0 : -std::expm1(-x) / x;
  if (std::fabs(x) < 0.5) {
    // sum_{j>=0} (-x)^j / (j+2)!
    double term = 0.5, sum = 0.5;
    for (int j = 1; j <= 40; ++j) {
      term = term * (-x) / double(j + 2);
      double next = sum + term;
      if (next == sum) break;
      sum = next;
    }
    *phi2 = sum;
  } else {
    *phi2 = (std::expm1(-x) + x) / (x * x);
  }
}

struct Coef {
  std::vector<double> ca, cj, ch, ka, kb, kc;
  double chh, m;
};

// S0 — the six per-cell coefficients of SURVEY §8(a) row a0.  Derivation:
// write (11) as J' = a J + (b-c) E + c E', put it into (12), collect E'
// (this is eq. (13) with the 1/D the print drops restored — SURVEY G1).
//
// scheme 1 — the first-order ETD variant the paper derives but does not use (eqs. (8)-(9), PAPER.md:55-60;
// SURVEY §8(f) NEXT-4): F held at F_n over the step, J' = a J + b E.  Put into (12): D = 1,
// ca = 1 - wp^2 beta dt/2, cj = (dt/2 eps0)(1 + a), ch = dt/(eps0 dz), ka = a, kb = b, kc = 0.
void coefficients(int64_t n, const double* wp, const double* nu, double dz, double dt,
                  double* ca, double* cj, double* ch, double* ka, double* kb, double* kc,
                  double* chh, double* m, int scheme = 0) {
  for (int64_t k = 0; k < n && scheme == 1; ++k) {
    const double x = nu[k] * dt;
    const double a = std::exp(-x);
    double p1, p2;
    phi(x, &p1, &p2);
    const double beta = dt * p1;                 // (1 - a)/nu
    const double wp2 = wp[k] * wp[k];
    ca[k] = 1.0 - wp2 * beta * dt / 2.0;
    cj[k] = (dt / (2.0 * kEps0)) * (1.0 + a);
    ch[k] = dt / (kEps0 * dz);
    ka[k] = a;
    kb[k] = kEps0 * wp2 * beta;                  // eq. (9): F_n (1 - a)/nu
    kc[k] = 0.0;
  }
  for (int64_t k = 0; k < n && scheme == 0; ++k) {
    const double x = nu[k] * dt;
    const double a = std::exp(-x);
    double p1, p2;
    phi(x, &p1, &p2);
    const double beta = dt * p1;                 // (1 - a)/nu
    const double gamma = dt * p2;                // (a - 1 + x)/(nu^2 dt)
    const double wp2 = wp[k] * wp[k];
    const double b = kEps0 * wp2 * beta;
    const double c = kEps0 * wp2 * gamma;
    const double D = 1.0 + wp2 * gamma * dt / 2.0;
    ca[k] = 1.0 - (wp2 * beta * dt / 2.0) / D;
    cj[k] = (dt / (2.0 * kEps0)) * (1.0 + a) / D;
    ch[k] = (dt / (kEps0 * dz)) / D;
    ka[k] = a;
    kb[k] = b - c;
    kc[k] = c;
  }
  *chh = dt / (kMu0 * dz);                        // eq. (14), PAPER.md:84 ("dx" is dz, G3)
  const double S = kC0 * dt / dz;
  *m = (S - 1.0) / (S + 1.0);                     // Mur first order
}

// Source sample added to E^{n+1}: s[n+1], s[i] = s(i dt).
// kind 0: eq. (15) PAPER.md:125 normalised to unit peak:
//   s(t) = A ((t-t0)/tau) exp(1/2 - (t-t0)^2/(2 tau^2)),  params = {tau, t0, A}.
// kind 1: table; params[i] is the value added at step index i (0-based), 0 beyond.
double source_sample(int kind, const double* params, int64_t nparams, int64_t step_index, double dt) {
  if (kind == 0) {
    const double tau = params[0], t0 = params[1], A = params[2];
    const double t = double(step_index + 1) * dt;
    const double u = (t - t0) / tau;
    return A * u * std::exp(0.5 - 0.5 * u * u);
  }
  if (kind == 1) return (step_index >= 0 && step_index < nparams) ? params[step_index] : 0.0;
  return 0.0;
}

}  // namespace

extern "C" {

void oracle_constants(double* c0, double* mu0, double* eps0) {
  *c0 = kC0; *mu0 = kMu0; *eps0 = kEps0;
}

void oracle_phi(double x, double* phi1, double* phi2) { phi(x, phi1, phi2); }

// scheme: 0 = second-order ETD, eq. (11) (the paper's method); 1 = first-order ETD, eq. (9)
int oracle_coefficients_scheme(int64_t n, const double* wp, const double* nu, double dz, double dt,
                               double* ca, double* cj, double* ch, double* ka, double* kb, double* kc,
                               double* chh, double* m, int scheme) {
  if (n < 0 || dz <= 0 || dt <= 0 || scheme < 0 || scheme > 1) return 1;
  coefficients(n, wp, nu, dz, dt, ca, cj, ch, ka, kb, kc, chh, m, scheme);
  return 0;
}

int oracle_coefficients(int64_t n, const double* wp, const double* nu, double dz, double dt,
                        double* ca, double* cj, double* ch, double* ka, double* kb, double* kc,
                        double* chh, double* m) {
  return oracle_coefficients_scheme(n, wp, nu, dz, dt, ca, cj, ch, ka, kb, kc, chh, m, 0);
}

double oracle_source(int kind, const double* params, int64_t nparams, int64_t step_index, double dt) {
  return source_sample(kind, params, nparams, step_index, dt);
}

// Advance nbatch independent grids by nsteps steps, continuing from global step
// index step0 (so that repeated calls continue the same run).
//   wp, nu          [nbatch][ncells]  rad/s, 1/s
//   E, H, J         [nbatch][ncells]  in/out (state at step step0 in, step0+nsteps out)
//   probes          [nprobes]         cells, the same in every grid (may be NULL if nprobes==0)
//   rec, recJ       [nbatch][nprobes][nsteps]  E' resp. J' at the probe cells, sample n <-> time
//                   (step0+n+1) dt; either may be NULL
//   freqs           [nfreq] Hz; dft_re/dft_im [nbatch][nprobes][nfreq] accumulators (in/out), NULL = off
//   boundary        0 = Mur first order (a3), 1 = PEC (E[0] = E[N-1] = 0; oracle-only, for pin P3)
//   scheme          0 = eq. (11) (second-order ETD), 1 = eq. (9) (first-order ETD): only S0 differs
//   boundary 2      PML (the paper's choice: "PML absorbing boundary conditions [29] ... at both
//                   ends of 5 cells").  The paper gives no conductivity profile; the reading
//                    is Berenger's layer at normal incidence with polynomial grading:
//                     E nodes k < npml (and mirrored at the right end): depth rho = (npml - k)/npml,
//                     H nodes k + 1/2, k < npml:                        depth rho = (npml - k - 1/2)/npml,
//                     sigma(rho) = sigma_max rho^m,  sigma_max = -(m + 1) eps0 c ln(R0) / (2 npml dz),
//                     matched magnetic conductivity sigma* = sigma mu0/eps0; with s = sigma dt / (2 eps0):
//                       E'[k] = ((1 - s)/(1 + s)) E[k] - ((dt/(eps0 dz))/(1 + s)) (H[k] - H[k-1])     (PML E nodes: vacuum,
//                       H'[k] = ((1 - s)/(1 + s)) H[k] - ((dt/(mu0 dz))/(1 + s)) (E[k+1] - E[k])       media there ignored)
//                   and a perfect conductor behind the layer: E[0] = E[N-1] = 0.  In 1-D the split fields of [29]
//                   have one non-trivial part each, so "split" and "unsplit" coincide.
int oracle_run_bc(int64_t ncells, int64_t nbatch, double dz, double dt,
                  const double* wp, const double* nu, double* E, double* H, double* J,
                  int src_kind, const double* src_params, int64_t nparams, int64_t src_cell,
                  const int64_t* probes, int nprobes, int64_t step0, int64_t nsteps,
                  double* rec, double* recJ,
                  const double* freqs, int nfreq, double* dft_re, double* dft_im,
                  int boundary, int scheme, int npml, double pml_m, double pml_R0) {
  const int64_t N = ncells;
  if (N < 3 || nbatch < 1 || nsteps < 0 || dz <= 0 || dt <= 0 || scheme < 0 || scheme > 1) return 1;
  if (boundary == 2 && (npml < 1 || 2 * (int64_t)npml + 1 > N || !(pml_R0 > 0.0) || pml_R0 > 1.0 || pml_m < 0.0)) return 1;
  // PML profile (the same for every grid): index j = distance in nodes from the outer end
  std::vector<double> pe_a(npml > 0 ? npml : 0), pe_b(npml > 0 ? npml : 0), ph_a(npml > 0 ? npml : 0), ph_b(npml > 0 ? npml : 0);
  if (boundary == 2) {
    const double smax = -(pml_m + 1.0) * kEps0 * kC0 * std::log(pml_R0) / (2.0 * double(npml) * dz);
    for (int j = 0; j < npml; ++j) {
      const double rho_e = double(npml - j) / double(npml);
      const double rho_h = (double(npml - j) - 0.5) / double(npml);
      const double se = smax * std::pow(rho_e, pml_m) * dt / (2.0 * kEps0);
      const double sh = smax * std::pow(rho_h, pml_m) * dt / (2.0 * kEps0);      // sigma* dt/(2 mu0) = sigma dt/(2 eps0)
      pe_a[j] = (1.0 - se) / (1.0 + se);
      pe_b[j] = (dt / (kEps0 * dz)) / (1.0 + se);
      ph_a[j] = (1.0 - sh) / (1.0 + sh);
      ph_b[j] = (dt / (kMu0 * dz)) / (1.0 + sh);
    }
  }
  if (src_kind >= 0 && (src_cell < 0 || src_cell >= N)) return 1;
  for (int p = 0; p < nprobes; ++p)
    if (probes[p] < 0 || probes[p] >= N) return 1;

  // Single grid: parallelise over k inside a step.  Batch: parallelise over grids.
  const bool par_cells = (nbatch == 1);
  (void)par_cells;

#pragma omp parallel for schedule(static) if (!par_cells)
  for (int64_t g = 0; g < nbatch; ++g) {
    const double* wpg = wp + g * N;
    const double* nug = nu + g * N;
    double* Eg = E + g * N;
    double* Hg = H + g * N;
    double* Jg = J + g * N;

    // S0
    Coef cf;
    cf.ca.resize(N); cf.cj.resize(N); cf.ch.resize(N); cf.ka.resize(N); cf.kb.resize(N); cf.kc.resize(N);
    coefficients(N, wpg, nug, dz, dt, cf.ca.data(), cf.cj.data(), cf.ch.data(), cf.ka.data(),
                 cf.kb.data(), cf.kc.data(), &cf.chh, &cf.m, scheme);
    if (boundary == 2) {   // PML E nodes: vacuum with electric conductivity (media there are ignored)
      for (int j = 0; j < npml; ++j) {
        const int64_t kk[2] = {int64_t(j), N - 1 - int64_t(j)};
        for (int64_t k : kk) {
          cf.ca[k] = pe_a[j]; cf.ch[k] = pe_b[j]; cf.cj[k] = 0.0; cf.ka[k] = 1.0; cf.kb[k] = 0.0; cf.kc[k] = 0.0;
        }
      }
    }
    const double* ca = cf.ca.data(); const double* cj = cf.cj.data(); const double* ch = cf.ch.data();
    const double* ka = cf.ka.data(); const double* kb = cf.kb.data(); const double* kc = cf.kc.data();
    const double chh = cf.chh, m = cf.m;
    std::vector<double> Eold_v(N);
    double* Eold = Eold_v.data();

    for (int64_t n = 0; n < nsteps; ++n) {
      const int64_t ng = step0 + n;             // global step index: advances E^{ng} -> E^{ng+1}

      // S1: H update, eq. (14)
#pragma omp parallel for schedule(static) if (par_cells)
      for (int64_t k = 0; k <= N - 2; ++k) {
        if (boundary == 2 && k < npml) Hg[k] = ph_a[k] * Hg[k] - ph_b[k] * (Eg[k + 1] - Eg[k]);
        else if (boundary == 2 && k > N - 2 - npml) Hg[k] = ph_a[N - 2 - k] * Hg[k] - ph_b[N - 2 - k] * (Eg[k + 1] - Eg[k]);
        else Hg[k] = Hg[k] - chh * (Eg[k + 1] - Eg[k]);
      }

      // S2: E update, eq. (12) with (11) substituted
#pragma omp parallel for schedule(static) if (par_cells)
      for (int64_t k = 0; k < N; ++k) Eold[k] = Eg[k];
#pragma omp parallel for schedule(static) if (par_cells)
      for (int64_t k = 1; k <= N - 2; ++k)
        Eg[k] = ca[k] * Eold[k] - cj[k] * Jg[k] - ch[k] * (Hg[k] - Hg[k - 1]);

      // S3: boundary cells (not in the paper, which uses PML: PAPER.md:123)
      if (boundary == 0) {
        Eg[0] = Eold[1] + m * (Eg[1] - Eold[0]);
        Eg[N - 1] = Eold[N - 2] + m * (Eg[N - 2] - Eold[N - 1]);
      } else {
        Eg[0] = 0.0;
        Eg[N - 1] = 0.0;
      }

      // S4: soft source, eq. (15)
      if (src_kind >= 0) Eg[src_cell] += source_sample(src_kind, src_params, nparams, ng, dt);

      // S5: J update, eq. (11)  PAPER.md:68 — every node, with the final E'
#pragma omp parallel for schedule(static) if (par_cells)
      for (int64_t k = 0; k < N; ++k) Jg[k] = ka[k] * Jg[k] + kb[k] * Eold[k] + kc[k] * Eg[k];

      // S6: probes (and the running DFT, evaluated directly — no phasor recurrence)
      for (int p = 0; p < nprobes; ++p) {
        const double v = Eg[probes[p]];
        if (rec) rec[(g * nprobes + p) * nsteps + n] = v;
        if (recJ) recJ[(g * nprobes + p) * nsteps + n] = Jg[probes[p]];
        if (dft_re && dft_im) {
          for (int q = 0; q < nfreq; ++q) {
            const double theta = 2.0 * kPi * freqs[q] * (double(ng + 1) * dt);
            dft_re[(g * nprobes + p) * nfreq + q] += v * std::cos(theta);
            dft_im[(g * nprobes + p) * nfreq + q] -= v * std::sin(theta);
          }
        }
      }
    }
  }
  return 0;
}

int oracle_run_scheme(int64_t ncells, int64_t nbatch, double dz, double dt,
                      const double* wp, const double* nu, double* E, double* H, double* J,
                      int src_kind, const double* src_params, int64_t nparams, int64_t src_cell,
                      const int64_t* probes, int nprobes, int64_t step0, int64_t nsteps,
                      double* rec, double* recJ,
                      const double* freqs, int nfreq, double* dft_re, double* dft_im,
                      int boundary, int scheme) {
  if (boundary == 2) return 1;     // PML needs its parameters: oracle_run_bc
  return oracle_run_bc(ncells, nbatch, dz, dt, wp, nu, E, H, J, src_kind, src_params, nparams, src_cell, probes,
                       nprobes, step0, nsteps, rec, recJ, freqs, nfreq, dft_re, dft_im, boundary, scheme, 0, 0.0, 1.0);
}

int oracle_run(int64_t ncells, int64_t nbatch, double dz, double dt,
               const double* wp, const double* nu, double* E, double* H, double* J,
               int src_kind, const double* src_params, int64_t nparams, int64_t src_cell,
               const int64_t* probes, int nprobes, int64_t step0, int64_t nsteps,
               double* rec, double* recJ,
               const double* freqs, int nfreq, double* dft_re, double* dft_im,
               int boundary) {
  return oracle_run_scheme(ncells, nbatch, dz, dt, wp, nu, E, H, J, src_kind, src_params, nparams, src_cell, probes,
                           nprobes, step0, nsteps, rec, recJ, freqs, nfreq, dft_re, dft_im, boundary, 0);
}


// ============================================================================
// 2-D TMz generalisation (the paper's stated next step).
// The paper writes the method for vector fields — eqs. (1)-(3), PAPER.md:33-37 — and then keeps one component
// pair.  Keeping the components (Ez, Hx, Hy, Jz) of fields that do not vary along z gives
//     mu0 dHx/dt = -dEz/dy,   mu0 dHy/dt = +dEz/dx,   eps0 dEz/dt + Jz = dHy/dx - dHx/dy,   dJz/dt + nu Jz = eps0 wp^2 Ez.
// J is advanced by the same recurrence, eq. (11), node by node, and E by eq. (12) PAPER.md:74 with the
// 1-D difference of H replaced by the z component of the discrete curl; substituting (11) into (12) as in 1-D gives
// the same D and the same six coefficients, with ch once per axis (cex with dx, cey with dy).
//
// Notation.  nx x ny Ez nodes (i, j), arrays row-major [ny][nx] (i fastest).  Ez[j][i] = Ez(i dx, j dy) and Jz at
// integer steps; Hx[j][i] = Hx(i dx, (j+1/2) dy), j <= ny-2 (row ny-1 is padding, kept 0); Hy[j][i] =
// Hy((i+1/2) dx, j dy), i <= nx-2 (column nx-1 is padding, kept 0); both at half steps.
// One step, in the order of the 1-D S1-S6:
//   S1  Hx[j][i] -= chy (Ez[j+1][i] - Ez[j][i])   chy = dt/(mu0 dy);   Hy[j][i] += chx (Ez[j][i+1] - Ez[j][i])   chx = dt/(mu0 dx)
//   S2  interior 1 <= i <= nx-2, 1 <= j <= ny-2:
//       Ez'[j][i] = ca Ez - cj Jz + cex (Hy[j][i] - Hy[j][i-1]) - cey (Hx[j][i] - Hx[j-1][i])
//   S3  edges: boundary 0 = first-order Mur normal to each edge, e.g. Ez'[j][0] = Ez[j][1] + mx (Ez'[j][1] - Ez[j][0]),
//       mx = (c dt - dx)/(c dt + dx), my likewise (the 1-D a3 applied along the normal; reading: the paper's PML has
//       no parameters); boundary 1 = perfect conductor, Ez' = 0 on the four edges.  The four corner
//       nodes are set to 0 in both cases: no interior update reads them (only edge H values do, and those feed
//       nothing), so the choice is unobservable.
//   S4  soft source Ez'[js][is] += s((n+1) dt);   S5  Jz' = ka Jz + kb Ez + kc Ez' at every node;   S6  probes.
// Pins (tests/test_oracle2d_pins.py): Q1 fields uniform along one axis reproduce the 1-D oracle bit for bit (both axes),
// Q2 discrete energy in a conducting box, Q3 cavity eigenmode against the scalar three-term recurrence of the Yee
// dispersion relation with dx != dy, Q4 RK4 brute force of eq. (6) on a recorded node, Q5 transposed problem gives the
// transposed result, Q7 domain of dependence (windowed run), Q8 OpenMP == serial.
// ============================================================================
int oracle2d_coefficients(int64_t n, const double* wp, const double* nu, double dx, double dy, double dt, int scheme,
                          double* ca, double* cj, double* cex, double* cey, double* ka, double* kb, double* kc,
                          double* chx_chy_mx_my) {
  if (n < 0 || dx <= 0 || dy <= 0 || dt <= 0 || scheme < 0 || scheme > 1) return 1;
  double chx, chy, mx, my;
  coefficients(n, wp, nu, dy, dt, ca, cj, cey, ka, kb, kc, &chy, &my, scheme);
  coefficients(n, wp, nu, dx, dt, ca, cj, cex, ka, kb, kc, &chx, &mx, scheme);
  chx_chy_mx_my[0] = chx; chx_chy_mx_my[1] = chy; chx_chy_mx_my[2] = mx; chx_chy_mx_my[3] = my;
  return 0;
}

//   wp, nu, Ez, Hx, Hy, Jz   [ny][nx]
//   probes                   [nprobes][2] = (i, j);  rec, recJ [nprobes][nsteps] (either may be NULL)
int oracle2d_run(int64_t nx, int64_t ny, double dx, double dy, double dt,
                 const double* wp, const double* nu, double* Ez, double* Hx, double* Hy, double* Jz,
                 int src_kind, const double* src_params, int64_t nparams, int64_t src_i, int64_t src_j,
                 const int64_t* probes, int nprobes, int64_t step0, int64_t nsteps,
                 double* rec, double* recJ, int boundary, int scheme) {
  if (nx < 3 || ny < 3 || nsteps < 0 || dx <= 0 || dy <= 0 || dt <= 0 || scheme < 0 || scheme > 1) return 1;
  if (boundary < 0 || boundary > 1) return 1;
  if (src_kind >= 0 && (src_i < 0 || src_i >= nx || src_j < 0 || src_j >= ny)) return 1;
  for (int p = 0; p < nprobes; ++p)
    if (probes[2 * p] < 0 || probes[2 * p] >= nx || probes[2 * p + 1] < 0 || probes[2 * p + 1] >= ny) return 1;
  const int64_t n = nx * ny;
  std::vector<double> ca(n), cj(n), cex(n), cey(n), ka(n), kb(n), kc(n), Eold(n);
  double g[4];
  oracle2d_coefficients(n, wp, nu, dx, dy, dt, scheme, ca.data(), cj.data(), cex.data(), cey.data(), ka.data(),
                        kb.data(), kc.data(), g);
  const double chx = g[0], chy = g[1], mx = g[2], my = g[3];
#define AT(j, i) ((j) * nx + (i))
  for (int64_t s = 0; s < nsteps; ++s) {
    const int64_t ng = step0 + s;
    // S1: H from the curl of E (eq. (2), discretised as eq. (14) PAPER.md:84 along each axis)
#pragma omp parallel for schedule(static)
    for (int64_t j = 0; j < ny; ++j)
      for (int64_t i = 0; i < nx; ++i) {
        if (j <= ny - 2) Hx[AT(j, i)] = Hx[AT(j, i)] - chy * (Ez[AT(j + 1, i)] - Ez[AT(j, i)]);
        if (i <= nx - 2) Hy[AT(j, i)] = Hy[AT(j, i)] + chx * (Ez[AT(j, i + 1)] - Ez[AT(j, i)]);
      }
    // S2: E from the curl of H and J (eq. (12) PAPER.md:74 with (11) substituted)
#pragma omp parallel for schedule(static)
    for (int64_t k = 0; k < n; ++k) Eold[k] = Ez[k];
#pragma omp parallel for schedule(static)
    for (int64_t j = 1; j <= ny - 2; ++j)
      for (int64_t i = 1; i <= nx - 2; ++i) {
        const int64_t k = AT(j, i);
        Ez[k] = ca[k] * Eold[k] - cj[k] * Jz[k] + cex[k] * (Hy[k] - Hy[AT(j, i - 1)]) - cey[k] * (Hx[k] - Hx[AT(j - 1, i)]);
      }
    // S3: the four edges, then the corners
    for (int64_t j = 1; j <= ny - 2; ++j) {
      if (boundary == 0) {
        Ez[AT(j, 0)] = Eold[AT(j, 1)] + mx * (Ez[AT(j, 1)] - Eold[AT(j, 0)]);
        Ez[AT(j, nx - 1)] = Eold[AT(j, nx - 2)] + mx * (Ez[AT(j, nx - 2)] - Eold[AT(j, nx - 1)]);
      } else {
        Ez[AT(j, 0)] = 0.0; Ez[AT(j, nx - 1)] = 0.0;
      }
    }
    for (int64_t i = 1; i <= nx - 2; ++i) {
      if (boundary == 0) {
        Ez[AT(0, i)] = Eold[AT(1, i)] + my * (Ez[AT(1, i)] - Eold[AT(0, i)]);
        Ez[AT(ny - 1, i)] = Eold[AT(ny - 2, i)] + my * (Ez[AT(ny - 2, i)] - Eold[AT(ny - 1, i)]);
      } else {
        Ez[AT(0, i)] = 0.0; Ez[AT(ny - 1, i)] = 0.0;
      }
    }
    Ez[AT(0, 0)] = 0.0; Ez[AT(0, nx - 1)] = 0.0; Ez[AT(ny - 1, 0)] = 0.0; Ez[AT(ny - 1, nx - 1)] = 0.0;
    // S4: soft source, eq. (15)
    if (src_kind >= 0) Ez[AT(src_j, src_i)] += source_sample(src_kind, src_params, nparams, ng, dt);
    // S5: J, eq. (11), every node, with the final E'
#pragma omp parallel for schedule(static)
    for (int64_t k = 0; k < n; ++k) Jz[k] = ka[k] * Jz[k] + kb[k] * Eold[k] + kc[k] * Ez[k];
    // S6: probes
    for (int p = 0; p < nprobes; ++p) {
      const int64_t k = AT(probes[2 * p + 1], probes[2 * p]);
      if (rec) rec[int64_t(p) * nsteps + s] = Ez[k];
      if (recJ) recJ[int64_t(p) * nsteps + s] = Jz[k];
    }
  }
#undef AT
  return 0;
}


// ============================================================================
// 2-D TEz: the other polarisation of fields that do not vary along z (SURVEY §8(f) NEXT-3 "2-D TMz/TEz";
// eqs. (1)-(3), kept in the components Ex, Ey, Hz, Jx, Jy):
//     mu0 dHz/dt = dEx/dy - dEy/dx,   eps0 dEx/dt + Jx = dHz/dy,   eps0 dEy/dt + Jy = -dHz/dx,
//     dJx/dt + nu Jx = eps0 wp^2 Ex,   dJy/dt + nu Jy = eps0 wp^2 Ey.
// J now has two components, each collocated with its E component (eq. (11) PAPER.md:68 per component, eq. (12)
// PAPER.md:74 per component with the 1-D difference of H replaced by the matching curl term) — a different stencil
// from TMz, where J sits on the one Ez node.
//
// Notation.  nx x ny cells (i, j), arrays row-major [ny][nx].  Ex[j][i] = Ex((i+1/2) dx, j dy), i <= nx-2 (column nx-1
// is padding, kept 0); Ey[j][i] = Ey(i dx, (j+1/2) dy), j <= ny-2 (row ny-1 is padding); Hz[j][i] = Hz((i+1/2) dx,
// (j+1/2) dy), i <= nx-2, j <= ny-2, at half steps.  Reading: the media are given per cell, wp[j][i], nu[j][i], and
// both components stored at [j][i] use that pair (the usual material-per-Yee-cell convention; the paper prints nothing
// 2-D).  The six coefficients are those of the 1-D method, `ch` once per axis (cex with dx, cey with dy).
// One step, in the order of the 1-D S1-S6:
//   S1  Hz[j][i] = Hz - chx (Ey[j][i+1] - Ey[j][i]) + chy (Ex[j+1][i] - Ex[j][i])          chx = dt/(mu0 dx), chy = dt/(mu0 dy)
//   S2  Ex'[j][i] = ca Ex - cj Jx + cey (Hz[j][i] - Hz[j-1][i])     1 <= j <= ny-2, i <= nx-2
//       Ey'[j][i] = ca Ey - cj Jy - cex (Hz[j][i] - Hz[j][i-1])     1 <= i <= nx-2, j <= ny-2
//   S3  tangential E on the four edges (Ex on rows 0 and ny-1, Ey on columns 0 and nx-1): boundary 0 = first-order
//       Mur along the normal, Ex'[0][i] = Ex[1][i] + my (Ex'[1][i] - Ex[0][i]) etc.; boundary 1 = conductor, 0.
//   S4  soft source added to component src_comp (0 = Ex, 1 = Ey) at (is, js);   S5  Jx, Jy by eq. (11);   S6  probes
//       (i, j, component).
// Pins (tests/test_oracle2d_te_pins.py): R1 fields uniform along one axis reproduce the 1-D oracle bit for bit (Ey, Hz
// along x; Ex, -Hz along y), R2 discrete energy in a conducting box, R3 cavity eigenmode TE_mn against the scalar
// recurrence of the Yee dispersion relation, R4 axis exchange, R5 first step by hand, R6 domain of dependence,
// R7 OpenMP == serial.
// ============================================================================
//   probes [nprobes][3] = (i, j, component);  rec [nprobes][nsteps]
int oracle2d_te_run(int64_t nx, int64_t ny, double dx, double dy, double dt,
                    const double* wp, const double* nu, double* Ex, double* Ey, double* Hz, double* Jx, double* Jy,
                    int src_kind, const double* src_params, int64_t nparams, int64_t src_i, int64_t src_j, int src_comp,
                    const int64_t* probes, int nprobes, int64_t step0, int64_t nsteps, double* rec, int boundary, int scheme) {
  if (nx < 3 || ny < 3 || nsteps < 0 || dx <= 0 || dy <= 0 || dt <= 0 || scheme < 0 || scheme > 1) return 1;
  if (boundary < 0 || boundary > 1 || src_comp < 0 || src_comp > 1) return 1;
  if (src_kind >= 0 && (src_i < 0 || src_i >= nx || src_j < 0 || src_j >= ny)) return 1;
  for (int p = 0; p < nprobes; ++p)
    if (probes[3 * p] < 0 || probes[3 * p] >= nx || probes[3 * p + 1] < 0 || probes[3 * p + 1] >= ny ||
        probes[3 * p + 2] < 0 || probes[3 * p + 2] > 1) return 1;
  const int64_t n = nx * ny;
  std::vector<double> ca(n), cj(n), cex(n), cey(n), ka(n), kb(n), kc(n), Exold(n), Eyold(n);
  double g[4];
  oracle2d_coefficients(n, wp, nu, dx, dy, dt, scheme, ca.data(), cj.data(), cex.data(), cey.data(), ka.data(),
                        kb.data(), kc.data(), g);
  const double chx = g[0], chy = g[1], mx = g[2], my = g[3];
#define AT(j, i) ((j) * nx + (i))
  for (int64_t s = 0; s < nsteps; ++s) {
    const int64_t ng = step0 + s;
    // S1: Hz from the z component of the curl of E (eq. (2); discretised as eq. (14) PAPER.md:84 along each axis)
#pragma omp parallel for schedule(static)
    for (int64_t j = 0; j <= ny - 2; ++j)
      for (int64_t i = 0; i <= nx - 2; ++i)
        Hz[AT(j, i)] = Hz[AT(j, i)] - chx * (Ey[AT(j, i + 1)] - Ey[AT(j, i)]) + chy * (Ex[AT(j + 1, i)] - Ex[AT(j, i)]);
    // S2: Ex, Ey from the curl of Hz and J (eq. (12) PAPER.md:74 with (11) substituted, per component)
#pragma omp parallel for schedule(static)
    for (int64_t k = 0; k < n; ++k) { Exold[k] = Ex[k]; Eyold[k] = Ey[k]; }
#pragma omp parallel for schedule(static)
    for (int64_t j = 0; j <= ny - 1; ++j)
      for (int64_t i = 0; i <= nx - 1; ++i) {
        const int64_t k = AT(j, i);
        if (j >= 1 && j <= ny - 2 && i <= nx - 2) Ex[k] = ca[k] * Exold[k] - cj[k] * Jx[k] + cey[k] * (Hz[k] - Hz[AT(j - 1, i)]);
        if (i >= 1 && i <= nx - 2 && j <= ny - 2) Ey[k] = ca[k] * Eyold[k] - cj[k] * Jy[k] - cex[k] * (Hz[k] - Hz[AT(j, i - 1)]);
      }
    // S3: tangential E on the edges
    for (int64_t i = 0; i <= nx - 2; ++i) {
      if (boundary == 0) {
        Ex[AT(0, i)] = Exold[AT(1, i)] + my * (Ex[AT(1, i)] - Exold[AT(0, i)]);
        Ex[AT(ny - 1, i)] = Exold[AT(ny - 2, i)] + my * (Ex[AT(ny - 2, i)] - Exold[AT(ny - 1, i)]);
      } else {
        Ex[AT(0, i)] = 0.0; Ex[AT(ny - 1, i)] = 0.0;
      }
    }
    for (int64_t j = 0; j <= ny - 2; ++j) {
      if (boundary == 0) {
        Ey[AT(j, 0)] = Eyold[AT(j, 1)] + mx * (Ey[AT(j, 1)] - Eyold[AT(j, 0)]);
        Ey[AT(j, nx - 1)] = Eyold[AT(j, nx - 2)] + mx * (Ey[AT(j, nx - 2)] - Eyold[AT(j, nx - 1)]);
      } else {
        Ey[AT(j, 0)] = 0.0; Ey[AT(j, nx - 1)] = 0.0;
      }
    }
    // S4: soft source, eq. (15), on one component
    if (src_kind >= 0) {
      const double sv = source_sample(src_kind, src_params, nparams, ng, dt);
      if (src_comp == 0) Ex[AT(src_j, src_i)] += sv; else Ey[AT(src_j, src_i)] += sv;
    }
    // S5: Jx, Jy, eq. (11), every stored node, with the final E'
#pragma omp parallel for schedule(static)
    for (int64_t k = 0; k < n; ++k) {
      Jx[k] = ka[k] * Jx[k] + kb[k] * Exold[k] + kc[k] * Ex[k];
      Jy[k] = ka[k] * Jy[k] + kb[k] * Eyold[k] + kc[k] * Ey[k];
    }
    // S6: probes
    for (int p = 0; p < nprobes; ++p) {
      const int64_t k = AT(probes[3 * p + 1], probes[3 * p]);
      if (rec) rec[int64_t(p) * nsteps + s] = probes[3 * p + 2] == 0 ? Ex[k] : Ey[k];
    }
  }
#undef AT
  return 0;
}


// ============================================================================
// 2-D TMz with the paper's boundary: Berenger's split-field layer on the four sides ("both the electric and
// magnetic fields are divided into two directions, both of which execute in their own kernel", :123 "PML ... of 5
// cells").  Reading: the 1-D reading of §12 applied per axis —
// sigma_x depends on x only, sigma_y on y only, polynomial grading sigma(rho) = sigma_max rho^m with sigma_max =
// -(m+1) eps0 c ln(R0) / (2 npml d) for the step d of that axis, matched sigma* = sigma mu0/eps0, a conductor behind
// the layer (Ez = 0 on the four edges), layer nodes vacuum (media there ignored, Jz = 0).  In the layer Ez = Ezx + Ezy:
//     Ezx' = ax[i] Ezx + bx[i] (Hy[j][i] - Hy[j][i-1]),   Ezy' = ay[j] Ezy - by[j] (Hx[j][i] - Hx[j-1][i]),
//     a = (1-s)/(1+s), b = (dt/(eps0 d))/(1+s), s = sigma dt/(2 eps0) at the E node;
//     Hx' = hay[j] Hx - hby[j] (Ez[j+1][i] - Ez[j][i]),   Hy' = hax[i] Hy + hbx[i] (Ez[j][i+1] - Ez[j][i])   everywhere,
//     ha = (1-s)/(1+s), hb = (dt/(mu0 d))/(1+s) with s at the H node (half a node deeper); outside the layers ha = 1,
//     hb = dt/(mu0 d) and the products with 1 are exact, so the interior is the plain update bit for bit.
// Nodes outside every layer take the unsplit plasma update of oracle2d_run.  Esplit = [2][ny][nx]: Ezx, Ezy (state,
// meaningful on layer nodes).  Pins (tests/test_oracle2d_pins.py, U1-U4): fields uniform along one axis reproduce the
// 1-D PML oracle bit for bit (both axes); R0 = 1 equals the conducting box up to rounding; the energy never grows;
// an obliquely incident pulse comes back smaller than from first-order Mur.
// ============================================================================
int oracle2d_run_pml(int64_t nx, int64_t ny, double dx, double dy, double dt,
                     const double* wp, const double* nu, double* Ez, double* Hx, double* Hy, double* Jz, double* Esplit,
                     int src_kind, const double* src_params, int64_t nparams, int64_t src_i, int64_t src_j,
                     const int64_t* probes, int nprobes, int64_t step0, int64_t nsteps,
                     double* rec, int npml, double pml_m, double pml_R0) {
  if (nx < 3 || ny < 3 || nsteps < 0 || dx <= 0 || dy <= 0 || dt <= 0 || !Esplit) return 1;
  if (npml < 1 || 2 * (int64_t)npml + 1 > nx || 2 * (int64_t)npml + 1 > ny || !(pml_R0 > 0.0) || pml_R0 > 1.0 || pml_m < 0.0) return 1;
  if (src_kind >= 0 && (src_i < 0 || src_i >= nx || src_j < 0 || src_j >= ny)) return 1;
  for (int p = 0; p < nprobes; ++p)
    if (probes[2 * p] < 0 || probes[2 * p] >= nx || probes[2 * p + 1] < 0 || probes[2 * p + 1] >= ny) return 1;
  const int64_t n = nx * ny;
  std::vector<double> ca(n), cj(n), cex(n), cey(n), ka(n), kb(n), kc(n), Eold(n);
  double g[4];
  oracle2d_coefficients(n, wp, nu, dx, dy, dt, 0, ca.data(), cj.data(), cex.data(), cey.data(), ka.data(), kb.data(), kc.data(), g);
  const double chx = g[0], chy = g[1];
  // per-axis tables over the whole axis: E nodes 0..N-1, H nodes 0..N-2 (value 1 / plain coefficient outside the layers)
  auto tables = [&](int64_t N, double d, std::vector<double>& ea, std::vector<double>& eb, std::vector<double>& ha,
                    std::vector<double>& hb, double ch) {
    ea.assign(N, 1.0); eb.assign(N, dt / (kEps0 * d)); ha.assign(N, 1.0); hb.assign(N, ch);
    const double smax = -(pml_m + 1.0) * kEps0 * kC0 * std::log(pml_R0) / (2.0 * double(npml) * d);
    for (int j = 0; j < npml; ++j) {
      const double rho_e = double(npml - j) / double(npml);
      const double rho_h = (double(npml - j) - 0.5) / double(npml);
      const double se = smax * std::pow(rho_e, pml_m) * dt / (2.0 * kEps0);
      const double sh = smax * std::pow(rho_h, pml_m) * dt / (2.0 * kEps0);
      ea[j] = ea[N - 1 - j] = (1.0 - se) / (1.0 + se);
      eb[j] = eb[N - 1 - j] = (dt / (kEps0 * d)) / (1.0 + se);
      ha[j] = ha[N - 2 - j] = (1.0 - sh) / (1.0 + sh);
      hb[j] = hb[N - 2 - j] = ch / (1.0 + sh);
    }
  };
  std::vector<double> eax, ebx, hax, hbx, eay, eby, hay, hby;
  tables(nx, dx, eax, ebx, hax, hbx, chx);
  tables(ny, dy, eay, eby, hay, hby, chy);
  double* Ezx = Esplit;
  double* Ezy = Esplit + n;
#define AT(j, i) ((j) * nx + (i))
  for (int64_t s = 0; s < nsteps; ++s) {
    const int64_t ng = step0 + s;
    // S1: H, damped inside the layers
#pragma omp parallel for schedule(static)
    for (int64_t j = 0; j < ny; ++j)
      for (int64_t i = 0; i < nx; ++i) {
        if (j <= ny - 2) Hx[AT(j, i)] = hay[j] * Hx[AT(j, i)] - hby[j] * (Ez[AT(j + 1, i)] - Ez[AT(j, i)]);
        if (i <= nx - 2) Hy[AT(j, i)] = hax[i] * Hy[AT(j, i)] + hbx[i] * (Ez[AT(j, i + 1)] - Ez[AT(j, i)]);
      }
    // S2: E — split in the layers, the plasma update elsewhere
#pragma omp parallel for schedule(static)
    for (int64_t k = 0; k < n; ++k) Eold[k] = Ez[k];
#pragma omp parallel for schedule(static)
    for (int64_t j = 1; j <= ny - 2; ++j)
      for (int64_t i = 1; i <= nx - 2; ++i) {
        const int64_t k = AT(j, i);
        const bool layer = i < npml || i > nx - 1 - npml || j < npml || j > ny - 1 - npml;
        if (layer) {
          Ezx[k] = eax[i] * Ezx[k] + ebx[i] * (Hy[k] - Hy[AT(j, i - 1)]);
          Ezy[k] = eay[j] * Ezy[k] - eby[j] * (Hx[k] - Hx[AT(j - 1, i)]);
          Ez[k] = Ezx[k] + Ezy[k];
        } else {
          Ez[k] = ca[k] * Eold[k] - cj[k] * Jz[k] + cex[k] * (Hy[k] - Hy[AT(j, i - 1)]) - cey[k] * (Hx[k] - Hx[AT(j - 1, i)]);
        }
      }
    // S3: the conductor behind the layer
    for (int64_t j = 0; j < ny; ++j) { Ez[AT(j, 0)] = 0.0; Ez[AT(j, nx - 1)] = 0.0; }
    for (int64_t i = 0; i < nx; ++i) { Ez[AT(0, i)] = 0.0; Ez[AT(ny - 1, i)] = 0.0; }
    // S4: soft source (a source inside a layer drives the x part)
    if (src_kind >= 0) {
      const double sv = source_sample(src_kind, src_params, nparams, ng, dt);
      const int64_t k = AT(src_j, src_i);
      Ez[k] += sv;
      Ezx[k] += sv;
    }
    // S5: J outside the layers (layer nodes are vacuum)
#pragma omp parallel for schedule(static)
    for (int64_t j = 0; j < ny; ++j)
      for (int64_t i = 0; i < nx; ++i) {
        const int64_t k = AT(j, i);
        const bool layer = i < npml || i > nx - 1 - npml || j < npml || j > ny - 1 - npml;
        Jz[k] = layer ? 0.0 : ka[k] * Jz[k] + kb[k] * Eold[k] + kc[k] * Ez[k];
      }
    for (int p = 0; p < nprobes; ++p)
      if (rec) rec[int64_t(p) * nsteps + s] = Ez[AT(probes[2 * p + 1], probes[2 * p])];
  }
#undef AT
  return 0;
}

}  // extern "C"
