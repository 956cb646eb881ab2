/* ============================================================================
 * rketd.h — C ABI of librketd: the per-time-step leapfrog hot path of the 1-D
 * RKETD-FDTD method for an unmagnetized collisional (Drude) plasma
 * (arxiv 1709.00821; citations are PAPER.md:<line> of /root/reference/PAPER.md
 * and SURVEY.md §8 rows).  sm_100a (B200) only; there is no CPU fallback: every
 * compute entry point returns RKETD_ECUDA when no CUDA device is usable.
 *
 * Conventions
 *   - Every call returns an int status (RKETD_OK = 0) and never throws.
 *   - The caller owns every buffer it passes; set_* copy, so the buffer may be
 *     freed or reused as soon as the call returns.  The library owns the handle
 *     and all device state.  One handle is used from one host thread.
 *   - "host or device" pointers: any pointer cudaMemcpy(..., cudaMemcpyDefault)
 *     accepts (pageable / pinned host memory, device memory, managed memory).
 *   - Grids: nbatch independent 1-D grids of ncells E-nodes each.  Node k holds
 *     E[k] = Ex(k dz) and J[k] = Jx(k dz) at integer time steps and
 *     H[k] = Hy((k+1/2) dz) at half steps (k = 0..ncells-2; H[ncells-1] is
 *     padding, reported as 0).  User arrays are row-major [nbatch][ncells].
 *   - Physical constants are fixed: c = 299792458 m/s, mu0 = 4 pi 1e-7 H/m,
 *     eps0 = 1/(mu0 c^2)  (the paper gives no values).
 *   - All work is enqueued on the CUDA stream given to rketd_create.
 * ========================================================================== */
#ifndef RKETD_H_
#define RKETD_H_

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct rketd_sim rketd_sim; /* opaque */

enum { RKETD_F64 = 0, RKETD_F32 = 1 };
enum { RKETD_OK = 0, RKETD_EINVAL = 1, RKETD_ENOMEM = 2, RKETD_ECUDA = 3, RKETD_ESTATE = 4 };
enum { RKETD_SRC_NONE = -1, RKETD_SRC_GAUSS_DERIV = 0, RKETD_SRC_TABLE = 1 };
/* current-density recurrence for rketd_set_scheme */
enum {
  RKETD_SCHEME_ETD2 = 0,     /* eq. (11): second-order ETD ("RKETD"), the paper's method; the default   */
  RKETD_SCHEME_ETD1 = 1      /* eq. (9)  PAPER.md:59: first-order ETD, F held at F_n over the step   */
};
/* grid ends for rketd_set_boundary */
enum {
  RKETD_BC_MUR = 0,          /* first-order Mur at both ends (BASELINE north_star); the default                    */
  RKETD_BC_PML = 1           /* absorbing layer + conductor, the paper's choice   */
};
/* kernel selection for rketd_set_plan */
enum {
  RKETD_KERNEL_AUTO = 0,     /* resident (K3) when a grid fits the registers of one cluster, else temporal blocking (K2) */
  RKETD_KERNEL_STEP = 1,     /* K1: one fused H/E/J launch per time step (baseline / cross-check)   */
  RKETD_KERNEL_TBLOCK = 2,   /* K2: T leapfrog steps per pass on a register-resident tile, TMA-staged */
  RKETD_KERNEL_RESIDENT = 3  /* K3: grids resident on chip (registers of a CTA or a cluster) for the whole run */
};
/* counters for rketd_get_counter */
enum {
  RKETD_CTR_LAUNCHES = 0,      /* kernels launched by this handle so far (all kinds)               */
  RKETD_CTR_STEP_LAUNCHES = 1, /* launches of the stencil kernel (K1/K2/K3) so far                  */
  RKETD_CTR_KERNEL_USED = 2,   /* RKETD_KERNEL_* the last rketd_run used                            */
  RKETD_CTR_DEPTH_USED = 3,    /* temporal depth T of the last run (K2: steps per pass; K3: per halo refresh) */
  RKETD_CTR_STEPS_DONE = 4,    /* global step counter                                               */
  RKETD_CTR_TILE_CELLS = 5,    /* cells per CTA tile, halo included, of the last K2/K3 run          */
  RKETD_CTR_HALO_CELLS = 6,    /* halo cells on each side of a K2 tile                              */
  RKETD_CTR_STATE_BYTES = 7,   /* device bytes held by this handle (fields + coefficients)          */
  RKETD_CTR_PIECES = 8         /* pieces the last rketd_run_from_host cut the line into (0: it ran as the plain sequence of calls) */
};

/* Create a simulation of nbatch grids of ncells nodes ("grid" of the north_star =
 * (ncells, nbatch)).  dz [m], dt [s]; dtype RKETD_F64 or RKETD_F32 (arithmetic and
 * storage type of fields, coefficients, probe records).  cuda_stream: a cudaStream_t
 * (e.g. torch.cuda.current_stream().cuda_stream) or NULL for the default stream.
 * Fields start at zero, step counter at 0, no source, no probes.
 * EINVAL: ncells < 3, nbatch < 1, dz <= 0, dt <= 0, c dt/dz > 1 (unstable), bad dtype.
 * Host code role: PAPER.md:93 (init, device alloc, copies). */
int rketd_create(rketd_sim **out, int64_t ncells, int64_t nbatch, double dz, double dt, int dtype,
                 void *cuda_stream);

/* Per-node plasma frequency wp [rad/s] and collision frequency nu [1/s], always fp64,
 * [nbatch][ncells], host or device.  Precomputes (in fp64, on the device) the per-node
 * coefficients of SURVEY §8(a) row a0, i.e. eq. (11) PAPER.md:68 written as
 * J' = ka J + kb E + kc E' and eq. (12) PAPER.md:74 with (11) substituted, solved for E'
 * (eq. (13) PAPER.md:79 with the missing 1/D restored): E' = ca E - cj J - ch (H[k]-H[k-1]),
 * and from them the four arrays the kernels read (rketd_get_kernel_coefficients).
 * The current fields E, H, J are kept.  EINVAL: any wp or nu negative or non-finite.  Synchronises. */
int rketd_set_media(rketd_sim *s, const double *wp, const double *nu);

/* Choose the recurrence that advances J (RKETD_SCHEME_*).  Only the coefficient precompute differs: with eq. (9),
 * J' = ka J + kb E (kc = 0) and eq. (12) solved for E' has D = 1.  Takes effect at the next rketd_set_media, which
 * derives the coefficients; call it before.  EINVAL: unknown scheme. */
int rketd_set_scheme(rketd_sim *s, int scheme);

/* Ends of every grid.  RKETD_BC_PML: Berenger's layer of npml nodes (paper: 5) at both ends, a perfect conductor
 * behind it (E[0] = E[ncells-1] = 0).  The paper gives no conductivity profile; the reading built:
 * sigma(rho) = sigma_max rho^grading at relative depth rho (E nodes at (npml-k)/npml, H nodes half a node less),
 * sigma_max = -(grading+1) eps0 c ln(R0) / (2 npml dz) (R0 = design reflection at normal incidence), matched magnetic
 * conductivity; layer nodes are vacuum: the media given for them are ignored and J stays 0 there.
 *   E'[k] = ((1-s)/(1+s)) E[k] - ((dt/(eps0 dz))/(1+s)) (H[k]-H[k-1]),  H likewise,  s = sigma dt/(2 eps0).
 * Takes effect at the next rketd_set_media (which derives the coefficients); call it before.  npml, grading, R0
 * are ignored for RKETD_BC_MUR.  EINVAL: unknown kind, npml outside 1..32, 2 npml + 1 > ncells, R0 outside (0, 1],
 * grading < 0. */
int rketd_set_boundary(rketd_sim *s, int kind, int npml, double grading, double R0);

/* Soft source added to E^{n+1}[cell] in every grid (eq. (15)).
 * kind RKETD_SRC_GAUSS_DERIV: params = {tau, t0, amplitude},
 *   s(t) = amplitude ((t-t0)/tau) exp(1/2 - (t-t0)^2/(2 tau^2)), sample added at step n: s((n+1) dt).
 * kind RKETD_SRC_TABLE: params[i] is added at step index i (0-based); 0 beyond nparams.
 * kind RKETD_SRC_NONE: no source.  params is a HOST pointer.  EINVAL: cell outside [0, ncells). */
int rketd_set_source(rketd_sim *s, int kind, const double *params, int64_t nparams, int64_t cell);

/* Probe nodes (host pointer), the same in every grid; at most 64.  Each step records
 * E^{n+1}[cell].  Discards earlier records.  EINVAL: cell outside [0, ncells). */
int rketd_set_probes(rketd_sim *s, const int64_t *cells, int nprobes);

/* Reduce the probe records on the device to DFT magnitudes (BASELINE config 5):
 * X[g][p][m] = sum_n rec[g][p][n] exp(-j 2 pi f_m (n+1) dt), accumulated in fp64.
 * freqs_hz host pointer; nfreq = 0 switches back to time-series mode.  Discards earlier records. */
int rketd_set_probe_dft(rketd_sim *s, const double *freqs_hz, int nfreq);

/* Overwrite the fields; arrays are [nbatch][ncells] in the handle's dtype, host or device;
 * NULL = zeros.  Does not touch the step counter or the probe records.  Synchronises. */
int rketd_set_fields(rketd_sim *s, const void *E, const void *H, const void *J);

/* Fields zero, step counter 0, probe records and DFT accumulators discarded; media, source and
 * probes kept. */
int rketd_reset(rketd_sim *s);

/* Drop the probe records (time-series chunks) and zero the DFT accumulators gathered so far; fields,
 * step counter, media, source and probes are kept.  The next rketd_run starts a fresh record.
 * Synchronises (device buffers are freed). */
int rketd_discard_records(rketd_sim *s);

/* Choose the kernel (RKETD_KERNEL_*), the temporal depth T (0 = default; K2: steps per pass, K3: steps between two halo
 * refreshes), and the launch variant (-1 = default).  K2: 6 = warp tiles (the default); 0, 2 = one tile per CTA of 128
 * or 256 threads with a block barrier per step (cross-checks).  K3: -1 = the library picks between warp tiles
 * (k3_wtile: few grids, or grids larger than one CTA) and the one-barrier-per-step kernel k3_resident (large batches
 * of grids of at most 512 rows); RKETD_RESIDENT_WTILE(nw, nc, k) = warp tiles with k whole grids per chunk held by a
 * cluster of nc CTAs x nw <= 8 warps (0 = chosen by the library); 0, 2 = k3_resident with the coefficients in
 * registers / in shared memory.  All choices compute identical bits.
 * EINVAL if the choice cannot run this grid (e.g. RESIDENT with a grid larger than a cluster can hold). */
#define RKETD_RESIDENT_WTILE_FLAG 0x40000000
#define RKETD_RESIDENT_WTILE_NOLEAN 0x20000000 /* or-ed in: the 232-register instantiation (coefficients in registers) */
#define RKETD_RESIDENT_WTILE_LEAN 0x10000000   /* or-ed in: the 168-register instantiation (E in place, coefficients from four
                                                  registers or shared memory); default for many grids */
#define RKETD_RESIDENT_WTILE_HALF 0x08000000   /* or-ed in: a lane holds half a 64-B row (twice the warps per grid, half the dependent
                                                  work per step); default for a few grids with Mur ends */
#define RKETD_RESIDENT_WTILE_NOHALF 0x04000000 /* or-ed in: whole rows per lane */
#define RKETD_RESIDENT_WTILE(nw, nc, k) (RKETD_RESIDENT_WTILE_FLAG | ((k) << 16) | ((nc) << 8) | (nw))   /* k < 1024 */
int rketd_set_plan(rketd_sim *s, int kernel, int depth, int variant);

/* Advance every grid by nsteps leapfrog steps (H eq. (14); E eq. (12)
 * with (11); Mur-1 at both ends; soft source; J eq. (11); probe record), asynchronously on the
 * stream.  Repeatable: time continues.  ESTATE before rketd_set_media. */
int rketd_run(rketd_sim *s, int64_t nsteps);

/* A whole job whose inputs live in HOST memory, in one call: the same result, bit for bit, as
 *     rketd_reset(s); rketd_set_media(s, wp, nu); rketd_set_fields(s, E0, NULL, NULL); rketd_run(s, nsteps);
 * (same steps: eq. (14), :76-:78 eqs. (11), (12)), but for one long line (nbatch = 1, temporal-blocking
 * kernel K2, no probe DFT) the line is cut into pieces of whole tiles, the host->device copies of later pieces run on a
 * second stream while earlier pieces step, and the K2 passes run in a time-skewed order: pass p of piece c covers the
 * tiles [b_c - p k, b_(c+1) - p k), k = ceil(halo rows / rows a tile writes), so that every tile finds the previous
 * level of its halo.  Other shapes run as the plain sequence above.
 * wp, nu: [ncells] doubles, E0: [ncells] elements of the handle's dtype or NULL (E = 0); host pointers (pinned memory
 * for the overlap; pageable and device pointers work, without overlap).  The buffers may be reused after the return:
 * the call synchronises the handle's stream.  npieces: 0 = chosen by the library (12, of at least 8 waves of tiles
 * each; measured flat between 8 and 16 on a 2^28-node line), > 0 = that many (tests).  Media are validated while the
 * pieces are staged: on EINVAL (negative or non-finite wp, nu) the handle is left reset and WITHOUT media — unlike
 * rketd_set_media the old media are gone.
 * Step counter restarts at 0, earlier records are discarded, source, probes, boundary and plan are kept. */
int rketd_run_from_host(rketd_sim *s, const double *wp, const double *nu, const void *E0, int64_t nsteps, int npieces);

/* Synchronise and copy out the probe records (host or device `out`, handle's dtype).
 * Time-series mode: [nbatch][nprobes][nsamples], nsamples = steps run since the records were last
 * discarded; sample n is E at time (n+1) dt.  DFT mode: [nbatch][nprobes][nfreq] magnitudes,
 * *nsamples = nfreq.  out may be NULL to query *nsamples.  EINVAL if out_bytes is too small. */
int rketd_read_probes(rketd_sim *s, void *out, int64_t out_bytes, int64_t *nsamples);

/* DFT mode only: the complex accumulators themselves, X = re + j im, each [nbatch][nprobes][nfreq] fp64 (host or
 * device), count = elements each buffer can hold.  Linear in the records, so reflection and transmission of a sweep
 * follow from two runs as |X_slab - X_vacuum| / |X_vacuum| and |X_slab| / |X_vacuum|.
 * Synchronises.  ESTATE outside DFT mode; EINVAL if count is too small. */
int rketd_read_probe_dft(rketd_sim *s, double *re, double *im, int64_t count);

/* Reflection and transmission magnitudes of a sweep, formed on the device: `s` holds
 * the slab grids, `vacuum` one all-vacuum grid (its grid 0 is used) run with the same source, probes, frequencies and
 * step count; both in DFT mode.  R[g][m] = |X_s[g][probe_r][m] - X_v[probe_r][m]| / |X_v[probe_r][m]|,
 * T[g][m] = |X_s[g][probe_t][m]| / |X_v[probe_t][m]|; probe_r, probe_t index the probe list; R, T [nbatch][nfreq] fp64
 * (host or device), count = elements each can hold.  Synchronises both handles' streams.
 * ESTATE outside DFT mode; EINVAL: different probes or frequencies, bad index, count too small. */
int rketd_read_sweep_rt(rketd_sim *s, rketd_sim *vacuum, int probe_r, int probe_t, double *R, double *T, int64_t count);

/* Copy the fields out ([nbatch][ncells], handle's dtype, host or device; any may be NULL).
 * Synchronises. */
int rketd_get_fields(rketd_sim *s, void *E, void *H, void *J);

/* The six coefficients of SURVEY a0 as fp64, order ca, cj, ch, ka, kb, kc (E' = ca E - cj J - ch dH,
 * J' = ka J + kb E + kc E'), computed on the device from the media: out[6][nbatch][ncells] (host or
 * device); chh_m[2] = {dt/(mu0 dz), Mur m} (host; may be NULL). */
int rketd_get_coefficients(rketd_sim *s, double *out, double *chh_m);

/* The four per-node coefficient arrays the stencil kernels actually read, converted to fp64, order
 * P = ca - cj kc, ch, ka, Q = ka cj kc + cj kb (the kernels carry G = cj J - cj kc E in place of J, for
 * which E' = P E - G - ch dH and G' = ka G + Q E hold exactly):
 * out[4][nbatch][ncells] (host or device).  In fp32 mode these are the fp64 values rounded once. */
int rketd_get_kernel_coefficients(rketd_sim *s, double *out);

/* RKETD_CTR_* counters (for bench.py's gpu_launches and roofline bookkeeping). */
int64_t rketd_get_counter(const rketd_sim *s, int which);

/* Microbenchmarks behind the "alu" roofline of bench.py ("builder must microbenchmark DFMA and
 * shared-memory peaks and use the measured values"); not on the hot path, needs no handle.  Runs `what` on the current
 * device for `iters` loop iterations (a few ms at 4000) on cuda_stream and synchronises.  out[4] (host):
 *   out[0]  thread-instructions per ns summed over the device (LDS128: bytes per ns = GB/s)
 *   out[1]  thread-instructions (bytes) per clock and SM — "lanes"
 *   out[2]  SM clock held during the run [MHz] (clock64 against globaltimer)
 *   out[3]  number of SMs
 * FMA forms differ in the number of DISTINCT register source operands per instruction (1, 2, 3, or 2 + one
 * constant-bank operand); MIX is the 7-instruction node update of the stencil kernels (H 2, E 3, G 2) on
 * a 64-B row per lane in registers, without shuffles or memory, at 12 warps per SM.  EINVAL: bad `what` or iters < 1. */
enum {
  RKETD_PEAK_DFMA_1REG = 0, RKETD_PEAK_DFMA_2REG = 1, RKETD_PEAK_DFMA_3REG = 2, RKETD_PEAK_DFMA_2REG_CONST = 3,
  RKETD_PEAK_FFMA_1REG = 4, RKETD_PEAK_FFMA_2REG = 5, RKETD_PEAK_FFMA_3REG = 6, RKETD_PEAK_FFMA_2REG_CONST = 7,
  RKETD_PEAK_MIX_F64 = 8, RKETD_PEAK_MIX_F32 = 9, RKETD_PEAK_LDS128 = 10,
  /* latencies: out[0] = ns, out[1] = cycles per operation (16 x iters operations in a dependent chain) */
  RKETD_LAT_DFMA = 11, RKETD_LAT_SHFL64 = 12,       /* dependent DFMA; 64-bit __shfl_up                                  */
  RKETD_LAT_STEP_F64 = 13, RKETD_LAT_STEP_F32 = 14, /* one leapfrog step of a warp tile, one warp per scheduler          */
  RKETD_LAT_BAR_SYNC = 15,                          /* bar.sync of 256 threads                                           */
  RKETD_LAT_CLUSTER_BARRIER = 16                    /* barrier.cluster arrive.release + wait.acquire, 8 CTAs x 128        */
};
int rketd_measure_peak(int what, int iters, double *out, void *cuda_stream);

/* Row a7 for callers that cannot allocate (code under CUDA graph capture, tight serving loops, harnesses that forbid
 * cudaMalloc): probe records -> DFT magnitudes in ONE call that allocates nothing and does not synchronise
 * (the records' "Fourier transform"; the definition of rketd_set_probe_dft):
 *   out[s][m] = | sum_{n < nsamples} rec[s][n] exp(-j 2 pi f_m (step0 + n + 1) dt) |,  sums in fp64.
 * rec [nseries][nsamples] and out [nseries][nfreq] in `dtype` (the layout rketd_read_probes gives with nseries =
 * nbatch x nprobes; step0 = step index of sample 0, 0 for a record from the start), freqs_hz [nfreq] fp64 — all three in
 * DEVICE memory of the current device, owned by the caller; cuda_stream as in rketd_create.  The twiddle table lives in a
 * static device array of RKETD_NOALLOC_MAX_TWIDDLES entries (8 MiB on every GPU that loads the library, until exit),
 * shared by all calls: a call rewrites what it reads, so nothing needs clearing, but calls that OVERLAP on the GPU
 * (different streams without ordering) race on it.  EINVAL (text: rketd_noalloc_last_error): bad dtype, negative size,
 * dt <= 0, NULL or host pointers, nsamples x nfreq > RKETD_NOALLOC_MAX_TWIDDLES, nseries > RKETD_NOALLOC_MAX_SERIES;
 * ECUDA: no device / launch failure.  nseries = 0 or nfreq = 0: nothing to do, OK. */
#define RKETD_NOALLOC_MAX_TWIDDLES (1 << 19)
#define RKETD_NOALLOC_MAX_SERIES (1 << 24)
int rketd_probe_dft_noalloc(int dtype, const void *rec, int64_t nseries, int64_t nsamples, int64_t step0, double dt,
                            const double *freqs_hz, int nfreq, void *out, void *cuda_stream);

/* Text of the calling thread's last failed rketd_probe_dft_noalloc ("" if none). */
const char *rketd_noalloc_last_error(void);

void rketd_destroy(rketd_sim *s);

/* Text of the last error on this handle (or of the last failed rketd_create when s is NULL). */
const char *rketd_last_error(const rketd_sim *s);

#ifdef __cplusplus
}
#endif
#endif /* RKETD_H_ */
