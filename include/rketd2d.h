/* ============================================================================
 * rketd2d.h — C ABI of the 2-D TMz generalisation of the RKETD-FDTD leapfrog (part of librketd.so).
 * SURVEY.md §8(f) NEXT-3; the paper names it as its next step and gives the vector equations
 * it follows from, eqs. (1)-(3) PAPER.md:33-37.  Fields that do not vary along z, components (Ez, Hx, Hy, Jz):
 *     mu0 dHx/dt = -dEz/dy,  mu0 dHy/dt = dEz/dx,  eps0 dEz/dt + Jz = dHy/dx - dHx/dy,  dJz/dt + nu Jz = eps0 wp^2 Ez.
 * Jz is advanced by eq. (11) PAPER.md:68 node by node, Ez by eq. (12) PAPER.md:74 with the difference of H replaced by
 * the z component of the discrete curl, H by eq. (14) PAPER.md:84 along each axis.  One step:
 *     Hx[j][i] -= (dt/(mu0 dy)) (Ez[j+1][i] - Ez[j][i]);      Hy[j][i] += (dt/(mu0 dx)) (Ez[j][i+1] - Ez[j][i])
 *     Ez'[j][i] = ca Ez - cj Jz + cex (Hy[j][i] - Hy[j][i-1]) - cey (Hx[j][i] - Hx[j-1][i])        (interior nodes)
 *     edges: first-order Mur along the normal, or a perfect conductor; the four corner nodes are 0
 *     Ez'[js][is] += s((n+1) dt);     Jz' = ka Jz + kb Ez + kc Ez' (every node);     rec[p][n] = Ez'[jp][ip]
 * with ca, cj, ka, kb, kc of rketd.h and cex, cey = its ch with dz = dx, dy.
 *
 * Conventions are those of rketd.h: int status returns (RKETD_* codes), caller owns its buffers, set_* copy,
 * "host or device" pointers, fixed SI constants, all work on the stream given at creation, no CPU fallback
 * (RKETD_ECUDA without a usable device).  Arrays are row-major [ny][nx], x fastest.  Ez[j][i] = Ez(i dx, j dy) and
 * Jz at integer steps; Hx[j][i] = Hx(i dx, (j+1/2) dy) (row ny-1 is padding, never updated); Hy[j][i] =
 * Hy((i+1/2) dx, j dy) (column nx-1 is padding, never updated); both at half steps.
 * ========================================================================== */
#ifndef RKETD2D_H_
#define RKETD2D_H_

#include <stdint.h>

#include "rketd.h"

#ifdef __cplusplus
extern "C" {
#endif

typedef struct rketd2d_sim rketd2d_sim; /* opaque */

/* grid edges for rketd2d_set_boundary */
enum {
  RKETD2D_BC_MUR = 0,        /* first-order Mur along the normal of each edge (the 1-D rule a3 per edge); the default */
  RKETD2D_BC_PEC = 1,        /* perfect conductor: Ez = 0 on the four edges                                            */
  RKETD2D_BC_PML = 2         /* the paper's split-field layer + conductor: set by rketd2d_set_boundary_pml only         */
};
/* kernel selection for rketd2d_set_plan */
enum {
  RKETD2D_KERNEL_AUTO = 0,   /* the streaming kernel                                                                   */
  RKETD2D_KERNEL_STEP = 1,   /* one fused H/E/J launch per time step (baseline / cross-check)                          */
  RKETD2D_KERNEL_STREAM = 2  /* temporal blocking: T steps per pass, rows streamed through a register pipeline        */
};
/* counters for rketd2d_get_counter */
enum {
  RKETD2D_CTR_LAUNCHES = 0,      /* kernels launched by this handle so far                                  */
  RKETD2D_CTR_STEP_LAUNCHES = 1, /* launches of the stencil kernels so far                                  */
  RKETD2D_CTR_KERNEL_USED = 2,   /* RKETD2D_KERNEL_* the last rketd2d_run used                              */
  RKETD2D_CTR_DEPTH_USED = 3,    /* temporal depth T of the last streaming run                              */
  RKETD2D_CTR_STEPS_DONE = 4,    /* global step counter                                                     */
  RKETD2D_CTR_STRIP_COLS = 5,    /* columns a CTA of the streaming kernel holds (halo included)             */
  RKETD2D_CTR_HALO_COLS = 6,     /* halo columns on each side of a strip                                    */
  RKETD2D_CTR_SEG_ROWS = 7,      /* rows of one streamed segment (its 2 T halo rows not included)            */
  RKETD2D_CTR_STATE_BYTES = 8    /* device bytes held by this handle                                        */
};

/* nx x ny Ez nodes; dx, dy [m], dt [s]; dtype RKETD_F64 / RKETD_F32; cuda_stream as in rketd_create.
 * Fields zero, step counter 0, no source, no probes, Mur edges.
 * EINVAL: nx < 3, ny < 3, nx or ny > 2^30, steps <= 0, c dt sqrt(1/dx^2 + 1/dy^2) > 1 (unstable), bad dtype. */
int rketd2d_create(rketd2d_sim **out, int64_t nx, int64_t ny, double dx, double dy, double dt, int dtype,
                   void *cuda_stream);

/* Per-node wp [rad/s], nu [1/s], fp64 [ny][nx], host or device.  Derives on the device, in fp64, the six
 * coefficients of SURVEY a0 per node and from them the four arrays the kernels read
 * (rketd2d_get_kernel_coefficients).  Current fields are kept.  EINVAL: negative or non-finite values.  Synchronises. */
int rketd2d_set_media(rketd2d_sim *s, const double *wp, const double *nu);

/* RKETD2D_BC_*; takes effect at the next rketd2d_run.  EINVAL: unknown kind. */
int rketd2d_set_boundary(rketd2d_sim *s, int kind);

/* Soft source added to Ez^{n+1}[j][i]; kinds and params as rketd_set_source.  EINVAL: node outside the grid. */
int rketd2d_set_source(rketd2d_sim *s, int kind, const double *params, int64_t nparams, int64_t i, int64_t j);

/* Probe nodes, ij[p] = {i, j} (host pointer, [nprobes][2]); at most 64.  Each step records Ez^{n+1} there.
 * Discards earlier records.  EINVAL: node outside the grid. */
int rketd2d_set_probes(rketd2d_sim *s, const int64_t *ij, int nprobes);

/* Overwrite the fields ([ny][nx], handle's dtype, host or device; NULL = zeros).  Synchronises. */
int rketd2d_set_fields(rketd2d_sim *s, const void *Ez, const void *Hx, const void *Hy, const void *Jz);

/* Copy the fields out ([ny][nx], handle's dtype, host or device; any may be NULL).  Synchronises. */
int rketd2d_get_fields(rketd2d_sim *s, void *Ez, void *Hx, void *Hy, void *Jz);

/* Fields zero, step counter 0, records discarded; media, source, probes, boundary kept. */
int rketd2d_reset(rketd2d_sim *s);

/* Drop the probe records gathered so far (their device buffers are freed); fields, step counter, media, source and
 * probes are kept.  The next rketd2d_run starts a fresh record.  Synchronises. */
int rketd2d_discard_records(rketd2d_sim *s);

/* Kernel (RKETD2D_KERNEL_*) and, for the streaming kernel, the temporal depth T in {1, 2, 4, 6, 8} or, fp32 only, 16
 * (0 = default: 8).  All choices compute identical bits.  EINVAL otherwise. */
int rketd2d_set_plan(rketd2d_sim *s, int kernel, int depth);

/* Advance by nsteps leapfrog steps, asynchronously on the stream.  Repeatable.  ESTATE before rketd2d_set_media. */
int rketd2d_run(rketd2d_sim *s, int64_t nsteps);

/* The paper's boundary (PAPER.md:93 "both the electric and magnetic fields are divided into two directions", :123 "PML
 * ... of 5 cells"): Berenger's split-field layer of npml nodes on the four sides, a conductor behind it.  The paper gives
 * no conductivity profile; the reading built is the 1-D one (rketd_set_boundary) per axis: sigma_x(x),
 * sigma_y(y) = sigma_max rho^grading, sigma_max = -(grading+1) eps0 c ln(R0) / (2 npml d) for the step d of the axis,
 * matched magnetic conductivity; Ez = Ezx + Ezy on layer nodes, which are vacuum (media given there are ignored, Jz = 0).
 * Takes effect at the next rketd2d_set_media (which derives the coefficients): call it before; rketd2d_set_boundary
 * with MUR / PEC switches back (again at the next rketd2d_set_media).  Runs in the one-step kernel (the streaming
 * kernel has no layer).  EINVAL: npml outside 1..64, 2 npml + 1 > nx or ny, R0 outside (0, 1], grading < 0. */
int rketd2d_set_boundary_pml(rketd2d_sim *s, int npml, double grading, double R0);

/* Synchronise and copy out the probe records: [nprobes][nsamples] in the handle's dtype (host or device), sample n
 * is Ez at time (n+1) dt.  out may be NULL to query *nsamples.  EINVAL if out_bytes is too small. */
int rketd2d_read_probes(rketd2d_sim *s, void *out, int64_t out_bytes, int64_t *nsamples);

/* The four per-node arrays the stencil kernels read, as fp64 [4][ny][nx] (host or device), order
 * P = ca - cj kc, ce = cex, ka, Q = ka cj kc + cj kb: with G = cj Jz - cj kc Ez in place of Jz,
 * Ez' = P Ez - G + ce ((Hy[i] - Hy[i-1]) - (dx/dy) (Hx[j] - Hx[j-1])) and G' = ka G + Q Ez hold exactly
 * (cey = cex dx/dy).  globals[4] = {dt/(mu0 dx), dt/(mu0 dy), Mur mx, Mur my} (host; may be NULL). */
int rketd2d_get_kernel_coefficients(rketd2d_sim *s, double *out, double *globals);

int64_t rketd2d_get_counter(const rketd2d_sim *s, int which);

void rketd2d_destroy(rketd2d_sim *s);

/* Text of the last error on this handle (or of the last failed rketd2d_create when s is NULL). */
const char *rketd2d_last_error(const rketd2d_sim *s);

/* ============================================================================
 * 2-D TEz: the other polarisation (SURVEY.md §8(f) NEXT-3 "2-D TMz/TEz"; eqs. (1)-(3), kept in the
 * components Ex, Ey, Hz, Jx, Jy of fields that do not vary along z):
 *     mu0 dHz/dt = dEx/dy - dEy/dx,   eps0 dEx/dt + Jx = dHz/dy,   eps0 dEy/dt + Jy = -dHz/dx,
 *     dJ/dt + nu J = eps0 wp^2 E per component (eq. (11); eq. (12) PAPER.md:74 per component).
 * nx x ny cells, arrays row-major [ny][nx].  Ex[j][i] = Ex((i+1/2) dx, j dy) (column nx-1 is padding, reported as 0),
 * Ey[j][i] = Ey(i dx, (j+1/2) dy) (row ny-1 is padding), Hz[j][i] = Hz((i+1/2) dx, (j+1/2) dy) at half steps (row ny-1
 * and column nx-1 are padding); Jx, Jy collocated with Ex, Ey.  The media are given per cell and both components stored
 * at [j][i] use that pair.  One step, in the order of the 1-D path:
 *     Hz[j][i] = Hz - (dt/(mu0 dx)) (Ey[j][i+1] - Ey[j][i]) + (dt/(mu0 dy)) (Ex[j+1][i] - Ex[j][i])
 *     Ex'[j][i] = ca Ex - cj Jx + cey (Hz[j][i] - Hz[j-1][i])      Ey'[j][i] = ca Ey - cj Jy - cex (Hz[j][i] - Hz[j][i-1])
 *     tangential E on the edges (Ex on rows 0 and ny-1, Ey on columns 0 and nx-1): first-order Mur along the normal, or 0
 *     soft source on one component at one cell;  Jx, Jy by eq. (11) with the final E';  probes (i, j, component).
 * One fused launch per step (k1_te); same conventions, error codes and ownership rules as the TMz calls above.
 * ========================================================================== */
typedef struct rketd2d_te_sim rketd2d_te_sim; /* opaque */
enum { RKETD2D_EX = 0, RKETD2D_EY = 1 };      /* component ids of the source and the probes */

/* as rketd2d_create */
int rketd2d_te_create(rketd2d_te_sim **out, int64_t nx, int64_t ny, double dx, double dy, double dt, int dtype,
                      void *cuda_stream);
/* wp [rad/s], nu [1/s] per cell, fp64 [ny][nx], host or device.  Validates before anything changes; EINVAL: negative or
 * non-finite values.  The physical Jx, Jy of live fields are kept.  Synchronises. */
int rketd2d_te_set_media(rketd2d_te_sim *s, const double *wp, const double *nu);
/* RKETD2D_BC_MUR (default) or RKETD2D_BC_PEC */
int rketd2d_te_set_boundary(rketd2d_te_sim *s, int kind);
/* soft source (kinds and params as rketd_set_source) added to component `component` at cell (i, j) */
int rketd2d_te_set_source(rketd2d_te_sim *s, int kind, const double *params, int64_t nparams, int64_t i, int64_t j,
                          int component);
/* probes: triples (i, j, component), host pointer, at most 64; discards earlier records */
int rketd2d_te_set_probes(rketd2d_te_sim *s, const int64_t *ijc, int nprobes);
/* [ny][nx] arrays in the handle's dtype, host or device; NULL = zeros.  Synchronises. */
int rketd2d_te_set_fields(rketd2d_te_sim *s, const void *Ex, const void *Ey, const void *Hz, const void *Jx, const void *Jy);
int rketd2d_te_get_fields(rketd2d_te_sim *s, void *Ex, void *Ey, void *Hz, void *Jx, void *Jy);
/* advance nsteps steps, asynchronously on the stream; ESTATE before rketd2d_te_set_media */
int rketd2d_te_run(rketd2d_te_sim *s, int64_t nsteps);
/* [nprobes][nsamples] in the handle's dtype; out may be NULL to query *nsamples.  Synchronises. */
int rketd2d_te_read_probes(rketd2d_te_sim *s, void *out, int64_t out_bytes, int64_t *nsamples);
/* RKETD2D_CTR_LAUNCHES, _STEP_LAUNCHES, _STEPS_DONE, _STATE_BYTES */
int64_t rketd2d_te_get_counter(const rketd2d_te_sim *s, int which);
void rketd2d_te_destroy(rketd2d_te_sim *s);
const char *rketd2d_te_last_error(const rketd2d_te_sim *s);

#ifdef __cplusplus
}
#endif
#endif /* RKETD2D_H_ */
