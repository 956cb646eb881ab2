// rketd_internal.h — host-side types shared by the API (rketd_api.cu) and the kernel
// launchers (rketd_kernels.cu, rketd_aux.cu).  Not part of the public boundary.
#pragma once
#include <cuda.h>            // CUtensorMap type only; libcuda is reached through cudaGetDriverEntryPoint
#include <cuda_runtime.h>
#include <stdint.h>

namespace rketd {

// HBM layout of every per-node array (fields E, H, G x2 for ping-pong; four coefficient arrays P, ch, ka, Q;
// the media wp, nu in fp64):
//   [nbatch][nrows][C] with rows of 64 B (C = 8 fp64 / 16 fp32 nodes) — one row is what one thread
//   (or half of what) one thread owns in registers.  Node k of grid g sits at physical in-grid
//   index off + k.  off is 0, or 1 when (ncells-1) % (C/2) == 0, so that nodes {0,1} sit in the same
//   half row and so do nodes {ncells-2, ncells-1} (Mur needs both in one thread).  Padding nodes carry zero fields and zero
//   coefficients and never influence real nodes (they sit behind the Mur nodes).
struct Layout {
  int64_t ncells = 0, nbatch = 0;
  int esize = 8;       // bytes per value
  int C = 8;           // nodes per row
  int off = 0;         // physical index of node 0
  int64_t nrows = 0;   // rows per grid
  int64_t gstride = 0; // physical nodes per grid = nrows * C
};

struct FieldPtrs { void *E, *H, *J; };

// E-node coefficients of the absorbing layer, index = distance in nodes from the outer end (npml = 0: none)
struct PmlE {
  int npml;
  double a[32], b[32];     // E' = a E - b (H[k] - H[k-1])
};

// dtype-agnostic description of what a step needs (converted to StepParams<R> by the launchers)
struct StepCommon {
  double nchh, mur_m;
  int64_t cellL, cellR, cellS;
  int nprobes;
  int64_t rec_stride, n0;
  const void *src_tab;
  void *rec;
  const uint8_t *rowflag;
  int64_t probe_cell[64];
  int npml;                      // 0 = Mur ends
  double pml_ha[32], pml_hd[32]; // H pre-step coefficients of the absorbing layer (rketd_device.cuh StepParams)
};

// K2 (temporal blocking) plan: tiling + the TMA descriptors for one ping-pong direction.
struct K2Maps {
  CUtensorMap ld[7];   // E, H, G (source buffers), P, ch, ka, Q : box {C, rows, 1}, SWIZZLE_64B
  CUtensorMap st[3];   // E, H, G (destination buffers)         : box {C, rows_out, 1}
};
struct K2Plan {
  int variant = -1;        // K2 kernel variant (see rketd_kernels.cu)
  int rows = 0;            // rows per tile (halo included)
  int HR = 0;              // halo rows on each side (HR * nodes-per-row >= T)
  int rows_out = 0;        // rows - 2 HR
  int depth = 0;           // T, steps per pass
  int64_t tiles_per_grid = 0, total_tiles = 0;
  int grid = 0;            // CTAs launched (persistent)
  int ctas_per_sm = 0;
  int spread = 0;          // warp tiles dealt out across the SMs first (fewer tiles than one wave of warps)
  size_t smem_bytes = 0;
  K2Maps maps[2];          // maps[s]: read buffer s, write buffer 1-s
};

// K3 (resident warp tiles, rketd_resident.cu): a chunk of k whole grids lives in a cluster of nc CTAs x nw warps
struct K3WPlan {
  int T = 0, HR = 0, rows_out = 0;     // steps per round (between halo refreshes), halo rows, 32 - 2 HR
  int k = 1, nc = 1, nw = 1;           // grids per chunk, CTAs per cluster, warps per CTA
  int64_t chunk_rows = 0, nchunks = 0;
  int tiles_per_chunk = 0;
  uint32_t smem_bytes = 0;
  bool lean = false;                   // the <= 128-register instantiation (E in place, coefficients from 4 registers / shared memory)
  bool half = false;                   // a lane holds half a 64-B row: rows above count half rows (few grids: shorter dependent steps)
};
// false when the grid cannot stay resident (a grid needs more than 16 CTAs x 12 warp tiles) or the wish cannot be met;
// want_* = 0: chosen here
bool k3w_few_grids(const Layout &L, int sms);
bool k3w_plan(const Layout &L, int depth, int sms, int64_t want_nw, int64_t want_nc, int64_t want_k, bool lean, bool half, K3WPlan *out);
cudaError_t launch_k3w(int dtype, const Layout &L, const K3WPlan &P, FieldPtrs fld, void *const coef[4], const StepCommon &sc,
                       int64_t nsteps, cudaStream_t st);
cudaError_t k3w_max_clusters(int dtype, const K3WPlan &P, int *nclusters);

constexpr int kK2Variants = 8;
constexpr int kNumCoefArrays = 4;                                 // P, ch, ka, Q (rketd_device.cuh COEF_*)
int k2_tile_rows(int variant);                                    // rows per tile of a K2 variant, 0 if none
int k2_tiles_per_cta(int variant);                               // tiles a CTA works on at a time (warp tiles)
size_t k2_smem_bytes(int variant);
int k3_threads_for_rows(int dtype, int64_t nrows, int variant);   // threads per CTA of the K3 kernel, or 0

cudaError_t launch_k1(int dtype, const Layout &L, FieldPtrs src, FieldPtrs dst, void *const coef[kNumCoefArrays],
                      const StepCommon &sc, cudaStream_t st);
// tile_end >= 0: only the tiles [tile_begin, tile_end) of the plan (rketd_run_from_host)
cudaError_t launch_k2(int dtype, const Layout &L, const K2Plan &plan, int src_buf, FieldPtrs dst, const StepCommon &sc,
                      int steps, cudaStream_t st, int64_t tile_begin = 0, int64_t tile_end = -1);
// tile_flags[t]: OR of the row flags of the grid's rows 32 t .. 32 t + 31 (host copy; nullptr or balance = false: tile t on
// warp t)
cudaError_t launch_k3(int dtype, const Layout &L, FieldPtrs fld, void *const coef[kNumCoefArrays], const StepCommon &sc,
                      int64_t nsteps, int NT, int variant, cudaStream_t st, const uint8_t *tile_flags = nullptr,
                      bool balance = false);
cudaError_t k2_configure(int dtype, int variant, int *ctas_per_sm);   // sets smem attribute, returns occupancy

// auxiliary kernels (rketd_aux.cu)
// media: user wp, nu [nbatch][ncells] -> padded fp64 copies wp_p, nu_p + the four kernel coefficients
cudaError_t launch_coefficients(int dtype, const Layout &L, const double *wp, const double *nu, double dz,
                                double dt, int scheme, const PmlE &pml, double *wp_p, double *nu_p, void *const coef[kNumCoefArrays],
                                int *d_bad,
                                cudaStream_t st);
// sets *d_bad when any wp or nu (user layout, n values each) is negative or not finite; reads only
cudaError_t launch_validate_media(const double *wp, const double *nu, int64_t n, int *d_bad, cudaStream_t st);
// the six coefficients of SURVEY a0 (ca, cj, ch, ka, kb, kc), recomputed in fp64 from the padded media
cudaError_t launch_six_coefficients(const Layout &L, const double *wp_p, const double *nu_p, double dz, double dt,
                                    int scheme, const PmlE &pml, double *out, cudaStream_t st);
// the four kernel coefficients as stored (P, ch, ka, Q), converted to fp64, user layout
cudaError_t launch_unpack_coefficients(int dtype, const Layout &L, void *const coef[kNumCoefArrays], double *out,
                                       cudaStream_t st);
// J <-> G = cj J - cj kc E on the padded arrays (in place on the third field array)
cudaError_t launch_stage_piece(int dtype, const Layout &L, int64_t i0, int64_t i1, double dz, double dt, int scheme, const PmlE &pml,
                               double *wp_p, double *nu_p, void *const coef[kNumCoefArrays], const void *E, void *G, int *d_bad,
                               cudaStream_t st);
cudaError_t launch_current_to_G(int dtype, const Layout &L, const double *wp_p, const double *nu_p, double dz,
                                double dt, int scheme, const PmlE &pml, const void *E, void *JG, cudaStream_t st);
cudaError_t launch_G_to_current(int dtype, const Layout &L, const double *wp_p, const double *nu_p, double dz,
                                double dt, int scheme, const PmlE &pml, const void *E, const void *G, void *J_user, cudaStream_t st);
cudaError_t launch_twiddles(const double *d_freqs, int nfreq, int64_t step0, int64_t nsteps, double dt,
                            double2 *tw, cudaStream_t st);
cudaError_t launch_dft_accumulate(int dtype, const void *rec, int64_t nseries, int64_t nsteps, const double2 *tw,
                                  int nfreq, double *re, double *im, cudaStream_t st);
cudaError_t launch_dft_magnitude(int dtype, const double *re, const double *im, int64_t n, void *out,
                                 cudaStream_t st);

cudaError_t launch_sweep_rt(const double *sre, const double *sim, const double *vre, const double *vim, int64_t nbatch,
                            int nprobes, int nfreq, int pr, int pt, double *R, double *T, cudaStream_t st);

extern const double kC0, kMu0, kEps0;

}  // namespace rketd
