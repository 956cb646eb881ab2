// rketd_api.cu — the C ABI of librketd (include/rketd.h): handle, device state, plans, launches.
// Host-side logic only; every step of the hot path runs in the kernels of rketd_kernels.cu.
#include <algorithm>
#include <cmath>
#include <cstdio>
#include <cstring>
#include <string>
#include <vector>

#include "../../include/rketd.h"
#include "rketd_device.cuh"
#include "rketd_internal.h"

using namespace rketd;

namespace {
std::string g_create_error;

struct Chunk {
  void *buf;
  int64_t nsteps;
  size_t bytes;
};
}  // namespace

struct rketd_sim {
  Layout L;
  double dz = 0, dt = 0;
  int dtype = 0;
  int scheme = RKETD_SCHEME_ETD2, media_scheme = RKETD_SCHEME_ETD2;   // requested / the one the live coefficients use
  int bc_npml = 0;                 // requested boundary: 0 = first-order Mur, > 0 = absorbing layer of that many nodes
  double bc_m = 3.0, bc_R0 = 1e-6;
  PmlE pml{};                      // the layer the live coefficients use (npml = 0: Mur)
  double pml_ha[kMaxPml] = {}, pml_hd[kMaxPml] = {};
  cudaStream_t stream = nullptr;
  void *fld[2][3] = {{nullptr, nullptr, nullptr}, {nullptr, nullptr, nullptr}};
  int cur = 0;
  void *coef[kNumCoefArrays] = {nullptr, nullptr, nullptr, nullptr};   // P, ch, ka, Q (rketd_device.cuh)
  double *wp_p = nullptr, *nu_p = nullptr;                              // media in the padded layout, fp64
  uint8_t *rowflag = nullptr;
  std::vector<uint8_t> h_rowflag;  // host copy (k3_resident: which warps carry a boundary, the source, a probe)
  bool flags_dirty = true;
  bool have_media = false;
  bool fields_zero = true;      // E = H = J = 0 (after create / reset): no J <-> G conversion needed
  bool third_is_J = false;      // the third field array holds J, not G (fields set before the media)
  int *d_bad = nullptr;
  int src_kind = RKETD_SRC_NONE;
  std::vector<double> src_params;
  int64_t src_cell = -1;
  // source samples of the global steps [srctab_step0, srctab_step0 + srctab_len): device table + the pinned host
  // buffer it was uploaded from; kept across runs, so that a repeated run (rketd_reset + rketd_run) enqueues nothing
  void *d_srctab = nullptr, *h_srctab = nullptr;
  int64_t srctab_cap = 0, srctab_step0 = 0, srctab_len = 0;
  bool srctab_valid = false;
  // DFT mode: record segment and twiddle table, grow-only (no allocation or synchronisation inside rketd_run)
  void *dft_rec = nullptr;
  double2 *dft_tw = nullptr;
  size_t dft_rec_bytes = 0, dft_tw_bytes = 0;
  void *dft_out = nullptr;       // magnitudes staged for rketd_read_probes
  size_t dft_out_bytes = 0;
  std::vector<int64_t> probes;
  std::vector<double> freqs;
  double *d_freqs = nullptr, *dft_re = nullptr, *dft_im = nullptr;
  std::vector<Chunk> chunks;
  void *spare_buf = nullptr;     // one discarded record buffer kept for the next rketd_run (no cudaMalloc per run)
  size_t spare_bytes = 0;
  int64_t nsamples = 0;
  int64_t step = 0;
  int plan_kernel = RKETD_KERNEL_AUTO, plan_depth = 0, plan_variant = -1;
  K2Plan k2;
  bool k2_valid = false;
  int sms = 0;                   // multiprocessors of the device the handle lives on
  // rketd_run_from_host: the copies of later pieces run on a stream of their own, one event per piece
  cudaStream_t copy_stream = nullptr;
  cudaEvent_t ev_ready = nullptr;
  std::vector<cudaEvent_t> ev_piece;
  int64_t ctr_pieces = 0;
  int64_t ctr_launches = 0, ctr_step_launches = 0, ctr_kernel_used = 0, ctr_depth_used = 0, ctr_tile_cells = 0,
          ctr_halo_cells = 0, state_bytes = 0;
  std::string err;
};

namespace {

int fail(rketd_sim *s, int code, const std::string &msg) {
  if (s) s->err = msg; else g_create_error = msg;
  return code;
}
#define CU_TRY(s, expr)                                                                          \
  do {                                                                                           \
    cudaError_t e__ = (expr);                                                                    \
    if (e__ != cudaSuccess)                                                                      \
      return fail(s, e__ == cudaErrorMemoryAllocation ? RKETD_ENOMEM : RKETD_ECUDA,              \
                  std::string(#expr) + ": " + cudaGetErrorString(e__));                          \
  } while (0)

size_t arr_bytes(const Layout &L) { return (size_t)L.gstride * L.nbatch * L.esize; }

bool is_device_ptr(const void *p) {
  cudaPointerAttributes at;
  if (cudaPointerGetAttributes(&at, p) != cudaSuccess) { cudaGetLastError(); return false; }
  return at.type == cudaMemoryTypeDevice || at.type == cudaMemoryTypeManaged;
}

// pack / unpack between the user's [nbatch][ncells] and the padded physical layout
cudaError_t copy_in(const rketd_sim *s, void *dst_phys, const void *src_user) {
  const Layout &L = s->L;
  return cudaMemcpy2DAsync((char *)dst_phys + (size_t)L.off * L.esize, (size_t)L.gstride * L.esize, src_user,
                           (size_t)L.ncells * L.esize, (size_t)L.ncells * L.esize, (size_t)L.nbatch, cudaMemcpyDefault,
                           s->stream);
}
cudaError_t copy_out(const rketd_sim *s, void *dst_user, const void *src_phys) {
  const Layout &L = s->L;
  return cudaMemcpy2DAsync(dst_user, (size_t)L.ncells * L.esize, (const char *)src_phys + (size_t)L.off * L.esize,
                           (size_t)L.gstride * L.esize, (size_t)L.ncells * L.esize, (size_t)L.nbatch, cudaMemcpyDefault,
                           s->stream);
}

void discard_records(rketd_sim *s) {
  for (auto &c : s->chunks) {
    if (c.bytes > s->spare_bytes) {
      if (s->spare_buf) cudaFree(s->spare_buf);
      s->spare_buf = c.buf; s->spare_bytes = c.bytes;
    } else {
      cudaFree(c.buf);
    }
  }
  s->chunks.clear();
  s->nsamples = 0;
  if (s->dft_re) {
    const size_t n = (size_t)s->L.nbatch * s->probes.size() * s->freqs.size() * sizeof(double);
    cudaMemsetAsync(s->dft_re, 0, n, s->stream);
    cudaMemsetAsync(s->dft_im, 0, n, s->stream);
  }
}

int realloc_dft(rketd_sim *s) {
  if (s->dft_re) { cudaFree(s->dft_re); cudaFree(s->dft_im); s->dft_re = s->dft_im = nullptr; }
  if (s->d_freqs) { cudaFree(s->d_freqs); s->d_freqs = nullptr; }
  if (s->freqs.empty() || s->probes.empty()) return RKETD_OK;
  const size_t n = (size_t)s->L.nbatch * s->probes.size() * s->freqs.size() * sizeof(double);
  CU_TRY(s, cudaMalloc(&s->dft_re, n));
  CU_TRY(s, cudaMalloc(&s->dft_im, n));
  CU_TRY(s, cudaMalloc(&s->d_freqs, s->freqs.size() * sizeof(double)));
  CU_TRY(s, cudaMemcpyAsync(s->d_freqs, s->freqs.data(), s->freqs.size() * sizeof(double), cudaMemcpyHostToDevice,
                            s->stream));
  CU_TRY(s, cudaMemsetAsync(s->dft_re, 0, n, s->stream));
  CU_TRY(s, cudaMemsetAsync(s->dft_im, 0, n, s->stream));
  CU_TRY(s, cudaStreamSynchronize(s->stream));
  return RKETD_OK;
}

int rebuild_rowflags(rketd_sim *s) {
  const Layout &L = s->L;
  std::vector<uint8_t> f((size_t)L.nrows, 0);
  f[(size_t)(L.off / L.C)] |= F_MURL;
  f[(size_t)((L.off + L.ncells - 1) / L.C)] |= F_MURR;
  if (s->src_kind != RKETD_SRC_NONE) f[(size_t)((L.off + s->src_cell) / L.C)] |= F_SRC;
  for (int64_t c : s->probes) f[(size_t)((L.off + c) / L.C)] |= F_PROBE;
  for (int j = 0; j <= s->pml.npml && s->pml.npml > 0; ++j) {   // rows with H nodes of a layer, and the node right of the left layer
    f[(size_t)((L.off + j) / L.C)] |= F_PML;
    f[(size_t)((L.off + L.ncells - 1 - j) / L.C)] |= F_PML;
  }
  CU_TRY(s, cudaMemcpyAsync(s->rowflag, f.data(), f.size(), cudaMemcpyHostToDevice, s->stream));
  CU_TRY(s, cudaStreamSynchronize(s->stream));   // f is a local
  s->h_rowflag.swap(f);
  s->flags_dirty = false;
  return RKETD_OK;
}

double source_sample(const rketd_sim *s, int64_t step_index) {
  if (s->src_kind == RKETD_SRC_GAUSS_DERIV) {
    const double tau = s->src_params[0], t0 = s->src_params[1], A = s->src_params[2];
    const double u = ((double)(step_index + 1) * s->dt - t0) / tau;
    return A * u * std::exp(0.5 - 0.5 * u * u);
  }
  if (s->src_kind == RKETD_SRC_TABLE)
    return (step_index >= 0 && step_index < (int64_t)s->src_params.size()) ? s->src_params[(size_t)step_index] : 0.0;
  return 0.0;
}

typedef CUresult (*EncodeTiledFn)(CUtensorMap *, CUtensorMapDataType, cuuint32_t, void *, const cuuint64_t *,
                                  const cuuint64_t *, const cuuint32_t *, const cuuint32_t *, CUtensorMapInterleave,
                                  CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

EncodeTiledFn get_encode() {
  static EncodeTiledFn fn = nullptr;
  if (!fn) {
    void *p = nullptr;
    cudaDriverEntryPointQueryResult qres;
    if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &qres) == cudaSuccess &&
        qres == cudaDriverEntryPointSuccess)
      fn = (EncodeTiledFn)p;
  }
  return fn;
}

// 3-D view {C, nrows, nbatch} of one per-node array, rows of 64 B, box {C, box_rows, 1}, 64-B swizzle.
int make_map(rketd_sim *s, CUtensorMap *m, void *base, int box_rows) {
  EncodeTiledFn enc = get_encode();
  if (!enc) return fail(s, RKETD_ECUDA, "cuTensorMapEncodeTiled not available from the driver");
  const Layout &L = s->L;
  cuuint64_t dims[3] = {(cuuint64_t)L.C, (cuuint64_t)L.nrows, (cuuint64_t)L.nbatch};
  cuuint64_t strides[2] = {(cuuint64_t)kRowBytes, (cuuint64_t)L.nrows * kRowBytes};
  cuuint32_t box[3] = {(cuuint32_t)L.C, (cuuint32_t)box_rows, 1u};
  cuuint32_t estr[3] = {1u, 1u, 1u};
  CUresult r = enc(m, L.esize == 8 ? CU_TENSOR_MAP_DATA_TYPE_FLOAT64 : CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 3, base, dims,
                   strides, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_64B,
                   CU_TENSOR_MAP_L2_PROMOTION_L2_256B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
  if (r != CUDA_SUCCESS) return fail(s, RKETD_ECUDA, "cuTensorMapEncodeTiled failed: " + std::to_string((int)r));
  return RKETD_OK;
}

// Temporal depth T of K2.  Large problems: 16 (fp64) / 32 (fp32) steps per pass, the deepest setting that still
// sits on the HBM roofline.  Problems whose tiles do not even fill one wave of warps (148 SMs x 12
// warp tiles) are launch-latency bound (the paper's Table 2 sizes): there the deepest pass that still fits one
// wave wins, because it divides the number of launches.
int default_depth(const rketd_sim *s) {
  const int base = s->dtype == RKETD_F64 ? 16 : 32;
  const int64_t one_wave = (int64_t)s->sms * 12;
  for (int T = 4 * base; T > base; T -= base) {
    const int HR = (T + s->L.C - 1) / s->L.C, rows_out = 32 - 2 * HR;
    if (rows_out < 8) continue;
    if (((s->L.nrows + rows_out - 1) / rows_out) * s->L.nbatch <= one_wave) return T;
  }
  return base;
}
int default_k2_variant(const rketd_sim *) { return 6; }
int max_depth(const rketd_sim *s, int variant) { return (k2_tile_rows(variant) / 2 - 1) * s->L.C; }

int build_k2_plan(rketd_sim *s, int depth, int variant) {
  const Layout &L = s->L;
  K2Plan &P = s->k2;
  if (s->k2_valid && P.depth == depth && P.variant == variant) return RKETD_OK;
  const int rows = k2_tile_rows(variant);
  const int HR = (depth + L.C - 1) / L.C;
  if (rows - 2 * HR < 1) return fail(s, RKETD_EINVAL, "temporal depth too large for the tile");
  P.variant = variant; P.rows = rows; P.HR = HR; P.rows_out = rows - 2 * HR; P.depth = depth;
  P.tiles_per_grid = (L.nrows + P.rows_out - 1) / P.rows_out;
  P.total_tiles = P.tiles_per_grid * L.nbatch;
  if (P.total_tiles >= (int64_t)1 << 31) return fail(s, RKETD_EINVAL, "too many tiles for the temporal-blocking kernel");
  P.smem_bytes = k2_smem_bytes(variant);
  int ctas = 0;
  const int sms = s->sms;
  CU_TRY(s, k2_configure(s->dtype, variant, &ctas));
  if (ctas < 1) return fail(s, RKETD_ECUDA, "K2 kernel does not fit on an SM");
  P.ctas_per_sm = ctas;
  const int tpc = k2_tiles_per_cta(variant);
  P.grid = (int)std::min<int64_t>((P.total_tiles + tpc - 1) / tpc, (int64_t)sms * ctas);
  P.spread = 0;
  if (tpc > 1 && P.total_tiles < (int64_t)sms * ctas * tpc) {   // less than one wave of warp tiles
    P.spread = 1;
    P.grid = (int)std::min<int64_t>(P.total_tiles, (int64_t)sms * ctas);
  }
  for (int b = 0; b < 2; ++b) {
    for (int a = 0; a < 3; ++a) {
      int rc = make_map(s, &P.maps[b].ld[a], s->fld[b][a], rows);
      if (rc) return rc;
      rc = make_map(s, &P.maps[b].st[a], s->fld[1 - b][a], P.rows_out);
      if (rc) return rc;
    }
    for (int a = 0; a < kNumCoefArrays; ++a) {
      int rc = make_map(s, &P.maps[b].ld[3 + a], s->coef[a], rows);
      if (rc) return rc;
    }
  }
  s->k2_valid = true;
  return RKETD_OK;
}

// RESIDENT plans.  rketd_set_plan's variant: -1 = the warp-tile kernel k3_wtile with the packing chosen by k3w_plan;
// RKETD_RESIDENT_WTILE(nw, nc, k) = the same with an explicit packing; 0, 2 = the older one-barrier-per-step kernel
// k3_resident (kept as a structurally different cross-check).
// variant -1: warp tiles when the batch is a few grids (a run is then a chain of dependent steps: config 1 runs 1.9 x
// faster than with a barrier per step) or when a grid is too large for one CTA; the one-barrier-per-step kernel when
// many grids that each fit one CTA keep every SM busy — there four small CTAs per SM hide each other's barriers and it
// is still the faster of the two (config 3 1020 against 785 Gcell/s, config 5 863 against 701).
int legacy_k3_variant(const rketd_sim *s) {
  if (s->dtype == RKETD_F32 && s->L.nrows <= 64) return 0;      // (config 5 fp32, 64 rows: 1288 against 1230 Gcell/s)
  return (s->L.nrows > 32 && s->L.nrows <= 256) ? 2 : 0;
}
bool wtile_variant(const rketd_sim *s, int variant) {
  if (variant >= 0) return (variant & RKETD_RESIDENT_WTILE_FLAG) != 0;
  return k3w_few_grids(s->L, s->sms) || !k3_threads_for_rows(s->dtype, s->L.nrows, 0);
}
bool resident_wtile_plan(rketd_sim *s, int depth, int variant, K3WPlan *P) {
  int64_t nw = 0, nc = 0, k = 0;
  if (variant >= 0) { nw = variant & 0xff; nc = (variant >> 8) & 0xff; k = (variant >> 16) & 0x3ff; }
  const bool few = k3w_few_grids(s->L, s->sms), no_layer = s->bc_npml == 0 && s->pml.npml == 0;
  // the lean instantiation (<= 128 registers) serves Mur ends with at most two probes among the nodes of one lane
  // (measured: +26 % on config 3, +55 % on config 5 when many chunks share the SMs; 12 % slower on config 1, where one chunk is
  // a chain of dependent steps and the in-place update lengthens it — so: many grids only, unless the variant says otherwise)
  const bool ask_lean = variant >= 0 && (variant & RKETD_RESIDENT_WTILE_LEAN), ask_fat = variant >= 0 && (variant & RKETD_RESIDENT_WTILE_NOLEAN);
  const bool ask_half = variant >= 0 && (variant & RKETD_RESIDENT_WTILE_HALF), ask_full = variant >= 0 && (variant & RKETD_RESIDENT_WTILE_NOHALF);
  bool lean = no_layer && !ask_fat && !ask_half && (ask_lean || !few);
  if (lean) {
    std::vector<int64_t> rows;
    for (int64_t c : s->probes) rows.push_back((s->L.off + c) / s->L.C);
    std::sort(rows.begin(), rows.end());
    for (size_t i = 2; i < rows.size(); ++i) lean = lean && rows[i] != rows[i - 2];
  }
  // half rows per lane (a few grids = a chain of dependent steps: a step of 4 fp64 nodes per lane takes 75 cycles against 141,
  // profiles/r02_peaks.md); Mur ends only, at most two probes in one lane's nodes (else the general path, which is slower)
  bool half = no_layer && !lean && !ask_full && (ask_half || (few && variant < 0));
  auto schedulable = [&](K3WPlan *Q) {
    if (Q->nc <= 1 && !Q->half) return true;   // the cluster must be schedulable on this device (GPC size, registers, shared memory)
    int ncl = 0;
    if (k3w_max_clusters(s->dtype, *Q, &ncl) != cudaSuccess || ncl < 1) { cudaGetLastError(); return false; }
    return true;
  };
  if (half) {
    if (k3w_plan(s->L, depth, s->sms, nw, nc, k, false, true, P) && schedulable(P)) return true;
    if (ask_half) return false;
  }
  return k3w_plan(s->L, depth, s->sms, nw, nc, k, lean, false, P) && schedulable(P);
}

int resolve_kernel(rketd_sim *s) {
  if (s->plan_kernel != RKETD_KERNEL_AUTO) return s->plan_kernel;
  if (!wtile_variant(s, -1)) return RKETD_KERNEL_RESIDENT;          // many grids, each fits one CTA
  K3WPlan P;
  if (!resident_wtile_plan(s, 0, -1, &P)) return RKETD_KERNEL_TBLOCK;
  // one long line spread over most of a 16-CTA cluster: K2's deep passes (T = 64) win again from about 100 warp
  // tiles on (paper Table 2: 40 960 cells 0.44 ms against 0.54; 20 480 cells 0.47 against 0.41)
  if (k3w_few_grids(s->L, s->sms) && P.nc * P.nw > (P.half ? 128 : 96)) return RKETD_KERNEL_TBLOCK;
  return RKETD_KERNEL_RESIDENT;
}

// source table and launch-wide parameters of a segment of nsteps steps that starts at s->step
int prepare_common(rketd_sim *s, int64_t nsteps, void *rec, StepCommon &sc) {
  const Layout &L = s->L;
  // source samples of this segment: a slice of the kept table when it covers the steps, else the table is rebuilt
  const void *d_src = nullptr;
  if (s->src_kind != RKETD_SRC_NONE) {
    const bool covered = s->srctab_valid && s->step >= s->srctab_step0 && s->step + nsteps <= s->srctab_step0 + s->srctab_len;
    if (!covered) {
      if (s->srctab_cap < nsteps) {
        CU_TRY(s, cudaStreamSynchronize(s->stream));      // earlier launches may still read the old table
        if (s->d_srctab) cudaFree(s->d_srctab);
        if (s->h_srctab) cudaFreeHost(s->h_srctab);
        s->d_srctab = s->h_srctab = nullptr; s->srctab_cap = 0; s->srctab_valid = false;
        CU_TRY(s, cudaMalloc(&s->d_srctab, (size_t)nsteps * L.esize));
        CU_TRY(s, cudaMallocHost(&s->h_srctab, (size_t)nsteps * L.esize));
        s->srctab_cap = nsteps;
      } else if (s->srctab_valid) {
        CU_TRY(s, cudaStreamSynchronize(s->stream));      // the pinned buffer may still be in flight, the table in use
      }
      if (s->dtype == RKETD_F64) {
        double *tab = (double *)s->h_srctab;
        for (int64_t n = 0; n < nsteps; ++n) tab[n] = source_sample(s, s->step + n);
      } else {
        float *tab = (float *)s->h_srctab;
        for (int64_t n = 0; n < nsteps; ++n) tab[n] = (float)source_sample(s, s->step + n);
      }
      CU_TRY(s, cudaMemcpyAsync(s->d_srctab, s->h_srctab, (size_t)nsteps * L.esize, cudaMemcpyHostToDevice, s->stream));
      s->srctab_step0 = s->step; s->srctab_len = nsteps; s->srctab_valid = true;
    }
    d_src = (const char *)s->d_srctab + (size_t)(s->step - s->srctab_step0) * L.esize;
  }
  std::memset(&sc, 0, sizeof(sc));
  sc.nchh = -(s->dt / (kMu0 * s->dz));
  const double S = kC0 * s->dt / s->dz;
  sc.mur_m = (S - 1.0) / (S + 1.0);
  sc.cellL = L.off; sc.cellR = L.off + L.ncells - 1;
  sc.cellS = s->src_kind == RKETD_SRC_NONE ? -1 : L.off + s->src_cell;
  sc.nprobes = (int)s->probes.size();
  for (size_t i = 0; i < s->probes.size(); ++i) sc.probe_cell[i] = L.off + s->probes[i];
  sc.rec_stride = nsteps; sc.n0 = 0; sc.src_tab = d_src; sc.rec = rec; sc.rowflag = s->rowflag;
  sc.npml = s->pml.npml;
  std::memcpy(sc.pml_ha, s->pml_ha, sizeof(sc.pml_ha));
  std::memcpy(sc.pml_hd, s->pml_hd, sizeof(sc.pml_hd));
  return RKETD_OK;
}

// absorbing layer requested by rketd_set_boundary: tables of the E nodes (into the coefficient arrays) and of the H nodes
// (kernel parameters)
void make_pml_tables(const rketd_sim *s, PmlE &new_pml, double (&new_ha)[kMaxPml], double (&new_hd)[kMaxPml]) {
  new_pml.npml = s->bc_npml;
  if (s->bc_npml > 0) {
    const int np = s->bc_npml;
    const double smax = -(s->bc_m + 1.0) * kEps0 * kC0 * std::log(s->bc_R0) / (2.0 * (double)np * s->dz);
    const double nchh = -(s->dt / (kMu0 * s->dz));
    for (int j = 0; j < np; ++j) {
      const double rho_e = (double)(np - j) / (double)np, rho_h = ((double)(np - j) - 0.5) / (double)np;
      const double se = smax * std::pow(rho_e, s->bc_m) * s->dt / (2.0 * kEps0);
      const double sh = smax * std::pow(rho_h, s->bc_m) * s->dt / (2.0 * kEps0);
      new_pml.a[j] = (1.0 - se) / (1.0 + se);
      new_pml.b[j] = (s->dt / (kEps0 * s->dz)) / (1.0 + se);
      new_ha[j] = (1.0 - sh) / (1.0 + sh);
      new_hd[j] = nchh / (1.0 + sh) - nchh;
    }
  }
}

// run nsteps steps whose probe samples go to rec ([nbatch][nprobes][nsteps] or nullptr)
int run_segment(rketd_sim *s, int64_t nsteps, void *rec) {
  const Layout &L = s->L;
  StepCommon sc;
  { int rc = prepare_common(s, nsteps, rec, sc); if (rc) return rc; }

  const int kern = resolve_kernel(s);
  s->ctr_kernel_used = kern;
  if (kern == RKETD_KERNEL_STEP) {
    for (int64_t n = 0; n < nsteps; ++n) {
      sc.n0 = n;
      FieldPtrs src{s->fld[s->cur][0], s->fld[s->cur][1], s->fld[s->cur][2]};
      FieldPtrs dst{s->fld[1 - s->cur][0], s->fld[1 - s->cur][1], s->fld[1 - s->cur][2]};
      CU_TRY(s, launch_k1(s->dtype, L, src, dst, s->coef, sc, s->stream));
      s->cur ^= 1;
      ++s->ctr_launches; ++s->ctr_step_launches;
    }
    s->ctr_tile_cells = L.C; s->ctr_halo_cells = 1; s->ctr_depth_used = 1;
  } else if (kern == RKETD_KERNEL_RESIDENT) {
    FieldPtrs f{s->fld[s->cur][0], s->fld[s->cur][1], s->fld[s->cur][2]};
    if (wtile_variant(s, s->plan_variant)) {
      K3WPlan P;
      if (!resident_wtile_plan(s, s->plan_kernel == RKETD_KERNEL_RESIDENT ? s->plan_depth : 0, s->plan_variant, &P))
        return fail(s, RKETD_EINVAL, "grid too large for the resident kernel (or the requested packing cannot run)");
      CU_TRY(s, launch_k3w(s->dtype, L, P, f, s->coef, sc, nsteps, s->stream));
      // cells a chunk occupies on chip (halo and padding lanes included) against the cells it holds
      s->ctr_tile_cells = (int64_t)P.nc * P.nw * 32 * (P.half ? L.C / 2 : L.C);
      s->ctr_halo_cells = (s->ctr_tile_cells - P.k * L.gstride) / 2;
      s->ctr_depth_used = P.T;
    } else {
      int variant = s->plan_variant >= 0 ? s->plan_variant : legacy_k3_variant(s);
      if (!k3_threads_for_rows(s->dtype, L.nrows, variant)) variant = 0;
      const int NT = k3_threads_for_rows(s->dtype, L.nrows, variant);
      if (!NT) return fail(s, RKETD_EINVAL, "grid too large for the one-CTA resident kernel");
      // library's choice: the heavy tiles of a grid dealt over the SM's schedulers; an explicit variant keeps tile t on warp t
      uint8_t tile_flags[16] = {};
      for (int64_t r = 0; r < L.nrows && r < (int64_t)s->h_rowflag.size(); ++r) tile_flags[r / 32] |= s->h_rowflag[(size_t)r];
      CU_TRY(s, launch_k3(s->dtype, L, f, s->coef, sc, nsteps, NT, variant, s->stream, tile_flags, s->plan_variant < 0));
      s->ctr_tile_cells = L.gstride; s->ctr_halo_cells = 0; s->ctr_depth_used = nsteps;
    }
    ++s->ctr_launches; ++s->ctr_step_launches;
  } else {
    const int variant = s->plan_variant >= 0 ? s->plan_variant : default_k2_variant(s);
    int depth = s->plan_depth > 0 ? s->plan_depth : default_depth(s);
    depth = std::min<int>(depth, max_depth(s, variant));
    int rc = build_k2_plan(s, depth, variant);
    if (rc) return rc;
    for (int64_t n = 0; n < nsteps; n += depth) {
      const int steps = (int)std::min<int64_t>(depth, nsteps - n);
      sc.n0 = n;
      FieldPtrs dst{s->fld[1 - s->cur][0], s->fld[1 - s->cur][1], s->fld[1 - s->cur][2]};
      CU_TRY(s, launch_k2(s->dtype, L, s->k2, s->cur, dst, sc, steps, s->stream));
      s->cur ^= 1;
      ++s->ctr_launches; ++s->ctr_step_launches;
    }
    s->ctr_tile_cells = (int64_t)s->k2.rows * L.C; s->ctr_halo_cells = (int64_t)s->k2.HR * L.C; s->ctr_depth_used = depth;
  }
  s->step += nsteps;
  return RKETD_OK;
}

}  // namespace

extern "C" {

int rketd_create(rketd_sim **out, int64_t ncells, int64_t nbatch, double dz, double dt, int dtype, void *cuda_stream) {
  if (!out) return fail(nullptr, RKETD_EINVAL, "out is NULL");
  *out = nullptr;
  if (ncells < 3 || nbatch < 1 || !(dz > 0) || !(dt > 0) || (dtype != RKETD_F64 && dtype != RKETD_F32))
    return fail(nullptr, RKETD_EINVAL, "rketd_create: invalid argument");
  if (kC0 * dt / dz > 1.0 + 1e-12) return fail(nullptr, RKETD_EINVAL, "rketd_create: c dt/dz > 1 is unstable");
  int ndev = 0;
  if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev < 1) {
    cudaGetLastError();
    return fail(nullptr, RKETD_ECUDA, "rketd_create: no CUDA device (librketd has no CPU fallback)");
  }
  rketd_sim *s = new rketd_sim();
  {
    int dev = 0;
    if (cudaGetDevice(&dev) != cudaSuccess || cudaDeviceGetAttribute(&s->sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess ||
        s->sms < 1) {
      cudaGetLastError();
      delete s;
      return fail(nullptr, RKETD_ECUDA, "rketd_create: cannot query the device");
    }
  }
  Layout &L = s->L;
  L.ncells = ncells; L.nbatch = nbatch;
  L.esize = dtype == RKETD_F64 ? 8 : 4;
  L.C = kRowBytes / L.esize;
  L.off = ((ncells - 1) % (L.C / 2) == 0) ? 1 : 0;
  L.nrows = (L.off + ncells + L.C - 1) / L.C;
  L.gstride = L.nrows * L.C;
  if (L.nrows > 0x7fffff00LL || nbatch > 0x7fffff00LL) { delete s; return fail(nullptr, RKETD_EINVAL, "grid too large"); }
  s->dz = dz; s->dt = dt; s->dtype = dtype; s->stream = (cudaStream_t)cuda_stream;
  const size_t nb = arr_bytes(L);
  auto bail = [&](cudaError_t e) {
    std::string m = std::string("rketd_create: ") + cudaGetErrorString(e);
    rketd_destroy(s);
    return fail(nullptr, e == cudaErrorMemoryAllocation ? RKETD_ENOMEM : RKETD_ECUDA, m);
  };
  cudaError_t e;
  for (int b = 0; b < 2; ++b)
    for (int a = 0; a < 3; ++a) {
      if ((e = cudaMalloc(&s->fld[b][a], nb)) != cudaSuccess) return bail(e);
      if ((e = cudaMemsetAsync(s->fld[b][a], 0, nb, s->stream)) != cudaSuccess) return bail(e);
    }
  for (int a = 0; a < kNumCoefArrays; ++a) {
    if ((e = cudaMalloc(&s->coef[a], nb)) != cudaSuccess) return bail(e);
    if ((e = cudaMemsetAsync(s->coef[a], 0, nb, s->stream)) != cudaSuccess) return bail(e);
  }
  const size_t nb64 = (size_t)L.gstride * L.nbatch * sizeof(double);
  if ((e = cudaMalloc(&s->wp_p, nb64)) != cudaSuccess) return bail(e);
  if ((e = cudaMalloc(&s->nu_p, nb64)) != cudaSuccess) return bail(e);
  if ((e = cudaMalloc(&s->rowflag, (size_t)L.nrows)) != cudaSuccess) return bail(e);
  if ((e = cudaMalloc(&s->d_bad, sizeof(int))) != cudaSuccess) return bail(e);
  s->state_bytes = (int64_t)nb * (6 + kNumCoefArrays) + 2 * (int64_t)nb64 + L.nrows;
  *out = s;
  return RKETD_OK;
}

int rketd_set_media(rketd_sim *s, const double *wp, const double *nu) {
  if (!s || !wp || !nu) return fail(s, RKETD_EINVAL, "rketd_set_media: NULL argument");
  const Layout &L = s->L;
  const size_t n = (size_t)L.ncells * L.nbatch * sizeof(double);
  const double *dwp = wp, *dnu = nu;
  void *twp = nullptr, *tnu = nullptr, *tJ = nullptr;
  auto cleanup = [&]() { if (twp) cudaFree(twp); if (tnu) cudaFree(tnu); if (tJ) cudaFree(tJ); };
#define SM_TRY(expr) do { cudaError_t sm_e = (expr); if (sm_e != cudaSuccess) { cleanup(); CU_TRY(s, sm_e); } } while (0)
  if (!is_device_ptr(wp)) {
    SM_TRY(cudaMalloc(&twp, n));
    SM_TRY(cudaMemcpyAsync(twp, wp, n, cudaMemcpyDefault, s->stream));
    dwp = (const double *)twp;
  }
  if (!is_device_ptr(nu)) {
    SM_TRY(cudaMalloc(&tnu, n));
    SM_TRY(cudaMemcpyAsync(tnu, nu, n, cudaMemcpyDefault, s->stream));
    dnu = (const double *)tnu;
  }
  // read-only validation first: a rejected call leaves coefficients, media and fields exactly as they were
  int bad = 0;
  SM_TRY(cudaMemsetAsync(s->d_bad, 0, sizeof(int), s->stream));
  SM_TRY(launch_validate_media(dwp, dnu, (int64_t)L.ncells * L.nbatch, s->d_bad, s->stream));
  ++s->ctr_launches;
  SM_TRY(cudaMemcpyAsync(&bad, s->d_bad, sizeof(int), cudaMemcpyDeviceToHost, s->stream));
  SM_TRY(cudaStreamSynchronize(s->stream));
  if (bad) {
    cleanup();
    return fail(s, RKETD_EINVAL, "rketd_set_media: wp and nu must be finite and non-negative");
  }
  // live fields carry G = cj J - cj kc E of the OLD media: put J itself back into the third array before the
  // coefficients change, and say so in third_is_J at once, so that a CUDA failure further down leaves array and flag in
  // agreement (the next successful rketd_set_media converts J -> G)
  const bool reconvert = s->have_media && !s->fields_zero && !s->third_is_J;
  if (reconvert) {
    SM_TRY(cudaMalloc(&tJ, (size_t)L.ncells * L.nbatch * L.esize));
    SM_TRY(launch_G_to_current(s->dtype, L, s->wp_p, s->nu_p, s->dz, s->dt, s->media_scheme, s->pml, s->fld[s->cur][0], s->fld[s->cur][2], tJ,
                               s->stream));
    ++s->ctr_launches;
    SM_TRY(cudaMemsetAsync(s->fld[s->cur][2], 0, arr_bytes(L), s->stream));
    SM_TRY(copy_in(s, s->fld[s->cur][2], tJ));
    s->third_is_J = true;
  }
  // absorbing layer requested by rketd_set_boundary: tables of the E nodes (into the coefficient arrays) and of the
  // H nodes (kernel parameters).  Reading of PAPER.md:93, :123 in DESIGN.md §12: sigma(rho) = sigma_max rho^m,
  // sigma_max = -(m+1) eps0 c ln(R0) / (2 npml dz), rho = depth / thickness, matched sigma* = sigma mu0/eps0.
  PmlE new_pml{};
  double new_ha[kMaxPml] = {}, new_hd[kMaxPml] = {};
  make_pml_tables(s, new_pml, new_ha, new_hd);
  s->have_media = false;      // until the new coefficients are in place
  SM_TRY(launch_coefficients(s->dtype, L, dwp, dnu, s->dz, s->dt, s->scheme, new_pml, s->wp_p, s->nu_p, s->coef, s->d_bad, s->stream));
  ++s->ctr_launches;
  s->media_scheme = s->scheme;
  s->pml = new_pml;
  std::memcpy(s->pml_ha, new_ha, sizeof(new_ha));
  std::memcpy(s->pml_hd, new_hd, sizeof(new_hd));
  s->flags_dirty = true;
  if (s->third_is_J) {
    SM_TRY(launch_current_to_G(s->dtype, L, s->wp_p, s->nu_p, s->dz, s->dt, s->media_scheme, s->pml, s->fld[s->cur][0],
                               s->fld[s->cur][2], s->stream));
    ++s->ctr_launches;
  }
  SM_TRY(cudaStreamSynchronize(s->stream));     // the staging buffers are freed below
#undef SM_TRY
  cleanup();
  s->third_is_J = false;
  s->have_media = true;
  return RKETD_OK;
}

int rketd_set_scheme(rketd_sim *s, int scheme) {
  if (!s) return RKETD_EINVAL;
  if (scheme != RKETD_SCHEME_ETD2 && scheme != RKETD_SCHEME_ETD1) return fail(s, RKETD_EINVAL, "rketd_set_scheme: unknown scheme");
  s->scheme = scheme;
  return RKETD_OK;
}

int rketd_set_boundary(rketd_sim *s, int kind, int npml, double grading, double R0) {
  if (!s) return RKETD_EINVAL;
  if (kind == RKETD_BC_MUR) { s->bc_npml = 0; return RKETD_OK; }
  if (kind != RKETD_BC_PML) return fail(s, RKETD_EINVAL, "rketd_set_boundary: unknown kind");
  if (npml < 1 || npml > kMaxPml || 2 * (int64_t)npml + 1 > s->L.ncells || !(R0 > 0.0) || R0 > 1.0 || !(grading >= 0.0))
    return fail(s, RKETD_EINVAL, "rketd_set_boundary: need 1 <= npml <= 32, 2 npml + 1 <= ncells, 0 < R0 <= 1, grading >= 0");
  s->bc_npml = npml; s->bc_m = grading; s->bc_R0 = R0;
  return RKETD_OK;
}

int rketd_set_source(rketd_sim *s, int kind, const double *params, int64_t nparams, int64_t cell) {
  if (!s) return RKETD_EINVAL;
  s->srctab_valid = false;
  if (kind == RKETD_SRC_NONE) { s->src_kind = kind; s->src_params.clear(); s->src_cell = -1; s->flags_dirty = true; return RKETD_OK; }
  if (kind != RKETD_SRC_GAUSS_DERIV && kind != RKETD_SRC_TABLE) return fail(s, RKETD_EINVAL, "rketd_set_source: unknown kind");
  if (cell < 0 || cell >= s->L.ncells) return fail(s, RKETD_EINVAL, "rketd_set_source: cell outside the grid");
  if (nparams < 0 || (nparams > 0 && !params)) return fail(s, RKETD_EINVAL, "rketd_set_source: bad params");
  if (kind == RKETD_SRC_GAUSS_DERIV && (nparams != 3 || !(params[0] > 0)))
    return fail(s, RKETD_EINVAL, "rketd_set_source: GAUSS_DERIV needs {tau > 0, t0, amplitude}");
  s->src_kind = kind;
  s->src_params.assign(params, params + nparams);
  s->src_cell = cell;
  s->flags_dirty = true;
  return RKETD_OK;
}

int rketd_set_probes(rketd_sim *s, const int64_t *cells, int nprobes) {
  if (!s) return RKETD_EINVAL;
  if (nprobes < 0 || nprobes > kMaxProbes || (nprobes > 0 && !cells)) return fail(s, RKETD_EINVAL, "rketd_set_probes: 0..64 probes");
  for (int i = 0; i < nprobes; ++i)
    if (cells[i] < 0 || cells[i] >= s->L.ncells) return fail(s, RKETD_EINVAL, "rketd_set_probes: cell outside the grid");
  discard_records(s);
  s->probes.assign(cells, cells + nprobes);
  s->flags_dirty = true;
  return realloc_dft(s);
}

int rketd_set_probe_dft(rketd_sim *s, const double *freqs_hz, int nfreq) {
  if (!s) return RKETD_EINVAL;
  if (nfreq < 0 || (nfreq > 0 && !freqs_hz)) return fail(s, RKETD_EINVAL, "rketd_set_probe_dft: bad argument");
  discard_records(s);
  s->freqs.assign(freqs_hz, freqs_hz + nfreq);
  return realloc_dft(s);
}

int rketd_set_fields(rketd_sim *s, const void *E, const void *H, const void *J) {
  if (!s) return RKETD_EINVAL;
  const void *src[3] = {E, H, J};
  for (int a = 0; a < 3; ++a) {
    CU_TRY(s, cudaMemsetAsync(s->fld[s->cur][a], 0, arr_bytes(s->L), s->stream));
    if (src[a]) CU_TRY(s, copy_in(s, s->fld[s->cur][a], src[a]));
  }
  s->fields_zero = !E && !H && !J;
  s->third_is_J = false;
  if (E || J) {   // the kernels carry G = cj J - cj kc E in the third array (rketd_device.cuh)
    if (s->have_media) {
      CU_TRY(s, launch_current_to_G(s->dtype, s->L, s->wp_p, s->nu_p, s->dz, s->dt, s->media_scheme, s->pml, s->fld[s->cur][0],
                                    s->fld[s->cur][2], s->stream));
      ++s->ctr_launches;
    } else {
      s->third_is_J = true;   // converted by rketd_set_media
    }
  }
  CU_TRY(s, cudaStreamSynchronize(s->stream));
  return RKETD_OK;
}

int rketd_reset(rketd_sim *s) {
  if (!s) return RKETD_EINVAL;
  for (int a = 0; a < 3; ++a) CU_TRY(s, cudaMemsetAsync(s->fld[s->cur][a], 0, arr_bytes(s->L), s->stream));
  discard_records(s);
  s->step = 0;
  s->fields_zero = true;
  s->third_is_J = false;
  return RKETD_OK;
}

int rketd_discard_records(rketd_sim *s) {
  if (!s) return RKETD_EINVAL;
  CU_TRY(s, cudaStreamSynchronize(s->stream));
  discard_records(s);
  return RKETD_OK;
}

int rketd_set_plan(rketd_sim *s, int kernel, int depth, int variant) {
  if (!s) return RKETD_EINVAL;
  if (kernel < RKETD_KERNEL_AUTO || kernel > RKETD_KERNEL_RESIDENT || depth < 0) return fail(s, RKETD_EINVAL, "rketd_set_plan: bad argument");
  if (kernel == RKETD_KERNEL_RESIDENT) {
    K3WPlan P;
    if (wtile_variant(s, variant) ? !resident_wtile_plan(s, depth, variant, &P)
                                  : !k3_threads_for_rows(s->dtype, s->L.nrows, variant < 0 ? legacy_k3_variant(s) : variant))
      return fail(s, RKETD_EINVAL, "rketd_set_plan: grid does not fit the resident kernel (or bad depth / packing)");
  }
  if (kernel == RKETD_KERNEL_TBLOCK || kernel == RKETD_KERNEL_AUTO) {
    if (variant >= 0 && kernel == RKETD_KERNEL_TBLOCK && !k2_tile_rows(variant)) return fail(s, RKETD_EINVAL, "rketd_set_plan: unknown variant");
    const int v = (variant >= 0 && k2_tile_rows(variant)) ? variant : default_k2_variant(s);
    if (depth > max_depth(s, v)) return fail(s, RKETD_EINVAL, "rketd_set_plan: depth too large");
  }
  s->plan_kernel = kernel;
  s->plan_depth = depth;
  s->plan_variant = variant;
  return RKETD_OK;
}

int rketd_run(rketd_sim *s, int64_t nsteps) {
  if (!s) return RKETD_EINVAL;
  if (nsteps < 0) return fail(s, RKETD_EINVAL, "rketd_run: nsteps < 0");
  if (!s->have_media) return fail(s, RKETD_ESTATE, "rketd_run before rketd_set_media");
  if (nsteps == 0) return RKETD_OK;
  if (s->flags_dirty) { int rc = rebuild_rowflags(s); if (rc) return rc; }
  s->fields_zero = false;
  const Layout &L = s->L;
  const int64_t nseries = L.nbatch * (int64_t)s->probes.size();
  if (nseries == 0) return run_segment(s, nsteps, nullptr);
  if (s->freqs.empty()) {   // time-series mode: one record chunk per call
    void *buf = nullptr;
    size_t bytes = (size_t)nseries * nsteps * L.esize;
    if (s->spare_buf && s->spare_bytes >= bytes) {
      buf = s->spare_buf; bytes = s->spare_bytes;
      s->spare_buf = nullptr; s->spare_bytes = 0;
    } else {
      CU_TRY(s, cudaMalloc(&buf, bytes));
    }
    int rc = run_segment(s, nsteps, buf);
    if (rc) {             // a failed run records nothing: the chunk list and nsamples stay in step
      cudaStreamSynchronize(s->stream);
      cudaFree(buf);
      cudaGetLastError();
      return rc;
    }
    s->chunks.push_back(Chunk{buf, nsteps, bytes});
    s->nsamples += nsteps;
    return RKETD_OK;
  }
  // DFT mode (a7): the records of a segment are reduced into the accumulators by a second kernel on the same stream
  // and the segment buffer is reused; buffers live in the handle and only grow, so the call stays asynchronous
  const int nfreq = (int)s->freqs.size();
  const int64_t seg_max = std::max<int64_t>(64, std::min<int64_t>(nsteps, ((int64_t)1 << 29) / (nseries * L.esize)));
  const size_t need_rec = (size_t)nseries * std::min(seg_max, nsteps) * L.esize;
  const size_t need_tw = (size_t)std::min(seg_max, nsteps) * nfreq * sizeof(double2);
  if (need_rec > s->dft_rec_bytes || need_tw > s->dft_tw_bytes) {
    CU_TRY(s, cudaStreamSynchronize(s->stream));           // (growing only: an earlier run may still use the old buffers)
    if (need_rec > s->dft_rec_bytes) {
      if (s->dft_rec) cudaFree(s->dft_rec);
      s->dft_rec = nullptr; s->dft_rec_bytes = 0;
      CU_TRY(s, cudaMalloc(&s->dft_rec, need_rec));
      s->dft_rec_bytes = need_rec;
    }
    if (need_tw > s->dft_tw_bytes) {
      if (s->dft_tw) cudaFree(s->dft_tw);
      s->dft_tw = nullptr; s->dft_tw_bytes = 0;
      CU_TRY(s, cudaMalloc((void **)&s->dft_tw, need_tw));
      s->dft_tw_bytes = need_tw;
    }
  }
  for (int64_t n = 0; n < nsteps; n += seg_max) {
    const int64_t seg = std::min(seg_max, nsteps - n);
    const int64_t step0 = s->step;
    int rc = run_segment(s, seg, s->dft_rec);
    if (rc) return rc;
    cudaError_t e = launch_twiddles(s->d_freqs, nfreq, step0, seg, s->dt, s->dft_tw, s->stream);
    if (e == cudaSuccess) e = launch_dft_accumulate(s->dtype, s->dft_rec, nseries, seg, s->dft_tw, nfreq, s->dft_re, s->dft_im, s->stream);
    s->ctr_launches += 2;
    if (e != cudaSuccess) return fail(s, RKETD_ECUDA, std::string("dft: ") + cudaGetErrorString(e));
    s->nsamples += seg;
  }
  return RKETD_OK;
}

int rketd_run_from_host(rketd_sim *s, const double *wp, const double *nu, const void *E0, int64_t nsteps, int npieces) {
  if (!s || !wp || !nu) return fail(s, RKETD_EINVAL, "rketd_run_from_host: NULL argument");
  if (nsteps < 0 || npieces < 0) return fail(s, RKETD_EINVAL, "rketd_run_from_host: nsteps < 0 or npieces < 0");
  const Layout &L = s->L;
  s->ctr_pieces = 0;
  // the time-skewed order needs one line and the temporal-blocking kernel; everything else is the plain sequence
  if (L.nbatch != 1 || !s->freqs.empty() || nsteps == 0 || resolve_kernel(s) != RKETD_KERNEL_TBLOCK) {
    int rc = rketd_reset(s);
    if (!rc) rc = rketd_set_media(s, wp, nu);
    if (!rc) rc = rketd_set_fields(s, E0, nullptr, nullptr);
    if (!rc) rc = rketd_run(s, nsteps);
    return rc;
  }
  if (!s->copy_stream) {
    CU_TRY(s, cudaStreamCreateWithFlags(&s->copy_stream, cudaStreamNonBlocking));
    CU_TRY(s, cudaEventCreateWithFlags(&s->ev_ready, cudaEventDisableTiming));
  }
  int rc = rketd_reset(s);                       // E = H = G = 0 in the current buffers, records dropped, step 0
  if (rc) return rc;
  PmlE new_pml{};
  double new_ha[kMaxPml] = {}, new_hd[kMaxPml] = {};
  make_pml_tables(s, new_pml, new_ha, new_hd);
  if (std::memcmp(&new_pml, &s->pml, sizeof(PmlE)) != 0) s->flags_dirty = true;
  s->have_media = false;                         // until every piece has been staged and found valid
  s->media_scheme = s->scheme;
  s->pml = new_pml;
  std::memcpy(s->pml_ha, new_ha, sizeof(new_ha));
  std::memcpy(s->pml_hd, new_hd, sizeof(new_hd));
  if (s->flags_dirty) { rc = rebuild_rowflags(s); if (rc) return rc; }

  const int variant = s->plan_variant >= 0 ? s->plan_variant : default_k2_variant(s);
  int depth = s->plan_depth > 0 ? s->plan_depth : default_depth(s);
  depth = std::min<int>(depth, max_depth(s, variant));
  rc = build_k2_plan(s, depth, variant);
  if (rc) return rc;
  const K2Plan &P = s->k2;

  void *buf = nullptr;
  size_t bytes = 0;
  if (!s->probes.empty()) {
    bytes = s->probes.size() * (size_t)nsteps * L.esize;
    if (s->spare_buf && s->spare_bytes >= bytes) {
      buf = s->spare_buf; bytes = s->spare_bytes;
      s->spare_buf = nullptr; s->spare_bytes = 0;
    } else {
      CU_TRY(s, cudaMalloc(&buf, bytes));
    }
  }
  auto give_back = [&]() {                       // a failed job records nothing
    if (!buf) return;
    cudaStreamSynchronize(s->stream);
    if (!s->spare_buf) { s->spare_buf = buf; s->spare_bytes = bytes; } else cudaFree(buf);
    buf = nullptr;
  };
#define RH_TRY(expr) do { cudaError_t rh_e = (expr); if (rh_e != cudaSuccess) { cudaStreamSynchronize(s->copy_stream); give_back(); CU_TRY(s, rh_e); } } while (0)
  StepCommon sc;
  rc = prepare_common(s, nsteps, buf, sc);
  if (rc) { give_back(); return rc; }

  // pieces of whole tiles; a pass moves every piece boundary k tiles to the left (the tiles right of it lack their halo)
  const int64_t Tt = P.tiles_per_grid, k = (P.HR + P.rows_out - 1) / P.rows_out;
  const int64_t piece_tiles = npieces > 0 ? (Tt + npieces - 1) / npieces
                                          : std::max<int64_t>((Tt + 11) / 12, (int64_t)8 * s->sms * k2_tiles_per_cta(variant));
  const int64_t npc = (Tt + piece_tiles - 1) / piece_tiles;
  while ((int64_t)s->ev_piece.size() < npc) {
    cudaEvent_t e;
    RH_TRY(cudaEventCreateWithFlags(&e, cudaEventDisableTiming));
    s->ev_piece.push_back(e);
  }
  const int cur0 = s->cur;
  RH_TRY(cudaMemsetAsync(s->d_bad, 0, sizeof(int), s->stream));
  RH_TRY(cudaEventRecord(s->ev_ready, s->stream));                     // the cleared arrays, and everything before
  RH_TRY(cudaStreamWaitEvent(s->copy_stream, s->ev_ready, 0));
  const int64_t node_per_tile = (int64_t)P.rows_out * L.C;
  auto piece_nodes = [&](int64_t c, int64_t &i0, int64_t &i1) {       // physical nodes of piece c
    i0 = c * piece_tiles * node_per_tile;
    i1 = c == npc - 1 ? L.gstride : std::min<int64_t>(L.gstride, (c + 1) * piece_tiles * node_per_tile);
  };
  for (int64_t c = 0; c < npc; ++c) {
    int64_t i0, i1;
    piece_nodes(c, i0, i1);
    const int64_t k0 = std::max<int64_t>(i0 - L.off, 0), k1 = std::min<int64_t>(i1 - L.off, L.ncells);
    if (k1 > k0) {
      const size_t n = (size_t)(k1 - k0);
      RH_TRY(cudaMemcpyAsync(s->wp_p + L.off + k0, wp + k0, n * sizeof(double), cudaMemcpyDefault, s->copy_stream));
      RH_TRY(cudaMemcpyAsync(s->nu_p + L.off + k0, nu + k0, n * sizeof(double), cudaMemcpyDefault, s->copy_stream));
      if (E0)
        RH_TRY(cudaMemcpyAsync((char *)s->fld[cur0][0] + (size_t)(L.off + k0) * L.esize, (const char *)E0 + (size_t)k0 * L.esize,
                               n * L.esize, cudaMemcpyDefault, s->copy_stream));
    }
    RH_TRY(cudaEventRecord(s->ev_piece[(size_t)c], s->copy_stream));
  }
  const int64_t npass = (nsteps + depth - 1) / depth;
  for (int64_t c = 0; c < npc; ++c) {
    int64_t i0, i1;
    piece_nodes(c, i0, i1);
    RH_TRY(cudaStreamWaitEvent(s->stream, s->ev_piece[(size_t)c], 0));
    RH_TRY(launch_stage_piece(s->dtype, L, i0, i1, s->dz, s->dt, s->media_scheme, s->pml, s->wp_p, s->nu_p, s->coef,
                              s->fld[cur0][0], s->fld[cur0][2], s->d_bad, s->stream));
    ++s->ctr_launches;
    const int64_t b0 = c * piece_tiles, b1 = std::min<int64_t>(Tt, b0 + piece_tiles);
    for (int64_t p = 1; p <= npass; ++p) {
      const int64_t tb = std::max<int64_t>(0, b0 - p * k), te = c == npc - 1 ? Tt : b1 - p * k;
      if (te <= tb) continue;
      const int src_buf = (cur0 + (int)((p - 1) & 1)) & 1;
      sc.n0 = (p - 1) * depth;
      FieldPtrs dst{s->fld[1 - src_buf][0], s->fld[1 - src_buf][1], s->fld[1 - src_buf][2]};
      RH_TRY(launch_k2(s->dtype, L, P, src_buf, dst, sc, (int)std::min<int64_t>(depth, nsteps - sc.n0), s->stream, tb, te));
      ++s->ctr_launches; ++s->ctr_step_launches;
    }
  }
  int bad = 0;
  RH_TRY(cudaMemcpyAsync(&bad, s->d_bad, sizeof(int), cudaMemcpyDeviceToHost, s->stream));
  RH_TRY(cudaStreamSynchronize(s->stream));
#undef RH_TRY
  s->ctr_kernel_used = RKETD_KERNEL_TBLOCK;
  s->ctr_tile_cells = (int64_t)P.rows * L.C; s->ctr_halo_cells = (int64_t)P.HR * L.C; s->ctr_depth_used = depth;
  s->ctr_pieces = npc;
  if (bad) {                                     // the steps ran on garbage: nothing of this job is kept
    give_back();
    rketd_reset(s);
    return fail(s, RKETD_EINVAL, "rketd_run_from_host: wp and nu must be finite and non-negative (the handle now has no media)");
  }
  s->cur = (cur0 + (int)(npass & 1)) & 1;
  s->step = nsteps;
  s->have_media = true;
  s->fields_zero = false;
  s->third_is_J = false;
  if (buf) {
    s->chunks.push_back(Chunk{buf, nsteps, bytes});
    s->nsamples += nsteps;
  }
  return RKETD_OK;
}

int rketd_read_probes(rketd_sim *s, void *out, int64_t out_bytes, int64_t *nsamples) {
  if (!s) return RKETD_EINVAL;
  const Layout &L = s->L;
  const int64_t nseries = L.nbatch * (int64_t)s->probes.size();
  const bool dft = !s->freqs.empty();
  const int64_t per = dft ? (int64_t)s->freqs.size() : s->nsamples;
  if (nsamples) *nsamples = per;
  if (!out) { CU_TRY(s, cudaStreamSynchronize(s->stream)); return RKETD_OK; }
  const int64_t need = nseries * per * L.esize;
  if (out_bytes < need) return fail(s, RKETD_EINVAL, "rketd_read_probes: out buffer too small");
  if (need == 0) { CU_TRY(s, cudaStreamSynchronize(s->stream)); return RKETD_OK; }
  if (dft) {
    void *dst = out;
    if (!is_device_ptr(out)) {           // magnitudes are formed on the device, then copied out
      if ((size_t)need > s->dft_out_bytes) {
        if (s->dft_out) cudaFree(s->dft_out);
        s->dft_out = nullptr; s->dft_out_bytes = 0;
        CU_TRY(s, cudaMalloc(&s->dft_out, (size_t)need));
        s->dft_out_bytes = (size_t)need;
      }
      dst = s->dft_out;
    }
    CU_TRY(s, launch_dft_magnitude(s->dtype, s->dft_re, s->dft_im, nseries * per, dst, s->stream));
    ++s->ctr_launches;
    if (dst != out) CU_TRY(s, cudaMemcpyAsync(out, dst, (size_t)need, cudaMemcpyDefault, s->stream));
    CU_TRY(s, cudaStreamSynchronize(s->stream));
    return RKETD_OK;
  }
  int64_t o = 0;
  for (const Chunk &c : s->chunks) {
    CU_TRY(s, cudaMemcpy2DAsync((char *)out + o * L.esize, (size_t)per * L.esize, c.buf, (size_t)c.nsteps * L.esize,
                                (size_t)c.nsteps * L.esize, (size_t)nseries, cudaMemcpyDefault, s->stream));
    o += c.nsteps;
  }
  CU_TRY(s, cudaStreamSynchronize(s->stream));
  return RKETD_OK;
}

int rketd_read_probe_dft(rketd_sim *s, double *re, double *im, int64_t count) {
  if (!s) return RKETD_EINVAL;
  if (s->freqs.empty()) return fail(s, RKETD_ESTATE, "rketd_read_probe_dft: not in DFT mode (rketd_set_probe_dft)");
  const int64_t n = s->L.nbatch * (int64_t)s->probes.size() * (int64_t)s->freqs.size();
  if (count < n || (n > 0 && (!re || !im))) return fail(s, RKETD_EINVAL, "rketd_read_probe_dft: buffers too small");
  if (n > 0) {
    CU_TRY(s, cudaMemcpyAsync(re, s->dft_re, (size_t)n * sizeof(double), cudaMemcpyDefault, s->stream));
    CU_TRY(s, cudaMemcpyAsync(im, s->dft_im, (size_t)n * sizeof(double), cudaMemcpyDefault, s->stream));
  }
  CU_TRY(s, cudaStreamSynchronize(s->stream));
  return RKETD_OK;
}

int rketd_read_sweep_rt(rketd_sim *s, rketd_sim *vac, int probe_r, int probe_t, double *R, double *T, int64_t count) {
  if (!s || !vac) return fail(s, RKETD_EINVAL, "rketd_read_sweep_rt: NULL handle");
  if (s->freqs.empty() || vac->freqs.empty()) return fail(s, RKETD_ESTATE, "rketd_read_sweep_rt: both handles must be in DFT mode");
  const int np = (int)s->probes.size(), nf = (int)s->freqs.size();
  if (vac->probes != s->probes || vac->freqs != s->freqs)
    return fail(s, RKETD_EINVAL, "rketd_read_sweep_rt: the vacuum handle needs the same probes and frequencies");
  if (probe_r < 0 || probe_r >= np || probe_t < 0 || probe_t >= np || !R || !T || count < s->L.nbatch * (int64_t)nf)
    return fail(s, RKETD_EINVAL, "rketd_read_sweep_rt: bad probe index or buffers too small");
  CU_TRY(s, cudaStreamSynchronize(vac->stream));           // the two handles may live on different streams
  const size_t bytes = (size_t)s->L.nbatch * nf * sizeof(double);
  double *dR = R, *dT = T;
  void *tmp = nullptr;
  if (!is_device_ptr(R) || !is_device_ptr(T)) {
    CU_TRY(s, cudaMalloc(&tmp, 2 * bytes));
    dR = (double *)tmp; dT = dR + (size_t)s->L.nbatch * nf;
  }
  cudaError_t e = launch_sweep_rt(s->dft_re, s->dft_im, vac->dft_re, vac->dft_im, s->L.nbatch, np, nf, probe_r, probe_t, dR, dT, s->stream);
  ++s->ctr_launches;
  if (e == cudaSuccess && tmp) e = cudaMemcpyAsync(R, dR, bytes, cudaMemcpyDefault, s->stream);
  if (e == cudaSuccess && tmp) e = cudaMemcpyAsync(T, dT, bytes, cudaMemcpyDefault, s->stream);
  if (e == cudaSuccess) e = cudaStreamSynchronize(s->stream);
  if (tmp) cudaFree(tmp);
  CU_TRY(s, e);
  return RKETD_OK;
}

int rketd_get_fields(rketd_sim *s, void *E, void *H, void *J) {
  if (!s) return RKETD_EINVAL;
  if (E) CU_TRY(s, copy_out(s, E, s->fld[s->cur][0]));
  if (H) CU_TRY(s, copy_out(s, H, s->fld[s->cur][1]));
  void *tmp = nullptr;
  if (J) {
    if (!s->have_media || s->third_is_J) {   // nothing has run yet: the array still holds J itself
      CU_TRY(s, copy_out(s, J, s->fld[s->cur][2]));
    } else {                                 // J = (G + cj kc E)/cj
      const size_t n = (size_t)s->L.ncells * s->L.nbatch * s->L.esize;
      void *dst = J;
      if (!is_device_ptr(J)) { CU_TRY(s, cudaMalloc(&tmp, n)); dst = tmp; }
      cudaError_t e = launch_G_to_current(s->dtype, s->L, s->wp_p, s->nu_p, s->dz, s->dt, s->media_scheme, s->pml,
                                          s->fld[s->cur][0], s->fld[s->cur][2], dst, s->stream);
      ++s->ctr_launches;
      if (e == cudaSuccess && tmp) e = cudaMemcpyAsync(J, tmp, n, cudaMemcpyDefault, s->stream);
      if (e != cudaSuccess) { if (tmp) cudaFree(tmp); CU_TRY(s, e); }
    }
  }
  const cudaError_t e = cudaStreamSynchronize(s->stream);
  if (tmp) cudaFree(tmp);
  CU_TRY(s, e);
  return RKETD_OK;
}

int rketd_get_coefficients(rketd_sim *s, double *out, double *chh_m) {
  if (!s || !out) return fail(s, RKETD_EINVAL, "rketd_get_coefficients: NULL argument");
  if (!s->have_media) return fail(s, RKETD_ESTATE, "rketd_get_coefficients before rketd_set_media");
  const size_t n = (size_t)6 * s->L.ncells * s->L.nbatch * sizeof(double);
  void *tmp = nullptr;
  CU_TRY(s, cudaMalloc(&tmp, n));
  cudaError_t e = launch_six_coefficients(s->L, s->wp_p, s->nu_p, s->dz, s->dt, s->media_scheme, s->pml, (double *)tmp, s->stream);
  ++s->ctr_launches;
  if (e == cudaSuccess) e = cudaMemcpyAsync(out, tmp, n, cudaMemcpyDefault, s->stream);
  if (e == cudaSuccess) e = cudaStreamSynchronize(s->stream);
  cudaFree(tmp);
  CU_TRY(s, e);
  if (chh_m) {
    chh_m[0] = s->dt / (kMu0 * s->dz);
    const double S = kC0 * s->dt / s->dz;
    chh_m[1] = (S - 1.0) / (S + 1.0);
  }
  return RKETD_OK;
}

int rketd_get_kernel_coefficients(rketd_sim *s, double *out) {
  if (!s || !out) return fail(s, RKETD_EINVAL, "rketd_get_kernel_coefficients: NULL argument");
  if (!s->have_media) return fail(s, RKETD_ESTATE, "rketd_get_kernel_coefficients before rketd_set_media");
  const size_t n = (size_t)kNumCoefArrays * s->L.ncells * s->L.nbatch * sizeof(double);
  void *tmp = nullptr;
  CU_TRY(s, cudaMalloc(&tmp, n));
  cudaError_t e = launch_unpack_coefficients(s->dtype, s->L, s->coef, (double *)tmp, s->stream);
  ++s->ctr_launches;
  if (e == cudaSuccess) e = cudaMemcpyAsync(out, tmp, n, cudaMemcpyDefault, s->stream);
  if (e == cudaSuccess) e = cudaStreamSynchronize(s->stream);
  cudaFree(tmp);
  CU_TRY(s, e);
  return RKETD_OK;
}

int64_t rketd_get_counter(const rketd_sim *s, int which) {
  if (!s) return -1;
  switch (which) {
    case RKETD_CTR_LAUNCHES: return s->ctr_launches;
    case RKETD_CTR_STEP_LAUNCHES: return s->ctr_step_launches;
    case RKETD_CTR_KERNEL_USED: return s->ctr_kernel_used;
    case RKETD_CTR_DEPTH_USED: return s->ctr_depth_used;
    case RKETD_CTR_STEPS_DONE: return s->step;
    case RKETD_CTR_TILE_CELLS: return s->ctr_tile_cells;
    case RKETD_CTR_HALO_CELLS: return s->ctr_halo_cells;
    case RKETD_CTR_STATE_BYTES: return s->state_bytes;
    case RKETD_CTR_PIECES: return s->ctr_pieces;
  }
  return -1;
}

void rketd_destroy(rketd_sim *s) {
  if (!s) return;
  cudaStreamSynchronize(s->stream);
  if (s->copy_stream) { cudaStreamSynchronize(s->copy_stream); cudaStreamDestroy(s->copy_stream); }
  if (s->ev_ready) cudaEventDestroy(s->ev_ready);
  for (cudaEvent_t e : s->ev_piece) cudaEventDestroy(e);
  for (int b = 0; b < 2; ++b)
    for (int a = 0; a < 3; ++a)
      if (s->fld[b][a]) cudaFree(s->fld[b][a]);
  for (int a = 0; a < kNumCoefArrays; ++a)
    if (s->coef[a]) cudaFree(s->coef[a]);
  if (s->wp_p) cudaFree(s->wp_p);
  if (s->nu_p) cudaFree(s->nu_p);
  if (s->rowflag) cudaFree(s->rowflag);
  if (s->d_bad) cudaFree(s->d_bad);
  if (s->d_srctab) cudaFree(s->d_srctab);
  if (s->h_srctab) cudaFreeHost(s->h_srctab);
  if (s->dft_rec) cudaFree(s->dft_rec);
  if (s->dft_tw) cudaFree(s->dft_tw);
  if (s->dft_out) cudaFree(s->dft_out);
  for (auto &c : s->chunks) cudaFree(c.buf);
  if (s->spare_buf) cudaFree(s->spare_buf);
  if (s->dft_re) cudaFree(s->dft_re);
  if (s->dft_im) cudaFree(s->dft_im);
  if (s->d_freqs) cudaFree(s->d_freqs);
  cudaGetLastError();
  delete s;
}

const char *rketd_last_error(const rketd_sim *s) { return s ? s->err.c_str() : g_create_error.c_str(); }

}  // extern "C"
