// fe_api.cu -- C ABI of libfe (include/fe.h): handle, validation, launch logic.  No torch types, no CPU fallback.
#include <cuda_runtime.h>
#include <math.h>
#include <stdio.h>
#include <stdlib.h>
#include <string.h>

#include <mutex>
#include <new>

#include "../../include/fe.h"
#include "../../include/fe_debug.h"
#define FE_PLAIN_KERNELS
#include "fe_kernels.cuh"
#include "fe_bands3.cuh"
#include "fe_chi.cuh"
#include "fe_ksum_sp.cuh"
#include "fe_launch.h"

namespace {

using namespace fe;

thread_local char g_errbuf[512] = "no error";

int cuda_fail(cudaError_t e, const char* what) {
  snprintf(g_errbuf, sizeof g_errbuf, "CUDA error in %s: %s (%s)", what, cudaGetErrorName(e), cudaGetErrorString(e));
  return FE_ECUDA;
}
#define FE_CUDA(call)                                   \
  do {                                                  \
    cudaError_t e__ = (call);                           \
    if (e__ != cudaSuccess) return cuda_fail(e__, #call); \
  } while (0)

struct Tile { int th, td; };
constexpr Tile kTiles[] = {{8, 4}, {4, 4}, {2, 8}, {1, 8}, {16, 2}, {16, 4}};
constexpr int kNumTiles = sizeof(kTiles) / sizeof(kTiles[0]);
// Shapes of the block-cooperative kernel K1c: register tile TH x TD per thread, LH lanes of a warp along h, NW warps,
// KB k-points per shared-memory sub-batch, MINB resident blocks per SM.  Block tile = (TH LH) x (TD NW 32/LH).
struct CoopShape { int th, td, lh, nw, kb, minb; };
constexpr CoopShape kCoopShapes[] = {{16, 4, 4, 4, 4, 2}, {16, 4, 1, 4, 2, 2}, {8, 4, 4, 4, 4, 3}, {8, 4, 1, 4, 2, 2},
                                     {16, 4, 2, 4, 2, 2},    // 32 x 256 block tile (one- and two-band models)
                                     {16, 4, 4, 4, 2, 2}};   // 64 x 128 with a half-size sub-batch: the three-band model (12 slots
                                                             // per sub-batch would take 123 KB of shared memory: one block per SM)
constexpr int kNumCoopShapes = sizeof(kCoopShapes) / sizeof(kCoopShapes[0]);
constexpr int kStageSlots = 4;
constexpr int kSChunksMax = 128;
constexpr int kMaxQ = 65534;   // q sits on gridDim.y (<= 65535) of KS / KB; KB adds one row for the unshifted table

struct StageSlot {
  double* host = nullptr;    // pinned
  double* dev = nullptr;
  size_t cap = 0;            // doubles
  cudaEvent_t ev = nullptr;  // recorded after the H2D copy out of `host`
  bool pending = false;
};

}  // namespace

struct fe_handle {
  fe_model_params p;
  int32_t N = 0;
  double T = 0;
  int32_t mode = FE_EVAL_COOP_EO;
  int32_t tile = 0;            // 0 = auto, else 1 + index
  int32_t target_blocks = 0;   // 0 = auto
  int32_t debug_flags = 0;
  int32_t coop_shape = 0;      // 0 = auto, else 1 + index into kCoopShapes
  int32_t symmetry = 0;        // fe_set_symmetry: use a lattice mirror when every q of a launch is invariant under it
  int32_t last_sym = 0;        // CoopParams.sym of the most recent k-sum launch
  double chi_table_budget = 2.0e9;   // bytes of band tables one slice of fe_pair_susceptibility may hold (three-band model)
  int device = 0;
  int sm_count = 148;
  int nb = 1;
  // device scratch
  MathTabs* d_tabs = nullptr;
  double4* d_coltab = nullptr;
  double4* d_rowtab = nullptr;
  size_t coltab_cap = 0, rowtab_cap = 0;
  double* d_partial = nullptr;
  size_t partial_cap = 0;
  double* d_spart = nullptr;
  size_t spart_cap = 0;
  double* d_omega2 = nullptr;  // fe_scan_verified: fp64 Omega on the candidate Delta list
  size_t omega2_cap = 0;
  int32_t* d_flags = nullptr;  // fe_scan_verified: candidate flags per Delta index, then index scratch
  size_t flags_cap = 0;
  int32_t* h_flags = nullptr;  // pinned
  size_t hflags_cap = 0;
  double* d_etab = nullptr;    // three-band model: [1 + nq][3][N*N] eigenvalue tables
  size_t etab_cap = 0;
  bool etab_base_valid = false;   // table 0 (unshifted grid) already computed for this handle
  double* d_omega = nullptr;   // fe_scan_host only
  size_t omega_cap = 0;
  void* d_res = nullptr;       // fe_scan_host: idx | dstar | ostar
  size_t res_cap = 0;          // columns
  StageSlot slots[kStageSlots];
  int next_slot = 0;
  // timing
  bool timing = false;
  bool slot_counts = false;    // fe_enable_slot_counts: the cooperative kernel counts its slot kinds (atomics; off in timed runs)
  cudaEvent_t ev0 = nullptr, ev1 = nullptr;
  bool timing_valid = false;
  double last_band_evals = 0;
  int32_t last_info[6] = {0, 0, 0, 0, 0, 0};   // th, td, ksplit, grid, mode, rows_per_chunk
  unsigned long long* d_kinds = nullptr;       // 5 slot-kind counters of the most recent timed K1c launch
  bool kinds_valid = false;
  cudaStream_t kinds_stream = nullptr;         // stream of that launch: fe_get_slot_counts copies on it and waits for it
  int64_t launches = 0;
};

namespace {

int nbands(const fe_model_params& p) {
  return p.model == FE_MODEL_ONE_BAND ? 1 : (p.model == FE_MODEL_TWO_BAND ? 2 : 3);
}

// |E_k| <= Wb for every band and k (Gershgorin on the orbital matrix): used by the range guards of the k-sum.
double band_half_width(const fe_model_params& mp) {
  if (mp.model == FE_MODEL_ONE_BAND) return 4.0 * fabs(mp.t[0]);
  if (mp.model == FE_MODEL_TWO_BAND)
    return 2.0 * (fabs(mp.t[0]) + fabs(mp.t[1])) + 4.0 * fabs(mp.t[2]) + 4.0 * fabs(mp.t[3]);
  const double* t = mp.tb3;   // t[i-1] = t_i
  const double d12 = 2.0 * (fabs(t[0]) + fabs(t[1])) + 4.0 * fabs(t[2]) + 4.0 * fabs(t[10]) + 4.0 * fabs(t[11]);
  const double d3 = fabs(t[12]) + 4.0 * fabs(t[4]) + 4.0 * fabs(t[5]) + 4.0 * fabs(t[8]) + 8.0 * fabs(t[9]);
  const double o12 = 4.0 * fabs(t[3]), o3 = 2.0 * fabs(t[6]) + 4.0 * fabs(t[7]);
  return fmax(d12 + o12 + o3, d3 + 2.0 * o3);
}

bool finite_pos(double x) { return isfinite(x) && x > 0.0; }

int validate_params(const fe_model_params* p, int32_t N, double T) {
  if (!p) { snprintf(g_errbuf, sizeof g_errbuf, "params is NULL"); return FE_EINVAL; }
  if (p->model != FE_MODEL_ONE_BAND && p->model != FE_MODEL_TWO_BAND && p->model != FE_MODEL_THREE_BAND) {
    snprintf(g_errbuf, sizeof g_errbuf, "unknown model %d", p->model); return FE_EINVAL; }
  if (p->form_factor != FE_FORM_S && p->form_factor != FE_FORM_SPM) {
    snprintf(g_errbuf, sizeof g_errbuf, "unknown form_factor %d", p->form_factor); return FE_EINVAL; }
  if (p->const_mode != 0 && p->const_mode != 1) {
    snprintf(g_errbuf, sizeof g_errbuf, "const_mode must be 0 or 1"); return FE_EINVAL; }
  if (N < 1 || N > 65536) { snprintf(g_errbuf, sizeof g_errbuf, "N must be in [1, 65536]"); return FE_EINVAL; }
  if (!finite_pos(T)) { snprintf(g_errbuf, sizeof g_errbuf, "T must be finite and > 0"); return FE_EINVAL; }
  if (!finite_pos(p->U)) { snprintf(g_errbuf, sizeof g_errbuf, "U must be finite and > 0"); return FE_EINVAL; }
  const int nb = nbands(*p);
  for (int i = 0; i < (nb == 1 ? 1 : 4) && nb < 3; ++i)
    if (!isfinite(p->t[i])) { snprintf(g_errbuf, sizeof g_errbuf, "t[%d] is not finite", i); return FE_EINVAL; }
  for (int i = 0; i < 13 && nb == 3; ++i)
    if (!isfinite(p->tb3[i])) { snprintf(g_errbuf, sizeof g_errbuf, "tb3[%d] is not finite", i); return FE_EINVAL; }
  if (!isfinite(p->mu) || !isfinite(p->eta_scale) || !isfinite(p->cond_mult)) {
    snprintf(g_errbuf, sizeof g_errbuf, "mu, eta_scale, cond_mult must be finite"); return FE_EINVAL; }
  if (p->band_mask < 0 || p->band_mask >= (1 << nb)) {
    snprintf(g_errbuf, sizeof g_errbuf, "band_mask out of range for %d band(s)", nb); return FE_EINVAL; }
  return FE_OK;
}

void build_tabs(MathTabs* t) {
  for (int j = 0; j < kExpTabN; ++j) t->exp2_j64[j] = (double)exp2l((long double)j / 64.0L);
  for (int j = 0; j < 256; ++j) t->exp2_j256[j] = (double)exp2l((long double)j / 256.0L);
  for (int idx = 0; idx < kLogTabN; ++idx) {
    const int e = idx >> 7, i = idx & 127;
    const long double c = ldexpl(1.0L + ((long double)i + 0.5L) / 128.0L, e);
    const double inv = (double)(1.0L / c);
    t->log_tab[idx].x = inv;
    t->log_tab[idx].y = (double)(-logl((long double)inv));   // ln of the centre actually used (1/inv), not of c
  }
}

ModelConsts make_consts(const fe_model_params& p) {
  ModelConsts mc;
  if (p.model == FE_MODEL_ONE_BAND) {
    mc.tp = -2.0 * p.t[0]; mc.tm = 0; mc.t3x4 = 0; mc.t4x4 = 0;
  } else if (p.model == FE_MODEL_THREE_BAND) {
    mc.tp = 0; mc.tm = 0; mc.t3x4 = 0; mc.t4x4 = 0;      // bands come from the tables (fe_bands3.cuh)
  } else {
    mc.tp = -(p.t[0] + p.t[1]);
    mc.tm = -(p.t[0] - p.t[1]);
    mc.t3x4 = -4.0 * p.t[2];
    mc.t4x4 = -4.0 * p.t[3];
  }
  mc.mu = p.mu; mc.eta_scale = p.eta_scale; mc.band_mask = p.band_mask; mc.const_mode = p.const_mode;
  return mc;
}

template <typename T>
int ensure(T*& ptr, size_t& cap, size_t need) {
  if (need <= cap && ptr) return FE_OK;
  if (ptr) { cudaFree(ptr); ptr = nullptr; cap = 0; }
  // grow geometrically to avoid reallocation on slowly growing grids
  size_t want = need + need / 4;
  cudaError_t e = cudaMalloc((void**)&ptr, want * sizeof(T));
  if (e != cudaSuccess) {
    e = cudaMalloc((void**)&ptr, need * sizeof(T));
    want = need;
  }
  if (e != cudaSuccess) {
    cudaGetLastError();
    snprintf(g_errbuf, sizeof g_errbuf, "device allocation of %zu bytes failed", need * sizeof(T));
    ptr = nullptr;
    return FE_ENOMEM;
  }
  cap = want;
  return FE_OK;
}

// Copy `n` doubles assembled by `fill` into a pinned slot and enqueue the H2D copy.  Returns the device pointer.
int stage_lists(fe_handle* h, size_t n, cudaStream_t st, double** host_out, double** dev_out, StageSlot** slot_out) {
  StageSlot& s = h->slots[h->next_slot];
  h->next_slot = (h->next_slot + 1) % kStageSlots;
  if (s.pending) { FE_CUDA(cudaEventSynchronize(s.ev)); s.pending = false; }
  if (n > s.cap) {
    if (s.host) cudaFreeHost(s.host);
    if (s.dev) cudaFree(s.dev);
    s.host = nullptr; s.dev = nullptr; s.cap = 0;
    const size_t want = n + 256;
    if (cudaMallocHost((void**)&s.host, want * sizeof(double)) != cudaSuccess ||
        cudaMalloc((void**)&s.dev, want * sizeof(double)) != cudaSuccess) {
      cudaGetLastError();
      snprintf(g_errbuf, sizeof g_errbuf, "staging allocation of %zu doubles failed", want);
      return FE_ENOMEM;
    }
    s.cap = want;
  }
  if (!s.ev) FE_CUDA(cudaEventCreateWithFlags(&s.ev, cudaEventDisableTiming));
  (void)st;
  *host_out = s.host; *dev_out = s.dev; *slot_out = &s;
  return FE_OK;
}

// Relative cost per evaluated term of each tile (measured on B200, config-4 slice).
// kTiles order: (8,4) (4,4) (2,8) (1,8) (16,2) (16,4).
constexpr double kTileCostFactored[] = {1.00, 1.72, 2.30, 3.40, 0.91, 0.73};
constexpr double kTileCostDirect[]   = {1.51, 1.00, 1.12, 1.30, 2.00, 3.00};

// cost of one K1c pair relative to kTileCostFactored's unit (measured, config-4 step)
constexpr double kCoopVsFactored = 0.28;

int choose_tile_mode(int forced_tile, int mode, int nh, int nd) {
  if (forced_tile > 0) return forced_tile - 1;
  const double* cost_tab = mode == FE_EVAL_FACTORED ? kTileCostFactored : kTileCostDirect;
  int best = 0; double best_cost = 1e300;
  for (int t = 0; t < kNumTiles; ++t) {
    const double padded = (double)((nh + kTiles[t].th - 1) / kTiles[t].th * kTiles[t].th) *
                          (double)((nd + kTiles[t].td - 1) / kTiles[t].td * kTiles[t].td);
    const double cost = padded * cost_tab[t];          // padded (clamped duplicate) terms are still evaluated
    if (cost < best_cost * (1.0 - 1e-12)) { best_cost = cost; best = t; }
  }
  return best;
}


cudaError_t launch_ksum(int tile, int nb, int form, int mode, int grid, cudaStream_t st, const KsumParams& P) {
  switch (tile) {      // kTiles order
    case 0: return launch_ksum_tile_0(nb, form, mode, grid, st, P);
    case 1: return launch_ksum_tile_1(nb, form, mode, grid, st, P);
    case 2: return launch_ksum_tile_2(nb, form, mode, grid, st, P);
    case 3: return launch_ksum_tile_3(nb, form, mode, grid, st, P);
    case 4: return launch_ksum_tile_4(nb, form, mode, grid, st, P);
    default: return launch_ksum_tile_5(nb, form, mode, grid, st, P);
  }
}

cudaError_t launch_coop(int shape, int nb, int form, int grid, cudaStream_t st, const CoopParams& P) {
  switch (shape) {     // kCoopShapes order
    case 0: return launch_coop_shape_0(nb, form, grid, st, P);
    case 1: return launch_coop_shape_1(nb, form, grid, st, P);
    case 2: return launch_coop_shape_2(nb, form, grid, st, P);
    case 3: return launch_coop_shape_3(nb, form, grid, st, P);
    case 4: return launch_coop_shape_4(nb, form, grid, st, P);
    default: return launch_coop_shape_5(nb, form, grid, st, P);
  }
}

// Relative cost per evaluated pair of each coop shape: pair work 2 TH TD per slot and thread plus the thread's share
// of the (WD + WH) exponentials (~20 FP64 instructions each).
double coop_shape_cost(const CoopShape& s) {
  const int nt = s.nw * 32, wh = s.th * s.lh, wd = s.td * s.nw * (32 / s.lh);
  const double pair = 2.0 * s.th * s.td, expo = 20.0 * (wh + wd) / nt;
  return (pair + expo) / pair * (s.th * s.td >= 64 ? 1.0 : 1.08);
}

// Sizes of the symmetry-reduced k set (CoopParams.sym): n2 points counted twice, n1 fixed points of the mirror counted once.
void sym_counts(int sym, int N, unsigned long long& n2, unsigned long long& n1) {
  const unsigned long long uN = (unsigned long long)N;
  if (sym == 3) { n2 = uN * (uN - 1) / 2; n1 = uN; }
  else { n2 = uN * ((uN - 1) / 2); n1 = (N % 2 == 0) ? 2 * uN : uN; }
}

int choose_coop_shape(const fe_handle* h, const double* h_list, int nh, int nd, bool early_out) {
  if (h->coop_shape > 0) return h->coop_shape - 1;
  int best = 0; double best_cost = 1e300;
  for (int t = 0; t < 5; ++t) {                 // (shape 5 is shape 0 with another sub-batch: chosen below, not by cost)
    const CoopShape& s = kCoopShapes[t];
    if (h->nb == 3 && s.lh != 4) continue;
    const int wh = s.th * s.lh, wd = s.td * s.nw * (32 / s.lh);
    const double padded = (double)((nh + wh - 1) / wh * wh) * (double)((nd + wd - 1) / wd * wd);
    const double cost = padded * coop_shape_cost(s);
    if (cost < best_cost * (1.0 - 1e-12)) { best_cost = cost; best = t; }
  }
  // Early-out mode classifies a (k, band) slot for a whole block tile, so a tile that is narrower along h leaves fewer
  // slots dense when the dominance window kDomGap T ln2 is small against the h range of the tile; the 32 x 256 tile pays
  // ~12 % more per dense slot (WD + WH = 288 instead of 192 exponentials per 8192 pairs).  Measured on config 4 (h range
  // 0.3 per 64 values; launches in ms, 64 x 128 vs 32 x 256): T = 0.0005 63.1 / 46.8, 0.001 58.6 / 47.6, 0.002 56.4 / 52.7,
  // 0.004 63.7 / 62.7, 0.006 70.4 / 72.3, 0.01 83.6 / 88.6, 0.02 117.6 / 128.9: the narrow tile wins below window / range ~ 0.5.
  if (h->nb == 3 && best == 0) best = 5;        // two resident blocks per SM (measured: dense 625 -> see DESIGN.md section 11 f-1)
  if (early_out && best == 0 && h->nb < 3 && nh > 32 && (nd + 255) / 256 * 2 <= (nd + 127) / 128) {   // (no extra Delta padding)
    double range = 0.0;
    for (int t0 = 0; t0 < nh; t0 += 64) {
      double lo = h_list[t0], hi = h_list[t0];
      for (int i = t0; i < nh && i < t0 + 64; ++i) { lo = fmin(lo, h_list[i]); hi = fmax(hi, h_list[i]); }
      range = fmax(range, hi - lo);
    }
    if ((double)kDomGap * h->T * 0.6931471805599453 < 0.5 * range) best = 4;
  }
  return best;
}

int check_lists(const double* q_xy, int32_t nq, const double* h_list, int32_t nh, const double* delta, int32_t nd) {
  if (!q_xy || !h_list || !delta) { snprintf(g_errbuf, sizeof g_errbuf, "a list pointer is NULL"); return FE_EINVAL; }
  if (nq < 1 || nh < 1 || nd < 1) { snprintf(g_errbuf, sizeof g_errbuf, "nq, nh, nd must be >= 1"); return FE_EINVAL; }
  if ((double)nq * nh * nd > 2.0e9) { snprintf(g_errbuf, sizeof g_errbuf, "grid too large (nq*nh*nd > 2e9)"); return FE_EINVAL; }
  if (nq > kMaxQ) { snprintf(g_errbuf, sizeof g_errbuf, "nq must be <= %d (q is a grid dimension of the table kernels)", kMaxQ); return FE_EINVAL; }
  for (int i = 0; i < 2 * nq; ++i) if (!isfinite(q_xy[i])) { snprintf(g_errbuf, sizeof g_errbuf, "q[%d] not finite", i); return FE_EINVAL; }
  for (int i = 0; i < nh; ++i) if (!isfinite(h_list[i])) { snprintf(g_errbuf, sizeof g_errbuf, "h[%d] not finite", i); return FE_EINVAL; }
  for (int i = 0; i < nd; ++i) if (!isfinite(delta[i])) { snprintf(g_errbuf, sizeof g_errbuf, "delta[%d] not finite", i); return FE_EINVAL; }
  return FE_OK;
}

// sp: 0 = the handle's fp64 evaluation mode; 1 = K1s SP; 2 = K1s SPFM (fe_ksum_sp.cuh)
int check_device(const fe_handle* h) {
  int dev = -1;
  FE_CUDA(cudaGetDevice(&dev));
  if (dev != h->device) {
    snprintf(g_errbuf, sizeof g_errbuf, "handle was created on device %d but device %d is current", h->device, dev);
    return FE_EINVAL;
  }
  return FE_OK;
}

int omega_grid_impl(fe_handle* h, const double* q_xy, int32_t nq, const double* h_list, int32_t nh,
                    const double* delta, int32_t nd, double* omega_dev, cudaStream_t st, int sp = 0) {
  const int N = h->N;
  if (int rcd = check_device(h)) return rcd;
  h->last_sym = 0;
  // ---- K1c or a per-thread kernel?  (K1c pads to its block tile; tiny h lists are cheaper on K1f) ----
  int mode = h->mode;
  if (sp) {
    if (h->nb == 3) { snprintf(g_errbuf, sizeof g_errbuf, "the single-precision kernels cover the one- and two-band models"); return FE_EINVAL; }
    mode = FE_EVAL_DIRECT;                                  // K1's geometry, tile (4, 4)
  }
  int cshape = 0;
  const bool early_out = mode == FE_EVAL_COOP_EO;
  if (early_out) mode = FE_EVAL_COOP;                       // same kernel, CoopParams.early_out = 1
  if (h->nb == 3 && mode != FE_EVAL_COOP) {
    snprintf(g_errbuf, sizeof g_errbuf, "FE_MODEL_THREE_BAND supports FE_EVAL_COOP / FE_EVAL_COOP_EO only"); return FE_EINVAL; }
  if (mode == FE_EVAL_COOP) {
    cshape = choose_coop_shape(h, h_list, nh, nd, early_out);
    if (h->nb == 3 && kCoopShapes[cshape].lh != 4) {
      snprintf(g_errbuf, sizeof g_errbuf, "FE_MODEL_THREE_BAND needs a coop shape with 4 lanes along h"); return FE_EINVAL; }
    if (h->coop_shape == 0 && h->nb < 3) {
      const CoopShape& cs = kCoopShapes[cshape];
      const int wh = cs.th * cs.lh, wd = cs.td * cs.nw * (32 / cs.lh);
      double coop_cost = (double)((nh + wh - 1) / wh * wh) * (double)((nd + wd - 1) / wd * wd) *
                         coop_shape_cost(cs) * kCoopVsFactored;
      if (early_out) {
        // Early-out leaves only the slots within the dominance window of the Fermi surface for the pair products: of the
        // dense cost roughly 0.1 (classification, dominated sums) + (h range + 2 windows) / band half-width remains
        // (config 4: 0.13 at T = 0.001, 0.18 at T = 0.01; measured 0.13 / 0.22).  At low T that makes K1c the cheaper
        // kernel even on grids far smaller than its block tile (the paper's benchmark shape, 1 h x 200 Delta at N = 2000:
        // 3.8 ms per-thread kernel, 2.7 ms K1c with the 8 x 512 tile).
        double hlo = h_list[0], hhi = h_list[0];
        for (int i = 1; i < nh; ++i) { hlo = fmin(hlo, h_list[i]); hhi = fmax(hhi, h_list[i]); }
        const double window = (double)kDomGap * h->T * 0.6931471805599453;
        coop_cost *= fmin(1.0, 0.1 + (hhi - hlo + 2.0 * window) / band_half_width(h->p));
      }
      const int lt = choose_tile_mode(0, FE_EVAL_FACTORED, nh, nd);
      const double legacy_cost = (double)((nh + kTiles[lt].th - 1) / kTiles[lt].th * kTiles[lt].th) *
                                 (double)((nd + kTiles[lt].td - 1) / kTiles[lt].td * kTiles[lt].td) * kTileCostFactored[lt];
      if (legacy_cost < coop_cost) mode = FE_EVAL_FACTORED;
    }
  }
  const bool coop = mode == FE_EVAL_COOP;
  // ---- stage lists: [q (2nq) | h (nh) | delta^2 (nd)] ----
  const int tile = sp ? 1 : choose_tile_mode((mode == h->mode || (early_out && mode == FE_EVAL_COOP)) ? h->tile : 0, mode, nh, nd);
  const int TH = kTiles[tile].th, TD = kTiles[tile].td;
  const int ntile_h = (nh + TH - 1) / TH;
  const int hstride = htile_stride(TH);
  const size_t nlist = (size_t)2 * nq + nh + nd + (size_t)ntile_h * hstride + (sp ? nd : 0);
  double *hs, *ds; StageSlot* slot;
  int rc = stage_lists(h, nlist, st, &hs, &ds, &slot);
  if (rc) return rc;
  memcpy(hs, q_xy, sizeof(double) * 2 * nq);
  memcpy(hs + 2 * nq, h_list, sizeof(double) * nh);
  for (int i = 0; i < nd; ++i) hs[2 * nq + nh + i] = delta[i] * delta[i];
  {
    // per-h-tile table of the factored kernel (fe_kernels.cuh "Per-h-tile table"), in long double
    double* ht = hs + 2 * nq + nh + nd;
    const long double Tl = (long double)h->T;
    for (int t = 0; t < ntile_h; ++t, ht += hstride) {
      double hmin = h_list[t * TH], hmax = hmin;
      for (int i = 0; i < TH; ++i) {
        const double hi = h_list[(t * TH + i < nh) ? t * TH + i : nh - 1];
        hmin = fmin(hmin, hi); hmax = fmax(hmax, hi);
      }
      for (int i = 0; i < TH; ++i) {
        const double hi = h_list[(t * TH + i < nh) ? t * TH + i : nh - 1];
        ht[4 + i] = (double)expl(-((long double)hi - (long double)hmin) / Tl);
        ht[4 + TH + i] = (double)expl(-((long double)hmax - (long double)hi) / Tl);
      }
      const long double l2 = ((long double)hmax - (long double)hmin) / Tl * 1.442695040888963407359924681001892137L;
      const long double fl = floorl(l2);
      ht[0] = hmin; ht[1] = hmax;
      ht[2] = (double)exp2l(l2 - fl);              // mC in [1, 2)
      ht[3] = (double)fl;                          // eC (< 2^31: max|h|/T < 1e9 is enforced below)
    }
  }
  if (sp) memcpy(hs + nlist - nd, delta, sizeof(double) * nd);       // K1s squares Delta in float itself
  FE_CUDA(cudaMemcpyAsync(ds, hs, nlist * sizeof(double), cudaMemcpyHostToDevice, st));
  FE_CUDA(cudaEventRecord(slot->ev, st));
  slot->pending = true;
  const double* d_q = ds;
  const double* d_h = ds + 2 * nq;
  const double* d_d2 = ds + 2 * nq + nh;
  const double* d_htile = ds + 2 * nq + nh + nd;

  // ---- geometry ----
  KsumParams P;
  P.mc = make_consts(h->p);
  P.T = h->T; P.neg_beta = -1.0 / h->T; P.window = 37.0 * h->T;
  P.N = N; P.nq = nq; P.nh = nh; P.nd = nd;
  P.debug_flags = h->debug_flags;
  P.ntile_h = (nh + TH - 1) / TH;
  P.ntile_d = (nd + TD - 1) / TD;
  const int bthreads = mode == FE_EVAL_FACTORED ? kFThreads : kThreads;
  int bxl = 0;
  while ((1 << bxl) < bthreads) ++bxl;           // all threads along kx when N allows it
  while (bxl > 5 && (1 << (bxl - 1)) >= N) --bxl;
  P.bx_log2 = bxl;
  const int bx = 1 << bxl, by = bthreads >> bxl;
  P.ncg = (N + bx - 1) / bx;
  const long long ntiles = (long long)nq * P.ntile_h * P.ntile_d;
  const long long target = h->target_blocks > 0 ? h->target_blocks : (long long)h->sm_count * 2 * 24;
  long long nrs = (target + ntiles * P.ncg - 1) / (ntiles * P.ncg);
  const int max_nrs = (N + by - 1) / by;         // at least one row per row lane
  if (nrs > max_nrs) nrs = max_nrs;
  if (nrs < 1) nrs = 1;
  int rpc = (int)((N + nrs - 1) / nrs);
  rpc = (rpc + by - 1) / by * by;                // whole row-lane strides per chunk
  double coop_max_k = 1e18;                      // k-points per chunk K1c may sum into its int32 exponent sums
  {
    // Range guards of the factored kernel: binary exponents x/(T ln2) are summed in int32 per thread, and the
    // range reduction needs x/T * 64/ln2 < 2^37.  |E_k| <= W, so R <= W + |mu| + |Delta eta|, |d| <= W + |h|.
    const fe_model_params& mp = h->p;
    const double Wb = band_half_width(mp);
    double hmax = 0, dmax = 0;
    for (int i = 0; i < nh; ++i) hmax = fmax(hmax, fabs(h_list[i]));
    for (int i = 0; i < nd; ++i) dmax = fmax(dmax, fabs(delta[i]));
    const double xmax = fmax(Wb + fabs(mp.mu) + dmax * fabs(mp.eta_scale), Wb + hmax) / h->T;
    if (!(xmax < 1.0e9)) {
      snprintf(g_errbuf, sizeof g_errbuf, "T = %g is too small for the energy scale (max x/T = %.3g >= 1e9)", h->T, xmax);
      return FE_EINVAL;
    }
    const double ebound = xmax / 0.6931471805599453 + 4.0;            // max binary exponent of one term
    const double max_terms = 2.0e9 / ebound;                          // per thread and accumulator
    coop_max_k = floor(max_terms / h->nb);
    int max_rows = (int)fmin((double)N, floor(max_terms / h->nb)) * by;
    if (max_rows < by) max_rows = by;
    if (rpc > max_rows) rpc = max_rows / by * by;
  }
  P.rows_per_chunk = rpc;
  P.nrs = (N + rpc - 1) / rpc;
  P.ksplit = P.ncg * P.nrs;
  long long grid_ll = ntiles * P.ksplit;

  // ---- K1c geometry: block tiles x k-chunks; the grid is sized to whole waves of resident blocks ----
  CoopParams CP;
  if (coop) {
    const CoopShape& cs = kCoopShapes[cshape];
    const int nt = cs.nw * 32, wh = cs.th * cs.lh, wd = cs.td * cs.nw * (32 / cs.lh);
    CP.mc = P.mc; CP.fc = make_factored(h->T); CP.T = h->T;
    CP.N = N; CP.nq = nq; CP.nh = nh; CP.nd = nd;
    CP.ntile_h = (nh + wh - 1) / wh; CP.ntile_d = (nd + wd - 1) / wd;
    CP.debug_flags = h->debug_flags;
    CP.early_out = early_out ? 1 : 0;
    CP.nk = (unsigned long long)N * (unsigned long long)N;
    // mirror-symmetry reduction (fe_set_symmetry): needs a mirror of the lattice that leaves EVERY q of the launch
    // unchanged (compared exactly); one- and two-band models (E and eta are invariant under all three mirrors)
    CP.sym = 0; CP.ksplit2 = 0; CP.n2 = 0; CP.n1 = 0;
    if (h->symmetry && h->nb < 3 && N >= 3) {
      bool diag = true, my = true, mx = true;
      for (int i = 0; i < nq; ++i) {
        diag = diag && q_xy[2 * i] == q_xy[2 * i + 1];
        my = my && q_xy[2 * i + 1] == 0.0;
        mx = mx && q_xy[2 * i] == 0.0;
      }
      CP.sym = diag ? 3 : (my ? 1 : (mx ? 2 : 0));
      if (CP.sym) sym_counts(CP.sym, N, CP.n2, CP.n1);
    }
    const unsigned long long nk_eff = CP.sym ? CP.n2 + CP.n1 : CP.nk;       // k-points actually visited
    const long long ctiles = (long long)nq * CP.ntile_h * CP.ntile_d;
    const long long wave = (long long)h->sm_count * cs.minb;
    const long long max_split = (long long)((nk_eff + nt - 1) / nt);         // at least one thread-batch per chunk
    long long min_split = (long long)ceil((double)nk_eff / fmax(1.0, floor(coop_max_k / nt) * nt));
    if (min_split < 1) min_split = 1;
    long long ks;
    if (h->target_blocks > 0) {
      ks = (h->target_blocks + ctiles - 1) / ctiles;
    } else {
      // >= 24 waves (the dense share of a k-chunk varies with where it lies in the zone, so block durations differ: many
      // short blocks keep the last waves full; measured on the config-4 step: 8 waves 71.0 / 102.4 ms, 24 waves 69.3 / 99.8 ms
      // for T = 0.001 / 0.01); among the next candidates take the split whose last wave is fullest
      const long long ks0 = (24 * wave + ctiles - 1) / ctiles;
      ks = ks0; double best_eff = 0;
      for (long long c = ks0; c <= 2 * ks0 + 1; ++c) {
        const long long g = ctiles * c, waves = (g + wave - 1) / wave;
        const double eff = (double)g / (double)(waves * wave);
        if (eff > best_eff + 1e-9) { best_eff = eff; ks = c; }
      }
    }
    if (ks < min_split) ks = min_split;
    if (ks > max_split) ks = max_split;
    if (ks < 1) ks = 1;
    unsigned long long kc = (nk_eff + ks - 1) / ks;
    kc = (kc + nt - 1) / nt * nt;
    CP.kc = kc;
    CP.ksplit = (int32_t)((CP.nk + kc - 1) / kc);
    if (CP.sym) {                                                              // weight-2 chunks first, then the weight-1 chunks
      CP.ksplit2 = (int32_t)((CP.n2 + kc - 1) / kc);
      CP.ksplit = CP.ksplit2 + (int32_t)((CP.n1 + kc - 1) / kc);
    }
    h->last_sym = CP.sym;
    P.ksplit = CP.ksplit;
    grid_ll = ctiles * CP.ksplit;
  }
  if (grid_ll > 2147483647LL) { snprintf(g_errbuf, sizeof g_errbuf, "grid too large"); return FE_EINVAL; }

  const size_t nout = (size_t)nq * nh * nd;
  if ((rc = ensure(h->d_coltab, h->coltab_cap, (size_t)nq * N))) return rc;
  if ((rc = ensure(h->d_rowtab, h->rowtab_cap, (size_t)nq * N))) return rc;
  if ((rc = ensure(h->d_partial, h->partial_cap, (size_t)P.ksplit * nout))) return rc;
  int nschunk = N < kSChunksMax ? N : kSChunksMax;
  const int srpc = (N + nschunk - 1) / nschunk;
  nschunk = (N + srpc - 1) / srpc;
  if ((rc = ensure(h->d_spart, h->spart_cap, (size_t)nq * nschunk))) return rc;
  if (h->nb == 3) {
    const size_t need = (size_t)(1 + nq) * 3 * N * N;
    if (need > h->etab_cap || !h->d_etab) h->etab_base_valid = false;      // reallocation drops table 0
    if ((rc = ensure(h->d_etab, h->etab_cap, need))) return rc;
  }

  P.coltab = h->d_coltab; P.rowtab = h->d_rowtab; P.h = d_h; P.d2 = d_d2; P.htile = d_htile; P.tabs = h->d_tabs;
  P.partial = h->d_partial;

  // ---- K0 trig, KS constant sum, K1 k-sum, K2 finish ----
  {
    const int n = N * nq;
    fe_trig_kernel<<<(n + 255) / 256, 256, 0, st>>>(N, nq, d_q, h->d_coltab, h->d_rowtab);
    FE_CUDA(cudaGetLastError());
    h->launches++;
  }
  if (sp) {
    nschunk = 0;                                           // K1s sums the whole Eq. 5 term: no separate constant sum
  } else if (h->nb == 3) {
    // KB: numerical band diagonalisation into the per-q tables (table 0 = unshifted grid, once per handle)
    Band3Consts bc;
    for (int i = 0; i < 12; ++i) bc.t[i] = h->p.tb3[i];
    bc.e0 = h->p.tb3[12];
    const int y0 = h->etab_base_valid ? 1 : 0;
    dim3 g((unsigned)(((size_t)N * N + 255) / 256), (unsigned)(1 + nq - y0));
    fe_bands3_kernel<<<g, 256, 0, st>>>(bc, N, y0, h->d_coltab, h->d_rowtab, nullptr, h->d_etab);
    FE_CUDA(cudaGetLastError());
    h->etab_base_valid = true;
    h->launches++;
    dim3 gs(nschunk, nq);
    fe_ssum3_kernel<<<gs, kThreads, 0, st>>>(P.mc, N, srpc, h->d_etab, h->d_spart);
    FE_CUDA(cudaGetLastError());
    h->launches++;
  } else {
    dim3 g(nschunk, nq);
    if (h->nb == 1) fe_ssum_kernel<1><<<g, kThreads, 0, st>>>(P.mc, N, srpc, h->d_coltab, h->d_rowtab, h->d_spart);
    else            fe_ssum_kernel<2><<<g, kThreads, 0, st>>>(P.mc, N, srpc, h->d_coltab, h->d_rowtab, h->d_spart);
    FE_CUDA(cudaGetLastError());
    h->launches++;
  }
  h->last_info[0] = TH; h->last_info[1] = TD; h->last_info[2] = P.ksplit; h->last_info[3] = (int32_t)grid_ll;
  h->last_info[4] = (coop && early_out) ? FE_EVAL_COOP_EO : mode; h->last_info[5] = P.rows_per_chunk;
  if (coop) {
    const CoopShape& cs = kCoopShapes[cshape];
    h->last_info[0] = cs.th * cs.lh; h->last_info[1] = cs.td * cs.nw * (32 / cs.lh);     // block tile WH x WD
    h->last_info[5] = (int32_t)(CP.kc < 2147483647ULL ? CP.kc : 2147483647ULL);          // k-points per chunk
    CP.coltab = h->d_coltab; CP.rowtab = h->d_rowtab; CP.h = d_h; CP.d2 = d_d2; CP.tabs = h->d_tabs;
    CP.partial = h->d_partial; CP.etab = h->d_etab;
    CP.kind_counts = nullptr;
    h->kinds_valid = false;
    if (h->slot_counts) {
      if (!h->d_kinds) FE_CUDA(cudaMalloc((void**)&h->d_kinds, 5 * sizeof(unsigned long long)));
      FE_CUDA(cudaMemsetAsync(h->d_kinds, 0, 5 * sizeof(unsigned long long), st));
      CP.kind_counts = h->d_kinds;
      h->kinds_valid = true;
      h->kinds_stream = st;
    }
  }
  if (h->timing) FE_CUDA(cudaEventRecord(h->ev0, st));
  if (sp) {
    SpConsts sc;
    for (int i = 0; i < 4; ++i) sc.t[i] = (float)h->p.t[i];
    sc.mu = (float)h->p.mu; sc.eta_scale = (float)h->p.eta_scale; sc.T = (float)h->T;
    P.d2 = ds + nlist - nd;                                // raw Delta list
    const int g = (int)grid_ll, form = h->p.form_factor;
#define FE_SP(NB_, F_, X_) fe_ksum_sp_kernel<NB_, F_, X_><<<g, kThreads, 0, st>>>(P, sc)
    if (h->nb == 1) { if (form == 0) { if (sp == 2) FE_SP(1, 0, true); else FE_SP(1, 0, false); }
                      else           { if (sp == 2) FE_SP(1, 1, true); else FE_SP(1, 1, false); } }
    else            { if (form == 0) { if (sp == 2) FE_SP(2, 0, true); else FE_SP(2, 0, false); }
                      else           { if (sp == 2) FE_SP(2, 1, true); else FE_SP(2, 1, false); } }
#undef FE_SP
    FE_CUDA(cudaGetLastError());
    h->last_info[4] = 100 + sp;
  }
  else if (coop) FE_CUDA(launch_coop(cshape, h->nb, h->p.form_factor, (int)grid_ll, st, CP));
  else      FE_CUDA(launch_ksum(tile, h->nb, h->p.form_factor, mode, (int)grid_ll, st, P));
  h->launches++;
  if (h->timing) {
    FE_CUDA(cudaEventRecord(h->ev1, st));
    h->timing_valid = true;
    int nbm = 0;
    for (int e = 0; e < h->nb; ++e) nbm += (h->p.band_mask >> e) & 1;
    h->last_band_evals = (double)N * N * nbm * (double)nout;
  }
  {
    const double condc = h->p.cond_mult * (double)N * (double)N / h->p.U;
    fe_finish_kernel<<<(unsigned)((nout + 255) / 256), 256, 0, st>>>(nq, nh, nd, P.ksplit, nschunk, condc,
                                                                      h->d_partial, h->d_spart, d_d2, omega_dev);
    FE_CUDA(cudaGetLastError());
    h->launches++;
  }
  return FE_OK;
}

int argmin_impl(fe_handle* h, const double* omega_dev, const double* delta, int32_t ncol, int32_t nd,
                int32_t* idx_dev, double* dstar_dev, double* ostar_dev, cudaStream_t st) {
  double *hs, *ds; StageSlot* slot;
  int rc = stage_lists(h, (size_t)nd, st, &hs, &ds, &slot);
  if (rc) return rc;
  memcpy(hs, delta, sizeof(double) * nd);
  FE_CUDA(cudaMemcpyAsync(ds, hs, (size_t)nd * sizeof(double), cudaMemcpyHostToDevice, st));
  FE_CUDA(cudaEventRecord(slot->ev, st));
  slot->pending = true;
  const int wpb = 8;
  fe_argmin_kernel<<<(ncol + wpb - 1) / wpb, wpb * 32, 0, st>>>(ncol, nd, omega_dev, ds, idx_dev, dstar_dev, ostar_dev);
  FE_CUDA(cudaGetLastError());
  h->launches++;
  return FE_OK;
}

}  // namespace

// =====================================================================================================
// C ABI
// =====================================================================================================
extern "C" {

int fe_create(const fe_model_params* params, int32_t N, double T, fe_handle** out) {
  if (!out) { snprintf(g_errbuf, sizeof g_errbuf, "out is NULL"); return FE_EINVAL; }
  int rc = validate_params(params, N, T);
  if (rc) return rc;
  int dev = 0;
  FE_CUDA(cudaGetDevice(&dev));
  cudaDeviceProp prop;
  FE_CUDA(cudaGetDeviceProperties(&prop, dev));
  if (prop.major != 10) {
    snprintf(g_errbuf, sizeof g_errbuf, "device %d (%s) is compute capability %d.%d; libfe is built for sm_100a only",
             dev, prop.name, prop.major, prop.minor);
    return FE_EARCH;
  }
  fe_handle* h = new (std::nothrow) fe_handle();
  if (!h) { snprintf(g_errbuf, sizeof g_errbuf, "host allocation failed"); return FE_ENOMEM; }
  h->p = *params; h->N = N; h->T = T; h->device = dev; h->sm_count = prop.multiProcessorCount;
  h->nb = nbands(*params);
  MathTabs host_tabs;
  memset(&host_tabs, 0, sizeof host_tabs);
  build_tabs(&host_tabs);
  cudaError_t e = cudaMalloc((void**)&h->d_tabs, sizeof(MathTabs));
  if (e == cudaSuccess) e = cudaMemcpy(h->d_tabs, &host_tabs, sizeof(MathTabs), cudaMemcpyHostToDevice);
  if (e == cudaSuccess) e = cudaEventCreate(&h->ev0);
  if (e == cudaSuccess) e = cudaEventCreate(&h->ev1);
  if (e != cudaSuccess) { rc = cuda_fail(e, "fe_create setup"); fe_destroy(h); return rc; }
  *out = h;
  return FE_OK;
}

int fe_set_temperature(fe_handle* h, double T) {
  if (!h) { snprintf(g_errbuf, sizeof g_errbuf, "handle is NULL"); return FE_EINVAL; }
  if (!finite_pos(T)) { snprintf(g_errbuf, sizeof g_errbuf, "T must be finite and > 0"); return FE_EINVAL; }
  h->T = T;
  return FE_OK;
}

int fe_set_eval_mode(fe_handle* h, int32_t mode) {
  if (!h) { snprintf(g_errbuf, sizeof g_errbuf, "handle is NULL"); return FE_EINVAL; }
  if (mode != FE_EVAL_FACTORED && mode != FE_EVAL_DIRECT && mode != FE_EVAL_WINDOWED && mode != FE_EVAL_COOP &&
      mode != FE_EVAL_COOP_EO) {
    snprintf(g_errbuf, sizeof g_errbuf, "unknown eval mode %d", mode); return FE_EINVAL; }
  h->mode = mode;
  return FE_OK;
}

int fe_set_tuning(fe_handle* h, int32_t tile, int32_t target_blocks) {
  if (!h) { snprintf(g_errbuf, sizeof g_errbuf, "handle is NULL"); return FE_EINVAL; }
  if (tile < 0 || tile > kNumTiles || target_blocks < 0) {
    snprintf(g_errbuf, sizeof g_errbuf, "tile must be in [0, %d], target_blocks >= 0", kNumTiles); return FE_EINVAL; }
  h->tile = tile; h->target_blocks = target_blocks;
  return FE_OK;
}

int fe_debug_sym_index(int32_t sym, int32_t N, int64_t i, int32_t* row, int32_t* col, int64_t* counts2) {
  if (sym < 1 || sym > 3 || N < 3) { snprintf(g_errbuf, sizeof g_errbuf, "sym must be 1, 2 or 3 and N >= 3"); return FE_EINVAL; }
  unsigned long long n2, n1;
  sym_counts(sym, N, n2, n1);
  if (counts2) { counts2[0] = (int64_t)n2; counts2[1] = (int64_t)n1; }
  if (row || col) {
    if (i < 0 || (unsigned long long)i >= n2 + n1) { snprintf(g_errbuf, sizeof g_errbuf, "index out of range"); return FE_EINVAL; }
    int r, c;
    coop_sym_index(sym, N, n2, (unsigned long long)i, r, c);
    if (row) *row = r;
    if (col) *col = c;
  }
  return FE_OK;
}

int fe_set_symmetry(fe_handle* h, int32_t on) {
  if (!h) { snprintf(g_errbuf, sizeof g_errbuf, "handle is NULL"); return FE_EINVAL; }
  h->symmetry = on ? 1 : 0;
  return FE_OK;
}

int fe_get_last_symmetry(fe_handle* h, int32_t* sym) {
  if (!h || !sym) { snprintf(g_errbuf, sizeof g_errbuf, "NULL argument"); return FE_EINVAL; }
  *sym = h->last_sym;
  return FE_OK;
}

int fe_set_coop_shape(fe_handle* h, int32_t shape) {
  if (!h) { snprintf(g_errbuf, sizeof g_errbuf, "handle is NULL"); return FE_EINVAL; }
  if (shape < 0 || shape > kNumCoopShapes) {
    snprintf(g_errbuf, sizeof g_errbuf, "shape must be in [0, %d]", kNumCoopShapes); return FE_EINVAL; }
  h->coop_shape = shape;
  return FE_OK;
}

int fe_debug_coop_occupancy(int32_t shape, int32_t nbands, int32_t form_factor, int32_t sym, int32_t* blocks_per_sm) {
  if (shape < 1 || shape > kNumCoopShapes || nbands < 1 || nbands > 3 || form_factor < 0 || form_factor > 1 || !blocks_per_sm) {
    snprintf(g_errbuf, sizeof g_errbuf, "no such instance"); return FE_EINVAL; }
  int blocks = 0;
  cudaError_t e;
  switch (shape - 1) {
    case 0: e = occupancy_coop_shape_0(nbands, form_factor, sym, &blocks); break;
    case 1: e = occupancy_coop_shape_1(nbands, form_factor, sym, &blocks); break;
    case 2: e = occupancy_coop_shape_2(nbands, form_factor, sym, &blocks); break;
    case 3: e = occupancy_coop_shape_3(nbands, form_factor, sym, &blocks); break;
    case 4: e = occupancy_coop_shape_4(nbands, form_factor, sym, &blocks); break;
    default: e = occupancy_coop_shape_5(nbands, form_factor, sym, &blocks); break;
  }
  if (e == cudaErrorInvalidConfiguration) { cudaGetLastError(); snprintf(g_errbuf, sizeof g_errbuf, "this shape has no instance for %d bands", nbands); return FE_EINVAL; }
  FE_CUDA(e);
  *blocks_per_sm = blocks;
  return FE_OK;
}

int fe_coop_shape_info(int32_t shape, int32_t* info6) {
  if (shape < 1 || shape > kNumCoopShapes || !info6) { snprintf(g_errbuf, sizeof g_errbuf, "no such shape"); return FE_EINVAL; }
  const CoopShape& s = kCoopShapes[shape - 1];
  info6[0] = s.th; info6[1] = s.td; info6[2] = s.th * s.lh; info6[3] = s.td * s.nw * (32 / s.lh);
  info6[4] = s.nw * 32; info6[5] = s.minb;
  return FE_OK;
}

int fe_set_chi_table_budget(fe_handle* h, double bytes) {
  if (!h || !(bytes >= 0.0) || !isfinite(bytes)) { snprintf(g_errbuf, sizeof g_errbuf, "handle is NULL or bytes is not finite and >= 0"); return FE_EINVAL; }
  h->chi_table_budget = bytes;
  return FE_OK;
}

int fe_set_debug_flags(fe_handle* h, int32_t flags) {
  if (!h) { snprintf(g_errbuf, sizeof g_errbuf, "handle is NULL"); return FE_EINVAL; }
  if (flags < 0 || flags > 3) { snprintf(g_errbuf, sizeof g_errbuf, "flags must be in [0, 3]"); return FE_EINVAL; }
  h->debug_flags = flags;
  return FE_OK;
}

int fe_tile_info(int32_t tile, int32_t* th, int32_t* td) {
  if (tile < 1 || tile > kNumTiles) { snprintf(g_errbuf, sizeof g_errbuf, "no such tile"); return FE_EINVAL; }
  if (th) *th = kTiles[tile - 1].th;
  if (td) *td = kTiles[tile - 1].td;
  return FE_OK;
}

int fe_omega_grid(fe_handle* h, const double* q_xy, int32_t nq, const double* h_list, int32_t nh,
                  const double* delta, int32_t nd, double* omega_dev, void* cuda_stream) {
  if (!h || !omega_dev) { snprintf(g_errbuf, sizeof g_errbuf, "handle or omega_dev is NULL"); return FE_EINVAL; }
  int rc = check_lists(q_xy, nq, h_list, nh, delta, nd);
  if (rc) return rc;
  return omega_grid_impl(h, q_xy, nq, h_list, nh, delta, nd, omega_dev, (cudaStream_t)cuda_stream);
}

int fe_argmin(fe_handle* h, const double* omega_dev, const double* delta, int32_t ncol, int32_t nd,
              int32_t* idx_dev, double* delta_star_dev, double* omega_star_dev, void* cuda_stream) {
  if (!h || !omega_dev || !delta) { snprintf(g_errbuf, sizeof g_errbuf, "handle, omega_dev or delta is NULL"); return FE_EINVAL; }
  if (ncol < 1 || nd < 1) { snprintf(g_errbuf, sizeof g_errbuf, "ncol, nd must be >= 1"); return FE_EINVAL; }
  return argmin_impl(h, omega_dev, delta, ncol, nd, idx_dev, delta_star_dev, omega_star_dev, (cudaStream_t)cuda_stream);
}

int fe_argmin_q(fe_handle* h, const double* omega_dev, int32_t nq, int32_t nh, int32_t nd, int32_t ref_id,
                int32_t* iq_dev, int32_t* id_dev, double* value_dev, void* cuda_stream) {
  if (!h || !omega_dev) { snprintf(g_errbuf, sizeof g_errbuf, "handle or omega_dev is NULL"); return FE_EINVAL; }
  if (nq < 1 || nh < 1 || nd < 1 || ref_id < -1 || ref_id >= nd) {
    snprintf(g_errbuf, sizeof g_errbuf, "nq, nh, nd must be >= 1 and ref_id in [-1, nd)"); return FE_EINVAL; }
  fe_argmin_q_kernel<<<nh, 256, 0, (cudaStream_t)cuda_stream>>>(nq, nh, nd, ref_id, omega_dev, iq_dev, id_dev, value_dev);
  FE_CUDA(cudaGetLastError());
  h->launches++;
  return FE_OK;
}

// q on the k-grid?  (then E(k + q) is the unshifted band table read at a shifted index: no table of its own.)  The ONE
// predicate both the slicing of fe_pair_susceptibility and the shift codes of chi_slice use; *sx, *sy = grid shift in [0, N).
static bool chi_q_on_grid(const double* q, int N, long long* sx, long long* sy) {
  const double mx = q[0] * N / (2.0 * 3.14159265358979323846), my = q[1] * N / (2.0 * 3.14159265358979323846);
  const double rx = nearbyint(mx), ry = nearbyint(my);
  if (!(fabs(mx - rx) <= 1e-9 && fabs(my - ry) <= 1e-9 && fabs(rx) < 1e15 && fabs(ry) < 1e15)) return false;
  if (sx) *sx = (((long long)rx % N) + N) % N;
  if (sy) *sy = (((long long)ry % N) + N) % N;
  return true;
}

static int chi_slice(fe_handle* h, const double* q_xy, int32_t nq, double hz, double* chi_dev, void* cuda_stream, bool first_slice) {
  cudaStream_t st = (cudaStream_t)cuda_stream;
  const int N = h->N, nb = h->nb, nbb = nb * nb;
  if (int rcd = check_device(h)) return rcd;
  double *hs, *ds; StageSlot* slot;
  int rc = stage_lists(h, (size_t)3 * nq, st, &hs, &ds, &slot);
  if (rc) return rc;
  for (int i = 0; i < 2 * nq; ++i) hs[i] = -q_xy[i];          // tables of k - (-q) = k + q; E, eta even: = -k - q
  int noff = 0;                                               // q-values off the k-grid: they need a band table each
  for (int i = 0; i < nq; ++i) {                              // q on the k-grid: shift code sx + sy N, else -(table index)
    long long sx = 0, sy = 0;
    double code = -(double)(1 + noff);
    if (chi_q_on_grid(q_xy + 2 * i, N, &sx, &sy)) code = (double)(sx + sy * (long long)N);
    else ++noff;
    hs[2 * nq + i] = code;
  }
  FE_CUDA(cudaMemcpyAsync(ds, hs, (size_t)3 * nq * sizeof(double), cudaMemcpyHostToDevice, st));
  FE_CUDA(cudaEventRecord(slot->ev, st));
  slot->pending = true;
  const unsigned long long nk = (unsigned long long)N * N;
  long long nchunk = ((long long)h->sm_count * 16 + nq - 1) / nq;                  // >= 16 blocks per SM in total
  const long long max_chunk = (long long)((nk + 4 * kThreads - 1) / (4 * kThreads));  // >= 4 k-points per thread
  if (nchunk > max_chunk) nchunk = max_chunk;
  if (nchunk < 1) nchunk = 1;
  if (nchunk > 65535) nchunk = 65535;
  unsigned long long kc = (nk + nchunk - 1) / nchunk;
  kc = (kc + kThreads - 1) / kThreads * kThreads;
  nchunk = (long long)((nk + kc - 1) / kc);
  if ((rc = ensure(h->d_coltab, h->coltab_cap, (size_t)nq * N))) return rc;
  if ((rc = ensure(h->d_rowtab, h->rowtab_cap, (size_t)nq * N))) return rc;
  if ((rc = ensure(h->d_partial, h->partial_cap, (size_t)nchunk * nq * nbb))) return rc;
  if (nb == 3) {
    const size_t need = (size_t)(1 + noff) * 3 * N * N;
    if (need > h->etab_cap || !h->d_etab) h->etab_base_valid = false;
    if ((rc = ensure(h->d_etab, h->etab_cap, need))) return rc;
  }
  fe_trig_kernel<<<(N * nq + 255) / 256, 256, 0, st>>>(N, nq, ds, h->d_coltab, h->d_rowtab);
  FE_CUDA(cudaGetLastError());
  h->launches++;
  if (nb == 3) {
    Band3Consts bc;
    for (int i = 0; i < 12; ++i) bc.t[i] = h->p.tb3[i];
    bc.e0 = h->p.tb3[12];
    const int y0 = h->etab_base_valid ? 1 : 0;
    dim3 g((unsigned)((nk + 255) / 256), (unsigned)(1 + nq - y0));
    fe_bands3_kernel<<<g, 256, 0, st>>>(bc, N, y0, h->d_coltab, h->d_rowtab, ds + 2 * nq, h->d_etab);
    FE_CUDA(cudaGetLastError());
    h->etab_base_valid = true;
    h->launches++;
  }
  const ModelConsts mc = make_consts(h->p);
  dim3 grid((unsigned)nchunk, (unsigned)nq);
  if (h->timing && first_slice) FE_CUDA(cudaEventRecord(h->ev0, st));
  const int form = h->p.form_factor;
#define FE_CHI(NB_, F_) fe_chi_kernel<NB_, F_><<<grid, kThreads, 0, st>>>(mc, h->T, hz, N, nq, kc, h->d_coltab, h->d_rowtab, h->d_etab, ds + 2 * nq, h->d_tabs, h->d_partial)
  if (nb == 1) { if (form == 0) FE_CHI(1, 0); else FE_CHI(1, 1); }
  else if (nb == 2) { if (form == 0) FE_CHI(2, 0); else FE_CHI(2, 1); }
  else { if (form == 0) FE_CHI(3, 0); else FE_CHI(3, 1); }
#undef FE_CHI
  FE_CUDA(cudaGetLastError());
  h->launches++;
  if (h->timing) {
    FE_CUDA(cudaEventRecord(h->ev1, st));
    h->timing_valid = true;
    h->last_band_evals = (first_slice ? 0.0 : h->last_band_evals) + (double)nk * nq * nbb;
  }
  h->last_info[0] = nb; h->last_info[1] = nb; h->last_info[2] = (int32_t)nchunk;
  h->last_info[3] = (first_slice ? 0 : h->last_info[3]) + (int32_t)(nchunk * nq);                 // blocks of all slices
  h->last_info[4] = -1; h->last_info[5] = (int32_t)(kc < 2147483647ULL ? kc : 2147483647ULL);
  const int nout = nq * nbb;
  fe_chi_finish_kernel<<<(nout + 255) / 256, 256, 0, st>>>(nout, (int)nchunk, 1.0 / ((double)N * (double)N), h->d_partial, chi_dev);
  FE_CUDA(cudaGetLastError());
  h->launches++;
  return FE_OK;
}

int fe_pair_susceptibility(fe_handle* h, const double* q_xy, int32_t nq, double hz, double* chi_dev, void* cuda_stream) {
  if (!h || !q_xy || !chi_dev) { snprintf(g_errbuf, sizeof g_errbuf, "handle, q_xy or chi_dev is NULL"); return FE_EINVAL; }
  if (nq < 1 || nq > kMaxQ || !isfinite(hz)) { snprintf(g_errbuf, sizeof g_errbuf, "nq must be in [1, %d], hz finite", kMaxQ); return FE_EINVAL; }
  for (int i = 0; i < 2 * nq; ++i) if (!isfinite(q_xy[i])) { snprintf(g_errbuf, sizeof g_errbuf, "q[%d] not finite", i); return FE_EINVAL; }
  if (h->nb < 3) return chi_slice(h, q_xy, nq, hz, chi_dev, cuda_stream, true);
  // Three-band model: every q OFF the k-grid needs a band table of its own (24 MB at N = 1024).  The q list is processed
  // in consecutive slices that hold at most `maxoff` such q-values, so the table scratch stays below ~2 GB (chi_table_budget) whatever the
  // size of the map (a 48 x 48 off-grid map would otherwise need 55 GB); slices reuse the scratch in stream order.
  const double table_bytes = 3.0 * (double)h->N * (double)h->N * sizeof(double);
  int maxoff = (int)fmin(1.0e9, h->chi_table_budget / table_bytes) - 1;
  if (maxoff < 1) maxoff = 1;
  const int nbb = h->nb * h->nb;
  int q0 = 0;
  while (q0 < nq) {
    int q1 = q0, noff = 0;
    while (q1 < nq) {
      const int off = chi_q_on_grid(q_xy + 2 * q1, h->N, nullptr, nullptr) ? 0 : 1;
      if (noff + off > maxoff) break;
      noff += off; ++q1;
    }
    const int rc = chi_slice(h, q_xy + 2 * q0, q1 - q0, hz, chi_dev + (size_t)q0 * nbb, cuda_stream, q0 == 0);
    if (rc) return rc;
    q0 = q1;
  }
  return FE_OK;
}

int fe_omega_grid_sp(fe_handle* h, const double* q_xy, int32_t nq, const double* h_list, int32_t nh,
                     const double* delta, int32_t nd, int32_t fast_math, double* omega_dev, void* cuda_stream) {
  if (!h || !omega_dev) { snprintf(g_errbuf, sizeof g_errbuf, "handle or omega_dev is NULL"); return FE_EINVAL; }
  if (fast_math != 0 && fast_math != 1) { snprintf(g_errbuf, sizeof g_errbuf, "fast_math must be 0 or 1"); return FE_EINVAL; }
  int rc = check_lists(q_xy, nq, h_list, nh, delta, nd);
  if (rc) return rc;
  return omega_grid_impl(h, q_xy, nq, h_list, nh, delta, nd, omega_dev, (cudaStream_t)cuda_stream, 1 + fast_math);
}

int fe_scan_verified(fe_handle* h, const double* q_xy, int32_t nq, const double* h_list, int32_t nh,
                     const double* delta, int32_t nd, int32_t fast_math, double margin_rel,
                     int32_t* idx_dev, double* delta_star_dev, double* omega_star_dev,
                     int32_t* n_verified_host, int32_t* n_changed_host, void* cuda_stream) {
  if (!h) { snprintf(g_errbuf, sizeof g_errbuf, "handle is NULL"); return FE_EINVAL; }
  if (n_changed_host) *n_changed_host = -1;
  if (fast_math != 0 && fast_math != 1) { snprintf(g_errbuf, sizeof g_errbuf, "fast_math must be 0 or 1"); return FE_EINVAL; }
  if (!(margin_rel >= 0.0) || !isfinite(margin_rel)) { snprintf(g_errbuf, sizeof g_errbuf, "margin_rel must be finite and >= 0"); return FE_EINVAL; }
  int rc = check_lists(q_xy, nq, h_list, nh, delta, nd);
  if (rc) return rc;
  cudaStream_t st = (cudaStream_t)cuda_stream;
  const size_t nout = (size_t)nq * nh * nd;
  const int ncol = nq * nh;
  if ((rc = ensure(h->d_omega, h->omega_cap, nout))) return rc;
  // flags: [0, max(nd, ncol)) candidate flags then the index map; behind it ncol low-precision minima and one counter
  const size_t nflag = (size_t)(nd > ncol ? nd : ncol);
  if ((rc = ensure(h->d_flags, h->flags_cap, nflag + (size_t)ncol + 1))) return rc;
  int32_t* const d_idx_lo = h->d_flags + nflag;
  int32_t* const d_changed = d_idx_lo + ncol;
  if ((size_t)nd > h->hflags_cap) {
    if (h->h_flags) cudaFreeHost(h->h_flags);
    h->h_flags = nullptr; h->hflags_cap = 0;
    if (cudaMallocHost((void**)&h->h_flags, sizeof(int32_t) * (size_t)nd) != cudaSuccess) {
      cudaGetLastError(); snprintf(g_errbuf, sizeof g_errbuf, "pinned allocation failed"); return FE_ENOMEM; }
    h->hflags_cap = nd;
  }
  // 1. screening pass in single precision
  if ((rc = omega_grid_impl(h, q_xy, nq, h_list, nh, delta, nd, h->d_omega, st, 1 + fast_math))) return rc;
  if (n_changed_host && idx_dev) {           // the screening pass's own minima, to report how many the verification moves
    if ((rc = argmin_impl(h, h->d_omega, delta, ncol, nd, d_idx_lo, nullptr, nullptr, st))) return rc;
    FE_CUDA(cudaMemsetAsync(d_changed, 0, sizeof(int32_t), st));
  }
  // 2. candidates
  FE_CUDA(cudaMemsetAsync(h->d_flags, 0, sizeof(int32_t) * (size_t)nd, st));
  // the low-precision error scales with the magnitude of the summed terms (~ N^2 (band half-width + |mu|) per band),
  // not with |Omega_min|, which can be close to zero: the margin is relative to the larger of the two
  int nbm = 0;
  for (int e = 0; e < h->nb; ++e) nbm += (h->p.band_mask >> e) & 1;
  const double abs_scale = (double)h->N * (double)h->N * nbm * (band_half_width(h->p) + fabs(h->p.mu));
  fe_mark_candidates_kernel<<<(ncol + 7) / 8, 256, 0, st>>>(ncol, nd, margin_rel, abs_scale, h->d_omega, h->d_flags);
  FE_CUDA(cudaGetLastError());
  h->launches++;
  FE_CUDA(cudaMemcpyAsync(h->h_flags, h->d_flags, sizeof(int32_t) * (size_t)nd, cudaMemcpyDeviceToHost, st));
  FE_CUDA(cudaStreamSynchronize(st));
  int nu = 0;
  for (int i = 0; i < nd; ++i) nu += h->h_flags[i] != 0;
  if (nu == 0) { snprintf(g_errbuf, sizeof g_errbuf, "screening pass produced no finite minimum"); return FE_EINVAL; }
  double* du = (double*)malloc(sizeof(double) * (size_t)nu);
  if (!du) { snprintf(g_errbuf, sizeof g_errbuf, "host allocation failed"); return FE_ENOMEM; }
  for (int i = 0, u = 0; i < nd; ++i) if (h->h_flags[i]) { du[u] = delta[i]; h->h_flags[u] = i; ++u; }   // u <= i: in place
  if (n_verified_host) *n_verified_host = nu;
  // 3. fp64 on the candidate list, 4. minima, mapped back
  rc = ensure(h->d_omega2, h->omega2_cap, (size_t)ncol * nu);
  if (!rc) rc = omega_grid_impl(h, q_xy, nq, h_list, nh, du, nu, h->d_omega2, st, 0);
  if (!rc) rc = argmin_impl(h, h->d_omega2, du, ncol, nu, idx_dev, delta_star_dev, omega_star_dev, st);
  free(du);
  if (rc) return rc;
  if (idx_dev) {
    FE_CUDA(cudaMemcpyAsync(h->d_flags, h->h_flags, sizeof(int32_t) * (size_t)nu, cudaMemcpyHostToDevice, st));
    fe_map_index_kernel<<<(ncol + 255) / 256, 256, 0, st>>>(ncol, h->d_flags, idx_dev);
    FE_CUDA(cudaGetLastError());
    h->launches++;
    if (n_changed_host) {
      fe_count_changed_kernel<<<(ncol + 255) / 256, 256, 0, st>>>(ncol, d_idx_lo, idx_dev, d_changed);
      FE_CUDA(cudaGetLastError());
      h->launches++;
      FE_CUDA(cudaMemcpyAsync(n_changed_host, d_changed, sizeof(int32_t), cudaMemcpyDeviceToHost, st));
    }
    FE_CUDA(cudaStreamSynchronize(st));        // h_flags (pinned map) may be reused by the next call
  }
  return FE_OK;
}

int fe_scan_host(fe_handle* h, const double* q_xy, int32_t nq, const double* h_list, int32_t nh,
                 const double* delta, int32_t nd, double* omega_host, int32_t* idx_host,
                 double* delta_star_host, double* omega_star_host, void* cuda_stream) {
  if (!h) { snprintf(g_errbuf, sizeof g_errbuf, "handle is NULL"); return FE_EINVAL; }
  int rc = check_lists(q_xy, nq, h_list, nh, delta, nd);
  if (rc) return rc;
  cudaStream_t st = (cudaStream_t)cuda_stream;
  const size_t nout = (size_t)nq * nh * nd;
  const size_t ncol = (size_t)nq * nh;
  if ((rc = ensure(h->d_omega, h->omega_cap, nout))) return rc;
  {
    char* p = (char*)h->d_res;
    size_t cap = h->res_cap;
    if (ncol > cap || !p) {
      if (p) cudaFree(p);
      h->d_res = nullptr; h->res_cap = 0;
      if (cudaMalloc(&h->d_res, ncol * 24) != cudaSuccess) {
        cudaGetLastError(); snprintf(g_errbuf, sizeof g_errbuf, "device allocation failed"); return FE_ENOMEM; }
      h->res_cap = ncol;
    }
  }
  double* d_dstar = (double*)h->d_res;
  double* d_ostar = d_dstar + h->res_cap;
  int32_t* d_idx = (int32_t*)(d_ostar + h->res_cap);
  if ((rc = omega_grid_impl(h, q_xy, nq, h_list, nh, delta, nd, h->d_omega, st))) return rc;
  if ((rc = argmin_impl(h, h->d_omega, delta, (int32_t)ncol, nd, d_idx, d_dstar, d_ostar, st))) return rc;
  if (omega_host) FE_CUDA(cudaMemcpyAsync(omega_host, h->d_omega, nout * sizeof(double), cudaMemcpyDeviceToHost, st));
  if (idx_host) FE_CUDA(cudaMemcpyAsync(idx_host, d_idx, ncol * sizeof(int32_t), cudaMemcpyDeviceToHost, st));
  if (delta_star_host) FE_CUDA(cudaMemcpyAsync(delta_star_host, d_dstar, ncol * sizeof(double), cudaMemcpyDeviceToHost, st));
  if (omega_star_host) FE_CUDA(cudaMemcpyAsync(omega_star_host, d_ostar, ncol * sizeof(double), cudaMemcpyDeviceToHost, st));
  FE_CUDA(cudaStreamSynchronize(st));
  return FE_OK;
}

int fe_enable_timing(fe_handle* h, int32_t on) {
  if (!h) { snprintf(g_errbuf, sizeof g_errbuf, "handle is NULL"); return FE_EINVAL; }
  h->timing = on != 0;
  h->timing_valid = false;
  return FE_OK;
}

int fe_enable_slot_counts(fe_handle* h, int32_t on) {
  if (!h) { snprintf(g_errbuf, sizeof g_errbuf, "handle is NULL"); return FE_EINVAL; }
  h->slot_counts = on != 0;
  h->kinds_valid = false;
  return FE_OK;
}

int fe_get_timing(fe_handle* h, float* ksum_ms, double* band_evals) {
  if (!h) { snprintf(g_errbuf, sizeof g_errbuf, "handle is NULL"); return FE_EINVAL; }
  if (!h->timing_valid) { snprintf(g_errbuf, sizeof g_errbuf, "no timed launch recorded"); return FE_EINVAL; }
  float ms = 0;
  FE_CUDA(cudaEventElapsedTime(&ms, h->ev0, h->ev1));
  if (ksum_ms) *ksum_ms = ms;
  if (band_evals) *band_evals = h->last_band_evals;
  return FE_OK;
}

int fe_get_slot_counts(fe_handle* h, double* counts5) {
  if (!h || !counts5) { snprintf(g_errbuf, sizeof g_errbuf, "NULL argument"); return FE_EINVAL; }
  if (!h->kinds_valid || !h->d_kinds) { snprintf(g_errbuf, sizeof g_errbuf, "no counted cooperative k-sum launch recorded (fe_enable_slot_counts)"); return FE_EINVAL; }
  unsigned long long c[5];
  // on the stream of the counted launch, then wait for it: a non-blocking user stream is not ordered with the default stream
  FE_CUDA(cudaMemcpyAsync(c, h->d_kinds, sizeof c, cudaMemcpyDeviceToHost, h->kinds_stream));
  FE_CUDA(cudaStreamSynchronize(h->kinds_stream));
  for (int i = 0; i < 5; ++i) counts5[i] = (double)c[i];
  return FE_OK;
}

int fe_get_last_launch_info(fe_handle* h, int32_t* info6) {
  if (!h || !info6) { snprintf(g_errbuf, sizeof g_errbuf, "NULL argument"); return FE_EINVAL; }
  for (int i = 0; i < 6; ++i) info6[i] = h->last_info[i];
  return FE_OK;
}

int fe_get_launch_count(fe_handle* h, int64_t* launches) {
  if (!h || !launches) { snprintf(g_errbuf, sizeof g_errbuf, "NULL argument"); return FE_EINVAL; }
  *launches = h->launches;
  return FE_OK;
}

int fe_fp64_peak_probe(int32_t blocks, int32_t iters, float* ms, double* dfma_count, void* cuda_stream) {
  if (blocks < 1 || iters < 1 || !ms || !dfma_count) { snprintf(g_errbuf, sizeof g_errbuf, "bad argument"); return FE_EINVAL; }
  cudaStream_t st = (cudaStream_t)cuda_stream;
  double* sink = nullptr;
  cudaEvent_t a = nullptr, b = nullptr;
  FE_CUDA(cudaMalloc((void**)&sink, sizeof(double)));
  cudaError_t e = cudaEventCreate(&a);
  if (e == cudaSuccess) e = cudaEventCreate(&b);
  if (e == cudaSuccess) { fe_dfma_probe_kernel<<<blocks, 256, 0, st>>>(16, 1.0, sink); e = cudaGetLastError(); }  // warm-up
  if (e == cudaSuccess) e = cudaEventRecord(a, st);
  if (e == cudaSuccess) { fe_dfma_probe_kernel<<<blocks, 256, 0, st>>>(iters, 1.0, sink); e = cudaGetLastError(); }
  if (e == cudaSuccess) e = cudaEventRecord(b, st);
  if (e == cudaSuccess) e = cudaEventSynchronize(b);
  if (e == cudaSuccess) e = cudaEventElapsedTime(ms, a, b);
  if (a) cudaEventDestroy(a);
  if (b) cudaEventDestroy(b);
  cudaFree(sink);
  if (e != cudaSuccess) return cuda_fail(e, "fe_fp64_peak_probe");
  *dfma_count = (double)blocks * 256.0 * (double)iters * 16.0;
  return FE_OK;
}

// Diagnostic entry used by the GPU tests: y[i] = exp_nonpos(x[i]) (which = 0), log_1p_w(x[i]) (which = 1), sqrt_pos(x[i]) (2).
// x_dev, y_dev: DEVICE arrays of n doubles.  Not part of the method; exported so the device math can be
// checked in isolation against numpy.
int fe_debug_math(fe_handle* h, int32_t which, int32_t n, const double* x_dev, double* y_dev, void* cuda_stream) {
  if (!h || !x_dev || !y_dev || n < 1 || which < 0 || which > 2) { snprintf(g_errbuf, sizeof g_errbuf, "bad argument"); return FE_EINVAL; }
  fe_math_probe_kernel<<<(n + 255) / 256, 256, 0, (cudaStream_t)cuda_stream>>>(which, n, x_dev, y_dev, h->d_tabs);
  FE_CUDA(cudaGetLastError());
  h->launches++;
  return FE_OK;
}

void fe_destroy(fe_handle* h) {
  if (!h) return;
  cudaFree(h->d_tabs); cudaFree(h->d_coltab); cudaFree(h->d_rowtab); cudaFree(h->d_partial);
  cudaFree(h->d_kinds);
  cudaFree(h->d_spart); cudaFree(h->d_etab); cudaFree(h->d_omega); cudaFree(h->d_omega2); cudaFree(h->d_flags);
  if (h->h_flags) cudaFreeHost(h->h_flags); cudaFree(h->d_res);
  for (auto& s : h->slots) {
    if (s.pending && s.ev) cudaEventSynchronize(s.ev);
    if (s.host) cudaFreeHost(s.host);
    if (s.dev) cudaFree(s.dev);
    if (s.ev) cudaEventDestroy(s.ev);
  }
  if (h->ev0) cudaEventDestroy(h->ev0);
  if (h->ev1) cudaEventDestroy(h->ev1);
  cudaGetLastError();
  delete h;
}

#ifndef FE_SOURCE_HASH
#define FE_SOURCE_HASH "unknown"
#endif
const char* fe_build_source_hash(void) { return FE_SOURCE_HASH; }

const char* fe_strerror(int code) {
  switch (code) {
    case FE_OK: return "ok";
    case FE_EINVAL: case FE_ENOMEM: case FE_ECUDA: case FE_EARCH: return g_errbuf;
    default: return "unknown error code";
  }
}

}  // extern "C"

// =====================================================================================================
// fe_omega_grid_static: Omega on a small grid for callers that must not allocate (include/fe.h has the contract)
// =====================================================================================================
//
// Everything fe_omega_grid keeps in cudaMalloc'ed handle scratch (the exp / log tables, the device copy of the parameter
// lists, the trig tables of K0, the constant-term partial sums of KS and the [k-chunk][q, h, Delta] partial sums that K1
// writes and K2 adds up) lives here in ONE fixed array that is part of the library image: the driver places it when the
// library's code is loaded onto a device and it stays there, on every device that loads the library, until the process
// exits.  The kernels are the ones fe_omega_grid uses in FE_EVAL_DIRECT mode (K0, KS, K1 with the 4 x 4 register tile,
// K2); only where their scratch comes from differs.
namespace {

constexpr size_t kStTabsBytes = 8192;                    // MathTabs (6.7 KB), padded
constexpr size_t kStListMax = FE_STATIC_MAX_LIST;        // doubles: q (2 nq) | h (nh) | Delta^2 (nd)
constexpr size_t kStTrigMax = FE_STATIC_MAX_TRIG;        // entries of each trig table: nq * N
constexpr size_t kStOutMax = FE_STATIC_MAX_OUT;          // nq * nh * nd
constexpr size_t kStPartialMax = FE_STATIC_MAX_PARTIAL;  // doubles: k-chunks * nq * nh * nd
constexpr size_t kStOffList = kStTabsBytes;
constexpr size_t kStOffCol = kStOffList + kStListMax * sizeof(double);
constexpr size_t kStOffRow = kStOffCol + kStTrigMax * sizeof(double4);
constexpr size_t kStOffSpart = kStOffRow + kStTrigMax * sizeof(double4);
constexpr size_t kStOffPartial = kStOffSpart + kStTrigMax * sizeof(double);     // nq * min(N, 128) <= nq * N
constexpr size_t kStBytes = kStOffPartial + kStPartialMax * sizeof(double);
static_assert(sizeof(MathTabs) <= kStTabsBytes, "table block too small");
static_assert(kStOffList % 256 == 0 && kStOffCol % 256 == 0 && kStOffRow % 256 == 0 && kStOffSpart % 256 == 0 &&
              kStOffPartial % 256 == 0, "sub-blocks keep the 256-byte alignment of the array");
static_assert(kStBytes <= (size_t)8 << 20, "the fixed scratch is meant to stay modest (8 MiB)");

}  // namespace

// The scratch itself.  In HOST code the name `fe_static_scratch` is only the runtime's handle for the symbol, NOT a device
// address: it must go through cudaGetSymbolAddress (static_setup below) before a kernel can be given a pointer into it.
static __device__ __align__(256) unsigned char fe_static_scratch[kStBytes];

namespace {

constexpr int kStMaxDevices = 64;
struct StaticDev {
  bool ready = false;
  unsigned char* base = nullptr;   // device address of fe_static_scratch on this device
  int sm_count = 0;
};
StaticDev g_static_dev[kStMaxDevices];      // plain static storage: no allocation at first use
std::mutex g_static_mutex;                  // two host threads making the first call on a device at once

// Once per device, with that device current: resolve the device address of the array and fill its table block.
// Host-synchronous (a pageable cudaMemcpy), which is why the first call on a device belongs before any stream capture.
int static_setup(int dev, StaticDev** out) {
  if (dev < 0 || dev >= kStMaxDevices) { snprintf(g_errbuf, sizeof g_errbuf, "device ordinal %d is beyond the %d this entry point keeps state for", dev, kStMaxDevices); return FE_EINVAL; }
  StaticDev& sd = g_static_dev[dev];
  std::lock_guard<std::mutex> lock(g_static_mutex);
  if (!sd.ready) {
    int major = 0, sms = 0;
    FE_CUDA(cudaDeviceGetAttribute(&major, cudaDevAttrComputeCapabilityMajor, dev));
    FE_CUDA(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
    if (major != 10) { snprintf(g_errbuf, sizeof g_errbuf, "device %d is compute capability %d.x; libfe is built for sm_100a only", dev, major); return FE_EARCH; }
    unsigned char* base = nullptr;
    FE_CUDA(cudaGetSymbolAddress((void**)&base, fe_static_scratch));
    if (!base) { snprintf(g_errbuf, sizeof g_errbuf, "cudaGetSymbolAddress returned a null address for the fixed scratch"); return FE_ECUDA; }
    MathTabs host_tabs;                                     // 6.7 KB on the stack
    memset(&host_tabs, 0, sizeof host_tabs);
    build_tabs(&host_tabs);
    FE_CUDA(cudaMemcpy(base, &host_tabs, sizeof(MathTabs), cudaMemcpyHostToDevice));
    sd.base = base; sd.sm_count = sms; sd.ready = true;
  }
  *out = &sd;
  return FE_OK;
}

}  // namespace

extern "C" {

int fe_static_limits(int64_t* limits5) {
  if (!limits5) { snprintf(g_errbuf, sizeof g_errbuf, "NULL argument"); return FE_EINVAL; }
  limits5[0] = (int64_t)kStListMax; limits5[1] = (int64_t)kStTrigMax; limits5[2] = (int64_t)kStOutMax;
  limits5[3] = (int64_t)kStPartialMax; limits5[4] = (int64_t)kStBytes;
  return FE_OK;
}

int fe_omega_grid_static(const fe_model_params* params, int32_t N, double T,
                         const double* q_xy, int32_t nq, const double* h_list, int32_t nh,
                         const double* delta, int32_t nd, double* omega_dev, void* cuda_stream) {
  if (!omega_dev) { snprintf(g_errbuf, sizeof g_errbuf, "omega_dev is NULL"); return FE_EINVAL; }
  int rc = validate_params(params, N, T);
  if (rc) return rc;
  if ((rc = check_lists(q_xy, nq, h_list, nh, delta, nd))) return rc;
  const int nb = nbands(*params);
  if (nb == 3) { snprintf(g_errbuf, sizeof g_errbuf, "fe_omega_grid_static covers the one- and two-band models (the three-band model needs per-q band tables of 3 N^2 doubles)"); return FE_EINVAL; }
  // ---- the fixed limits, checked before anything touches the device ----
  const size_t nlist = (size_t)2 * nq + nh + nd, ntrig = (size_t)nq * N, nout = (size_t)nq * nh * nd;
  if (nlist > kStListMax || ntrig > kStTrigMax || nout > kStOutMax) {
    snprintf(g_errbuf, sizeof g_errbuf, "too large for the fixed scratch of fe_omega_grid_static: 2 nq + nh + nd = %zu (limit %zu), nq N = %zu (limit %zu), "
             "nq nh nd = %zu (limit %zu); use fe_omega_grid, which allocates", nlist, kStListMax, ntrig, kStTrigMax, nout, kStOutMax);
    return FE_EINVAL;
  }
  // ---- geometry of K1 (as fe_omega_grid in FE_EVAL_DIRECT mode: 4 x 4 register tile, 256 threads), k-chunks capped by the scratch ----
  constexpr int tile = 1;
  const int TH = kTiles[tile].th, TD = kTiles[tile].td;
  KsumParams P;
  P.mc = make_consts(*params);
  P.T = T; P.neg_beta = -1.0 / T; P.window = 37.0 * T;
  P.N = N; P.nq = nq; P.nh = nh; P.nd = nd;
  P.debug_flags = 0;
  P.ntile_h = (nh + TH - 1) / TH;
  P.ntile_d = (nd + TD - 1) / TD;
  int bxl = 8;                                        // 256 threads: all along kx when N allows it
  while (bxl > 5 && (1 << (bxl - 1)) >= N) --bxl;
  P.bx_log2 = bxl;
  const int bx = 1 << bxl, by = kThreads >> bxl;
  P.ncg = (N + bx - 1) / bx;
  if ((size_t)P.ncg * nout > kStPartialMax) {
    snprintf(g_errbuf, sizeof g_errbuf, "too large for the fixed scratch of fe_omega_grid_static: %d column groups x %zu outputs = %zu partial sums (limit %zu); "
             "use fe_omega_grid, which allocates", P.ncg, nout, (size_t)P.ncg * nout, kStPartialMax);
    return FE_EINVAL;
  }
  int dev = -1;
  FE_CUDA(cudaGetDevice(&dev));
  StaticDev* sd = nullptr;
  if ((rc = static_setup(dev, &sd))) return rc;
  cudaStream_t st = (cudaStream_t)cuda_stream;
  const long long ntiles = (long long)nq * P.ntile_h * P.ntile_d;
  long long nrs = ((long long)sd->sm_count * 2 * 24 + ntiles * P.ncg - 1) / (ntiles * P.ncg);
  const long long cap_nrs = (long long)(kStPartialMax / ((size_t)P.ncg * nout));   // >= 1 (checked above)
  if (nrs > cap_nrs) nrs = cap_nrs;
  if (nrs > (N + by - 1) / by) nrs = (N + by - 1) / by;
  if (nrs < 1) nrs = 1;
  int rpc = (int)((N + nrs - 1) / nrs);
  rpc = (rpc + by - 1) / by * by;
  P.rows_per_chunk = rpc;
  P.nrs = (N + rpc - 1) / rpc;
  P.ksplit = P.ncg * P.nrs;
  const long long grid_ll = ntiles * P.ksplit;
  if (grid_ll > 2147483647LL) { snprintf(g_errbuf, sizeof g_errbuf, "grid too large"); return FE_EINVAL; }
  // ---- carve the array ----
  double* d_list = reinterpret_cast<double*>(sd->base + kStOffList);
  double4* d_col = reinterpret_cast<double4*>(sd->base + kStOffCol);
  double4* d_row = reinterpret_cast<double4*>(sd->base + kStOffRow);
  double* d_spart = reinterpret_cast<double*>(sd->base + kStOffSpart);
  double* d_partial = reinterpret_cast<double*>(sd->base + kStOffPartial);
  // ---- lists: assembled on the stack, copied from pageable memory (the copy call returns once the source may be reused) ----
  double hs[kStListMax];
  memcpy(hs, q_xy, sizeof(double) * 2 * nq);
  memcpy(hs + 2 * nq, h_list, sizeof(double) * nh);
  for (int i = 0; i < nd; ++i) hs[2 * nq + nh + i] = delta[i] * delta[i];
  FE_CUDA(cudaMemcpyAsync(d_list, hs, nlist * sizeof(double), cudaMemcpyHostToDevice, st));
  const double* d_q = d_list;
  P.h = d_list + 2 * nq; P.d2 = d_list + 2 * nq + nh; P.htile = nullptr;
  P.coltab = d_col; P.rowtab = d_row; P.tabs = reinterpret_cast<const MathTabs*>(sd->base); P.partial = d_partial;
  // ---- K0, KS, K1, K2.  Each of them writes every scratch word that a later one reads (all nq N table entries, all nq x
  // nschunk constant sums, all ksplit x nout partial sums, empty chunks included), so nothing has to start at zero and what
  // an earlier, larger call left behind is never read. ----
  fe_trig_kernel<<<(N * nq + 255) / 256, 256, 0, st>>>(N, nq, d_q, d_col, d_row);
  FE_CUDA(cudaGetLastError());
  int nschunk = N < kSChunksMax ? N : kSChunksMax;
  const int srpc = (N + nschunk - 1) / nschunk;
  nschunk = (N + srpc - 1) / srpc;
  {
    dim3 g(nschunk, nq);
    if (nb == 1) fe_ssum_kernel<1><<<g, kThreads, 0, st>>>(P.mc, N, srpc, d_col, d_row, d_spart);
    else         fe_ssum_kernel<2><<<g, kThreads, 0, st>>>(P.mc, N, srpc, d_col, d_row, d_spart);
    FE_CUDA(cudaGetLastError());
  }
  FE_CUDA(launch_ksum(tile, nb, params->form_factor, FE_EVAL_DIRECT, (int)grid_ll, st, P));
  const double condc = params->cond_mult * (double)N * (double)N / params->U;
  fe_finish_kernel<<<(unsigned)((nout + 255) / 256), 256, 0, st>>>(nq, nh, nd, P.ksplit, nschunk, condc, d_partial, d_spart, P.d2, omega_dev);
  FE_CUDA(cudaGetLastError());
  return FE_OK;
}

}  // extern "C"
