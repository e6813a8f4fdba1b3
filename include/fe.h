/*
 * fe.h -- C ABI of libfe: B200-native (sm_100a) evaluation of the mean-field grand potential
 * Omega(Delta; q, h, T) of a lattice superconductor over an N x N Brillouin-zone grid, for every
 * point of a (q, h, Delta) parameter grid, and the per-(q, h) global-minimum search over Delta.
 *
 * Method: Januszewski, Ptok, Crivelli, Gardas, "GPU-based acceleration of free energy calculations
 * in solid state physics" (arXiv 1412.8754); citations are PAPER.md:<line> of the reference text.
 *
 *   Omega = sum_{eps in bands} sum_{k in grid} [ f(E+) + f(E-) + C_{eps k} ] + cond_mult N^2 Delta^2 / U
 *   f(x)  = -T ln(1 + exp(-x/T))                                              (Eq. 5)
 *   E+-   = (a-b)/2 +- sqrt(((a+b)/2)^2 + (Delta eta_k)^2)                    (Eq. 4)
 *   a = E_{eps,k} - mu - h (spin up),  b = E_{eps,-k+q} - mu + h (spin down)
 *   k = 2 pi (i, j)/N, i, j = 0..N-1;  q is any real vector (need not be on the grid).
 *
 * Everything is fp64.  All device work is enqueued on the CUDA stream the caller passes and the
 * calls return without synchronising (except fe_scan_host, which is the host-buffer convenience
 * path and returns with results in host memory).  Results are deterministic: the k-sum uses a fixed
 * k -> thread map, a fixed shuffle tree and a fixed chunk order; there are no floating-point atomics,
 * so the same inputs give bit-identical Omega on every run.
 *
 * There is NO CPU fallback: without a compute-capability 10.x device fe_create fails.
 *
 * Thread-safety: one handle must be used by one host thread and one stream at a time; distinct
 * handles are independent.  No function throws or aborts across this boundary.
 */
#ifndef FE_H_
#define FE_H_

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

/* ---- error codes (fe_strerror gives text; for FE_ECUDA it includes the CUDA error string) ---- */
#define FE_OK      0
#define FE_EINVAL (-1) /* null pointer, N < 1, T <= 0 or non-finite, U <= 0, list length < 1, unknown model/mode */
#define FE_ENOMEM (-2) /* host or device allocation failed                                                       */
#define FE_ECUDA  (-3) /* a CUDA runtime call or kernel launch failed                                            */
#define FE_EARCH  (-4) /* current device is not compute capability 10.x (B200)                                   */

/* ---- model selectors ---- */
#define FE_MODEL_ONE_BAND 1 /* E_k = -2 t[0] (cos kx + cos ky): nearest-neighbour square lattice (BCS use) */
#define FE_MODEL_TWO_BAND 2 /* Raghu et al. two-orbital model, Eqs. A.1-A.4, t[0..3] = t1..t4;
                               band 0 = E_+ (electron-like), band 1 = E_- (hole-like)             */
#define FE_MODEL_THREE_BAND 3 /* Daghofer et al. three-orbital model, Eqs. B.1-B.6, hoppings in tb3[];
                                 the 3x3 complex-Hermitian T_k is diagonalised numerically on the device and the
                                 eigenvalues are stored in per-q tables in HBM, as the paper proposes for more than two
                                 bands; band e = e-th eigenvalue in ascending order.
                                 FE_EVAL_COOP / FE_EVAL_COOP_EO only.                                              */
#define FE_FORM_S   0       /* eta(k) = eta_scale                       (homogeneous s-wave)                      */
#define FE_FORM_SPM 1       /* eta(k) = eta_scale * cos kx * cos ky     (s+-)                        */

/* ---- evaluation mode of the k-sum kernel (fe_set_eval_mode); both compute the same sums ----
 * COOP_EO : default.  The block-cooperative factored kernel with a block-uniform early-out: a (k, band) slot whose
 *           2cosh(R_j/T) exceeds 2cosh(|d_i|/T) by more than 2^42 over the whole block tile contributes
 *           T ln Z_ij = R_j (what is neglected is below 5.1e-15 of the term and one-signed), so it needs no pair products; the
 *           other slots are compacted and run through the dense pipeline.  Same results to ~1e-15 relative; several
 *           times fewer FP64 instructions at low T.
 * COOP    : the dense variant (every pair of every slot is multiplied out).  Uses 2cosh(d/T) + 2cosh(R/T) =
 *           B(h) + A(Delta): a thread block owns one (h, Delta) block tile and a chunk of k-points; the exponentials
 *           per (k, band) are computed once per block and shared through shared memory; every thread keeps a register
 *           tile of running products over all k of the chunk (no cross-thread reduction).
 * Three further formulations of the same sums (per-thread factored, direct Eq. 4 / Eq. 5 per term, windowed) are kept
 * as cross-checks for the tests; their selectors are in fe_debug.h.                                           */
#define FE_EVAL_COOP     3
#define FE_EVAL_COOP_EO  4

typedef struct fe_handle fe_handle; /* opaque; owns device scratch (trig tables, partial sums, staging) */

typedef struct {
  int32_t model;       /* FE_MODEL_*                                                                       */
  int32_t form_factor; /* FE_FORM_*                                                                        */
  double  t[4];        /* hoppings; unused entries ignored                                                 */
  double  mu;          /* chemical potential                                                               */
  double  U;           /* pairing strength, > 0; enters only the condensation term                         */
  double  eta_scale;   /* 1.0 for Delta_k = Delta cos kx cos ky; 4.0 reproduces eta of PAPER.md:289        */
  double  cond_mult;   /* condensation term = cond_mult * N^2 * Delta^2 / U; Eq. 5 per band => #bands      */
  int32_t band_mask;   /* bit e set => band e contributes (Omega = sum_eps Omega_eps)         */
  int32_t const_mode;  /* 0: constant of Eq. 5 = sum_k xi_{eps,-k+q,dn} (what the Bogoliubov transformation
                             of Eq. 3 gives for any q)   1: sum_k xi_{eps,k,dn} (Eq. 5 as printed; equal for
                             on-grid q)                                                                     */
  double  tb3[13];     /* FE_MODEL_THREE_BAND: t1..t12 = tb3[0..11], eps0 = tb3[12]; else ignored */
} fe_model_params;

/* Create a handle for an N x N k-grid at temperature T (k_B = 1, energies in units of |t1|).
 * Uses the CURRENT CUDA device.  *out is set only on success.  Errors: FE_EINVAL, FE_EARCH, FE_ENOMEM, FE_ECUDA. */
int fe_create(const fe_model_params* params, int32_t N, double T, fe_handle** out);

/* Change T (> 0, finite) for subsequent calls (config 4 scans two temperatures).  Host-only, cheap. */
int fe_set_temperature(fe_handle* h, double T);

/* Select FE_EVAL_COOP_EO (default) or FE_EVAL_COOP (or one of the cross-check modes of fe_debug.h) for subsequent
 * fe_omega_grid calls.  Unknown mode: FE_EINVAL. */
int fe_set_eval_mode(fe_handle* h, int32_t mode);

/* Opt-in mirror-symmetry reduction of the k-sum (default off).  The paper notes that symmetries of the dispersion can
 * shorten Algorithm 1 (E(-k) = E(k) for q = 0, scans along specific q directions).  When on,
 * every fe_omega_grid call whose q list is invariant, element by element and compared exactly, under one mirror M of the
 * square lattice -- k_x <-> k_y (all q_x == q_y), k_y -> -k_y (all q_y == 0) or k_x -> -k_x (all q_x == 0) -- sums only
 * the k-points with M k "above" k with weight 2 and the fixed points of M with weight 1: E_k, E_{k-q} and eta_k are the same
 * at k and M k, so the terms are equal and half of the zone is visited.  Mathematically the same Omega; the summation order
 * differs, so the result differs from the full-zone sum by rounding (~1e-15 relative).  One- and two-band models with the
 * cooperative kernel (FE_EVAL_COOP / FE_EVAL_COOP_EO); other calls ignore the setting.  fe_get_last_symmetry reports
 * what the most recent fe_omega_grid launch used: 0 none, 1 k_y -> -k_y, 2 k_x -> -k_x, 3 k_x <-> k_y.            */
int fe_set_symmetry(fe_handle* h, int32_t on);
int fe_get_last_symmetry(fe_handle* h, int32_t* sym);

/* Omega on the full grid  (steps S1-S9 of DESIGN.md: k generation, dispersion A.1-A.4, Eq. 4, Eq. 5,
 * deterministic two-stage k-sum; Algorithm 1 lines 1-5, Algorithm 2).
 *   q_xy  : HOST, nq pairs (qx, qy), radians.            h_list : HOST, nh Zeeman fields.
 *   delta : HOST, nd order-parameter amplitudes (any sign; Omega is even in Delta).
 *   omega_dev : DEVICE, nq*nh*nd doubles, index (iq*nh + ih)*nd + id (Delta fastest); caller-owned.
 *   cuda_stream : cudaStream_t cast to void* (NULL = legacy default stream).
 * The three host lists are copied before the call returns and may be reused immediately.
 * Omega is extensive (sum over k and bands, not per site).  Asynchronous w.r.t. the host.          */
int fe_omega_grid(fe_handle* h,
                  const double* q_xy, int32_t nq,
                  const double* h_list, int32_t nh,
                  const double* delta, int32_t nd,
                  double* omega_dev, void* cuda_stream);

/* Per-(q, h) global minimum over Delta (Algorithm 1 line 6; step 3 of PAPER.md:169, moved on-device).
 *   omega_dev : DEVICE, ncol*nd doubles, Delta fastest (the layout fe_omega_grid writes; ncol = nq*nh).
 *   delta     : HOST, nd values (copied before return).
 *   idx_dev (int32), delta_star_dev, omega_star_dev : DEVICE, ncol each; any of them may be NULL.
 * Lowest Omega wins; among exactly equal values the lowest index wins.  NaN never wins.             */
int fe_argmin(fe_handle* h, const double* omega_dev, const double* delta,
              int32_t ncol, int32_t nd,
              int32_t* idx_dev, double* delta_star_dev, double* omega_star_dev, void* cuda_stream);

/* Global ground state per field h: minimum over (q, Delta) (outer loops of Algorithm 1, PAPER.md:133-153 lines 1, 6-9;
 * "minimizing the free energy over the set of Delta and q").
 *   omega_dev : DEVICE, nq*nh*nd doubles in the layout fe_omega_grid writes.
 *   ref_id    : >= 0: the quantity compared across q is the condensation energy
 *               Omega(q, h, Delta) - Omega(q, h, delta[ref_id]) (give the index of Delta = 0; for off-grid q the
 *               normal-state Omega itself depends on q at finite N, reading G17);
 *               -1: Omega itself, Algorithm 1 as printed.  Other values: FE_EINVAL.
 *   iq_dev, id_dev (int32), value_dev (double) : DEVICE, nh each; any may be NULL.
 * Lowest value wins; among exactly equal values the lowest iq, then the lowest Delta index.  NaN never wins.
 * For the paper's per-band minimisation run one handle per band (band_mask).                        */
int fe_argmin_q(fe_handle* h, const double* omega_dev, int32_t nq, int32_t nh, int32_t nd, int32_t ref_id,
                int32_t* iq_dev, int32_t* id_dev, double* value_dev, void* cuda_stream);

/* Static Cooper-pair susceptibility of Appendix C, Eqs. C.2-C.3 at omega -> 0, at the handle's
 * temperature and one Zeeman field hz:
 *   chi_{e f}(q) = (1/N^2) sum_k eta(-k-q)^2 [f(-E_{e,k,up}) - f(E_{f,-k-q,down})] / (E_{e,k,up} + E_{f,-k-q,down}),
 * f = Fermi function, E_{e,k,sigma} = E_e(k) - mu - sigma hz, eta from form_factor / eta_scale (4.0 = the paper's C.3).
 *   q_xy    : HOST, nq pairs (qx, qy), any real vectors (copied before return).
 *   chi_dev : DEVICE, nq * nb * nb doubles, index (iq*nb + e)*nb + f, nb = number of bands (band_mask is ignored).
 * Asynchronous on cuda_stream; deterministic.  With fe_enable_timing the k-sum kernel of this call is the one
 * fe_get_timing reports (its second value is then the number of (k, q, e, f) pair terms).  Three-band model: q-values on
 * the k-grid read the unshifted band table at a shifted index; q-values off the grid need a table each (3 N^2 doubles),
 * so the list is worked through in consecutive slices whose tables fit ~2 GB of scratch; fe_get_timing then reports the
 * pair terms of ALL slices and the time from the start of the first slice's k-sum kernel to the end of the last one's (the
 * table and finishing kernels of the slices in between are inside that interval).               */
int fe_pair_susceptibility(fe_handle* h, const double* q_xy, int32_t nq, double hz, double* chi_dev, void* cuda_stream);

/* The paper's single-precision builds: Omega on the full grid with every per-term
 * operation of Eq. 4 / Eq. 5 in binary32 -- fast_math = 0: "SP" (accurate expf / log1pf / sqrtf), 1: "SPFM" (fast
 * intrinsics).  Only the sum over k is kept in double (fixed order).  Arguments as fe_omega_grid; omega_dev receives
 * doubles.  One- and two-band models only (FE_EINVAL for the three-band model).  Expect ~1e-7 relative accuracy.  */
int fe_omega_grid_sp(fe_handle* h,
                     const double* q_xy, int32_t nq, const double* h_list, int32_t nh,
                     const double* delta, int32_t nd, int32_t fast_math,
                     double* omega_dev, void* cuda_stream);

/* Low-precision screening + selective double-precision verification ("run larger parameter scans at
 * lower precision and then selectively verify with double precision calculations"):
 *   1. fe_omega_grid_sp over the whole grid;  2. every Delta index that comes within margin_rel * M of the minimum of ANY
 *   (q, h) column is a candidate, M = max(|column minimum|, N^2 (#bands in band_mask) (band half-width + |mu|)): the
 *   single-precision error scales with the magnitude of the summed terms, not with |Omega_min|, which may be near zero;
 *   3. fe_omega_grid (fp64, the handle's evaluation mode) on the candidate Delta list only;  4. fe_argmin on that, indices
 *   mapped back to the full list.
 * Guarantee: the minima equal those of a full fp64 scan whenever the single-precision Omega is within margin_rel * M / 2 of
 * the fp64 Omega on every grid point (measured error ~1e-7 M: the default 1e-5 is ample).  All list pointers HOST;
 * idx_dev / delta_star_dev / omega_star_dev DEVICE, nq*nh each, any may be NULL; HOST outputs, either may be NULL:
 * *n_verified_host = number of Delta values evaluated in fp64; *n_changed_host = number of (q, h) columns whose minimum
 * index the verification moved away from the single-precision argmin (-1 if idx_dev is NULL) -- the quantity PAPER.md:198
 * asks to watch ("we advise careful experimentation").  Synchronises the stream between steps 2 and 3 (the candidate list
 * is built on the host) and before returning.            */
int fe_scan_verified(fe_handle* h,
                     const double* q_xy, int32_t nq, const double* h_list, int32_t nh,
                     const double* delta, int32_t nd, int32_t fast_math, double margin_rel,
                     int32_t* idx_dev, double* delta_star_dev, double* omega_star_dev,
                     int32_t* n_verified_host, int32_t* n_changed_host, void* cuda_stream);

/* Host-buffer end-to-end path: copies the lists to the device, runs fe_omega_grid and fe_argmin,
 * copies results back and SYNCHRONISES the stream.  All pointers are HOST memory (pinned or pageable).
 *   omega_host : nq*nh*nd doubles or NULL (skip the Omega copy-back);
 *   idx_host / delta_star_host / omega_star_host : nq*nh each, any may be NULL.                     */
int fe_scan_host(fe_handle* h,
                 const double* q_xy, int32_t nq, const double* h_list, int32_t nh,
                 const double* delta, int32_t nd,
                 double* omega_host, int32_t* idx_host, double* delta_star_host, double* omega_star_host,
                 void* cuda_stream);

/* Omega on a SMALL grid without any allocation, for callers that cannot let this library call cudaMalloc.
 *
 * Who that is.  Every other entry point works on an fe_handle, and a handle allocates: fe_create makes the math tables,
 * and fe_omega_grid releases and re-makes the handle's scratch (cudaFree + cudaMalloc, plus pinned staging) whenever a call
 * needs more than any earlier call did.  That does not suit
 *   - a process in which something else already owns the device memory -- typically a framework's caching allocator (the
 *     PyTorch one this library's Python binding sits next to) that has reserved nearly all of HBM: a cudaMalloc from
 *     outside that pool then fails although the job as a whole has memory to spare;
 *   - a caller that runs other work on the same GPU at the same time: cudaMalloc and cudaFree make the whole device wait,
 *     so a scan that grows its grid stalls the other streams at a moment the caller does not choose;
 *   - a caller whose memory budget is fixed when the job starts (a service with a hard per-process limit) and who
 *     therefore needs the library's footprint to be a constant known in advance.
 * For them this function computes the same Omega (Eq. 4 / Eq. 5; steps S1-S9) with all of its working
 * memory in ONE fixed array compiled into the library (a file-scope __device__ array of FE_STATIC_BYTES_MAX bytes or less,
 * about 7.8 MiB).  That array is part of the library image: every GPU on which the library's code gets loaded holds it
 * from then until the process exits, whether or not this function is ever called.  The function takes no handle and calls
 * no cudaMalloc, cudaFree, cudaMallocHost or other allocating routine; the caller brings the inputs and the output.
 *
 *   params, N, T : as fe_create (same validation).  One- and two-band models only; FE_MODEL_THREE_BAND is FE_EINVAL
 *                  (its per-q band tables do not fit a fixed array of this size).
 *   q_xy, h_list, delta : HOST lists as fe_omega_grid; copied before the call returns (from pageable memory, so the
 *                  copy call may first wait for earlier work on cuda_stream).
 *   omega_dev    : DEVICE, nq*nh*nd doubles, layout as fe_omega_grid; caller-owned.
 * Limits (fe_static_limits reports them; beyond any of them the call returns FE_EINVAL with a message that names the
 * quantity, its value and the limit, and touches nothing):
 *   2 nq + nh + nd <= FE_STATIC_MAX_LIST,  nq N <= FE_STATIC_MAX_TRIG,  nq nh nd <= FE_STATIC_MAX_OUT,
 *   ceil(N / 256) nq nh nd <= FE_STATIC_MAX_PARTIAL.   Example that fits: N = 1024, 1 q, 16 h, 512 Delta.
 * It evaluates every term directly (the FE_EVAL_DIRECT formulation of fe_debug.h, the slowest and most literal one):
 * the example above takes 57 ms on a B200 where fe_omega_grid's default kernel takes 2.5 ms, so this is the path for
 * callers who cannot allocate, not a fast path.  Results agree with fe_omega_grid to rounding (5e-15 relative measured
 * on that example) and are deterministic.
 *
 * First call on a device: it looks up the device address of the array (cudaGetSymbolAddress, once per device, with that
 * device current) and copies the math tables into it with a host-synchronous cudaMemcpy.  Make that first call during
 * start-up, before any stream capture begins and before the phase in which the device must not be disturbed.
 * Later calls only enqueue work on cuda_stream and return without synchronising.
 *
 * Sharing: all calls on a device use the SAME array, and it keeps what the last call left in it.  Each call rewrites every
 * word it later reads (tables, lists, partial sums), so stale contents never reach a result and nothing needs to be zeroed.
 * But two calls whose GPU work overlaps -- different streams, or different host threads -- overwrite each other's
 * partial sums and both results are garbage: keep all calls of a device on one stream, or order them with events.
 * Errors: FE_EINVAL (arguments, limits), FE_EARCH, FE_ECUDA.                                                     */
#define FE_STATIC_MAX_LIST    4096      /* doubles */
#define FE_STATIC_MAX_TRIG    32768     /* table entries */
#define FE_STATIC_MAX_OUT     32768     /* Omega values per call */
#define FE_STATIC_MAX_PARTIAL 720896    /* doubles: k-chunks x Omega values */
#define FE_STATIC_BYTES_MAX   (8u << 20)
int fe_omega_grid_static(const fe_model_params* params, int32_t N, double T,
                         const double* q_xy, int32_t nq, const double* h_list, int32_t nh,
                         const double* delta, int32_t nd, double* omega_dev, void* cuda_stream);
/* limits5 (HOST) = {FE_STATIC_MAX_LIST, FE_STATIC_MAX_TRIG, FE_STATIC_MAX_OUT, FE_STATIC_MAX_PARTIAL, bytes of the fixed
 * array as built}.  Host-only, no CUDA call. */
int fe_static_limits(int64_t* limits5);

/* Kernel timing for roofline reports.  When enabled, fe_omega_grid brackets its k-sum kernel (K1) with
 * CUDA events on the launching stream; after the caller has synchronised the stream, fe_get_timing returns
 * the duration of the most recent K1 launch (ms) and the number of (k, band, q, h, Delta) terms it evaluated. */
int fe_enable_timing(fe_handle* h, int32_t on);
int fe_get_timing(fe_handle* h, float* ksum_ms, double* band_evals);

/* What a cooperative k-sum launch (FE_EVAL_COOP / FE_EVAL_COOP_EO) was made of.  fe_enable_slot_counts(h, 1) makes every
 * following launch count its (k, band) slots by kind -- a few global atomics per group of k-points, so leave it OFF (the
 * default) in launches whose duration is being measured; fe_enable_timing does not switch it on.  fe_get_slot_counts then
 * returns, for the most recent counted launch, counts5 = {dense, A-dominated (summed as square roots per Delta_j),
 * B-dominated, padding, A-dominated (summed through the moment series)} slots, each counted once per block tile it was
 * classified for (a slot of a 64 x 128 block tile stands for 8192 (h, Delta) pairs).  Dense and padding slots run through
 * the pair products, dominated slots are summed without exponentials (FE_EVAL_COOP_EO; FE_EVAL_COOP has none).  HOST
 * doubles.  The call copies the five counters on the stream of that launch and waits for that stream.  FE_EINVAL if there
 * is no counted launch. */
int fe_enable_slot_counts(fe_handle* h, int32_t on);
int fe_get_slot_counts(fe_handle* h, double* counts5);

/* Launch configuration of the most recent k-sum kernel: info6 = {TH, TD, ksplit, grid blocks, eval mode actually
 * used, rows per k-chunk}; for FE_EVAL_COOP / FE_EVAL_COOP_EO: {WH, WD, ksplit, grid blocks, mode, k-points per chunk};
 * after fe_omega_grid_sp the mode entry is 101 (SP) or 102 (SPFM); after fe_pair_susceptibility
 * {nb, nb, k-chunks, grid blocks (summed over the slices of the call), -1, k-points per chunk}.  Host-only. */
int fe_get_last_launch_info(fe_handle* h, int32_t* info6);

/* Number of kernel launches this handle has issued since creation (all kernels of this library). */
int fe_get_launch_count(fe_handle* h, int64_t* launches);

/* FP64 DFMA-chain microbenchmark on the current device (register-resident, no memory traffic):
 * runs `blocks` blocks of 256 threads, each thread `iters` x 16 dependent-chain-interleaved DFMAs,
 * and returns elapsed ms and the number of DFMA instructions (thread-level) executed.
 * Used to measure the FP64 roofline denominator in the same run as the benchmark.                  */
int fe_fp64_peak_probe(int32_t blocks, int32_t iters, float* ms, double* dfma_count, void* cuda_stream);

/* First 16 hex digits of the sha256 of the kernel sources this library was compiled from (comments and white space
 * removed; paper_1412_8754_b200/build.py source_hash).  bench.py uses it to tell whether committed profiler counts
 * describe the kernels that are running.  Static string, never NULL. */
const char* fe_build_source_hash(void);

void fe_destroy(fe_handle* h);          /* frees all device/host scratch; NULL is a no-op */
const char* fe_strerror(int code);      /* static or thread-local string; never NULL      */

#ifdef __cplusplus
}
#endif
#endif /* FE_H_ */
