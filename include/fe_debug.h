/*
 * fe_debug.h -- test and tuning hooks of libfe.  NOT part of the boundary SURVEY.md 8(b) lists (that is include/fe.h):
 * included only by the tests, bench.py's binding and the library itself.  Same conventions as fe.h (C ABI, int error
 * codes, fe_strerror).  Nothing here changes WHAT is computed, only which kernel formulation / launch shape computes it.
 */
#ifndef FE_DEBUG_H_
#define FE_DEBUG_H_

#include "fe.h"

#ifdef __cplusplus
extern "C" {
#endif

/* ---- cross-check formulations of the k-sum (fe_set_eval_mode); same sums as FE_EVAL_COOP (Eq. 4 / Eq. 5) ----
 * FACTORED: per-thread version of the factored form.  Per (k, band) TH + TD exponentials in extended range (fp64
 *           mantissa + int exponent), per term one add and one multiply into a running product; the logarithm is
 *           taken once per thread at the end.  fe_omega_grid falls back to it when the (h, Delta) grid is much smaller
 *           than a block tile of FE_EVAL_COOP (e.g. a single h value) unless a shape is forced with fe_set_coop_shape.
 * DIRECT  : every (k, band, q, h, Delta) term evaluates both exponentials and the logarithm of Eq. 5
 *           (the stable form max(R,|d|) + T ln(1 + u + v + uv)).
 * WINDOWED: DIRECT, but a term whose thermal part is below half an ulp of its T=0 part (|R-|d|| >= 37 T) adds
 *           only max(R,|d|); the decision is taken per warp.  Bit-identical to DIRECT.                      */
#define FE_EVAL_FACTORED 0
#define FE_EVAL_DIRECT   1
#define FE_EVAL_WINDOWED 2

/* Tuning knobs (optional).  tile: 0 = auto, else index into the built-in tile table (see fe_tile_info);
 * target_blocks: minimum number of thread blocks K1 should be split into (0 = auto).               */
int fe_set_tuning(fe_handle* h, int32_t tile, int32_t target_blocks);
int fe_tile_info(int32_t tile, int32_t* th, int32_t* td);   /* FE_EINVAL past the end of the table */
/* FE_EVAL_COOP block shape: 0 = auto, else index (from 1) into the built-in shape table; forcing a shape also
 * disables the fallback to FE_EVAL_FACTORED.  fe_coop_shape_info: info6 = {TH, TD, WH, WD, threads per block,
 * resident blocks per SM}; FE_EINVAL past the end of the table. */
int fe_set_coop_shape(fe_handle* h, int32_t shape);
int fe_coop_shape_info(int32_t shape, int32_t* info6);
/* Resident blocks per SM of one instance of the cooperative kernel on the CURRENT device (occupancy query with the
 * instance's shared memory and registers): shape from 1 as above, nbands 1..3, form_factor FE_FORM_*, sym 0 / 1 (the
 * fe_set_symmetry instance).  A test compares it with the launch bound of fe_coop_shape_info, so that an instance that
 * stops fitting (more shared memory, more registers) is noticed.  FE_EINVAL if the shape has no such instance.       */
int fe_debug_coop_occupancy(int32_t shape, int32_t nbands, int32_t form_factor, int32_t sym, int32_t* blocks_per_sm);
/* Test hook for FE_EVAL_FACTORED / FE_EVAL_COOP(_EO): bit 0 = always take the robust per-pair path (this also switches
 * the early-out of FE_EVAL_COOP_EO off), bit 1 = never use the per-tile h recurrence (FACTORED).  Results are the same
 * sums; only the code path changes (lets tests cover each path).                                            */
int fe_set_debug_flags(fe_handle* h, int32_t flags);

/* fe_pair_susceptibility, three-band model: bytes of per-q band tables one slice of the q list may hold (default 2e9;
 * a slice always holds at least one off-grid q).  Lets tests force the slicing on small grids.  Results do not depend on it. */
int fe_set_chi_table_budget(fe_handle* h, double bytes);

/* Host-only test hook for fe_set_symmetry: the symmetry-reduced k enumeration the cooperative kernel walks.  sym = 1, 2, 3 as
 * fe_get_last_symmetry reports.  counts2 = {n2, n1}: indices [0, n2) are the k-points summed with weight 2, [n2, n2 + n1)
 * those with weight 1; for 0 <= i < n2 + n1, (row, col) = (k_y, k_x) grid indices of entry i.  Any pointer may be NULL.
 * FE_EINVAL for another sym, N < 3 or i out of range.  No CUDA call. */
int fe_debug_sym_index(int32_t sym, int32_t N, int64_t i, int32_t* row, int32_t* col, int64_t* counts2);

/* Diagnostic (not part of the method): evaluate the library's device math on DEVICE arrays of n doubles,
 * y[i] = exp(x[i]) for x <= 0 (which = 0), ln(1 + x[i]) for 0 <= x <= 3 (which = 1), exactly as the direct k-sum
 * kernel evaluates the thermal term of Eq. 5, or sqrt(x[i]) for normal x > 0 (which = 2) as every kernel
 * evaluates the radicand of Eq. 4.  Lets tests check them in isolation.       */
int fe_debug_math(fe_handle* h, int32_t which, int32_t n, const double* x_dev, double* y_dev, void* cuda_stream);

#ifdef __cplusplus
}
#endif
#endif /* FE_DEBUG_H_ */
