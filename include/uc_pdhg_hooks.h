/*
 * uc_pdhg_hooks.h -- measurement and test hooks of libuc_pdhg.so.
 *
 * Not part of the product ABI (include/uc_pdhg.h): these entry points exist for bench.py (kernel times for
 * the roofline), for the timeline tool behind profiles/, and for the tests (layout checks of ingest step A1,
 * the scaled matrix for R1, the double-double log / exp of R11).  Same conventions as uc_pdhg.h: 0 or a negative uc_error,
 * uc_last_error() for the text, HOST pointers unless the name says otherwise.
 */
#ifndef UC_PDHG_HOOKS_H
#define UC_PDHG_HOOKS_H

#include "uc_pdhg.h"

#ifdef __cplusplus
extern "C" {
#endif

/* Measurement hook: from the initial point, run `attempts` attempts as plain stream
   launches with a CUDA event between the two kernels and return the average device time, in ms, of
   the primal kernel (K' pass, A5+A6) and of the dual kernel (K pass, A7..A9).  stream: cudaStream_t or
   NULL.  The handle's iterate state is overwritten. */
int uc_pdhg_time_kernels(uc_lp* lp, void* stream, int32_t attempts, double* primal_ms, double* dual_ms);

/* Measurement hook, only in a library built with -DUC_TIMELINE (otherwise UC_ERR_INVALID): run `attempts` attempts from
   the initial point as plain stream launches (programmatic dependent launch, no events in between) and return the
   %globaltimer marks (ns) that every warp of the two kernels of the LAST attempt recorded:
   out[((cta * 32 + warp) * 8) + i], i = 0 kernel entry, 1 grid dependency resolved, 2 own steps done, 3 block sum done
   (for the warp that ran the step rule: attempt decided), 4 ticket taken, 5 partials of all CTAs loaded, 6 final sums
   done (4-6: warp 0 of the dual kernel only); the dual kernel's block starts at out + grid_primal * 32 * 8.
   out: HOST buffer of `cap` entries, cap >= (grid_primal + grid_dual) * 256; unused entries stay 0.
   and profiles/ use it for the timeline of an attempt. */
int uc_pdhg_timeline(uc_lp* lp, void* stream, int32_t attempts, uint64_t* out, int64_t cap, int32_t* grid_primal, int32_t* grid_dual);

/* Scaled matrix values Ktilde in the caller's CSR order (val_out[nnz]) read back from the K layout
   (from_transpose = 0) or from the explicit K' layout (from_transpose = 1).  HOST out.  Test hook
   for R1 and for "K' equals the CSC of K bit-exactly". */
int uc_lp_get_scaled_values(uc_lp* lp, int32_t from_transpose, double* val_out);

/* Host-only self-check of ingest step A1 (no GPU needed): builds the row / column permutations, the explicit
   transpose, both SELL-32 layouts and both attempt schedules (for `sched_ctas` CTAs of `warps_per_cta` consumer warps)
   exactly as uc_lp_create does, and verifies them entry by entry against the caller's CSR: stored entries are the
   caller's, in the caller's order (K' rows in ascending caller row index), padding is (0, 0.0), every slice is scheduled
   exactly once as consecutive chunks, and the slices of a CTA form one contiguous range (CTA c's before CTA c+1's).
   Returns UC_OK, or UC_ERR_INVALID with the violated property in uc_last_error(). */
int uc_host_layout_selftest(int64_t m, int64_t n, int64_t nnz, const int64_t* row_ptr, const int32_t* col_idx, const double* val,
                            int32_t sell_window, int32_t long_row_threshold, int32_t sched_ctas, int32_t warps_per_cta);

/* Test hook for ingest step A1 (needs the GPU): rebuilds the permutations, both layouts (16-bit offsets included) and both
   attempt schedules from the caller's CSR with the HOST builders that uc_host_layout_selftest verifies, downloads what
   the handle holds on the device and compares bit for bit (the matrix values only if the handle was created with
   ruiz_iters = 0 and pc_alpha = 0: uc_lp_create scales them in place).  UC_OK, or UC_ERR_INVALID naming the first
   difference.  With host_ingest = 0 this is the parity test of the device-side ingest kernels. */
int uc_lp_compare_layout(uc_lp* lp, int64_t m, int64_t n, int64_t nnz, const int64_t* row_ptr, const int32_t* col_idx, const double* val);

/* Host evaluation of the double-double log / exp that the primal-weight update (R11) runs on the
   device (same source, csrc/uc_dd.cuh).  Test hooks: no GPU needed. */
double uc_host_log_rounded(double a);
double uc_host_exp_rounded(double x);

#ifdef __cplusplus
}
#endif
#endif /* UC_PDHG_HOOKS_H */
