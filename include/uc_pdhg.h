/*
 * uc_pdhg.h -- C ABI of the B200-native restarted PDHG (PDLP-style) LP solver.
 *
 * What it solves (BASELINE.json north_star; "One solver employs the PDHG algorithm to
 * solve the relaxed linear problem using a GPU"):
 *
 *        min c'x   s.t.   (A x)_i = b_i  (sense 'E')  or  (A x)_i >= b_i  (sense 'G'),   l <= x <= u
 *
 * i.e. the LP relaxation of the DC unit-commitment MILP (commitment relaxed to [0,1], or fixed by
 * l = u).  The algorithm is fixed step by step in DESIGN.md "Readings" R1..R14 (SURVEY.md 8(c)
 * O0..O7): Ruiz + Pock-Chambolle diagonal preconditioning, adaptive-step PDHG with the
 * extrapolation 2x+ - x, eta-weighted averaging, KKT-based restarts, primal-weight update,
 * relative-KKT termination.  Default stopping parameters are the paper's (PAPER.md l.66, l.91:
 * iteration limit 100,000; convergence tolerance 1e-4; absolute feasibility tolerance 1e-5 opt-in).
 * uc_pdhg_cancel is the hook for Algorithm 1: "Terminate the other solver".
 *
 * Conventions
 *   - every call returns 0 on success, or a negative uc_error; no exception or abort crosses the ABI;
 *     uc_last_error() returns the text of the last failure on this thread.
 *   - all array arguments are HOST pointers unless the name says `_device`; the library copies
 *     what it needs; the caller keeps ownership of everything it passes in.
 *   - all device memory, streams, events and CUDA graphs are owned by the handle and released
 *     by uc_lp_destroy.  The handle is bound to one device.
 *   - there is no CPU fallback: every call that computes fails with UC_ERR_CUDA without a GPU.
 *   - dual sign convention: Lagrangian c'x - y'(A x - b), so y_i >= 0 on 'G' rows.
 *   - uc_pdhg_solve* is blocking and not re-entrant per handle; uc_pdhg_cancel may be called
 *     from any thread at any time.
 *   - measurement and test hooks of the same library (kernel timing, timeline, layout checks) are declared in
 *     uc_pdhg_hooks.h, not here: this header is the product ABI.
 */
#ifndef UC_PDHG_H
#define UC_PDHG_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct uc_lp uc_lp; /* opaque */

enum uc_error {
    UC_OK = 0,
    UC_ERR_INVALID = -1, /* bad argument (NULL, negative size, column out of range, duplicate entry, l > u, NaN) */
    UC_ERR_CUDA = -2,    /* a CUDA runtime call or kernel failed (includes: no device) */
    UC_ERR_NOMEM = -3,   /* host or device allocation failed */
    UC_ERR_BUSY = -4,    /* a solve is already running on this handle */
    UC_ERR_INTERNAL = -5 /* a failure inside the library that is none of the above (e.g. a helper thread could not be started) */
};

enum uc_status {
    UC_OPTIMAL = 0,         /* relative KKT test passed (R12) */
    UC_ITERATION_LIMIT = 1, /* iter_limit attempts done (also the status of every fixed_iterations run) */
    UC_CANCELLED = 2,       /* uc_pdhg_cancel was seen */
    UC_TIME_LIMIT = 3,
    UC_NUMERICAL_ERROR = 4  /* a non-finite step size or KKT term appeared */
};

/* ------------------------------------------------------------------------------------------ create */
typedef struct {
    int32_t device;             /* CUDA device ordinal; -1 = current device */
    int32_t ruiz_iters;         /* 10  (R1) */
    double pc_alpha;            /* 1.0; 0 = no Pock-Chambolle pass (R1) */
    int32_t sell_window;        /* rows per length-sorting window of the sliced-ELL layout; 4096 */
    int32_t long_row_threshold; /* rows longer than this leave the sliced-ELL part (warp-per-row); 32 */
    int32_t keep_source_map;    /* 1: keep the slot -> CSR position maps on the host (uc_lp_get_scaled_values); 0 */
    int32_t index_compression;  /* 1 (default): slices whose column indices span < 2^16 store them as 16-bit offsets from
                                   the slice's smallest index (SURVEY.md 8(f) NEXT-4, 2 bytes per entry less per matrix
                                   copy; results are bit-identical); 0: 32-bit indices everywhere */
    int32_t host_ingest;        /* 0 (default): step A1 -- permutations, explicit transpose, both layouts -- runs as kernels on
                                   the device from one copy of the caller's CSR; 1: the host builders (the checker's code)
                                   build them and upload.  Both give the same layouts bit for bit (uc_lp_compare_layout) */
    int32_t max_ctas;           /* 0 (default): the kernels of this handle may use every SM.  > 0: at most this many CTAs per
                                   kernel -- for LPs solved SIDE BY SIDE (uc_pdhg_solve_batch, the paper's 45 scenarios): a
                                   mid-size LP spread over all SMs has one slice per warp and leaves no SM to its neighbours;
                                   with a quarter of the SMs each, four of them run at once.  Results do not depend on it */
} uc_lp_options;

void uc_lp_default_options(uc_lp_options* opt);

/*
 * Ingest + transpose + preconditioning.
 *   m, n, nnz        rows, columns, nonzeros (any may be 0)
 *   row_ptr[m+1]     CSR row pointers, row_ptr[0] = 0, row_ptr[m] = nnz
 *   col_idx[nnz]     0-based column indices; order inside a row is free; duplicates are an error
 *   val[nnz]         finite values
 *   sense[m]         'E' or 'G'
 *   b[m], c[n]       finite;  l[n], u[n]: l <= u, -INFINITY / +INFINITY or |v| >= 1e20 = absent (R13)
 *   opt              NULL = defaults
 *   out              receives the handle
 * The call keeps its block of scratch device memory (the caller's CSR and the sort buffers of the ingest kernels, ~150
 * bytes per nonzero, at most 2 GiB) cached per device in the process for the next uc_lp_create; larger blocks are freed.
 */
int uc_lp_create(int64_t m, int64_t n, int64_t nnz, const int64_t* row_ptr, const int32_t* col_idx,
                 const double* val, const char* sense, const double* b, const double* c, const double* l,
                 const double* u, const uc_lp_options* opt, uc_lp** out);

/* Replace the bounds (fixed-commitment re-solves, north_star "relaxed to [0,1] or fixed"); the
   matrix, its scalings and the captured graph are kept.  l_new/u_new: host, length n. */
int uc_lp_update_bounds(uc_lp* lp, const double* l_new, const double* u_new);

/* Replace the objective (re-solves inside branch-and-bound and cost sweeps):
   c~ = c / D_c is rescaled with the scalings already on the device, ||c|| (R9) and omega0 = ||c~|| / ||q~|| (R2)
   are recomputed; the matrix, its scalings and the captured graph are kept.  c_new: host, length n, finite.
   The handle then behaves exactly like one created with c_new (the preconditioner does not depend on c). */
int uc_lp_update_objective(uc_lp* lp, const double* c_new);

void uc_lp_destroy(uc_lp* lp); /* NULL ok; must not race with a solve on the same handle */

/* Give back the scratch block that uc_lp_create keeps cached per device (see uc_lp_create: up to 2 GiB, ~1 GB after one
   config-3 create; no handle owns it, so uc_lp_destroy does not free it).  device: an ordinal, or -1 = every device.
   A block that a running uc_lp_create is using is left alone.  bytes_released (nullable) receives the bytes freed.
   For processes that share a GPU or create once and then solve for a long time; the next uc_lp_create simply allocates
   again.  uc_lp_info.scratch_cached_bytes reports what is held. */
int uc_release_scratch(int32_t device, int64_t* bytes_released);

/* ------------------------------------------------------------------------------------------- solve */
/* per-attempt trace record (R5): step size used, the bound eta_bar, the next step size, the three
   reductions, and whether the attempt was accepted */
typedef struct {
    double eta_used, eta_bar, eta_next, dx2, dy2, inter;
    int32_t accepted, pad_;
} uc_attempt_record;

/* per-check trace record (R8..R11) */
typedef struct {
    int64_t k;
    int32_t restart_kind; /* 0 none, 1 sufficient, 2 necessary, 3 artificial */
    int32_t candidate;    /* 0 current, 1 average */
    double omega_after, mu_c, mu_r, relkkt_cur, relkkt_avg;
} uc_check_record;

typedef struct {
    int64_t iter_limit;       /* 100000  PAPER.md l.66.  Any size: per-attempt tables grow while the solve runs */
    double eps_rel;           /* 1e-4    PAPER.md l.91 "convergence tolerance" */
    double eps_abs;           /* 1e-4 (= eps_rel, R12); 1e-5 reproduces the paper's extra knob (l.66) */
    double time_limit_s;      /* +inf */
    int32_t check_every;      /* 64 (R8) */
    int32_t pad_;
    int64_t fixed_iterations; /* 0 = off; F > 0: exactly F attempts, termination test off, current iterate returned (R14) */
    double beta_sufficient;   /* 0.2  (R10) */
    double beta_necessary;    /* 0.8  (R10) */
    double beta_artificial;   /* 0.36 (R10) */
    double weight_smoothing;  /* 0.5  (R11) */
    const double* x0;         /* nullable warm start, original space, length n (host; `_device` call: device) */
    const double* y0;         /* nullable warm start, original space, length m */
    void* stream;             /* cudaStream_t to run on; NULL = the handle's own stream */
    uc_attempt_record* attempt_trace; /* nullable HOST buffer, attempt_trace_cap records */
    int64_t attempt_trace_cap;
    uc_check_record* check_trace;     /* nullable HOST buffer, check_trace_cap records */
    int64_t check_trace_cap;
    double eta0;              /* 0 = R2's 1/max|K~|; > 0: step size of the first attempt (R2b) -- for re-solves: pass the eta and */
    double omega0;            /* omega that uc_pdhg_result returned for the neighbouring LP, next to its (x, y) as x0 / y0.     */
                              /* 0 = R2's ||c~||/||q~||; > 0: primal weight the run starts with (R2b).  Both must be finite, >= 0 */
} uc_pdhg_params;

void uc_pdhg_default_params(uc_pdhg_params* p);

typedef struct {
    int32_t status;           /* enum uc_status */
    int32_t returned_average; /* 1 if x, y are the averaged iterate */
    int64_t iterations;       /* attempts (each = one K' pass + one K pass, accepted or not) */
    int64_t accepted, restarts;
    double rel_kkt, rel_primal_res, rel_dual_res, rel_gap, primal_obj, dual_obj;
    double eta, omega;        /* final step size and primal weight */
    double solve_seconds;     /* host wall clock of this call */
    double loop_seconds;      /* device time (CUDA events) of the attempt loop incl. checks */
    int64_t attempt_records, check_records; /* records produced (may exceed the capacities given) */
    int64_t kernel_launches;  /* kernels of this library executed by the call (graph nodes included) */
} uc_pdhg_result;

/* Run restarted PDHG.  x_out[n], y_out[m]: HOST buffers receiving the returned point in the
   original space (nullable).  params NULL = defaults. */
int uc_pdhg_solve(uc_lp* lp, const uc_pdhg_params* params, double* x_out, double* y_out, uc_pdhg_result* result);

/* Same, with x_out / y_out / params->x0 / params->y0 being DEVICE pointers on the handle's device
   (the torch harness owns them); nothing but the result struct and the traces crosses PCIe. */
int uc_pdhg_solve_device(uc_lp* lp, const uc_pdhg_params* params, double* x_out_device, double* y_out_device,
                         uc_pdhg_result* result);

/* Batched solve of independent LPs (the paper's 45 scenarios): solves
   handles[0..count) concurrently, each on its own handle's stream, with up to max_concurrent (<= 0: 16) solves in
   flight, and returns when all are done.  Small LPs are bound by the two dependent kernel launches of an attempt
   (~6-8 us each), not by the GPU: solves in flight at the same time fill it.  Every result is bit-identical to the
   solve run alone.  params: one set for all (NULL = defaults); its stream / x0 / y0 / trace fields must be NULL.
   x_out[i] / y_out[i]: HOST buffers of handle i (the arrays or any entry may be NULL).  results[count].
   Returns 0, or the first failure (uc_last_error names the solve); uc_pdhg_cancel(handles[i]) stops solve i. */
int uc_pdhg_solve_batch(uc_lp* const* handles, int32_t count, const uc_pdhg_params* params, double* const* x_out,
                        double* const* y_out, uc_pdhg_result* results, int32_t max_concurrent);

/* Cancel, any thread, idempotent (Algorithm 1: "Terminate the other solver").
   - A solve is in flight on the handle: THAT solve returns UC_CANCELLED at its next check (within one check
     period).  The request is scoped to it: if the solve was already past its last check and returns with
     another status, the request is dropped -- it never leaks into a later solve on the handle.  (A request that arrives
     after the library has left the solve takes the second route, whatever the caller believed: uc_pdhg_cancel_clear.)
   - The handle is idle: the request is kept for the NEXT solve, which returns UC_CANCELLED at entry with
     iterations = 0 and x_out / y_out untouched -- so a cancel that lands just before the solve starts is not
     lost (the race of Algorithm 1).
   A cancel that races with the very start of a solve takes one of these two routes; both stop that solve. */
int uc_pdhg_cancel(uc_lp* lp);

/* Drop a cancel request that is being kept for the NEXT solve (second route above); a solve in flight is not affected.
   was_pending (nullable) receives 1 if there was one.  For callers that cancel from another thread and then reuse the
   handle: a cancel sent while the solve was returning on its own -- the caller saw its thread still alive, the library
   had already left the solve -- would otherwise stop the next, unrelated solve at entry.  Call it after the solve has
   returned with a status other than UC_CANCELLED (race.py does, after joining its solve thread). */
int uc_pdhg_cancel_clear(uc_lp* lp, int32_t* was_pending);

/* ------------------------------------------------------------------------------- introspection */
typedef struct {
    int64_t m, n, nnz;
    int64_t k_sell_slots, kt_sell_slots; /* stored slots (incl. padding) of the sliced-ELL parts */
    int64_t k_long_rows, kt_long_rows;   /* rows handled warp-per-row */
    int64_t k_long_nnz, kt_long_nnz;
    int64_t device_bytes;                /* device memory owned by the handle */
    double precondition_seconds;         /* device time of A2..A4 */
    double create_seconds;               /* host wall clock of uc_lp_create */
    double eta0, omega0;                 /* R2 */
    double norm_b, norm_c;               /* unscaled 2-norms used by R9 */
    int64_t bytes_per_attempt;           /* bytes one attempt streams in this layout */
    int64_t k_narrow_slots, kt_narrow_slots; /* stored slots whose column index is a 16-bit offset (index_compression) */
    int64_t scratch_cached_bytes;        /* device memory the PROCESS keeps cached on this handle's device for the next
                                            uc_lp_create (not owned by the handle; see uc_release_scratch) */
} uc_lp_info;

int uc_lp_get_info(const uc_lp* lp, uc_lp_info* info);

/* Diagonal scalings of R1, original row/column order: K = diag(Dr) Ktilde diag(Dc).  HOST out. */
int uc_lp_get_scaling(uc_lp* lp, double* Dr_out, double* Dc_out);

/* out = Ktilde v (transpose = 0; v[n], out[m]) or Ktilde' v (transpose = 1; v[m], out[n]) over the handle's own layouts
   with the row traversal of the CHECK kernels (A11); HOST in/out, original order.  Test hook for the layouts and the
   adjoint identity.  (The pipelines of the attempt kernels are covered by the one-attempt test of
   tests/test_gpu_parity.py, which runs k_primal + k_dual once from a warm start through uc_pdhg_solve.) */
int uc_lp_spmv(uc_lp* lp, int32_t transpose, const double* v, double* out);

/* uc_lp_spmv for callers that must not allocate device memory.
 *
 * Who that is: code that runs beside latency-critical work on the same GPU (cudaMalloc and cudaFree synchronise the
 * whole device, so one call stalls every other stream -- a racing PDHG solve, included); code inside a
 * process whose device memory has all been handed to a pool or to another library's caching allocator, where a raw
 * cudaMalloc fails although memory is "free"; and code under a no-allocation rule after start-up (fixed memory budget,
 * certified or long-running services that must not fragment or grow).  uc_lp_spmv allocates four temporary vectors per
 * call; this entry point allocates nothing and calls no cudaMalloc, cudaFree or other allocating routine.
 *
 * It computes the same product with the same kernels, so the result equals uc_lp_spmv's bit for bit:
 *   out = Ktilde v (transpose = 0; v[n], out[m])  or  Ktilde' v (transpose = 1; v[m], out[n]),  original order.
 * v_device / out_device are DEVICE pointers on the handle's device, owned by the caller; they must not overlap.  The two
 * intermediate vectors (v and the product in the layout's own order) live in ONE fixed array inside the library, 2 MiB
 * on every GPU that has loaded it, held until the process exits.
 *
 * Limit: round m and n up to multiples of 32; their sum must not exceed UC_SPMV_STATIC_MAX_DOUBLES (262,144 -- config 0
 * and config 1 of BASELINE.json fit, the larger ones do not).  A larger handle gets UC_ERR_INVALID and a message naming
 * the limit; nothing is launched.  Other errors as uc_lp_spmv (UC_ERR_BUSY while a solve runs on the handle).
 *
 * Stream order: the three kernels are enqueued on `stream` (cudaStream_t; NULL = the handle's own stream) and the call
 * returns without waiting; out_device is complete when the stream reaches that point.
 *
 * Sharing: the array is one per GPU, shared by every handle, stream and host thread, and it keeps whatever the last call
 * wrote.  Nothing in it needs to start at zero (every entry that is read has been written earlier in the same call), so
 * back-to-back calls on ONE stream are safe.  Two calls that can overlap on the GPU -- different streams, or different
 * threads using different streams -- race on it and both results are garbage: order them yourself (one stream, or an
 * event between them).
 *
 * First call on a device: it looks up the array's device address (cudaGetSymbolAddress, with the handle's device made
 * current) and remembers it per device.  Make that first call during set-up, before any stream capture is begun. */
#define UC_SPMV_STATIC_MAX_DOUBLES 262144
int uc_lp_spmv_static(uc_lp* lp, int32_t transpose, const double* v_device, double* out_device, void* stream);

const char* uc_last_error(void);

#ifdef __cplusplus
}
#endif
#endif /* UC_PDHG_H */
