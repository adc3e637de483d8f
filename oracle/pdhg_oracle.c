/*
 * pdhg_oracle.c -- TEST INFRASTRUCTURE, NOT PRODUCT.
 *
 * A plain, slow, sequential CPU fp64 implementation of the restarted PDHG (PDLP-style) LP
 * solver that BASELINE.json `north_star` names as the GPU half of the paper's concurrent
 * solver ("One solver employs the PDHG algorithm to solve the relaxed linear
 * problem using a GPU"; l.66/l.91: iteration limit 100,000, tolerances 1e-5 / 1e-4).
 * The paper prints no PDHG equations; the algorithm below is the reading fixed in
 * DESIGN.md section "Readings" (R1..R14), i.e. SURVEY.md 8(c) O0..O7, followed step by step
 * in that order and notation.  One thread, no blocking, no fusion, no reordering.
 *
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs
 * may build, load or call this file.  It shares no code, header, table or helper with
 * paper_2607_03627_b200/ (the CUDA path) and neither includes the other.
 *
 * Pins (tests/test_oracle_pins.py; DESIGN.md section 4 lists which reading each one covers): brute-force vertex
 * enumeration (n <= 8), HiGHS objective, box-only and merit-order closed forms, the worked 1x1 step example and
 * the worked 2x2 preconditioner example of SURVEY.md 8(c) (tests/golden/), sigma_max <= 1 after Pock-Chambolle,
 * Fejer monotonicity with a frozen step, explicit weighted averages, KKT / complementary slackness.  The restart
 * rule and the primal-weight update (R10, R11) are pinned by the worked restart example
 * (tests/golden/restart_1x1.txt, derived by hand in DESIGN.md: all three restart kinds, restarts to the average,
 * a moving primal weight) and by an independent dense-numpy recomputation of every decision and of the closed
 * form omega_new = (Dy/Dx)^theta omega^(1-theta) from the iterates dumped at each check (tests/helpers.py
 * restart_replay).  Every function of this file has a pin.
 *
 * Numerics: IEEE fp64, round to nearest, compiled with -ffp-contract=off.  SpMV row sums run
 * in CSR order; every long reduction (norm, dot, objective) is Neumaier-compensated so that
 * the oracle sums more accurately than the GPU's tree reductions.
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

#define ORACLE_OPTIMAL 0
#define ORACLE_ITERATION_LIMIT 1
#define ORACLE_NUMERICAL_ERROR 4

typedef struct {
    int64_t iter_limit;        /* 100000 */
    double eps_rel;            /* 1e-4   ("convergence tolerance") */
    double eps_abs;            /* = eps_rel by default (R12) */
    int32_t check_every;       /* 64 (R8) */
    int32_t ruiz_iters;        /* 10 (R1) */
    double pc_alpha;           /* 1.0; 0 = Pock-Chambolle off (R1) */
    int64_t fixed_iterations;  /* 0 = off; F > 0: exactly F attempts, termination test off (R14) */
    double beta_sufficient;    /* 0.2  (R10) */
    double beta_necessary;     /* 0.8  (R10) */
    double beta_artificial;    /* 0.36 (R10) */
    double weight_smoothing;   /* 0.5  (R11) */
    int32_t restarts_enabled;  /* 1; 0 = checks still run, never restart (test hook) */
    int32_t pad_;
    double frozen_eta;         /* 0 = adaptive rule (R5); > 0: constant step, always accept (test hook) */
    double eta0;               /* 0 = R2's 1/max|K~|; > 0: the step size the first attempt uses (R2b: state carried from an earlier solve) */
    double omega0;             /* 0 = R2's ||c~||/||q~||; > 0: the primal weight the run starts with (R2b) */
} oracle_params;

typedef struct {
    int32_t status;
    int32_t returned_average;
    int64_t iterations, accepted, restarts;
    double rel_kkt, rel_primal_res, rel_dual_res, rel_gap, primal_obj, dual_obj;
    double eta, omega;         /* final step size and primal weight */
} oracle_result;

/* per-attempt trace record (R5) */
typedef struct {
    double eta_used, eta_bar, eta_next, dx2, dy2, inter;
    int32_t accepted, pad_;
} oracle_attempt;

/* per-check trace record (R8..R11) */
typedef struct {
    int64_t k;
    int32_t restart_kind;      /* 0 none, 1 sufficient, 2 necessary, 3 artificial */
    int32_t candidate;         /* 0 current, 1 average */
    double omega_after, mu_c, mu_r, relkkt_cur, relkkt_avg;
} oracle_check;

void oracle_default_params(oracle_params* p) {
    p->iter_limit = 100000; p->eps_rel = 1e-4; p->eps_abs = 1e-4; p->check_every = 64;
    p->ruiz_iters = 10; p->pc_alpha = 1.0; p->fixed_iterations = 0;
    p->beta_sufficient = 0.2; p->beta_necessary = 0.8; p->beta_artificial = 0.36;
    p->weight_smoothing = 0.5; p->restarts_enabled = 1; p->pad_ = 0; p->frozen_eta = 0.0;
    p->eta0 = 0.0; p->omega0 = 0.0;
}

/* ---------------------------------------------------------------- compensated sums */
typedef struct { double s, c; } nsum;                 /* Neumaier running sum */
static void ns_add(nsum* a, double v) {
    double t = a->s + v;
    if (fabs(a->s) >= fabs(v)) a->c += (a->s - t) + v; else a->c += (v - t) + a->s;
    a->s = t;
}
static double ns_get(const nsum* a) { return a->s + a->c; }

static double dot(int64_t n, const double* a, const double* b) {
    nsum s = {0, 0};
    for (int64_t i = 0; i < n; ++i) ns_add(&s, a[i] * b[i]);
    return ns_get(&s);
}
static double norm2sq(int64_t n, const double* a) { return dot(n, a, a); }
static double clampd(double v, double lo, double hi) { return v < lo ? lo : (v > hi ? hi : v); }

/* ---------------------------------------------------------------- SpMV (CSR order) */
/* out = K v  (K m x n in CSR) */
void oracle_spmv(int64_t m, const int64_t* row_ptr, const int32_t* col, const double* val,
                 const double* v, double* out) {
    for (int64_t i = 0; i < m; ++i) {
        double s = 0.0;
        for (int64_t p = row_ptr[i]; p < row_ptr[i + 1]; ++p) s += val[p] * v[col[p]];
        out[i] = s;
    }
}
/* out = K' y, written out as the definition (K'y)_j = sum_i K_ij y_i: a column-wise scatter over
   the same CSR -- no transposed copy is ever built here. */
void oracle_spmv_t(int64_t m, int64_t n, const int64_t* row_ptr, const int32_t* col, const double* val,
                   const double* y, double* out) {
    for (int64_t j = 0; j < n; ++j) out[j] = 0.0;
    for (int64_t i = 0; i < m; ++i)
        for (int64_t p = row_ptr[i]; p < row_ptr[i + 1]; ++p) out[col[p]] += val[p] * y[i];
}

/* ---------------------------------------------------------------- R1 preconditioning (O1) */
/* Ruiz (inf-norm) x ruiz_iters, then one Pock-Chambolle pass with exponent alpha (north_star (a)).
   val_s <- scaled values (same pattern); Dr[m], Dc[n] with K = diag(Dr) Ktilde diag(Dc). */
void oracle_precondition(int64_t m, int64_t n, const int64_t* row_ptr, const int32_t* col,
                         const double* val, int32_t ruiz_iters, double pc_alpha,
                         double* val_s, double* Dr, double* Dc) {
    int64_t nnz = row_ptr[m];
    double* r = (double*)malloc(sizeof(double) * (size_t)(m > 0 ? m : 1));
    double* s = (double*)malloc(sizeof(double) * (size_t)(n > 0 ? n : 1));
    for (int64_t p = 0; p < nnz; ++p) val_s[p] = val[p];
    for (int64_t i = 0; i < m; ++i) Dr[i] = 1.0;
    for (int64_t j = 0; j < n; ++j) Dc[j] = 1.0;
    for (int pass = 0; pass < ruiz_iters + (pc_alpha > 0.0 ? 1 : 0); ++pass) {
        int ruiz = pass < ruiz_iters;
        for (int64_t i = 0; i < m; ++i) r[i] = 0.0;
        for (int64_t j = 0; j < n; ++j) s[j] = 0.0;
        for (int64_t i = 0; i < m; ++i)
            for (int64_t p = row_ptr[i]; p < row_ptr[i + 1]; ++p) {
                double a = fabs(val_s[p]);
                if (ruiz) {                         /* r_i = max_j |K_ij|, s_j = max_i |K_ij| */
                    if (a > r[i]) r[i] = a;
                    if (a > s[col[p]]) s[col[p]] = a;
                } else {                            /* r_i = sum_j |K_ij|^(2-alpha), s_j = sum_i |K_ij|^alpha */
                    r[i] += (pc_alpha == 1.0) ? a : pow(a, 2.0 - pc_alpha);
                    s[col[p]] += (pc_alpha == 1.0) ? a : pow(a, pc_alpha);
                }
            }
        for (int64_t i = 0; i < m; ++i) r[i] = (r[i] > 0.0) ? sqrt(r[i]) : 1.0;   /* empty row -> 1 */
        for (int64_t j = 0; j < n; ++j) s[j] = (s[j] > 0.0) ? sqrt(s[j]) : 1.0;   /* empty col -> 1 */
        for (int64_t i = 0; i < m; ++i)
            for (int64_t p = row_ptr[i]; p < row_ptr[i + 1]; ++p) val_s[p] = val_s[p] / (r[i] * s[col[p]]);
        for (int64_t i = 0; i < m; ++i) Dr[i] *= r[i];
        for (int64_t j = 0; j < n; ++j) Dc[j] *= s[j];
    }
    free(r); free(s);
}

/* ---------------------------------------------------------------- scaled problem */
typedef struct {
    int64_t m, n;
    const int64_t* row_ptr; const int32_t* col;
    double* val;                    /* Ktilde */
    const unsigned char* sense;
    double *q, *c, *l, *u;          /* scaled */
    double *Dr, *Dc;
    double norm_q, norm_c;          /* UNSCALED ||q||_2, ||c||_2 (R9) */
} sprob;

typedef struct { double rp2_s, rd2_s, rp2_u, rd2_u, pobj, dobj; } kkt_terms;

/* R9 (O4): residuals, objectives of the scaled point (x,y); scratch a[m], rho[n]. */
static void kkt_eval(const sprob* P, const double* x, const double* y, double* a, double* rho, kkt_terms* t) {
    nsum rp_s = {0, 0}, rp_u = {0, 0}, rd_s = {0, 0}, rd_u = {0, 0}, po = {0, 0}, dob = {0, 0};
    oracle_spmv(P->m, P->row_ptr, P->col, P->val, x, a);
    for (int64_t i = 0; i < P->m; ++i) {
        double ai = a[i] - P->q[i];
        double r = (P->sense[i] == 'E') ? ai : (ai < 0.0 ? ai : 0.0);
        ns_add(&rp_s, r * r);
        ns_add(&rp_u, (P->Dr[i] * r) * (P->Dr[i] * r));
        ns_add(&dob, P->q[i] * y[i]);
    }
    oracle_spmv_t(P->m, P->n, P->row_ptr, P->col, P->val, y, rho);
    for (int64_t j = 0; j < P->n; ++j) {
        double rj = P->c[j] - rho[j];
        double lam = 0.0;
        if (rj > 0.0 && isfinite(P->l[j])) lam = rj;
        if (rj < 0.0 && isfinite(P->u[j])) lam = rj;
        double rd = rj - lam;
        ns_add(&rd_s, rd * rd);
        ns_add(&rd_u, (P->Dc[j] * rd) * (P->Dc[j] * rd));
        ns_add(&po, P->c[j] * x[j]);
        if (lam > 0.0) ns_add(&dob, P->l[j] * lam);
        if (lam < 0.0) ns_add(&dob, P->u[j] * lam);
    }
    t->rp2_s = ns_get(&rp_s); t->rp2_u = ns_get(&rp_u);
    t->rd2_s = ns_get(&rd_s); t->rd2_u = ns_get(&rd_u);
    t->pobj = ns_get(&po); t->dobj = ns_get(&dob);
}
static double kkt_omega(const kkt_terms* t, double w) {   /* restart measure KKT_omega (R9) */
    double g = t->pobj - t->dobj;
    return sqrt(w * w * t->rp2_s + t->rd2_s / (w * w) + g * g);
}
static void rel_terms(const sprob* P, const kkt_terms* t, double* rp, double* rd, double* gap) {
    *rp = sqrt(t->rp2_u) / (1.0 + P->norm_q);
    *rd = sqrt(t->rd2_u) / (1.0 + P->norm_c);
    *gap = fabs(t->pobj - t->dobj) / (1.0 + fabs(t->pobj) + fabs(t->dobj));
}
static double rel_kkt(const sprob* P, const kkt_terms* t) {
    double a, b, c; rel_terms(P, t, &a, &b, &c);
    double r = a > b ? a : b; return r > c ? r : c;
}
static int converged(const sprob* P, const kkt_terms* t, double ea, double er) {   /* R12 */
    return sqrt(t->rp2_u) <= ea + er * P->norm_q && sqrt(t->rd2_u) <= ea + er * P->norm_c &&
           fabs(t->pobj - t->dobj) <= ea + er * (fabs(t->pobj) + fabs(t->dobj));
}

/* Unscaled-space KKT terms written directly from the LP's definition (no scaling involved):
   out[0]=||r_p||_2, out[1]=||r_d||_2, out[2]=c'x, out[3]=dual objective, out[4]=relKKT (R9). */
void oracle_kkt_unscaled(int64_t m, int64_t n, const int64_t* row_ptr, const int32_t* col, const double* val,
                         const unsigned char* sense, const double* b, const double* c, const double* l,
                         const double* u, const double* x, const double* y, double* out) {
    double* a = (double*)malloc(sizeof(double) * (size_t)(m > 0 ? m : 1));
    double* g = (double*)malloc(sizeof(double) * (size_t)(n > 0 ? n : 1));
    nsum rp = {0, 0}, rd = {0, 0}, po = {0, 0}, dob = {0, 0};
    oracle_spmv(m, row_ptr, col, val, x, a);
    for (int64_t i = 0; i < m; ++i) {
        double ai = a[i] - b[i];
        double r = (sense[i] == 'E') ? ai : (ai < 0.0 ? ai : 0.0);
        ns_add(&rp, r * r); ns_add(&dob, b[i] * y[i]);
    }
    oracle_spmv_t(m, n, row_ptr, col, val, y, g);
    for (int64_t j = 0; j < n; ++j) {
        double rj = c[j] - g[j], lam = 0.0;
        if (rj > 0.0 && isfinite(l[j])) lam = rj;
        if (rj < 0.0 && isfinite(u[j])) lam = rj;
        ns_add(&rd, (rj - lam) * (rj - lam)); ns_add(&po, c[j] * x[j]);
        if (lam > 0.0) ns_add(&dob, l[j] * lam);
        if (lam < 0.0) ns_add(&dob, u[j] * lam);
    }
    double nq = sqrt(norm2sq(m, b)), nc = sqrt(norm2sq(n, c));
    out[0] = sqrt(ns_get(&rp)); out[1] = sqrt(ns_get(&rd)); out[2] = ns_get(&po); out[3] = ns_get(&dob);
    double e1 = out[0] / (1.0 + nq), e2 = out[1] / (1.0 + nc);
    double e3 = fabs(out[2] - out[3]) / (1.0 + fabs(out[2]) + fabs(out[3]));
    out[4] = e1 > e2 ? (e1 > e3 ? e1 : e3) : (e2 > e3 ? e2 : e3);
    free(a); free(g);
}

static double* dalloc(int64_t k) { return (double*)calloc((size_t)(k > 0 ? k : 1), sizeof(double)); }

/* ---------------------------------------------------------------- the solver (O2..O7) */
/*
 * All array arguments are caller-owned host memory.  x0/y0 (nullable): warm start in the
 * ORIGINAL space.  x_out[n], y_out[m]: returned point, original space.  Optional traces:
 * att[att_cap], chk[chk_cap] (counts written to *n_att, *n_chk; records beyond capacity are
 * dropped); dump_x[dump_cap*n], dump_y[dump_cap*m]: the SCALED current iterate after each of
 * the first dump_cap attempts; avg_x[n], avg_y[m], *avg_w: final scaled weighted sums / w.
 * Dr_out[m], Dc_out[n] (nullable): the scalings used.
 * Check dumps (nullable, TRACE ONLY -- they read the state, they never change it): for each of the first
 * cdump_cap checks, cdump_x[i*n..], cdump_y[i*m..] = the SCALED current iterate as the check sees it (before any
 * restart is applied), cdump_ax / cdump_ay = the SCALED average x_sum/w, y_sum/w (the current iterate if w = 0),
 * cdump_w[i] = w.  They let a test recompute every restart decision and primal-weight update (R10, R11) from
 * the iterates with its own algebra.
 * Returns 0, or -1 on bad arguments.
 */
int oracle_pdhg_solve(int64_t m, int64_t n, const int64_t* row_ptr, const int32_t* col, const double* val,
                      const unsigned char* sense, const double* b, const double* c, const double* l,
                      const double* u, const oracle_params* prm, const double* x0, const double* y0,
                      double* x_out, double* y_out, oracle_result* res,
                      oracle_attempt* att, int64_t att_cap, int64_t* n_att,
                      oracle_check* chk, int64_t chk_cap, int64_t* n_chk,
                      double* dump_x, double* dump_y, int64_t dump_cap,
                      double* avg_x, double* avg_y, double* avg_w,
                      double* Dr_out, double* Dc_out,
                      double* cdump_x, double* cdump_y, double* cdump_ax, double* cdump_ay, double* cdump_w,
                      int64_t cdump_cap) {
    if (m < 0 || n < 0 || !prm || !res || prm->check_every <= 0) return -1;
    int64_t nnz = row_ptr[m];
    sprob P; memset(&P, 0, sizeof P);
    P.m = m; P.n = n; P.row_ptr = row_ptr; P.col = col; P.sense = sense;
    P.val = dalloc(nnz); P.Dr = dalloc(m); P.Dc = dalloc(n);
    P.q = dalloc(m); P.c = dalloc(n); P.l = dalloc(n); P.u = dalloc(n);

    /* R1 (O1): scale the problem */
    oracle_precondition(m, n, row_ptr, col, val, prm->ruiz_iters, prm->pc_alpha, P.val, P.Dr, P.Dc);
    for (int64_t i = 0; i < m; ++i) P.q[i] = b[i] / P.Dr[i];
    for (int64_t j = 0; j < n; ++j) {
        P.c[j] = c[j] / P.Dc[j];
        P.l[j] = (l[j] <= -1e20) ? -INFINITY : l[j] * P.Dc[j];      /* R13: |bound| >= 1e20 = absent */
        P.u[j] = (u[j] >= 1e20) ? INFINITY : u[j] * P.Dc[j];
    }
    P.norm_q = sqrt(norm2sq(m, b)); P.norm_c = sqrt(norm2sq(n, c));
    if (Dr_out) memcpy(Dr_out, P.Dr, sizeof(double) * (size_t)m);
    if (Dc_out) memcpy(Dc_out, P.Dc, sizeof(double) * (size_t)n);

    double *x = dalloc(n), *y = dalloc(m), *xn = dalloc(n), *yn = dalloc(m), *xbar = dalloc(n);
    double *xsum = dalloc(n), *ysum = dalloc(m), *xavg = dalloc(n), *yavg = dalloc(m);
    double *xr = dalloc(n), *yr = dalloc(m);
    double *g = dalloc(n), *kx = dalloc(m), *dxv = dalloc(n), *kdx = dalloc(m);
    double *sa = dalloc(m), *srho = dalloc(n);

    /* R2 (O2): initial point, step size, primal weight */
    for (int64_t j = 0; j < n; ++j) x[j] = clampd(x0 ? x0[j] * P.Dc[j] : 0.0, P.l[j], P.u[j]);
    for (int64_t i = 0; i < m; ++i) {
        double v = y0 ? y0[i] * P.Dr[i] : 0.0;
        y[i] = (sense[i] == 'G' && v < 0.0) ? 0.0 : v;
    }
    double kmax = 0.0;
    for (int64_t p = 0; p < nnz; ++p) if (fabs(P.val[p]) > kmax) kmax = fabs(P.val[p]);
    double eta = (kmax > 0.0) ? 1.0 / kmax : 1.0;
    if (prm->frozen_eta > 0.0) eta = prm->frozen_eta;
    double ncs = sqrt(norm2sq(n, P.c)), nqs = sqrt(norm2sq(m, P.q));
    double omega = (ncs > 1e-10 && nqs > 1e-10) ? ncs / nqs : 1.0;
    /* R2b: a re-solve may start from the step size and primal weight an
       earlier solve of a neighbouring LP ended with, like it starts from its (x, y); everything else is R2..R14 unchanged */
    if (prm->eta0 > 0.0 && prm->frozen_eta <= 0.0) eta = prm->eta0;
    if (prm->omega0 > 0.0) omega = prm->omega0;

    int64_t k = 0, t0 = 0, accepted = 0, restarts = 0, na = 0, nc = 0;
    double w = 0.0, mu_prev = INFINITY;
    kkt_terms Tr, Tcur, Tavg;
    memcpy(xr, x, sizeof(double) * (size_t)n); memcpy(yr, y, sizeof(double) * (size_t)m);
    kkt_eval(&P, xr, yr, sa, srho, &Tr);                      /* components of the restart point z_r = z^0 */

    int fixed = prm->fixed_iterations > 0;
    int64_t limit = fixed ? prm->fixed_iterations : prm->iter_limit;
    int status = ORACLE_ITERATION_LIMIT, ret_avg = 0;
    Tcur = Tr; Tavg = Tr;
    int have_avg = 0;

    while (k < limit) {
        /* ---- R3..R6 (O3): one attempt */
        k += 1;
        double tau = eta / omega, sig = eta * omega;
        oracle_spmv_t(m, n, row_ptr, col, P.val, y, g);                            /* g = K'y */
        for (int64_t j = 0; j < n; ++j) {
            xn[j] = clampd(x[j] - tau * (P.c[j] - g[j]), P.l[j], P.u[j]);          /* primal step + projection */
            xbar[j] = 2.0 * xn[j] - x[j];                                          /* extrapolation */
        }
        oracle_spmv(m, row_ptr, col, P.val, xbar, kx);                             /* K xbar */
        for (int64_t i = 0; i < m; ++i) {
            double v = y[i] + sig * (P.q[i] - kx[i]);                              /* dual step */
            yn[i] = (sense[i] == 'G' && v < 0.0) ? 0.0 : v;                        /* projection on Y */
        }
        nsum sdx = {0, 0}, sdy = {0, 0}, sin_ = {0, 0};
        for (int64_t j = 0; j < n; ++j) { dxv[j] = xn[j] - x[j]; ns_add(&sdx, dxv[j] * dxv[j]); }
        oracle_spmv(m, row_ptr, col, P.val, dxv, kdx);                             /* K dx (own SpMV) */
        for (int64_t i = 0; i < m; ++i) {
            double dy = yn[i] - y[i];
            ns_add(&sdy, dy * dy); ns_add(&sin_, dy * kdx[i]);
        }
        double dx2 = ns_get(&sdx), dy2 = ns_get(&sdy), inter = fabs(ns_get(&sin_));
        double N = omega * dx2 + dy2 / omega;
        double eta_bar = (inter > 0.0) ? N / (2.0 * inter) : INFINITY;             /* R5 */
        double grow = (1.0 + pow((double)(k + 1), -0.6)) * eta;
        double eta_next = isinf(eta_bar) ? grow : fmin((1.0 - pow((double)(k + 1), -0.3)) * eta_bar, grow);
        int accept = eta <= eta_bar;
        if (prm->frozen_eta > 0.0) { accept = 1; eta_next = eta; }
        if (att && na < att_cap) {
            oracle_attempt* r = &att[na];
            r->eta_used = eta; r->eta_bar = eta_bar; r->eta_next = eta_next;
            r->dx2 = dx2; r->dy2 = dy2; r->inter = inter; r->accepted = accept; r->pad_ = 0;
        }
        na += 1;
        if (accept) {                                                              /* R6 */
            for (int64_t j = 0; j < n; ++j) { x[j] = xn[j]; xsum[j] += eta * xn[j]; }
            for (int64_t i = 0; i < m; ++i) { y[i] = yn[i]; ysum[i] += eta * yn[i]; }
            w += eta; accepted += 1;
        }
        eta = eta_next;
        if (dump_x && k <= dump_cap) memcpy(dump_x + (k - 1) * n, x, sizeof(double) * (size_t)n);
        if (dump_y && k <= dump_cap) memcpy(dump_y + (k - 1) * m, y, sizeof(double) * (size_t)m);
        if (!isfinite(eta) || !(eta > 0.0)) { status = ORACLE_NUMERICAL_ERROR; break; }

        /* ---- R8 (O4): check cadence */
        int do_check = (k % prm->check_every == 0) || (!fixed && k == limit);
        if (!do_check) continue;
        kkt_eval(&P, x, y, sa, srho, &Tcur);
        have_avg = w > 0.0;
        if (have_avg) {
            for (int64_t j = 0; j < n; ++j) xavg[j] = xsum[j] / w;
            for (int64_t i = 0; i < m; ++i) yavg[i] = ysum[i] / w;
            kkt_eval(&P, xavg, yavg, sa, srho, &Tavg);
        }
        if (nc < cdump_cap) {                                  /* trace only */
            if (cdump_x) memcpy(cdump_x + nc * n, x, sizeof(double) * (size_t)n);
            if (cdump_y) memcpy(cdump_y + nc * m, y, sizeof(double) * (size_t)m);
            if (cdump_ax) memcpy(cdump_ax + nc * n, have_avg ? xavg : x, sizeof(double) * (size_t)n);
            if (cdump_ay) memcpy(cdump_ay + nc * m, have_avg ? yavg : y, sizeof(double) * (size_t)m);
            if (cdump_w) cdump_w[nc] = w;
        }
        double rk_cur = rel_kkt(&P, &Tcur), rk_avg = have_avg ? rel_kkt(&P, &Tavg) : INFINITY;
        if (!isfinite(rk_cur)) { status = ORACLE_NUMERICAL_ERROR; break; }
        /* ---- R12 (O5): termination */
        if (!fixed) {
            if (have_avg && converged(&P, &Tavg, prm->eps_abs, prm->eps_rel)) { status = ORACLE_OPTIMAL; ret_avg = 1; }
            else if (converged(&P, &Tcur, prm->eps_abs, prm->eps_rel)) { status = ORACLE_OPTIMAL; ret_avg = 0; }
        }
        /* ---- R10, R11 (O6): restart test and primal weight */
        oracle_check rec; memset(&rec, 0, sizeof rec);
        rec.k = k; rec.relkkt_cur = rk_cur; rec.relkkt_avg = rk_avg;
        if (status != ORACLE_OPTIMAL && k < limit) {
            int cand_avg = have_avg && (kkt_omega(&Tavg, omega) < kkt_omega(&Tcur, omega));
            const kkt_terms* Tc = cand_avg ? &Tavg : &Tcur;
            double mu_c = kkt_omega(Tc, omega), mu_r = kkt_omega(&Tr, omega);
            int64_t t = k - t0;
            int kind = 0;
            if (mu_c <= prm->beta_sufficient * mu_r) kind = 1;
            else if (mu_c <= prm->beta_necessary * mu_r && mu_c > mu_prev) kind = 2;
            else if ((double)t >= prm->beta_artificial * (double)k) kind = 3;
            if (!prm->restarts_enabled) kind = 0;
            rec.candidate = cand_avg; rec.mu_c = mu_c; rec.mu_r = mu_r; rec.restart_kind = kind;
            if (kind) {
                const double* xc = cand_avg ? xavg : x; const double* yc = cand_avg ? yavg : y;
                nsum ddx = {0, 0}, ddy = {0, 0};
                for (int64_t j = 0; j < n; ++j) ns_add(&ddx, (xc[j] - xr[j]) * (xc[j] - xr[j]));
                for (int64_t i = 0; i < m; ++i) ns_add(&ddy, (yc[i] - yr[i]) * (yc[i] - yr[i]));
                double Dx = sqrt(ns_get(&ddx)), Dy = sqrt(ns_get(&ddy));
                if (Dx > 1e-10 && Dy > 1e-10)
                    omega = exp(prm->weight_smoothing * log(Dy / Dx) + (1.0 - prm->weight_smoothing) * log(omega));
                if (cand_avg) { memcpy(x, xavg, sizeof(double) * (size_t)n); memcpy(y, yavg, sizeof(double) * (size_t)m); }
                memcpy(xr, x, sizeof(double) * (size_t)n); memcpy(yr, y, sizeof(double) * (size_t)m);
                Tr = *Tc;
                memset(xsum, 0, sizeof(double) * (size_t)n); memset(ysum, 0, sizeof(double) * (size_t)m);
                w = 0.0; t0 = k; mu_prev = INFINITY; restarts += 1;
            } else {
                mu_prev = mu_c;
            }
        }
        rec.omega_after = omega;
        if (chk && nc < chk_cap) chk[nc] = rec;
        nc += 1;
        if (status == ORACLE_OPTIMAL) break;
    }

    /* ---- R12/R14: which point is returned */
    const double* xs = x; const double* ys = y; const kkt_terms* Tf = &Tcur;
    if (fixed) {
        kkt_eval(&P, x, y, sa, srho, &Tcur);                 /* report only; current iterate returned */
    } else if (status == ORACLE_OPTIMAL) {
        if (ret_avg) { xs = xavg; ys = yavg; Tf = &Tavg; }
    } else if (status == ORACLE_ITERATION_LIMIT && k > 0) {
        /* last check ran at k == limit: return the better of cur / avg */
        if (have_avg && w > 0.0 && rel_kkt(&P, &Tavg) < rel_kkt(&P, &Tcur)) { xs = xavg; ys = yavg; Tf = &Tavg; ret_avg = 1; }
    } else {
        kkt_eval(&P, x, y, sa, srho, &Tcur);
    }
    for (int64_t j = 0; j < n; ++j) x_out[j] = xs[j] / P.Dc[j];
    for (int64_t i = 0; i < m; ++i) y_out[i] = ys[i] / P.Dr[i];
    res->status = status; res->returned_average = ret_avg;
    res->iterations = k; res->accepted = accepted; res->restarts = restarts;
    rel_terms(&P, Tf, &res->rel_primal_res, &res->rel_dual_res, &res->rel_gap);
    res->rel_kkt = rel_kkt(&P, Tf); res->primal_obj = Tf->pobj; res->dual_obj = Tf->dobj;
    res->eta = eta; res->omega = omega;
    if (n_att) *n_att = na;
    if (n_chk) *n_chk = nc;
    if (avg_w) *avg_w = w;
    if (avg_x) for (int64_t j = 0; j < n; ++j) avg_x[j] = (w > 0.0) ? xsum[j] / w : x[j];
    if (avg_y) for (int64_t i = 0; i < m; ++i) avg_y[i] = (w > 0.0) ? ysum[i] / w : y[i];

    free(P.val); free(P.Dr); free(P.Dc); free(P.q); free(P.c); free(P.l); free(P.u);
    free(x); free(y); free(xn); free(yn); free(xbar); free(xsum); free(ysum); free(xavg); free(yavg);
    free(xr); free(yr); free(g); free(kx); free(dxv); free(kdx); free(sa); free(srho);
    return 0;
}
