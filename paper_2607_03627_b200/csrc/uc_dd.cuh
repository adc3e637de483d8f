// uc_dd.cuh -- double-double helpers for the device side.
//
// Why: the adaptive step rule makes the PDHG trajectory exponentially sensitive to rounding (DESIGN.md
// "Numerics"): a 1-ulp difference in one reduction is 1e-8 after 200 attempts.  The sequential
// statement of the method sums its long reductions with compensated (Neumaier) accumulators, i.e. it
// returns the exactly rounded sum in all but freak cases.  A parallel tree cannot follow a sequential
// order, but it can be exact too: every block / grid reduction here carries (hi, lo) pairs with
// error-free transformations, so the rounded result is the same number whatever the order.
// log / exp below are evaluated in double-double and rounded once (used only by the primal-weight
// update, once per restart, by one thread).
//
// The translation unit is compiled with -fmad=false: no a*b+c is contracted behind our back; the
// explicit fma() calls below are intended.
#pragma once
#include <cuda_runtime.h>
#include <math.h>

namespace ucpdhg {

struct dd { double hi, lo; };

__host__ __device__ __forceinline__ dd two_sum(double a, double b) {
    double s = a + b, bb = s - a;
    double e = (a - (s - bb)) + (b - bb);
    return dd{s, e};
}
__host__ __device__ __forceinline__ dd quick_two_sum(double a, double b) {   // |a| >= |b|
    double s = a + b;
    return dd{s, b - (s - a)};
}
__host__ __device__ __forceinline__ dd two_prod(double a, double b) {
    double p = a * b;
    return dd{p, fma(a, b, -p)};
}
__host__ __device__ __forceinline__ dd dd_add(dd a, dd b) {
    dd s = two_sum(a.hi, b.hi), t = two_sum(a.lo, b.lo);
    s.lo += t.hi; s = quick_two_sum(s.hi, s.lo);
    s.lo += t.lo; return quick_two_sum(s.hi, s.lo);
}
__host__ __device__ __forceinline__ dd dd_add_d(dd a, double b) {
    dd s = two_sum(a.hi, b);
    s.lo += a.lo; return quick_two_sum(s.hi, s.lo);
}
// Cascaded addition for the SERIAL TAIL of an attempt (the reductions between the last row and the step rule): the high
// parts are added with an error-free transformation, the error and the low parts in plain double.  One fp64 operation
// on the dependent chain per addition instead of ~13 (an fp64 add has ~20 cycles of latency on B200 and these chains
// run in ONE warp while the whole GPU waits); the pair is not renormalised -- dd_round adds the two parts once.  The
// low part carries n * 2^-53 relative error of ITSELF, i.e. ~2^-99 of the largest partial sum: the rounded result is
// still the correctly rounded exact sum unless that lies within ~1e-29 (relative) of a rounding boundary.
__host__ __device__ __forceinline__ dd dd_acc(dd a, dd b) {
    dd s = two_sum(a.hi, b.hi);
    s.lo += a.lo + b.lo;
    return s;
}
__host__ __device__ __forceinline__ dd dd_neg(dd a) { return dd{-a.hi, -a.lo}; }
__host__ __device__ __forceinline__ dd dd_mul(dd a, dd b) {
    dd p = two_prod(a.hi, b.hi);
    p.lo += a.hi * b.lo + a.lo * b.hi;
    return quick_two_sum(p.hi, p.lo);
}
__host__ __device__ __forceinline__ dd dd_mul_d(dd a, double b) {
    dd p = two_prod(a.hi, b);
    p.lo += a.lo * b;
    return quick_two_sum(p.hi, p.lo);
}
__host__ __device__ __forceinline__ dd dd_div(dd a, dd b) {
    double q1 = a.hi / b.hi;
    dd r = dd_add(a, dd_neg(dd_mul_d(b, q1)));
    double q2 = r.hi / b.hi;
    r = dd_add(r, dd_neg(dd_mul_d(b, q2)));
    double q3 = r.hi / b.hi;
    dd q = quick_two_sum(q1, q2);
    return dd_add_d(q, q3);
}
__host__ __device__ __forceinline__ double dd_round(dd a) { return a.hi + a.lo; }

// ln 2 to ~106 bits
__host__ __device__ __forceinline__ dd dd_ln2() { return dd{0.6931471805599453094, 2.3190468138462995584e-17}; }

// log of a positive finite double, in double-double (relative error ~1e-31)
__host__ __device__ inline dd dd_log(double a) {
    int e;
    double m = frexp(a, &e);                       // a = m 2^e, m in [0.5, 1)
    if (m < 0.70710678118654752440) { m *= 2.0; e -= 1; }
    dd num = dd{m - 1.0, 0.0};                     // exact (Sterbenz)
    dd den = two_sum(m, 1.0);
    dd s = dd_div(num, den);                       // |s| <= 0.1716
    dd t = dd_mul(s, s);
    const int N = 24;                              // t^24 < 1e-36
    dd poly = dd_div(dd{1.0, 0.0}, dd{(double)(2 * N + 1), 0.0});
    for (int i = N - 1; i >= 0; --i)
        poly = dd_add(dd_mul(poly, t), dd_div(dd{1.0, 0.0}, dd{(double)(2 * i + 1), 0.0}));
    dd lm = dd_mul(s, poly);
    lm.hi *= 2.0; lm.lo *= 2.0;
    return dd_add(lm, dd_mul_d(dd_ln2(), (double)e));
}
// exp of a double-double argument with |x| < 700, in double-double
__host__ __device__ inline dd dd_exp(dd x) {
    double kf = rint(x.hi / 0.6931471805599453094);
    dd r = dd_add(x, dd_neg(dd_mul_d(dd_ln2(), kf)));   // |r| <= 0.35
    r.hi *= (1.0 / 256.0); r.lo *= (1.0 / 256.0);       // exact scaling
    const int N = 12;
    dd inv_fact[N + 1];
    inv_fact[0] = dd{1.0, 0.0};
    for (int i = 1; i <= N; ++i) inv_fact[i] = dd_div(inv_fact[i - 1], dd{(double)i, 0.0});
    dd p = inv_fact[N];
    for (int i = N - 1; i >= 0; --i) p = dd_add(dd_mul(p, r), inv_fact[i]);
    for (int i = 0; i < 8; ++i) p = dd_mul(p, p);
    int k = (int)kf;
    p.hi = ldexp(p.hi, k); p.lo = ldexp(p.lo, k);
    return p;
}
__host__ __device__ inline double log_rounded(double a) { return dd_round(dd_log(a)); }
__host__ __device__ inline double exp_rounded(double x) { return dd_round(dd_exp(dd{x, 0.0})); }

}  // namespace ucpdhg
