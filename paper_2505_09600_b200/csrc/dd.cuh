// dd.cuh -- double-double ("dd") arithmetic on the FP64 pipe: a value is the unevaluated sum hi + lo of two
// doubles, |lo| <= ulp(hi) / 2 after normalisation (about 106 significant bits).
//
// Why the library needs it.  The gen-2.0 LFA Michelson combination, Eq. (B33), takes a SECOND central
// difference of the single-link series y^LFA: white rounding noise of relative size s in y comes out as
// 2.45 s / (omega dt)^2 in X -- 4.5e4 s for config 3 (f = 2.35e-4 Hz, dt = 5 s).  The 1e-11 parity bar therefore
// needs y^LFA good to about one rounding (hard part 1), while a plain fp64 evaluation of the
// link geometry loses a factor 60 alone in n_l = (R_r - R_s) / |R_r - R_s| (two positions of 1.5e11 m rounded to
// 2e-5 m, subtracted to 2.5e9 m).  The orbit kernel (orbit.cuh) and the LFA link stage (fast.cuh) carry the
// quantities that enter y^LFA multiplicatively as dd values; everything else stays plain fp64.
//
// Error-free transformations (Knuth TwoSum, Dekker FastTwoSum, FMA TwoProduct) and the usual "sloppy" dd
// product / quotient (relative error a few 2^-104).
#pragma once

struct dd { double hi, lo; };

__host__ __device__ __forceinline__ dd dd_make(double hi, double lo) { dd r; r.hi = hi; r.lo = lo; return r; }

// a + b = s + e exactly
__device__ __forceinline__ dd two_sum(double a, double b)
{
    const double s = __dadd_rn(a, b);
    const double bb = __dadd_rn(s, -a);
    const double e = __dadd_rn(__dadd_rn(a, -__dadd_rn(s, -bb)), __dadd_rn(b, -bb));
    return dd_make(s, e);
}
// the same for |a| >= |b| (or a == 0)
__device__ __forceinline__ dd fast_two_sum(double a, double b)
{
    const double s = __dadd_rn(a, b);
    const double e = __dadd_rn(b, -__dadd_rn(s, -a));
    return dd_make(s, e);
}
// a * b = p + e exactly
__device__ __forceinline__ dd two_prod(double a, double b)
{
    const double p = __dmul_rn(a, b);
    return dd_make(p, __fma_rn(a, b, -p));
}

__device__ __forceinline__ dd dd_neg(dd a) { return dd_make(-a.hi, -a.lo); }

__device__ __forceinline__ dd dd_add(dd a, dd b)
{
    dd s = two_sum(a.hi, b.hi);
    const dd t = two_sum(a.lo, b.lo);
    s.lo = __dadd_rn(s.lo, t.hi);
    s = fast_two_sum(s.hi, s.lo);
    s.lo = __dadd_rn(s.lo, t.lo);
    return fast_two_sum(s.hi, s.lo);
}
__device__ __forceinline__ dd dd_sub(dd a, dd b) { return dd_add(a, dd_neg(b)); }
// a + b with an error of 2^-104 (|a| + |b|) instead of 2^-104 |a + b|: 11 additions instead of 20.  For sums whose terms
// do not cancel (Horner steps, combinations of O(1) terms with an O(1) result).
__device__ __forceinline__ dd dd_add_fast(dd a, dd b)
{
    dd s = two_sum(a.hi, b.hi);
    s.lo = __dadd_rn(s.lo, __dadd_rn(a.lo, b.lo));
    return fast_two_sum(s.hi, s.lo);
}
__device__ __forceinline__ dd dd_sub_fast(dd a, dd b) { return dd_add_fast(a, dd_neg(b)); }
__device__ __forceinline__ dd dd_add_d(dd a, double b)
{
    dd s = two_sum(a.hi, b);
    s.lo = __dadd_rn(s.lo, a.lo);
    return fast_two_sum(s.hi, s.lo);
}
__device__ __forceinline__ dd dd_mul(dd a, dd b)
{
    dd p = two_prod(a.hi, b.hi);
    p.lo = __fma_rn(a.hi, b.lo, p.lo);
    p.lo = __fma_rn(a.lo, b.hi, p.lo);
    return fast_two_sum(p.hi, p.lo);
}
__device__ __forceinline__ dd dd_mul_d(dd a, double b)
{
    dd p = two_prod(a.hi, b);
    p.lo = __fma_rn(a.lo, b, p.lo);
    return fast_two_sum(p.hi, p.lo);
}
// a / b: two Newton-style quotient digits
__device__ __forceinline__ dd dd_div(dd a, dd b)
{
    const double q1 = __ddiv_rn(a.hi, b.hi);
    const dd r = dd_sub(a, dd_mul_d(b, q1));
    const double q2 = __ddiv_rn(r.hi, b.hi);
    const dd r2 = dd_sub(r, dd_mul_d(b, q2));
    const double q3 = __ddiv_rn(r2.hi, b.hi);
    dd q = fast_two_sum(q1, q2);
    return dd_add_d(q, q3);
}
// sqrt(a), a > 0: one Newton step on the fp64 root (Karp-Markstein)
__device__ __forceinline__ dd dd_sqrt(dd a)
{
    const double x = __drcp_rn(__dsqrt_rn(a.hi));
    const double ax = __dmul_rn(a.hi, x);
    const dd sq = two_prod(ax, ax);
    const double r = dd_sub(a, sq).hi;
    return fast_two_sum(ax, __dmul_rn(r, __dmul_rn(x, 0.5)));
}
__device__ __forceinline__ double dd_to_double(dd a) { return __dadd_rn(a.hi, a.lo); }
