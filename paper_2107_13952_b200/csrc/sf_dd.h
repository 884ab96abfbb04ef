// sf_dd.h -- double-double arithmetic (two FP64 words, ~106-bit significand) for the Racah sum of the {6j} kernel.
// The Racah sum alternates in sign and cancels by up to ~2e5 for 2j <= 60 and ~6e10 for 2j <= 150 (SURVEY.md 7,
// "6j accuracy"), so plain FP64 summation misses the 1e-12 relative bound of north_star; error-free transforms
// (Knuth two-sum, FMA two-product) keep every term to ~1e-32 relative.
#pragma once
#include <math.h>

#ifdef __CUDACC__
#define SF_HD __host__ __device__ __forceinline__
#else
#define SF_HD inline
#endif

struct dd_t {
    double hi, lo;
};

// explicit round-to-nearest ops so that the compiler cannot contract the error-free transforms into FMAs
#ifdef __CUDA_ARCH__
#define SF_ADD(a, b) __dadd_rn((a), (b))
#define SF_SUB(a, b) __dsub_rn((a), (b))
#define SF_MUL(a, b) __dmul_rn((a), (b))
#define SF_FMA(a, b, c) __fma_rn((a), (b), (c))
#else
#define SF_ADD(a, b) ((a) + (b))
#define SF_SUB(a, b) ((a) - (b))
#define SF_MUL(a, b) ((a) * (b))
#define SF_FMA(a, b, c) fma((a), (b), (c))
#endif

SF_HD dd_t dd_make(double hi, double lo)
{
    dd_t r;
    r.hi = hi;
    r.lo = lo;
    return r;
}
SF_HD dd_t dd_quick_two_sum(double a, double b)   // |a| >= |b|
{
    double s = SF_ADD(a, b);
    return dd_make(s, SF_SUB(b, SF_SUB(s, a)));
}
SF_HD dd_t dd_two_sum(double a, double b)
{
    double s = SF_ADD(a, b);
    double bb = SF_SUB(s, a);
    double e = SF_ADD(SF_SUB(a, SF_SUB(s, bb)), SF_SUB(b, bb));
    return dd_make(s, e);
}
SF_HD dd_t dd_two_prod(double a, double b)
{
    double p = SF_MUL(a, b);
    return dd_make(p, SF_FMA(a, b, -p));
}
SF_HD dd_t dd_add(dd_t a, dd_t b)
{
    dd_t s = dd_two_sum(a.hi, b.hi);
    dd_t t = dd_two_sum(a.lo, b.lo);
    s.lo = SF_ADD(s.lo, t.hi);
    s = dd_quick_two_sum(s.hi, s.lo);
    s.lo = SF_ADD(s.lo, t.lo);
    return dd_quick_two_sum(s.hi, s.lo);
}
SF_HD dd_t dd_neg(dd_t a) { return dd_make(-a.hi, -a.lo); }
SF_HD dd_t dd_mul_d(dd_t a, double b)
{
    dd_t p = dd_two_prod(a.hi, b);
    p.lo = SF_FMA(a.lo, b, p.lo);
    return dd_quick_two_sum(p.hi, p.lo);
}
SF_HD dd_t dd_mul(dd_t a, dd_t b)
{
    dd_t p = dd_two_prod(a.hi, b.hi);
    p.lo = SF_ADD(p.lo, SF_FMA(a.hi, b.lo, SF_MUL(a.lo, b.hi)));
    return dd_quick_two_sum(p.hi, p.lo);
}
SF_HD dd_t dd_div_d(dd_t a, double b)
{
    double q1 = a.hi / b;
    dd_t p = dd_two_prod(q1, b);
    dd_t r = dd_add(a, dd_neg(p));
    double q2 = r.hi / b;
    p = dd_two_prod(q2, b);
    r = dd_add(r, dd_neg(p));
    double q3 = r.hi / b;
    dd_t q = dd_quick_two_sum(q1, q2);
    return dd_add(q, dd_make(q3, 0.0));
}
SF_HD dd_t dd_div(dd_t a, dd_t b)
{
    double q1 = a.hi / b.hi;
    dd_t r = dd_add(a, dd_neg(dd_mul_d(b, q1)));
    double q2 = r.hi / b.hi;
    r = dd_add(r, dd_neg(dd_mul_d(b, q2)));
    double q3 = r.hi / b.hi;
    dd_t q = dd_quick_two_sum(q1, q2);
    return dd_add(q, dd_make(q3, 0.0));
}
SF_HD dd_t dd_sqrt(dd_t a)   // a > 0
{
    double x = 1.0 / sqrt(a.hi);
    double ax = SF_MUL(a.hi, x);
    dd_t sq = dd_two_prod(ax, ax);
    dd_t r = dd_add(a, dd_neg(sq));
    return dd_two_sum(ax, SF_MUL(r.hi, SF_MUL(x, 0.5)));
}
