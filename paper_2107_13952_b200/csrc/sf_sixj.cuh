// sf_sixj.cuh -- device functions for the Wigner {6j} symbol (kernel (a) of north_star).
//
// The paper takes its {6j} from WIGXJPF / FASTWIGXJ tables (ref. [31] PAPER.md:621); what those
// evaluate is Racah's single-sum formula.  Here the formula is evaluated on the device:
//
//   {a b c; d e f} = sqrt(D2(abc) D2(aef) D2(dbf) D2(dec)) * sum_t (-1)^t (t+1)! / (prod_i (t-al_i)! prod_j (be_j-t)!)
//   D2(x y z) = (x+y-z)! (x-y+z)! (-x+y+z)! / (x+y+z+1)!        (arguments in units of spin; 2j integers in the code)
//   al = ((a+b+c),(a+e+f),(d+b+f),(d+e+c))/2,  be = ((a+b+d+e),(a+c+d+f),(b+c+e+f))/2,  t = max al .. min be.
//
// Factorials come from a table of double-double significands with separate binary exponents (n! = m * 2^e,
// 0.5 <= m < 1), so nothing overflows; the first term and the triangle coefficients are formed from that table and
// the remaining terms by the exact integer ratio term(t+1)/term(t) in double-double.
#pragma once
#include "sf_dd.h"
#include "sf_internal.h"

#define SF_NFACT 2048   // factorial table covers 0! .. 2047!

struct SfFact {
    double hi, lo;   // significand in [0.5, 1)
    int e;           // n! = (hi + lo) * 2^e
    int pad;
};
const SfFact* sf_fact_table(void);   // device pointer (sf_sixj.cu), valid after sf_sixj_module_init

__device__ __forceinline__ bool sf_triad(int x, int y, int z)
{
    return !((x + y + z) & 1) && z >= abs(x - y) && z <= x + y;
}
__device__ __forceinline__ bool sf_sixj_valid(int a, int b, int c, int d, int e, int f)
{
    return sf_triad(a, b, c) && sf_triad(a, e, f) && sf_triad(d, b, f) && sf_triad(d, e, c);
}

// product of factorial-table entries: acc (significand, exponent) *= n!
__device__ __forceinline__ void sf_fmul(dd_t& m, int& ex, const SfFact* __restrict__ F, int n)
{
    const SfFact v = F[n];
    m = dd_mul(m, dd_make(v.hi, v.lo));
    ex += v.e;
}

// direct evaluation; all arguments are 2j >= 0.  Returns 0 when a triad fails.
__device__ inline double sf_sixj_eval(const SfFact* __restrict__ F, int a, int b, int c, int d, int e, int f)
{
    if (!sf_sixj_valid(a, b, c, d, e, f)) return 0.0;
    const int al1 = (a + b + c) >> 1, al2 = (a + e + f) >> 1, al3 = (d + b + f) >> 1, al4 = (d + e + c) >> 1;
    const int be1 = (a + b + d + e) >> 1, be2 = (a + c + d + f) >> 1, be3 = (b + c + e + f) >> 1;
    const int tmin = max(max(al1, al2), max(al3, al4));
    const int tmax = min(be1, min(be2, be3));
    if (tmax + 1 >= SF_NFACT) return nan("");

    // first term of the sum, T0 = (tmin+1)! / (prod (tmin-al_i)! prod (be_j-tmin)!)
    dd_t num = dd_make(1.0, 0.0), den = dd_make(1.0, 0.0);
    int en = 0, ed = 0;
    sf_fmul(num, en, F, tmin + 1);
    sf_fmul(den, ed, F, tmin - al1);
    sf_fmul(den, ed, F, tmin - al2);
    sf_fmul(den, ed, F, tmin - al3);
    sf_fmul(den, ed, F, tmin - al4);
    sf_fmul(den, ed, F, be1 - tmin);
    sf_fmul(den, ed, F, be2 - tmin);
    sf_fmul(den, ed, F, be3 - tmin);
    dd_t T0 = dd_div(num, den);
    int eT = en - ed;

    // product of the four triangle coefficients squared
    num = dd_make(1.0, 0.0);
    den = dd_make(1.0, 0.0);
    en = 0;
    ed = 0;
#define SF_TRI(x, y, z)                            \
    sf_fmul(num, en, F, ((x) + (y) - (z)) >> 1);   \
    sf_fmul(num, en, F, ((x) - (y) + (z)) >> 1);   \
    sf_fmul(num, en, F, (-(x) + (y) + (z)) >> 1);  \
    sf_fmul(den, ed, F, (((x) + (y) + (z)) >> 1) + 1);
    SF_TRI(a, b, c)
    SF_TRI(a, e, f)
    SF_TRI(d, b, f)
    SF_TRI(d, e, c)
#undef SF_TRI
    dd_t D = dd_div(num, den);
    int eD = en - ed;
    if (eD & 1) {   // make the exponent even before the square root
        D = dd_make(D.hi * 2.0, D.lo * 2.0);
        eD -= 1;
    }
    const dd_t sD = dd_sqrt(D);

    // sum of term ratios r_t = term(t)/term(tmin); r_{t+1} = -r_t (t+2) prod(be_j - t) / prod(t+1-al_i)
    dd_t r = dd_make(1.0, 0.0), S = dd_make(1.0, 0.0);
    int sc = 0;
    for (int t = tmin; t < tmax; ++t) {
        const double rn = (double)(t + 2) * (double)(be1 - t) * (double)(be2 - t) * (double)(be3 - t);
        const double rd = (double)(t + 1 - al1) * (double)(t + 1 - al2) * (double)(t + 1 - al3) * (double)(t + 1 - al4);
        r = dd_div_d(dd_mul_d(r, -rn), rd);
        S = dd_add(S, r);
        if (fabs(r.hi) > 0x1p+500) {   // keep the running ratio inside the FP64 range (exact rescale)
            r = dd_make(r.hi * 0x1p-500, r.lo * 0x1p-500);
            S = dd_make(S.hi * 0x1p-500, S.lo * 0x1p-500);
            sc += 500;
        }
    }
    dd_t v = dd_mul(dd_mul(T0, sD), S);
    double val = v.hi + v.lo;
    if (tmin & 1) val = -val;
    return ldexp(val, eT + (eD >> 1) + sc);
}

// ---------------------------------------------------------------------------------------------------------
// Canonical form under the 24 tetrahedral symmetries (column permutations; row swap in two columns) and the
// dense table index.  Canonical: a = max of all six, b = max(b, c, e, f).  Then
//   c in [a-b, b], c = a+b (mod 2);   e in [a-b, b];   f in [a-e, b], f = a+e (mod 2);
//   d in [max(b-f, |e-c|), min(b+f, e+c, a)], d = b+f (mod 2).
// Slot = base4[group(a,b,c,e)] + sum_{f' < f} nd(f') + (d - dlo(f))/2.  Ties give several canonical tuples per
// class; every tuple that satisfies the constraints has its own (identical-valued) slot, so a lookup never misses.
// ---------------------------------------------------------------------------------------------------------
__host__ __device__ __forceinline__ void sf_swap(int& x, int& y)
{
    int t = x;
    x = y;
    y = t;
}
__host__ __device__ inline void sf_sixj_canon(int& a, int& b, int& c, int& d, int& e, int& f)
{
    int m = a;
    if (b > m) m = b;
    if (c > m) m = c;
    if (d > m) m = d;
    if (e > m) m = e;
    if (f > m) m = f;
    if (a == m) {
    } else if (b == m) {
        sf_swap(a, b);
        sf_swap(d, e);
    } else if (c == m) {
        sf_swap(a, c);
        sf_swap(d, f);
    } else if (d == m) {          // {a b c; d e f} = {d e c; a b f}
        sf_swap(a, d);
        sf_swap(b, e);
    } else if (e == m) {          // columns 1<->2, then the same row swap: {e d c; b a f}
        int na = e, nb = d, nd = b, ne = a;
        a = na; b = nb; d = nd; e = ne;
    } else {                      // columns 1<->3, then row swap of columns 1,2: {f e a; c b d}
        int na = f, nb = e, nc = a, nd = c, ne = b, nf = d;
        a = na; b = nb; c = nc; d = nd; e = ne; f = nf;
    }
    int m2 = b;
    if (c > m2) m2 = c;
    if (e > m2) m2 = e;
    if (f > m2) m2 = f;
    if (b == m2) {
    } else if (c == m2) {         // columns 2<->3
        sf_swap(b, c);
        sf_swap(e, f);
    } else if (e == m2) {         // row swap of columns 2,3: {a e f; d b c}
        sf_swap(b, e);
        sf_swap(c, f);
    } else {                      // both: {a f e; d c b}
        sf_swap(b, f);
        sf_swap(c, e);
    }
}
__host__ __device__ __forceinline__ int sf_sixj_nd(int a, int b, int c, int e, int f, int* dlo)
{
    int lo = b - f, l2 = e > c ? e - c : c - e;
    if (l2 > lo) lo = l2;
    int hi = b + f;
    if (e + c < hi) hi = e + c;
    if (a < hi) hi = a - ((a - (b + f)) & 1);
    *dlo = lo;
    return hi >= lo ? ((hi - lo) >> 1) + 1 : 0;
}
__host__ __device__ __forceinline__ long sf_sixj_group(int J, int a, int b, int c, int e)
{
    const long NC = J / 2 + 1, NE = J + 1;
    return (((long)a * (a + 1) / 2 + b) * NC + ((c - (a - b)) >> 1)) * NE + (e - (a - b));
}
// slot of a CANONICAL tuple
__device__ inline long sf_sixj_slot(const long* __restrict__ base4, int J, int a, int b, int c, int d, int e, int f)
{
    long s = base4[sf_sixj_group(J, a, b, c, e)];
    int dlo;
    for (int ff = a - e; ff < f; ff += 2) s += sf_sixj_nd(a, b, c, e, ff, &dlo);
    sf_sixj_nd(a, b, c, e, f, &dlo);
    return s + ((d - dlo) >> 1);
}
// value from the resident table; arguments need not be canonical; every argument must be <= tab.two_jmax
__device__ inline double sf_sixj_lookup(const SfSixjTable& tab, int a, int b, int c, int d, int e, int f)
{
    if (!sf_sixj_valid(a, b, c, d, e, f)) return 0.0;
    sf_sixj_canon(a, b, c, d, e, f);
    return tab.values[sf_sixj_slot(tab.base4, tab.two_jmax, a, b, c, d, e, f)];
}
