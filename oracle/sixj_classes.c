/* sixj_classes.c -- oracle side (test infrastructure, plain C, integers only): one representative of every class of {6j}
 * symbols {a b c; d e f} under the 24 tetrahedral symmetries, for all symbols with valid triads and every label 2j <= J.
 *
 * The symmetries are the textbook ones the paper's 6j tables rest on (tables of 6j symbols are precomputed
 * once per maximal spin; storing one value per symmetry class is what makes them small): any permutation of the three
 * columns (a d), (b e), (c f), and the exchange of the upper and lower label in any two columns.  The representative is the
 * image whose label sequence (a b c d e f) is lexicographically largest.  Triads: (a b c), (a e f), (d b f), (d e c).
 *
 * Nothing here is shared with the CUDA path (which has its own canonical form, sf_sixj.cuh); the exhaustive table test uses
 * this list only as "every distinct symbol once".  Pinned by tests/test_oracle_wigner.py against a brute-force grouping of
 * all tuples for small J.
 */
#include <stdlib.h>

static int triad(int a, int b, int c)
{
    if ((a + b + c) & 1) return 0;
    int lo = a > b ? a - b : b - a;
    return c >= lo && c <= a + b;
}

static long key6(const int t[6])
{
    long k = 0;
    for (int q = 0; q < 6; ++q) k = k * 1024 + t[q];
    return k;
}

/* 1 if (a b c d e f) is the lexicographically largest of its 24 images */
static int is_representative(int a, int b, int c, int d, int e, int f)
{
    static const int perm[6][3] = {{0, 1, 2}, {0, 2, 1}, {1, 0, 2}, {1, 2, 0}, {2, 0, 1}, {2, 1, 0}};
    static const int flip[4][3] = {{0, 0, 0}, {1, 1, 0}, {1, 0, 1}, {0, 1, 1}};
    const int up[3] = {a, b, c}, dn[3] = {d, e, f};
    const int self[6] = {a, b, c, d, e, f};
    const long k0 = key6(self);
    for (int p = 0; p < 6; ++p)
        for (int s = 0; s < 4; ++s) {
            int t[6];
            for (int q = 0; q < 3; ++q) {
                const int col = perm[p][q];
                t[q] = flip[s][q] ? dn[col] : up[col];
                t[q + 3] = flip[s][q] ? up[col] : dn[col];
            }
            if (key6(t) > k0) return 0;
        }
    return 1;
}

/* Representatives with first label a and second label b (labels <= J), written as six signed chars each to out (at most cap
 * symbols; out may be NULL to count only).  Returns their number.  A representative has a >= every label, b >= c, e, f. */
long orc_sixj_classes_ab(int J, int a, int b, signed char* out, long cap)
{
    long n = 0;
    if (a < 0 || a > J || b < 0 || b > a || J > 127) return 0;
    for (int c = 0; c <= b; ++c) {
        if (!triad(a, b, c)) continue;
        for (int d = 0; d <= a; ++d)
            for (int e = 0; e <= b; ++e) {
                if (!triad(d, e, c)) continue;
                for (int f = 0; f <= b; ++f) {
                    if (!triad(a, e, f) || !triad(d, b, f)) continue;
                    if (!is_representative(a, b, c, d, e, f)) continue;
                    if (out && n < cap) {
                        signed char* o = out + 6 * n;
                        o[0] = (signed char)a; o[1] = (signed char)b; o[2] = (signed char)c;
                        o[3] = (signed char)d; o[4] = (signed char)e; o[5] = (signed char)f;
                    }
                    ++n;
                }
            }
    }
    return n;
}
