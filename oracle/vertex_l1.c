/* ORACLE -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.  Shares nothing with the CUDA path.
 *
 * Level-L1 oracle for the EPRL vertex tensor: steps 5-7 of the vertex-tensor algorithm of
 * arXiv 2107.13952 written as plain nested loops, no blocking, no BLAS:
 *
 *   for every shell (l23 l24 l25 l34 l35 l45), canonical order, l45 fastest      [step 5]
 *     (i)   W[i1,k2,k3,k4,k5] = {15j} by direct summation of eq. (5) over x       [PAPER.md:178, 67-95]
 *     (ii)  select the four booster sub-matrices B_a[t_a(shell)]                  [PAPER.md:179]
 *     (iii) contract them with W over k5, k4, k3, k2, with the (2k_a+1) weights   [PAPER.md:180, eq. (3)]
 *     (iv)  accumulate                                                            [PAPER.md:181]
 *   finally multiply by prod_e sqrt(2 i_e + 1)                                    [eq. (3), PAPER.md:54]
 *
 * The {6j} values are NOT computed here: they arrive as the five dense arrays S1..S5 of step 4
 * (PAPER.md:173-175), filled by oracle/vertex.py with exact big-integer values rounded once to double.
 *
 * ACC_T is the accumulation type: long double for the parity reference, double for the timed baseline.
 * Spins are 2j integers.  Spin order (12 13 14 15 23 24 25 34 35 45).
 */
#include <math.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#ifndef ACC_T
#define ACC_T long double
#endif
typedef ACC_T acc_t;

enum { J12, J13, J14, J15, J23, J24, J25, J34, J35, J45 };

/* range of the spin recoupling (a b) with (c d): returns count, *lo = minimum (2j units) */
static int pair_range(int a, int b, int c, int d, int *lo)
{
    int l1 = abs(a - b), l2 = abs(c - d), h1 = a + b, h2 = c + d;
    int l = l1 > l2 ? l1 : l2, h = h1 < h2 ? h1 : h2;
    *lo = l;
    if (((a + b) ^ (c + d)) & 1) return 0;
    if (h < l) return 0;
    return (h - l) / 2 + 1;
}

typedef struct {
    int two_j[10], two_dl, nl;              /* nl = Delta_l + 1 */
    int two_i_min[5], n_i[5];               /* boundary intertwiners, nodes 1..5 */
    int two_k_base[4], n_k_pad[4];          /* padded k layout of edges 2..5 (boosters and S arrays) */
    int two_x_base, n_x_pad;
    const double *S1, *S2, *S3, *S4, *S5;   /* S1[o25][a1][q5][x] S2[o35][o45][q4][q5][x] S3[o24][o34][o35][q3][q4][x]
                                               S4[o23][o24][q2][q3][x] S5[o25][a1][q2][x]; q = (two_k - two_k_base)/2 */
    const double *B[4];                     /* B_a[t][ii][kk], edges 2..5 */
} problem_t;

static int imax(int a, int b) { return a > b ? a : b; }
static int imin(int a, int b) { return a < b ? a : b; }

/* one shell: adds its contribution to A (and to Aabs if non-NULL); returns 1 if the shell was non-empty */
static int do_shell(const problem_t *p, const int o[6], acc_t *A, acc_t *Aabs, acc_t **scratch)
{
    const int nl = p->nl;
    int l[10];
    memcpy(l, p->two_j, sizeof l);
    l[J23] += 2 * o[0]; l[J24] += 2 * o[1]; l[J25] += 2 * o[2];
    l[J34] += 2 * o[3]; l[J35] += 2 * o[4]; l[J45] += 2 * o[5];

    /* virtual intertwiner ranges at nodes 2..5 (node spin orders: see oracle/ranges.py) */
    int kmin[4], nk[4];
    nk[0] = pair_range(l[J23], l[J24], l[J25], l[J12], &kmin[0]);
    nk[1] = pair_range(l[J34], l[J35], l[J13], l[J23], &kmin[1]);
    nk[2] = pair_range(l[J45], l[J14], l[J24], l[J34], &kmin[2]);
    nk[3] = pair_range(l[J15], l[J25], l[J35], l[J45], &kmin[3]);
    if (!nk[0] || !nk[1] || !nk[2] || !nk[3]) return 0;

    /* booster triples, paper's superscript order */
    const long t2 = ((long)o[0] * nl + o[1]) * nl + o[2];   /* (l23 l24 l25) */
    const long t3 = ((long)o[3] * nl + o[4]) * nl + o[0];   /* (l34 l35 l23) */
    const long t4 = ((long)o[5] * nl + o[1]) * nl + o[3];   /* (l45 l24 l34) */
    const long t5 = ((long)o[2] * nl + o[4]) * nl + o[5];   /* (l25 l35 l45) */
    const long tt[4] = { t2, t3, t4, t5 };

    const int n1 = p->n_i[0], n2 = p->n_i[1], n3 = p->n_i[2], n4 = p->n_i[3], n5 = p->n_i[4];
    const int K2 = nk[0], K3 = nk[1], K4 = nk[2], K5 = nk[3];
    const int P2 = p->n_k_pad[0], P3 = p->n_k_pad[1], P4 = p->n_k_pad[2], P5 = p->n_k_pad[3];
    const int NX = p->n_x_pad;
    const int npass = Aabs ? 2 : 1;

    for (int pass = 0; pass < npass; ++pass) {
        /* (i) W[a1][q2][q3][q4][q5], eq. (5) */
        acc_t *W = scratch[0], *T = scratch[1];
        for (int a1 = 0; a1 < n1; ++a1) {
            const int i1 = p->two_i_min[0] + 2 * a1;
            for (int c2 = 0; c2 < K2; ++c2) { const int k2 = kmin[0] + 2 * c2, q2 = (k2 - p->two_k_base[0]) / 2;
            for (int c3 = 0; c3 < K3; ++c3) { const int k3 = kmin[1] + 2 * c3, q3 = (k3 - p->two_k_base[1]) / 2;
            for (int c4 = 0; c4 < K4; ++c4) { const int k4 = kmin[2] + 2 * c4, q4 = (k4 - p->two_k_base[2]) / 2;
            for (int c5 = 0; c5 < K5; ++c5) { const int k5 = kmin[3] + 2 * c5, q5 = (k5 - p->two_k_base[3]) / 2;
                /* x in the intersection of the five triads that contain it */
                int xlo = abs(i1 - l[J25]), xhi = i1 + l[J25];
                xlo = imax(xlo, abs(k5 - l[J14])); xhi = imin(xhi, k5 + l[J14]);
                xlo = imax(xlo, abs(k4 - l[J35])); xhi = imin(xhi, k4 + l[J35]);
                xlo = imax(xlo, abs(k3 - l[J24])); xhi = imin(xhi, k3 + l[J24]);
                xlo = imax(xlo, abs(k2 - l[J13])); xhi = imin(xhi, k2 + l[J13]);
                acc_t w = 0;
                for (int x = xlo; x <= xhi; x += 2) {
                    const int xx = (x - p->two_x_base) / 2;
                    const double s1 = p->S1[(((long)o[2] * n1 + a1) * P5 + q5) * NX + xx];
                    const double s2 = p->S2[((((long)o[4] * nl + o[5]) * P4 + q4) * P5 + q5) * NX + xx];
                    const double s3 = p->S3[(((((long)o[1] * nl + o[3]) * nl + o[4]) * P3 + q3) * P4 + q4) * NX + xx];
                    const double s4 = p->S4[((((long)o[0] * nl + o[1]) * P2 + q2) * P3 + q3) * NX + xx];
                    const double s5 = p->S5[(((long)o[2] * n1 + a1) * P2 + q2) * NX + xx];
                    acc_t term = (acc_t)(x + 1) * s1 * s2 * s3 * s4 * s5;
                    w += pass ? fabsl((long double)term) : term;
                }
                /* (-1)^R, R = sum of all fifteen labels (reading G1) */
                int twoR = i1 + k2 + k3 + k4 + k5;
                for (int s = 0; s < 10; ++s) twoR += l[s];
                if (!pass && ((twoR / 2) & 1)) w = -w;
                W[((((long)a1 * K2 + c2) * K3 + c3) * K4 + c4) * K5 + c5] = w;
            }}}}
        }
        /* (ii)+(iii) four mode products, k5 first; dims of the current tensor are d[0..4] */
        int d[5] = { n1, K2, K3, K4, K5 };
        const int nout[4] = { n2, n3, n4, n5 };
        acc_t *src = W, *dst = T;
        for (int mode = 4; mode >= 1; --mode) {          /* mode 4 = k5 ... mode 1 = k2 */
            const int e = mode - 1;                        /* edge index 0..3 for edges 2..5 */
            const int K = d[mode], N = nout[e], Pk = p->n_k_pad[e];
            const double *Bm = p->B[e] + tt[e] * (long)N * Pk;
            long outer = 1, inner = 1;
            for (int m = 0; m < mode; ++m) outer *= d[m];
            for (int m = mode + 1; m < 5; ++m) inner *= d[m];
            for (long u = 0; u < outer; ++u)
                for (int ii = 0; ii < N; ++ii)
                    for (long v = 0; v < inner; ++v) {
                        acc_t s = 0;
                        for (int c = 0; c < K; ++c) {
                            const int k = kmin[e] + 2 * c, kk = (k - p->two_k_base[e]) / 2;
                            double b = Bm[(long)ii * Pk + kk];
                            if (pass) b = fabs(b);
                            s += src[(u * K + c) * inner + v] * (acc_t)(k + 1) * b;
                        }
                        dst[(u * N + ii) * inner + v] = s;
                    }
            d[mode] = N;
            acc_t *tmp = src; src = dst; dst = tmp;
        }
        /* (iv) accumulate */
        const long ntot = (long)n1 * n2 * n3 * n4 * n5;
        acc_t *dstA = pass ? Aabs : A;
        for (long q = 0; q < ntot; ++q) dstA[q] += src[q];
    }
    return 1;
}

/* Exported entry point.  A_out / Aabs_out: n1*n2*n3*n4*n5 doubles, row-major [i1][i2][i3][i4][i5]
 * (= the paper's column-major A^{i5 i4 i3 i2 i1}).  Aabs_out may be NULL.
 * Shells [shell_lo, shell_hi) of the canonical order.  Returns the number of non-empty shells, <0 on error. */
long orc_vertex_range(const int *two_j, int two_dl,
                      const int *two_i_min, const int *n_i,
                      const int *two_k_base, const int *n_k_pad,
                      int two_x_base, int n_x_pad,
                      const double *S1, const double *S2, const double *S3, const double *S4, const double *S5,
                      const double *B2, const double *B3, const double *B4, const double *B5,
                      long shell_lo, long shell_hi, int nthreads,
                      double *A_out, double *Aabs_out)
{
    problem_t p;
    memcpy(p.two_j, two_j, sizeof p.two_j);
    p.two_dl = two_dl; p.nl = two_dl / 2 + 1;
    memcpy(p.two_i_min, two_i_min, sizeof p.two_i_min);
    memcpy(p.n_i, n_i, sizeof p.n_i);
    memcpy(p.two_k_base, two_k_base, sizeof p.two_k_base);
    memcpy(p.n_k_pad, n_k_pad, sizeof p.n_k_pad);
    p.two_x_base = two_x_base; p.n_x_pad = n_x_pad;
    p.S1 = S1; p.S2 = S2; p.S3 = S3; p.S4 = S4; p.S5 = S5;
    p.B[0] = B2; p.B[1] = B3; p.B[2] = B4; p.B[3] = B5;

    const long ntot = (long)n_i[0] * n_i[1] * n_i[2] * n_i[3] * n_i[4];
    long wmax = n_i[0];
    for (int e = 0; e < 4; ++e) wmax *= imax(n_k_pad[e], n_i[e + 1]);
    if (nthreads < 1) nthreads = 1;
    if (shell_hi - shell_lo < nthreads) nthreads = (int)imax(1, (int)(shell_hi - shell_lo));

    acc_t *part = calloc((size_t)ntot * nthreads * 2, sizeof(acc_t));
    long *cnt = calloc(nthreads, sizeof(long));
    if (!part || !cnt) return -1;
    int fail = 0;

#ifdef _OPENMP
#pragma omp parallel num_threads(nthreads)
#endif
    {
#ifdef _OPENMP
        const int tid = omp_get_thread_num();
#else
        const int tid = 0;
#endif
        acc_t *scratch[2];
        scratch[0] = malloc(sizeof(acc_t) * wmax);
        scratch[1] = malloc(sizeof(acc_t) * wmax);
        if (!scratch[0] || !scratch[1]) {
            fail = 1;
        } else {
            /* contiguous chunk of the canonical order per thread; partials are summed in thread order below */
            const long total = shell_hi - shell_lo;
            const long lo = shell_lo + total * tid / nthreads, hi = shell_lo + total * (tid + 1) / nthreads;
            acc_t *A = part + (size_t)ntot * (2 * tid), *Aabs = Aabs_out ? A + ntot : NULL;
            for (long s = lo; s < hi; ++s) {
                int o[6]; long r = s;
                for (int q = 5; q >= 0; --q) { o[q] = (int)(r % p.nl); r /= p.nl; }
                cnt[tid] += do_shell(&p, o, A, Aabs, scratch);
            }
        }
        free(scratch[0]); free(scratch[1]);
    }
    if (fail) { free(part); free(cnt); return -1; }

    long nonempty = 0;
    for (int t = 0; t < nthreads; ++t) nonempty += cnt[t];
    long q = 0;
    for (int a1 = 0; a1 < n_i[0]; ++a1) for (int a2 = 0; a2 < n_i[1]; ++a2) for (int a3 = 0; a3 < n_i[2]; ++a3)
    for (int a4 = 0; a4 < n_i[3]; ++a4) for (int a5 = 0; a5 < n_i[4]; ++a5, ++q) {
        acc_t s = 0, sa = 0;
        for (int t = 0; t < nthreads; ++t) { s += part[(size_t)ntot * (2 * t) + q]; sa += part[(size_t)ntot * (2 * t + 1) + q]; }
        const acc_t norm = sqrtl((long double)(two_i_min[0] + 2 * a1 + 1) * (two_i_min[1] + 2 * a2 + 1)
                                 * (two_i_min[2] + 2 * a3 + 1) * (two_i_min[3] + 2 * a4 + 1) * (two_i_min[4] + 2 * a5 + 1));
        A_out[q] = (double)(s * norm);
        if (Aabs_out) Aabs_out[q] = (double)(sa * norm);
    }
    free(part); free(cnt);
    return nonempty;
}
