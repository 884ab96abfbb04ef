// sf_ranges.cpp -- host integer logic of steps 1-2 of the vertex-tensor algorithm:
// intertwiner ranges of the boundary nodes, per-triple ranges of the virtual intertwiners k_a, array sizes,
// and the algorithmic work counts bench.py divides by.
//
// Node spin orders (first pair | second pair), read off the booster index sets and the 6j triads
// of eq. (5):
//   node 1 (j12 j13 | j14 j15)   node 2 (j23 j24 | j25 j12)   node 3 (j34 j35 | j13 j23)
//   node 4 (j45 j14 | j24 j34)   node 5 (j15 j25 | j35 j45)
#include <stdlib.h>
#include <string.h>

#include <vector>

#include "sf_internal.h"

static const int NODE[5][4] = {
    {J12, J13, J14, J15}, {J23, J24, J25, J12}, {J34, J35, J13, J23}, {J45, J14, J24, J34}, {J15, J25, J35, J45}};
// virtual spins of the booster of edge a = 2..5, in the paper's superscript order
static const int TRIPLE[4][3] = {{J23, J24, J25}, {J34, J35, J23}, {J45, J24, J34}, {J25, J35, J45}};

// range of the spin that recouples (a b) with (c d); returns the count, *lo = minimum (2j units)
int sf_host_pair_range(int a, int b, int c, int d, int* lo)
{
    int l1 = abs(a - b), l2 = abs(c - d), h1 = a + b, h2 = c + d;
    int l = l1 > l2 ? l1 : l2, h = h1 < h2 ? h1 : h2;
    *lo = l;
    if (((a + b) ^ (c + d)) & 1) return 0;
    if (h < l) return 0;
    return (h - l) / 2 + 1;
}

static int node_range(const int two_l[10], int node, int* lo)
{
    const int* s = NODE[node];
    return sf_host_pair_range(two_l[s[0]], two_l[s[1]], two_l[s[2]], two_l[s[3]], lo);
}

void sf_host_kranges(const SfDims& D, int e, SfKRange* out)
{
    const int nl = D.nl;
    int l[10];
    int t = 0;
    for (int u = 0; u < nl; ++u)
        for (int v = 0; v < nl; ++v)
            for (int w = 0; w < nl; ++w, ++t) {
                memcpy(l, D.two_j, sizeof l);
                l[TRIPLE[e][0]] += 2 * u;
                l[TRIPLE[e][1]] += 2 * v;
                l[TRIPLE[e][2]] += 2 * w;
                int lo;
                int n = node_range(l, e + 1, &lo);
                out[t].two_k_min = lo;
                out[t].n_k = n;
            }
}

int sf_host_dims(const int two_j[10], int two_dl, SfDims* D)
{
    if (!two_j || !D) return SF_EARG;
    if (two_dl < 0 || (two_dl & 1)) return SF_EARG;
    for (int s = 0; s < 10; ++s)
        if (two_j[s] < 0 || two_j[s] > 4096) return SF_EARG;
    memset(D, 0, sizeof *D);
    memcpy(D->two_j, two_j, sizeof D->two_j);
    D->two_dl = two_dl;
    D->nl = two_dl / 2 + 1;
    if (D->nl > 64) return SF_EARG;   // 64^6 shells is already far beyond any feasible call
    D->n_shells = 1;
    for (int q = 0; q < 6; ++q) D->n_shells *= D->nl;
    D->n_out = 1;
    for (int n = 0; n < 5; ++n) {
        D->n_i[n] = node_range(two_j, n, &D->two_i_min[n]);
        if (D->n_i[n] == 0) return SF_ESPIN;
        D->n_out *= D->n_i[n];
    }
    const int nt = D->nl * D->nl * D->nl;
    std::vector<SfKRange> kr(nt);
    for (int e = 0; e < 4; ++e) {
        sf_host_kranges(*D, e, kr.data());
        int base = 1 << 30, top = -1, kmax = 0;
        for (int t = 0; t < nt; ++t)
            if (kr[t].n_k > 0) {
                if (kr[t].two_k_min < base) base = kr[t].two_k_min;
                int hi = kr[t].two_k_min + 2 * (kr[t].n_k - 1);
                if (hi > top) top = hi;
                if (kr[t].n_k > kmax) kmax = kr[t].n_k;
            }
        if (top < 0) {
            D->two_k_base[e] = 0;
            D->n_k_pad[e] = 0;
        } else {
            D->two_k_base[e] = base;
            D->n_k_pad[e] = (top - base) / 2 + 1;
        }
        D->k_max[e] = kmax;
    }
    // union range of x from the triad (i1 l25 x) of eq. (5)
    int lo = 1 << 30, hi = -1;
    for (int a = 0; a < D->n_i[0]; ++a)
        for (int o = 0; o < D->nl; ++o) {
            int i1 = D->two_i_min[0] + 2 * a, l25 = two_j[J25] + 2 * o;
            int d = abs(i1 - l25), s = i1 + l25;
            if (d < lo) lo = d;
            if (s > hi) hi = s;
        }
    D->two_x_base = lo;
    D->n_x_pad = (hi - lo) / 2 + 1;
    return SF_OK;
}

void sf_host_shell_offsets(const SfDims& D, long shell, int o[6]) { sf_shell_offsets(shell, D.nl, o); }

// ---------------------------------------------------------------------------------------------------------
// C ABI: pure host integer helpers
// ---------------------------------------------------------------------------------------------------------
extern "C" int sf_vertex_dims(const int two_j[10], int two_i_min[5], int n_i[5])
{
    if (!two_j || !two_i_min || !n_i) return SF_EARG;
    SfDims D;
    int rc = sf_host_dims(two_j, 0, &D);
    if (rc != SF_OK) return rc;
    memcpy(two_i_min, D.two_i_min, sizeof D.two_i_min);
    memcpy(n_i, D.n_i, sizeof D.n_i);
    return SF_OK;
}

extern "C" int sf_booster_dims(const int two_j[10], int two_dl, int edge, int* n_triples, int* n_i, int* two_k_base,
                               int* n_k_pad)
{
    if (edge < 2 || edge > 5 || !n_triples || !n_i || !two_k_base || !n_k_pad) return SF_EARG;
    SfDims D;
    int rc = sf_host_dims(two_j, two_dl, &D);
    if (rc != SF_OK) return rc;
    *n_triples = D.nl * D.nl * D.nl;
    *n_i = D.n_i[edge - 1];
    *two_k_base = D.two_k_base[edge - 2];
    *n_k_pad = D.n_k_pad[edge - 2];
    return SF_OK;
}

extern "C" int sf_booster_krange(const int two_j[10], int two_dl, int edge, int t, int* two_k_min, int* n_k)
{
    if (edge < 2 || edge > 5 || !two_k_min || !n_k) return SF_EARG;
    SfDims D;
    int rc = sf_host_dims(two_j, two_dl, &D);
    if (rc != SF_OK) return rc;
    const int nl = D.nl;
    if (t < 0 || t >= nl * nl * nl) return SF_EARG;
    int l[10];
    memcpy(l, D.two_j, sizeof l);
    const int e = edge - 2;
    l[TRIPLE[e][0]] += 2 * (t / (nl * nl));
    l[TRIPLE[e][1]] += 2 * ((t / nl) % nl);
    l[TRIPLE[e][2]] += 2 * (t % nl);
    *n_k = node_range(l, e + 1, two_k_min);
    return SF_OK;
}

// all k-ranges of one edge in one call (binding convenience; same values as sf_booster_krange)
extern "C" int sf_booster_kranges(const int two_j[10], int two_dl, int edge, int* two_k_min, int* n_k)
{
    if (edge < 2 || edge > 5 || !two_k_min || !n_k) return SF_EARG;
    SfDims D;
    int rc = sf_host_dims(two_j, two_dl, &D);
    if (rc != SF_OK) return rc;
    const int nt = D.nl * D.nl * D.nl;
    std::vector<SfKRange> kr(nt);
    sf_host_kranges(D, edge - 2, kr.data());
    for (int t = 0; t < nt; ++t) {
        two_k_min[t] = kr[t].two_k_min;
        n_k[t] = kr[t].n_k;
    }
    return SF_OK;
}

extern "C" int sf_vertex_work(const int two_j[10], int two_dl, long shell_lo, long shell_hi, double* f_con,
                              long* n_nonempty, double* n_w)
{
    SfDims D;
    int rc = sf_host_dims(two_j, two_dl, &D);
    if (rc != SF_OK) return rc;
    if (shell_lo < 0 || shell_hi > D.n_shells || shell_lo > shell_hi) return SF_EARG;
    const int nt = D.nl * D.nl * D.nl;
    std::vector<SfKRange> kr[4];
    for (int e = 0; e < 4; ++e) {
        kr[e].resize(nt);
        sf_host_kranges(D, e, kr[e].data());
    }
    const double n1 = D.n_i[0], n2 = D.n_i[1], n3 = D.n_i[2], n4 = D.n_i[3], n5 = D.n_i[4];
    double f = 0, w = 0;
    long ne = 0;
    for (long s = shell_lo; s < shell_hi; ++s) {
        int o[6], t[4];
        sf_shell_offsets(s, D.nl, o);
        sf_triples(o, D.nl, t);
        const double K2 = kr[0][t[0]].n_k, K3 = kr[1][t[1]].n_k, K4 = kr[2][t[2]].n_k, K5 = kr[3][t[3]].n_k;
        if (K2 == 0 || K3 == 0 || K4 == 0 || K5 == 0) continue;
        ++ne;
        w += n1 * K2 * K3 * K4 * K5;
        f += 2.0 * (n1 * K2 * K3 * K4 * K5 * n5 + n1 * K2 * K3 * K4 * n4 * n5 + n1 * K2 * K3 * n3 * n4 * n5 +
                    n1 * K2 * n2 * n3 * n4 * n5);
    }
    if (f_con) *f_con = f;
    if (n_nonempty) *n_nonempty = ne;
    if (n_w) *n_w = w;
    return SF_OK;
}

// ---------------------------------------------------------------------------------------------------------
// useful work of the factorised path (include/sfoam_debug.h: sf_factor_work)
// ---------------------------------------------------------------------------------------------------------
// A term of a contraction counts when the triangle inequalities among the labels of BOTH operands hold (the {6j} of
// eq. (5) vanish otherwise, and a booster entry outside its triple's k-range is zero by reading G9) and, for an
// intermediate, when at least one term reaches the entry.  Sets of k values are bit masks (n_k_pad <= 128).
namespace {
struct Bits {
    unsigned long long w[2];
    Bits() { w[0] = w[1] = 0; }
    void set(int b) { w[b >> 6] |= 1ull << (b & 63); }
    bool test(int b) const { return (w[b >> 6] >> (b & 63)) & 1ull; }
    bool meets(const Bits& o) const { return (w[0] & o.w[0]) || (w[1] & o.w[1]); }
    void join(const Bits& o) { w[0] |= o.w[0]; w[1] |= o.w[1]; }
    int count() const { return __builtin_popcountll(w[0]) + __builtin_popcountll(w[1]); }
};
inline bool tri(int a, int b, int c)
{
    const int d = a > b ? a - b : b - a;
    return !((a + b + c) & 1) && c >= d && c <= a + b;
}
}   // namespace

extern "C" int sf_factor_work(const int two_j[10], int two_dl, double mac[6], double elems[4])
{
    if (!mac || !elems) return SF_EARG;
    SfDims D;
    int rc = sf_host_dims(two_j, two_dl, &D);
    if (rc != SF_OK) return rc;
    for (int e = 0; e < 4; ++e)
        if (D.n_k_pad[e] > 128) return SF_EARG;
    const int nl = D.nl, n1 = D.n_i[0], NX = D.n_x_pad;
    const double n2 = D.n_i[1], n3 = D.n_i[2], n4 = D.n_i[3], n5 = D.n_i[4];
    const int* j = D.two_j;
    const int P2 = D.n_k_pad[0], P3 = D.n_k_pad[1], P4 = D.n_k_pad[2], P5 = D.n_k_pad[3];
    auto L = [&](int s, int o) { return j[s] + 2 * o; };
    auto K = [&](int e, int q) { return D.two_k_base[e] + 2 * q; };
    auto I1 = [&](int a) { return D.two_i_min[0] + 2 * a; };
    auto X = [&](int xx) { return D.two_x_base + 2 * xx; };
    for (int q = 0; q < 6; ++q) mac[q] = 0.0;
    for (int q = 0; q < 4; ++q) elems[q] = 0.0;

    // ---- Z = sum_k5 S2 S1 Bw5:  S1 {i1 l25 x; k5 j14 j15}, S2 {j14 k5 x; l35 k4 l45}, B5 range (j15 l25 | l35 l45)
    // nk5[o25][xx][o35][o45] = number of k5 with (k5 l25 j15), (k5 j14 x), (l35 k5 l45)
    std::vector<int> nk5((size_t)nl * NX * nl * nl, 0);
    for (int o25 = 0; o25 < nl; ++o25)
        for (int xx = 0; xx < NX; ++xx)
            for (int o35 = 0; o35 < nl; ++o35)
                for (int o45 = 0; o45 < nl; ++o45) {
                    int n = 0;
                    for (int q = 0; q < P5; ++q)
                        n += tri(K(3, q), L(J25, o25), j[J15]) && tri(K(3, q), j[J14], X(xx)) &&
                             tri(L(J35, o35), K(3, q), L(J45, o45));
                    nk5[((size_t)(o25 * NX + xx) * nl + o35) * nl + o45] = n;
                }
    // k4 sets: (j14 k4 l45) per o45, (l35 k4 x) per (o35, xx), (l24 l34 k4) per (o24, o34)
    std::vector<Bits> k4_45(nl), k4_35x((size_t)nl * NX), k4_2434((size_t)nl * nl);
    for (int q = 0; q < P4; ++q) {
        for (int o = 0; o < nl; ++o)
            if (tri(j[J14], K(2, q), L(J45, o))) k4_45[o].set(q);
        for (int o = 0; o < nl; ++o)
            for (int xx = 0; xx < NX; ++xx)
                if (tri(L(J35, o), K(2, q), X(xx))) k4_35x[(size_t)o * NX + xx].set(q);
        for (int a = 0; a < nl; ++a)
            for (int b = 0; b < nl; ++b)
                if (tri(L(J24, a), L(J34, b), K(2, q))) k4_2434[(size_t)a * nl + b].set(q);
    }
    std::vector<double> npair4(P4, 0.0);             // number of (l24 l34) pairs that allow k4
    for (int q = 0; q < P4; ++q)
        for (int a = 0; a < nl * nl; ++a) npair4[q] += k4_2434[a].test(q);
    // k3 sets: (k3 l35 l34) per (o34, o35), (k3 l24 x) per (o24, xx); l23 counts per k3: (j13 k3 l23)
    std::vector<Bits> k3_3435((size_t)nl * nl), k3_24x((size_t)nl * NX);
    std::vector<double> nl23(P3, 0.0);
    for (int q = 0; q < P3; ++q) {
        for (int a = 0; a < nl; ++a)
            for (int b = 0; b < nl; ++b)
                if (tri(K(1, q), L(J35, b), L(J34, a))) k3_3435[(size_t)a * nl + b].set(q);
        for (int a = 0; a < nl; ++a)
            for (int xx = 0; xx < NX; ++xx)
                if (tri(K(1, q), L(J24, a), X(xx))) k3_24x[(size_t)a * NX + xx].set(q);
        for (int o = 0; o < nl; ++o) nl23[q] += tri(j[J13], K(1, q), L(J23, o));
    }
    // G operands: k2 with (l23 l24 k2), (l25 j12 k2), (k2 j13 x)
    std::vector<int> nk2((size_t)nl * nl * nl * NX, 0);
    for (int o23 = 0; o23 < nl; ++o23)
        for (int o24 = 0; o24 < nl; ++o24)
            for (int o25 = 0; o25 < nl; ++o25)
                for (int xx = 0; xx < NX; ++xx) {
                    int n = 0;
                    for (int q = 0; q < P2; ++q)
                        n += tri(L(J23, o23), L(J24, o24), K(0, q)) && tri(L(J25, o25), j[J12], K(0, q)) &&
                             tri(K(0, q), j[J13], X(xx));
                    nk2[((size_t)(o23 * nl + o24) * nl + o25) * NX + xx] = n;
                }

    std::vector<Bits> zk4((size_t)nl);               // per o35: the k4 for which Z[l25 i1 l35 . k4 x] has an entry
    std::vector<Bits> k3set((size_t)nl);             // per o24: the k3 for which R[l24 l25 i1 k3 x .] has an entry
    for (int o25 = 0; o25 < nl; ++o25)
        for (int a1 = 0; a1 < n1; ++a1)
            for (int xx = 0; xx < NX; ++xx) {
                if (!tri(I1(a1), L(J25, o25), X(xx))) continue;
                // Z and Q
                for (int o35 = 0; o35 < nl; ++o35) {
                    zk4[o35] = Bits();
                    const Bits& kx = k4_35x[(size_t)o35 * NX + xx];
                    for (int o45 = 0; o45 < nl; ++o45) {
                        const int n5k = nk5[((size_t)(o25 * NX + xx) * nl + o35) * nl + o45];
                        if (!n5k) continue;
                        Bits k4;
                        k4.w[0] = kx.w[0] & k4_45[o45].w[0];
                        k4.w[1] = kx.w[1] & k4_45[o45].w[1];
                        const int c = k4.count();
                        mac[0] += (double)n5k * c * n5;
                        elems[0] += (double)c * n5;
                        zk4[o35].join(k4);
                        for (int q = 0; q < P4; ++q)
                            if (k4.test(q)) mac[1] += npair4[q] * n5 * n4;          // Q: one term per l45, all (l24 l34) of k4
                    }
                    for (int q = 0; q < P4; ++q)
                        if (zk4[o35].test(q)) elems[1] += npair4[q] * n5 * n4;
                }
                // P, R, A' per l24
                for (int o24 = 0; o24 < nl; ++o24) {
                    k3set[o24] = Bits();
                    const Bits& k3x = k3_24x[(size_t)o24 * NX + xx];
                    for (int o34 = 0; o34 < nl; ++o34) {
                        const Bits& k4a = k4_2434[(size_t)o24 * nl + o34];
                        for (int o35 = 0; o35 < nl; ++o35) {
                            Bits k4;
                            k4.w[0] = zk4[o35].w[0] & k4a.w[0];
                            k4.w[1] = zk4[o35].w[1] & k4a.w[1];
                            const int c4 = k4.count();
                            if (!c4) continue;
                            Bits k3;
                            k3.w[0] = k3x.w[0] & k3_3435[(size_t)o34 * nl + o35].w[0];
                            k3.w[1] = k3x.w[1] & k3_3435[(size_t)o34 * nl + o35].w[1];
                            const int c3 = k3.count();
                            if (!c3) continue;
                            mac[2] += (double)c3 * c4 * n5 * n4;
                            elems[2] += (double)c3 * n5 * n4;
                            k3set[o24].join(k3);
                            for (int q = 0; q < P3; ++q)
                                if (k3.test(q)) mac[3] += nl23[q] * n3 * n4 * n5;   // R: one term per (l34 l35), all l23 of k3
                        }
                    }
                    for (int q = 0; q < P3; ++q) {
                        if (!k3x.test(q)) continue;
                        for (int o23 = 0; o23 < nl; ++o23) {
                            if (!tri(j[J13], K(1, q), L(J23, o23))) continue;
                            const int n2k = nk2[((size_t)(o23 * nl + o24) * nl + o25) * NX + xx];
                            mac[4] += (double)n2k * n2;                                 // G
                            if (k3set[o24].test(q)) {
                                elems[3] += n3 * n4 * n5;
                                if (n2k) mac[5] += n2 * n3 * n4 * n5;                   // A'
                            }
                        }
                    }
                }
            }
    return SF_OK;
}

/* Number of entries of the five S arrays of step 4 in the library's dense layout: the {6j} symbols one
 * vertex call gathers or evaluates.  Host integer function (include/sfoam_debug.h). */
extern "C" long sf_slice_elems(const int two_j[10], int two_dl)
{
    SfDims D;
    if (sf_host_dims(two_j, two_dl, &D) != SF_OK) return -1;
    const long nl = D.nl, n1 = D.n_i[0], NX = D.n_x_pad;
    const long P2 = D.n_k_pad[0], P3 = D.n_k_pad[1], P4 = D.n_k_pad[2], P5 = D.n_k_pad[3];
    return nl * n1 * P5 * NX + nl * nl * P4 * P5 * NX + nl * nl * nl * P3 * P4 * NX + nl * nl * P2 * P3 * NX + nl * n1 * P2 * NX;
}
