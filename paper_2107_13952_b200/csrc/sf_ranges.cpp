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
