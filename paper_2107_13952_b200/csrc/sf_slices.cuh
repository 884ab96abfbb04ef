// sf_slices.cuh -- index decoding of the five S arrays of step 4: entry q of array WHICH -> the six
// arguments of its {6j} symbol (the five {6j} of eq. (5)).  Shared by k_slices (sf_slices.cu) and the
// batched small-vertex kernel (sf_vertex_batch.cu).
#pragma once
#include "sf_internal.h"

struct SliceArgs {
    int two_j[10];
    int nl, n1, two_i1_min;
    int two_k_base[4], n_k_pad[4];
    int two_x_base, n_x_pad;
    long n[5];
    double* S[5];
};

template <int WHICH>
__device__ __forceinline__ void slice_args(const SliceArgs& A, long q, int& a, int& b, int& c, int& d, int& e, int& f)
{
    const int NX = A.n_x_pad, nl = A.nl;
    const int x = A.two_x_base + 2 * (int)(q % NX);
    q /= NX;
    const int* j = A.two_j;
    if (WHICH == 0) {          // S1[o25][a1][q5][xx] = {i1 l25 x; k5 j14 j15}
        const int k5 = A.two_k_base[3] + 2 * (int)(q % A.n_k_pad[3]);
        q /= A.n_k_pad[3];
        const int i1 = A.two_i1_min + 2 * (int)(q % A.n1);
        q /= A.n1;
        const int l25 = j[J25] + 2 * (int)q;
        a = i1; b = l25; c = x; d = k5; e = j[J14]; f = j[J15];
    } else if (WHICH == 1) {   // S2[o35][o45][q4][q5][xx] = {j14 k5 x; l35 k4 l45}
        const int k5 = A.two_k_base[3] + 2 * (int)(q % A.n_k_pad[3]);
        q /= A.n_k_pad[3];
        const int k4 = A.two_k_base[2] + 2 * (int)(q % A.n_k_pad[2]);
        q /= A.n_k_pad[2];
        const int l45 = j[J45] + 2 * (int)(q % nl);
        q /= nl;
        const int l35 = j[J35] + 2 * (int)q;
        a = j[J14]; b = k5; c = x; d = l35; e = k4; f = l45;
    } else if (WHICH == 2) {   // S3[o24][o34][o35][q3][q4][xx] = {k4 l35 x; k3 l24 l34}
        const int k4 = A.two_k_base[2] + 2 * (int)(q % A.n_k_pad[2]);
        q /= A.n_k_pad[2];
        const int k3 = A.two_k_base[1] + 2 * (int)(q % A.n_k_pad[1]);
        q /= A.n_k_pad[1];
        const int l35 = j[J35] + 2 * (int)(q % nl);
        q /= nl;
        const int l34 = j[J34] + 2 * (int)(q % nl);
        q /= nl;
        const int l24 = j[J24] + 2 * (int)q;
        a = k4; b = l35; c = x; d = k3; e = l24; f = l34;
    } else if (WHICH == 3) {   // S4[o23][o24][q2][q3][xx] = {l24 k3 x; j13 k2 l23}
        const int k3 = A.two_k_base[1] + 2 * (int)(q % A.n_k_pad[1]);
        q /= A.n_k_pad[1];
        const int k2 = A.two_k_base[0] + 2 * (int)(q % A.n_k_pad[0]);
        q /= A.n_k_pad[0];
        const int l24 = j[J24] + 2 * (int)(q % nl);
        q /= nl;
        const int l23 = j[J23] + 2 * (int)q;
        a = l24; b = k3; c = x; d = j[J13]; e = k2; f = l23;
    } else {                   // S5[o25][a1][q2][xx] = {k2 j13 x; i1 l25 j12}
        const int k2 = A.two_k_base[0] + 2 * (int)(q % A.n_k_pad[0]);
        q /= A.n_k_pad[0];
        const int i1 = A.two_i1_min + 2 * (int)(q % A.n1);
        q /= A.n1;
        const int l25 = j[J25] + 2 * (int)q;
        a = k2; b = j[J13]; c = x; d = i1; e = l25; f = j[J12];
    }
}


// ranges of the virtual intertwiners k_a for every booster triple (step 2): the node's recoupling pairs with
// the edge's three virtual spins at l = j + offset (superscript order of PAPER.md:171).  Entry q = e * nt + t.
__device__ __forceinline__ SfKRange sf_krange_entry(const int* j, int nl, int nt, int q)
{
    const int e = q / nt, t = q % nt;
    const int u = 2 * (t / (nl * nl)), v = 2 * ((t / nl) % nl), w = 2 * (t % nl);
    int a, b, c, d;
    if (e == 0) {          // node 2 (l23 l24 | l25 j12), triple (l23 l24 l25)
        a = j[J23] + u; b = j[J24] + v; c = j[J25] + w; d = j[J12];
    } else if (e == 1) {   // node 3 (l34 l35 | j13 l23), triple (l34 l35 l23)
        a = j[J34] + u; b = j[J35] + v; c = j[J13]; d = j[J23] + w;
    } else if (e == 2) {   // node 4 (l45 j14 | l24 l34), triple (l45 l24 l34)
        a = j[J45] + u; b = j[J14]; c = j[J24] + v; d = j[J34] + w;
    } else {               // node 5 (j15 l25 | l35 l45), triple (l25 l35 l45)
        a = j[J15]; b = j[J25] + u; c = j[J35] + v; d = j[J45] + w;
    }
    const int lo = max(abs(a - b), abs(c - d)), hi = min(a + b, c + d);
    SfKRange r;
    r.two_k_min = lo;
    r.n_k = (((a + b) ^ (c + d)) & 1) || hi < lo ? 0 : (hi - lo) / 2 + 1;
    return r;
}
