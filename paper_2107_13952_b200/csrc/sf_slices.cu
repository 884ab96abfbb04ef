// sf_slices.cu -- step 4 of the vertex-tensor algorithm: the five {6j} tensors, one per {6j} of
// eq. (5).  Dense, FP64, x fastest:
//
//   S1[o25][a1][q5][xx]           = {i1  l25 x; k5  j14 j15}
//   S2[o35][o45][q4][q5][xx]      = {j14 k5  x; l35 k4  l45}
//   S3[o24][o34][o35][q3][q4][xx] = {k4  l35 x; k3  l24 l34}
//   S4[o23][o24][q2][q3][xx]      = {l24 k3  x; j13 k2  l23}
//   S5[o25][a1][q2][xx]           = {k2  j13 x; i1  l25 j12}
//
// o = l - j shell offsets (units of 1), a1 = (i1 - i1_min), q_a = (k_a - k_base_a) over the booster's padded k
// layout, xx = (x - x_base) over the union range of x.  Entries whose triads fail are 0.  Values are gathered from
// the resident canonical table when every argument fits in it, and evaluated directly otherwise.
#include "sf_sixj.cuh"
#include "sf_slices.cuh"

void sf_slice_sizes(const SfDims& D, SfSliceSizes* sz)
{
    const long nl = D.nl, n1 = D.n_i[0], NX = D.n_x_pad;
    const long P2 = D.n_k_pad[0], P3 = D.n_k_pad[1], P4 = D.n_k_pad[2], P5 = D.n_k_pad[3];
    sz->n[0] = nl * n1 * P5 * NX;
    sz->n[1] = nl * nl * P4 * P5 * NX;
    sz->n[2] = nl * nl * nl * P3 * P4 * NX;
    sz->n[3] = nl * nl * P2 * P3 * NX;
    sz->n[4] = nl * n1 * P2 * NX;
}

template <int WHICH>
__global__ void __launch_bounds__(128) k_slices(SliceArgs A, SfSixjTable tab, const SfFact* __restrict__ F)
{
    const long q = blockIdx.x * (long)blockDim.x + threadIdx.x;
    if (q >= A.n[WHICH]) return;
    int a, b, c, d, e, f;
    slice_args<WHICH>(A, q, a, b, c, d, e, f);
    double v;
    const int m = max(max(max(a, b), max(c, d)), max(e, f));
    if (tab.two_jmax >= 0 && m <= tab.two_jmax)
        v = sf_sixj_lookup(tab, a, b, c, d, e, f);
    else
        v = sf_sixj_eval(F, a, b, c, d, e, f);
    A.S[WHICH][q] = v;
}

int sf_build_slices(const SfDims& D, double* const S[5], const SfSixjTable& tab, cudaStream_t st)
{
    SliceArgs A;
    for (int s = 0; s < 10; ++s) A.two_j[s] = D.two_j[s];
    A.nl = D.nl;
    A.n1 = D.n_i[0];
    A.two_i1_min = D.two_i_min[0];
    for (int e = 0; e < 4; ++e) {
        A.two_k_base[e] = D.two_k_base[e];
        A.n_k_pad[e] = D.n_k_pad[e];
    }
    A.two_x_base = D.two_x_base;
    A.n_x_pad = D.n_x_pad;
    SfSliceSizes sz;
    sf_slice_sizes(D, &sz);
    for (int w = 0; w < 5; ++w) {
        A.n[w] = sz.n[w];
        A.S[w] = S[w];
    }
    const SfFact* F = sf_fact_table();
    if (!F) return SF_ENOTINIT;
#define SF_LAUNCH(W)                                                                             \
    if (A.n[W] > 0) {                                                                            \
        k_slices<W><<<(unsigned)((A.n[W] + 127) / 128), 128, 0, st>>>(A, tab, F);                \
        sf_count_launch(1);                                                                      \
    }
    SF_LAUNCH(0)
    SF_LAUNCH(1)
    SF_LAUNCH(2)
    SF_LAUNCH(3)
    SF_LAUNCH(4)
#undef SF_LAUNCH
    return cudaGetLastError() == cudaSuccess ? SF_OK : SF_ECUDA;
}
