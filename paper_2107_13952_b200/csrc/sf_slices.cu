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
#include <string.h>

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
__device__ __forceinline__ void slice_entry(const SliceArgs& A, const SfSixjTable& tab, const SfFact* __restrict__ F, long q)
{
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

// ONE launch for steps 2 and 4: blocks [first[w], first[w + 1]) fill S array w (w = 0..4), the blocks from first[5] on the
// k-range tables of the four edges (small problems are bound by the number of dependent launches, not by their work)
struct SliceTasks {
    long first[7];
    int nt;                 // triples per edge (nl^3); 0: no k-range task
    SfKRange* kr;
};
__global__ void __launch_bounds__(128) k_slices(SliceArgs A, SfSixjTable tab, const SfFact* __restrict__ F, SliceTasks T)
{
    const long b = blockIdx.x;
    if (b >= T.first[5]) {
        const long q = (b - T.first[5]) * 128 + threadIdx.x;
        if (q < 4L * T.nt) T.kr[q] = sf_krange_entry(A.two_j, A.nl, T.nt, (int)q);
    } else if (b < T.first[1]) {
        slice_entry<0>(A, tab, F, (b - T.first[0]) * 128 + threadIdx.x);
    } else if (b < T.first[2]) {
        slice_entry<1>(A, tab, F, (b - T.first[1]) * 128 + threadIdx.x);
    } else if (b < T.first[3]) {
        slice_entry<2>(A, tab, F, (b - T.first[2]) * 128 + threadIdx.x);
    } else if (b < T.first[4]) {
        slice_entry<3>(A, tab, F, (b - T.first[3]) * 128 + threadIdx.x);
    } else {
        slice_entry<4>(A, tab, F, (b - T.first[4]) * 128 + threadIdx.x);
    }
}

// the k-range tables alone (callers that need no S arrays)
__global__ void k_kranges(SliceArgs A, int nt, SfKRange* __restrict__ out)
{
    const int q = blockIdx.x * blockDim.x + threadIdx.x;
    if (q < 4 * nt) out[q] = sf_krange_entry(A.two_j, A.nl, nt, q);
}
void sf_launch_kranges(const SfDims& D, SfKRange* out, cudaStream_t st)
{
    SliceArgs A;
    memset(&A, 0, sizeof A);
    for (int s = 0; s < 10; ++s) A.two_j[s] = D.two_j[s];
    A.nl = D.nl;
    const int nt = D.nl * D.nl * D.nl;
    k_kranges<<<(4 * nt + 127) / 128, 128, 0, st>>>(A, nt, out);
    sf_count_launch(1);
}

int sf_build_slices(const SfDims& D, double* const S[5], const SfSixjTable& tab, SfKRange* kr, cudaStream_t st)
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
    SliceTasks T;
    T.first[0] = 0;
    for (int w = 0; w < 5; ++w) T.first[w + 1] = T.first[w] + (A.n[w] + 127) / 128;
    T.nt = kr ? D.nl * D.nl * D.nl : 0;
    T.kr = kr;
    T.first[6] = T.first[5] + (4L * T.nt + 127) / 128;
    if (T.first[6] > 2147483647L) return SF_EARG;
    if (T.first[6] > 0) {
        k_slices<<<(unsigned)T.first[6], 128, 0, st>>>(A, tab, F, T);
        sf_count_launch(1);
    }
    return cudaGetLastError() == cudaSuccess ? SF_OK : SF_ECUDA;
}
