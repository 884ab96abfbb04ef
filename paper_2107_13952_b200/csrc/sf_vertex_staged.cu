// sf_vertex_staged.cu -- the general-size path of steps 5-7 of the vertex-tensor algorithm.
//
// For tensors too large for the fused on-chip path (sf_vertex_fused.cu) the per-shell intermediates go through
// global memory, a batch of shells at a time:
//   (i)   k_stage_asm   W[s][a1][c2][c3][c4][c5] = {15j}, eq. (5) summed over x
//   (ii)+(iii) k_stage_mode, four times (k5, k4, k3, k2): one mode product with the selected booster sub-matrix
//         and the (2k+1) weights, "loop over GEMM"
//   (iv)  k_stage_acc   acc += sum over the batch, in canonical shell order (fixed order => reproducible)
//   then  k_finalize    out = acc * prod_e sqrt(2 i_e + 1)                                  (eq. (3))
// c_a = (k_a - k_min_a(shell)) is the compact index of the shell's own k-range; strides use k_max_a.  The boundary
// intertwiner i1 is a pure batch index, so a tensor that exceeds the scratch budget is split along i1 (the paper's
// own way of batching).
#include <stdio.h>

#include "sf_internal.h"

struct StageShell {   // per-shell quantities every stage kernel derives from the shell index
    int o[6], t[4], kmin[4], K[4];
    bool empty;
};
__device__ __forceinline__ void stage_shell(const SfProblem& P, long shell, StageShell& S)
{
    sf_shell_offsets(shell, P.nl, S.o);
    sf_triples(S.o, P.nl, S.t);
    S.empty = false;
#pragma unroll
    for (int e = 0; e < 4; ++e) {
        const SfKRange r = P.kr[e][S.t[e]];
        S.kmin[e] = r.two_k_min;
        S.K[e] = r.n_k;
        if (r.n_k == 0) S.empty = true;
    }
}

// (i) assembly.  grid.y = shell of the batch, threads over entries (a1 c2 c3 c4 c5) of the max-size box.
__global__ void __launch_bounds__(256) k_stage_asm(SfProblem P, long shell0, int a1_lo, int n1c, double* __restrict__ W,
                                                   long stride)
{
    StageShell S;
    stage_shell(P, shell0 + blockIdx.y, S);
    if (S.empty) return;
    const int M2 = P.k_max[0], M3 = P.k_max[1], M4 = P.k_max[2], M5 = P.k_max[3];
    const long nbox = (long)n1c * M2 * M3 * M4 * M5;
    long q = blockIdx.x * (long)blockDim.x + threadIdx.x;
    if (q >= nbox) return;
    const long q0 = q;
    const int c5 = (int)(q % M5); q /= M5;
    const int c4 = (int)(q % M4); q /= M4;
    const int c3 = (int)(q % M3); q /= M3;
    const int c2 = (int)(q % M2); q /= M2;
    const int a1 = a1_lo + (int)q;
    if (c2 >= S.K[0] || c3 >= S.K[1] || c4 >= S.K[2] || c5 >= S.K[3]) return;
    const int i1 = P.two_i_min[0] + 2 * a1;
    const int k2 = S.kmin[0] + 2 * c2, k3 = S.kmin[1] + 2 * c3, k4 = S.kmin[2] + 2 * c4, k5 = S.kmin[3] + 2 * c5;
    const int l23 = P.two_j[J23] + 2 * S.o[0], l24 = P.two_j[J24] + 2 * S.o[1], l25 = P.two_j[J25] + 2 * S.o[2];
    const int l34 = P.two_j[J34] + 2 * S.o[3], l35 = P.two_j[J35] + 2 * S.o[4], l45 = P.two_j[J45] + 2 * S.o[5];
    const int j13 = P.two_j[J13], j14 = P.two_j[J14];
    // x in the intersection of the five triads of eq. (5) that contain it
    int xlo = abs(i1 - l25), xhi = i1 + l25;
    xlo = max(xlo, abs(k5 - j14)); xhi = min(xhi, k5 + j14);
    xlo = max(xlo, abs(k4 - l35)); xhi = min(xhi, k4 + l35);
    xlo = max(xlo, abs(k3 - l24)); xhi = min(xhi, k3 + l24);
    xlo = max(xlo, abs(k2 - j13)); xhi = min(xhi, k2 + j13);
    const int nl = P.nl, n1 = P.n_i[0], NX = P.n_x_pad;
    const int P2 = P.n_k_pad[0], P3 = P.n_k_pad[1], P4 = P.n_k_pad[2], P5 = P.n_k_pad[3];
    const int q2 = (k2 - P.two_k_base[0]) >> 1, q3 = (k3 - P.two_k_base[1]) >> 1;
    const int q4 = (k4 - P.two_k_base[2]) >> 1, q5 = (k5 - P.two_k_base[3]) >> 1;
    const double* s1 = P.S[0] + (((long)S.o[2] * n1 + a1) * P5 + q5) * NX;
    const double* s2 = P.S[1] + ((((long)S.o[4] * nl + S.o[5]) * P4 + q4) * P5 + q5) * NX;
    const double* s3 = P.S[2] + (((((long)S.o[1] * nl + S.o[3]) * nl + S.o[4]) * P3 + q3) * P4 + q4) * NX;
    const double* s4 = P.S[3] + ((((long)S.o[0] * nl + S.o[1]) * P2 + q2) * P3 + q3) * NX;
    const double* s5 = P.S[4] + (((long)S.o[2] * n1 + a1) * P2 + q2) * NX;
    double w = 0.0;
    for (int x = xlo; x <= xhi; x += 2) {
        const int xx = (x - P.two_x_base) >> 1;
        w += (double)(x + 1) * s1[xx] * s2[xx] * s3[xx] * s4[xx] * s5[xx];
    }
    // (-1)^R, R = sum of all fifteen labels of the symbol (reading G1 of DESIGN.md)
    const int twoR = i1 + k2 + k3 + k4 + k5 + P.two_j[J12] + j13 + j14 + P.two_j[J15] + l23 + l24 + l25 + l34 + l35 + l45;
    if ((twoR >> 1) & 1) w = -w;
    W[blockIdx.y * stride + q0] = w;
}

// (ii)+(iii) one mode product.  e = edge index 0..3 (k2..k5) = position e+1 of the five tensor indices.
// in:  [s][outer dims][k_max_e][inner]   out: [s][outer dims][n_i_e][inner]
// outer dims are (n1c, k_max of the not-yet-contracted edges before e), inner = prod n_i of the edges after e.
#define SF_IC 8
__global__ void __launch_bounds__(128) k_stage_mode(SfProblem P, long shell0, int e, int n1c, const double* __restrict__ Tin,
                                                    double* __restrict__ Tout, long stride)
{
    extern __shared__ double Bw[];   // [n_i][K] weighted sub-matrix (2k+1) B_e[t][ii][k]
    StageShell S;
    stage_shell(P, shell0 + blockIdx.y, S);
    if (S.empty) return;
    const int K = S.K[e], N = P.n_i[e + 1], Kmax = P.k_max[e];
    {
        const int kk0 = (S.kmin[e] - P.two_k_base[e]) >> 1, Pk = P.n_k_pad[e];
        const double* Bm = sf_brow(P, e, S.t[e], 0);
        for (int q = threadIdx.x; q < N * K; q += blockDim.x) {
            const int ii = q / K, c = q % K;
            Bw[q] = (double)(S.kmin[e] + 2 * c + 1) * Bm[(long)ii * Pk + kk0 + c];
        }
    }
    __syncthreads();
    long outer = n1c, inner = 1;
    for (int m = 0; m < e; ++m) outer *= P.k_max[m];
    for (int m = e + 1; m < 4; ++m) inner *= P.n_i[m + 1];
    const long nuv = outer * inner;
    const double* in = Tin + blockIdx.y * stride;
    double* out = Tout + blockIdx.y * stride;
    for (long q = blockIdx.x * (long)blockDim.x + threadIdx.x; q < nuv; q += (long)gridDim.x * blockDim.x) {
        const long v = q % inner, u = q / inner;
        // validity of the outer compact indices for this shell
        long r = u;
        bool ok = true;
        for (int m = e - 1; m >= 0; --m) {
            if ((int)(r % P.k_max[m]) >= S.K[m]) ok = false;
            r /= P.k_max[m];
        }
        if (!ok) continue;
        const double* src = in + (u * Kmax) * inner + v;
        for (int i0 = 0; i0 < N; i0 += SF_IC) {
            double acc[SF_IC];
#pragma unroll
            for (int r2 = 0; r2 < SF_IC; ++r2) acc[r2] = 0.0;
            for (int c = 0; c < K; ++c) {
                const double x = src[c * inner];
#pragma unroll
                for (int r2 = 0; r2 < SF_IC; ++r2)
                    if (i0 + r2 < N) acc[r2] = fma(x, Bw[(i0 + r2) * K + c], acc[r2]);
            }
#pragma unroll
            for (int r2 = 0; r2 < SF_IC; ++r2)
                if (i0 + r2 < N) out[(u * N + i0 + r2) * inner + v] = acc[r2];
        }
    }
}

// (iv) accumulate the batch in canonical shell order
__global__ void __launch_bounds__(256) k_stage_acc(SfProblem P, long shell0, int nb, long nchunk, const double* __restrict__ T1,
                                                   long stride, double* __restrict__ acc)
{
    const long q = blockIdx.x * (long)blockDim.x + threadIdx.x;
    if (q >= nchunk) return;
    double a = acc[q];
    for (int s = 0; s < nb; ++s) {
        StageShell S;
        stage_shell(P, shell0 + s, S);
        if (S.empty) continue;
        a += T1[s * stride + q];
    }
    acc[q] = a;
}

// out[i1..i5] = acc * prod_e sqrt(2 i_e + 1)   (eq. (3))
__global__ void __launch_bounds__(256) k_finalize(SfProblem P, long n_out, const double* __restrict__ acc, double* __restrict__ out)
{
    const long q = blockIdx.x * (long)blockDim.x + threadIdx.x;
    if (q >= n_out) return;
    long r = q;
    double d = 1.0;
    for (int n = 4; n >= 0; --n) {
        d *= (double)(P.two_i_min[n] + 2 * (int)(r % P.n_i[n]) + 1);
        r /= P.n_i[n];
    }
    out[q] = acc[q] * sqrt(d);
}

void sf_launch_finalize(const SfProblem& P, long n_out, const double* acc, double* out, cudaStream_t st)
{
    k_finalize<<<(unsigned)((n_out + 255) / 256), 256, 0, st>>>(P, n_out, acc, out);
    sf_count_launch(1);
}

static size_t g_staged_budget = (size_t)6 << 30;   // bytes for the two ping-pong buffers
extern "C" void sf_set_staged_budget(unsigned long bytes)
{
    SfHostLock lock;
    g_staged_budget = bytes;
    sf_bump_generation();
}

int sf_vertex_staged(const SfDims& D, const SfProblem& P, long shell_lo, long shell_hi, double* out, cudaStream_t st)
{
    const long n2 = D.n_i[1], n3 = D.n_i[2], n4 = D.n_i[3], n5 = D.n_i[4];
    const long M2 = D.k_max[0], M3 = D.k_max[1], M4 = D.k_max[2], M5 = D.k_max[3];
    double* acc = (double*)sf_scratch(0, sizeof(double) * D.n_out);
    if (!acc) return SF_ENOMEM;
    SF_CUDA_OK(cudaMemsetAsync(acc, 0, sizeof(double) * D.n_out, st));
    {   // k_stage_mode keeps one booster sub-matrix (n_i x k_max doubles) in dynamic shared memory: opt in above 48 KB
        size_t need = 0;
        for (int e = 0; e < 4; ++e) {
            const size_t b = sizeof(double) * (size_t)D.n_i[e + 1] * D.k_max[e];
            if (b > need) need = b;
        }
        static SfPerContext<size_t> attr_c(48 * 1024);
        size_t& attr = attr_c.get();
        if (need > 226 * 1024) return SF_EARG;       // a booster sub-matrix beyond one SM's shared memory: not held
        if (need > attr) {
            SF_CUDA_OK(cudaFuncSetAttribute(k_stage_mode, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)need));
            attr = need;
        }
    }
    if (M2 && M3 && M4 && M5 && shell_hi > shell_lo) {
        // per-i1 size of the largest intermediate
        long per1 = M2 * M3 * M4 * M5;
        if (M2 * M3 * M4 * n5 > per1) per1 = M2 * M3 * M4 * n5;
        if (M2 * M3 * n4 * n5 > per1) per1 = M2 * M3 * n4 * n5;
        if (M2 * n3 * n4 * n5 > per1) per1 = M2 * n3 * n4 * n5;
        if (n2 * n3 * n4 * n5 > per1) per1 = n2 * n3 * n4 * n5;
        const long budget_elems = (long)(g_staged_budget / (2 * sizeof(double)));
        if (per1 > budget_elems) return SF_ENOMEM;
        int n1c = (int)(budget_elems / per1);
        if (n1c > D.n_i[0]) n1c = D.n_i[0];
        for (int a1_lo = 0; a1_lo < D.n_i[0]; a1_lo += n1c) {
            const int nc = (a1_lo + n1c <= D.n_i[0]) ? n1c : D.n_i[0] - a1_lo;
            const long stride = per1 * nc;
            long nb_max = budget_elems / stride;
            if (nb_max < 1) nb_max = 1;
            if (nb_max > 32768) nb_max = 32768;
            if (nb_max > shell_hi - shell_lo) nb_max = shell_hi - shell_lo;
            double* buf0 = (double*)sf_scratch(1, sizeof(double) * stride * nb_max);
            double* buf1 = (double*)sf_scratch(2, sizeof(double) * stride * nb_max);
            if (!buf0 || !buf1) return SF_ENOMEM;
            const long nchunk = (long)nc * n2 * n3 * n4 * n5;
            for (long s0 = shell_lo; s0 < shell_hi; s0 += nb_max) {
                const int nb = (int)((s0 + nb_max <= shell_hi) ? nb_max : shell_hi - s0);
                const long nbox = (long)nc * M2 * M3 * M4 * M5;
                k_stage_asm<<<dim3((unsigned)((nbox + 255) / 256), nb), 256, 0, st>>>(P, s0, a1_lo, nc, buf0, stride);
                double *src = buf0, *dst = buf1;
                for (int e = 3; e >= 0; --e) {
                    long outer = nc, inner = 1;
                    for (int m = 0; m < e; ++m) outer *= D.k_max[m];
                    for (int m = e + 1; m < 4; ++m) inner *= D.n_i[m + 1];
                    long blocks = (outer * inner + 127) / 128;
                    if (blocks > 4096) blocks = 4096;
                    const size_t smem = sizeof(double) * D.n_i[e + 1] * D.k_max[e];
                    k_stage_mode<<<dim3((unsigned)blocks, nb), 128, smem, st>>>(P, s0, e, nc, src, dst, stride);
                    double* t = src;
                    src = dst;
                    dst = t;
                }
                k_stage_acc<<<(unsigned)((nchunk + 255) / 256), 256, 0, st>>>(P, s0, nb, nchunk, src, stride,
                                                                              acc + (long)a1_lo * n2 * n3 * n4 * n5);
                sf_count_launch(6);
            }
        }
    }
    sf_timing_mark(2, st);
    sf_launch_finalize(P, D.n_out, acc, out, st);
    return cudaGetLastError() == cudaSuccess ? SF_OK : SF_ECUDA;
}
