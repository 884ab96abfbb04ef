// sf_vertex_batch.cu -- many vertex tensors with few shells in ONE launch (the paper's own stated next step, PAPER.md:581;
// needed for graphs with internal faces, where a bulk spin is summed over and every value needs its own small vertex
// tensors).
//
// One CTA per vertex tensor runs the whole vertex-tensor algorithm on chip:
//   step 2    ranges of the virtual intertwiners per shell (integer arithmetic per shell)
//   step 4    the five S arrays of {6j} symbols into shared memory: gathered from the resident canonical table when every
//             argument fits in it, evaluated directly otherwise (double-double Racah sum, sf_sixj.cuh)
//   step 5-6  each WARP takes shells w, w + 8, ... of the canonical order: (i) W = {15j} by direct summation of eq. (5) over x,
//             (ii)-(iii) the four mode products with the shell's booster sub-matrices and the (2k+1) weights, in the order k5,
//             k4, k3, k2, ping-pong between two warp-private buffers, (iv) accumulation into the warp's partial tensor
//   step 7    out = prod_e sqrt(2 i_e + 1) * sum over the 8 partial tensors, in warp order
// The order of every sum is fixed by (two_j, two_dl) alone: bitwise reproducible.  Plain FP64 FMA arithmetic: these problems
// are far too small for MMA tiles (config 0: 243 entries per shell), the point is one launch instead of ~17 per tensor and
// no global scratch (the call is re-entrant: it touches only its arguments and a stream-ordered descriptor array).
//
// Problems whose S arrays and warp buffers exceed one SM's shared memory are handed to the single-tensor path afterwards.
#include <vector>

#include "sf_sixj.cuh"
#include "sf_slices.cuh"

#define SB_WARPS 8
#define SB_THREADS (32 * SB_WARPS)

struct SfBatchProb {
    int two_j[10];
    int nl;
    int two_i_min[5], n_i[5];
    int two_k_base[4], n_k_pad[4];
    int two_x_base, n_x_pad;
    int n_out, wmax;              // entries of the tensor; largest intermediate of a shell (entries)
    int k_cap[4], nbw;            // largest k-range of each edge; entries of a warp's weighted booster tables
    int large;                    // 1: not run by the kernel
    int s_off[6];                 // offsets (doubles) of S1..S5 in shared memory, s_off[5] = their end
    const double* B[4];
    double* out;
};

__device__ __forceinline__ int sb_pair_range(int a, int b, int c, int d, int& lo)
{
    const int l1 = abs(a - b), l2 = abs(c - d), h1 = a + b, h2 = c + d;
    lo = max(l1, l2);
    const int hi = min(h1, h2);
    if (((a + b) ^ (c + d)) & 1) return 0;
    return hi < lo ? 0 : (hi - lo) / 2 + 1;
}

// x / d for 0 <= x < 2^20 and small d through one float multiply with inv = 1 / d: exact, because the fractional part of
// (x + 0.5) / d is at least 0.5 / d, far above the rounding error of the float product
__device__ __forceinline__ int sb_div(int x, float inv) { return __float2int_rz(((float)x + 0.5f) * inv); }

template <int WHICH>
__device__ __forceinline__ void sb_fill(const SliceArgs& A, const SfSixjTable& tab, const SfFact* __restrict__ F,
                                        double* __restrict__ S, int n)
{
    for (int e = threadIdx.x; e < n; e += SB_THREADS) {
        int a, b, c, d, ee, f;
        slice_args<WHICH>(A, e, a, b, c, d, ee, f);
        const int m = max(max(max(a, b), max(c, d)), max(ee, f));
        // gathered from the resident canonical table when every argument fits in it, evaluated otherwise
        S[e] = (tab.two_jmax >= 0 && m <= tab.two_jmax) ? sf_sixj_lookup(tab, a, b, c, d, ee, f) : sf_sixj_eval(F, a, b, c, d, ee, f);
    }
}

__global__ void __launch_bounds__(SB_THREADS) k_vertex_batch(const SfBatchProb* __restrict__ probs, const SfSixjTable tab, const SfFact* __restrict__ F)
{
    extern __shared__ __align__(16) double smem[];
    __shared__ SfBatchProb p;
    if (threadIdx.x == 0) p = probs[blockIdx.x];
    __syncthreads();
    if (p.large) return;
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int nl = p.nl, n1 = p.n_i[0], NX = p.n_x_pad;
    const int P2 = p.n_k_pad[0], P3 = p.n_k_pad[1], P4 = p.n_k_pad[2], P5 = p.n_k_pad[3];

    // ---- step 4: the S arrays ----
    {
        SliceArgs A;
        for (int s = 0; s < 10; ++s) A.two_j[s] = p.two_j[s];
        A.nl = nl;
        A.n1 = n1;
        A.two_i1_min = p.two_i_min[0];
        for (int e = 0; e < 4; ++e) {
            A.two_k_base[e] = p.two_k_base[e];
            A.n_k_pad[e] = p.n_k_pad[e];
        }
        A.two_x_base = p.two_x_base;
        A.n_x_pad = NX;
        sb_fill<0>(A, tab, F, smem + p.s_off[0], p.s_off[1] - p.s_off[0]);
        sb_fill<1>(A, tab, F, smem + p.s_off[1], p.s_off[2] - p.s_off[1]);
        sb_fill<2>(A, tab, F, smem + p.s_off[2], p.s_off[3] - p.s_off[2]);
        sb_fill<3>(A, tab, F, smem + p.s_off[3], p.s_off[4] - p.s_off[3]);
        sb_fill<4>(A, tab, F, smem + p.s_off[4], p.s_off[5] - p.s_off[4]);
    }
    const double *S1 = smem + p.s_off[0], *S2 = smem + p.s_off[1], *S3 = smem + p.s_off[2], *S4 = smem + p.s_off[3],
                 *S5 = smem + p.s_off[4];
    const long pstride = 2 * p.wmax + p.n_out + p.nbw;
    double* buf0 = smem + p.s_off[5] + (long)warp * pstride;
    double* buf1 = buf0 + p.wmax;
    double* part = buf1 + p.wmax;
    double* bw = part + p.n_out;                             // the shell's four weighted booster sub-matrices
    for (int z = lane; z < p.n_out; z += 32) part[z] = 0.0;
    __syncthreads();

    // ---- steps 5-6: shells warp, warp + 8, ... of the canonical order (l45 fastest, eq. (9)) ----
    int n_shells = 1;                                        // nl <= 16: at most 2^24 shells
    for (int d = 0; d < 6; ++d) n_shells *= nl;
    const int* j = p.two_j;
    const float inl = 1.0f / (float)nl;
    for (int shell = warp; shell < n_shells; shell += SB_WARPS) {
        int o[6];
        {
            int r = shell;
#pragma unroll
            for (int d = 5; d >= 0; --d) {
                const int r2 = nl > 1 ? (r < (1 << 20) ? sb_div(r, inl) : r / nl) : 0;
                o[d] = r - r2 * nl;
                r = r2;
            }
        }
        const int l23 = j[J23] + 2 * o[0], l24 = j[J24] + 2 * o[1], l25 = j[J25] + 2 * o[2];
        const int l34 = j[J34] + 2 * o[3], l35 = j[J35] + 2 * o[4], l45 = j[J45] + 2 * o[5];
        int kmin[4], K[4];
        K[0] = sb_pair_range(l23, l24, l25, j[J12], kmin[0]);     // node 2 (l23 l24 | l25 j12)
        K[1] = sb_pair_range(l34, l35, j[J13], l23, kmin[1]);     // node 3 (l34 l35 | j13 l23)
        K[2] = sb_pair_range(l45, j[J14], l24, l34, kmin[2]);     // node 4 (l45 j14 | l24 l34)
        K[3] = sb_pair_range(j[J15], l25, l35, l45, kmin[3]);     // node 5 (j15 l25 | l35 l45)
        if (!K[0] || !K[1] || !K[2] || !K[3]) continue;           // an empty range: the shell contributes nothing (reading G10)
        const int tt[4] = {(o[0] * nl + o[1]) * nl + o[2], (o[3] * nl + o[4]) * nl + o[0], (o[5] * nl + o[1]) * nl + o[3],
                           (o[2] * nl + o[4]) * nl + o[5]};       // booster triples, superscript order of PAPER.md:171
        int lsum = 0;
        for (int s = 0; s < 4; ++s) lsum += j[s];
        lsum += l23 + l24 + l25 + l34 + l35 + l45;

        // (ii) the four booster sub-matrices of this shell with the weights of eq. (3): bw[e][ii][c] = (2k+1) B_e[t_e][ii][k]
        {
            int base = 0;
            for (int e = 0; e < 4; ++e) {
                const int N = p.n_i[e + 1], Pk = p.n_k_pad[e], Ke = K[e];
                const double* Bm = p.B[e] + ((long)tt[e] * N) * Pk + ((kmin[e] - p.two_k_base[e]) >> 1);
                const float invK = 1.0f / (float)Ke;
                for (int z = lane; z < N * Ke; z += 32) {
                    const int ii = sb_div(z, invK), c = z - ii * Ke;
                    bw[base + z] = (double)(kmin[e] + 2 * c + 1) * __ldg(Bm + ii * Pk + c);
                }
                base += p.n_i[e + 1] * p.k_cap[e];
            }
        }
        // (i) W[a1][c2][c3][c4][c5] = (-1)^R sum_x (2x+1) S1 S2 S3 S4 S5, eq. (5)
        const int EW = n1 * K[0] * K[1] * K[2] * K[3];
        {
            const float i5 = 1.0f / (float)K[3], i4 = 1.0f / (float)K[2], i3 = 1.0f / (float)K[1], i2 = 1.0f / (float)K[0];
            const int b1 = o[2] * n1, b2 = (o[4] * nl + o[5]) * P4, b3 = ((o[1] * nl + o[3]) * nl + o[4]) * P3,
                      b4 = (o[0] * nl + o[1]) * P2;
            const int kb2 = kmin[0] - p.two_k_base[0], kb3 = kmin[1] - p.two_k_base[1], kb4 = kmin[2] - p.two_k_base[2],
                      kb5 = kmin[3] - p.two_k_base[3];
            for (int e = lane; e < EW; e += 32) {
                int r = sb_div(e, i5);
                const int c5 = e - r * K[3];
                int r2 = sb_div(r, i4);
                const int c4 = r - r2 * K[2];
                r = sb_div(r2, i3);
                const int c3 = r2 - r * K[1];
                const int a1 = sb_div(r, i2), c2 = r - a1 * K[0];
                const int i1 = p.two_i_min[0] + 2 * a1;
                const int k2 = kmin[0] + 2 * c2, k3 = kmin[1] + 2 * c3, k4 = kmin[2] + 2 * c4, k5 = kmin[3] + 2 * c5;
                const int q2 = (kb2 >> 1) + c2, q3 = (kb3 >> 1) + c3, q4 = (kb4 >> 1) + c4, q5 = (kb5 >> 1) + c5;
                int xlo = abs(i1 - l25), xhi = i1 + l25;          // the five triads of eq. (5) that contain x
                xlo = max(xlo, abs(k5 - j[J14])); xhi = min(xhi, k5 + j[J14]);
                xlo = max(xlo, abs(k4 - l35)); xhi = min(xhi, k4 + l35);
                xlo = max(xlo, abs(k3 - l24)); xhi = min(xhi, k3 + l24);
                xlo = max(xlo, abs(k2 - j[J13])); xhi = min(xhi, k2 + j[J13]);
                const int xo = (xlo - p.two_x_base) >> 1;
                const double* s1 = S1 + ((b1 + a1) * P5 + q5) * NX + xo;
                const double* s2 = S2 + ((b2 + q4) * P5 + q5) * NX + xo;
                const double* s3 = S3 + ((b3 + q3) * P4 + q4) * NX + xo;
                const double* s4 = S4 + ((b4 + q2) * P3 + q3) * NX + xo;
                const double* s5 = S5 + ((b1 + a1) * P2 + q2) * NX + xo;
                double w = 0.0;
                const int nx = xhi >= xlo ? ((xhi - xlo) >> 1) + 1 : 0;
                for (int xx = 0; xx < nx; ++xx) w += (double)(xlo + 2 * xx + 1) * s1[xx] * s2[xx] * s3[xx] * s4[xx] * s5[xx];
                if (((lsum + i1 + k2 + k3 + k4 + k5) >> 1) & 1) w = -w;   // R = sum of all fifteen labels (reading G1)
                buf0[e] = w;
            }
        }
        __syncwarp();
        // (iii) the four mode products, k5 first; the current tensor has dims d[0..4]
        int d[5] = {n1, K[0], K[1], K[2], K[3]};
        double *src = buf0, *dst = buf1;
        int bbase = 0;
        for (int e = 0; e < 3; ++e) bbase += p.n_i[e + 1] * p.k_cap[e];
        for (int mode = 4; mode >= 1; --mode) {
            const int e = mode - 1, Kc = d[mode], N = p.n_i[mode];
            const double* bwe = bw + bbase;
            if (e > 0) bbase -= p.n_i[e] * p.k_cap[e - 1];
            int outer = 1, inner = 1;
            for (int m = 0; m < mode; ++m) outer *= d[m];
            for (int m = mode + 1; m < 5; ++m) inner *= d[m];
            const int total = outer * N * inner;
            const float iin = 1.0f / (float)inner, iN = 1.0f / (float)N;
            for (int z = lane; z < total; z += 32) {
                const int r = sb_div(z, iin), v = z - r * inner, u = sb_div(r, iN), ii = r - u * N;
                const double* sp = src + (u * Kc) * inner + v;
                const double* bp = bwe + ii * Kc;
                double s = 0.0;
                for (int c = 0; c < Kc; ++c) s += sp[c * inner] * bp[c];
                dst[z] = s;
            }
            d[mode] = N;
            double* t = src;
            src = dst;
            dst = t;
            __syncwarp();
        }
        // (iv) accumulate
        for (int z = lane; z < p.n_out; z += 32) part[z] += src[z];
        __syncwarp();
    }
    __syncthreads();
    // ---- step 7: fixed-order sum of the partial tensors and the normalisation of eq. (3) ----
    const double* part0 = smem + p.s_off[5] + 2 * p.wmax;
    for (int z = threadIdx.x; z < p.n_out; z += SB_THREADS) {
        double s = 0.0;
        for (int w = 0; w < SB_WARPS; ++w) s += part0[w * pstride + z];
        int r = z;
        double dd = 1.0;
        for (int n = 4; n >= 0; --n) {
            dd *= (double)(p.two_i_min[n] + 2 * (r % p.n_i[n]) + 1);
            r /= p.n_i[n];
        }
        p.out[z] = s * sqrt(dd);
    }
}

int sf_vertex_single(const int two_j[10], int two_dl, const sf_boosters* boosters, double* out, cudaStream_t st);   // sf_api.cu

/* The batched entry point behind sf_vertex_amplitude_batch (include/sfoam.h). */
int sf_vertex_batch_run(int n, const int* two_j, const int* two_dl, const sf_boosters* boosters, double* const* out,
                        cudaStream_t st)
{
    const SfFact* F = sf_fact_table();
    if (!F) return SF_ENOTINIT;
    std::vector<SfBatchProb> probs((size_t)n);
    size_t smem_max = 0;
    const size_t smem_cap = 200 * 1024;
    int n_small = 0;
    for (int q = 0; q < n; ++q) {
        SfDims D;
        const int rc = sf_host_dims(two_j + 10 * q, two_dl[q], &D);
        if (rc != SF_OK) return rc;
        {
            int m = 0;
            for (int s = 0; s < 10; ++s) m = D.two_j[s] > m ? D.two_j[s] : m;
            if (2 * (m + two_dl[q]) > SF_SIXJ_MAX_TWO_J) return SF_EARG;
        }
        if (!out[q]) return SF_EARG;
        SfBatchProb& p = probs[q];
        memset(&p, 0, sizeof p);
        memcpy(p.two_j, D.two_j, sizeof p.two_j);
        p.nl = D.nl;
        memcpy(p.two_i_min, D.two_i_min, sizeof p.two_i_min);
        memcpy(p.n_i, D.n_i, sizeof p.n_i);
        memcpy(p.two_k_base, D.two_k_base, sizeof p.two_k_base);
        memcpy(p.n_k_pad, D.n_k_pad, sizeof p.n_k_pad);
        p.two_x_base = D.two_x_base;
        p.n_x_pad = D.n_x_pad;
        for (int e = 0; e < 4; ++e) {
            if (!boosters[q].B[e]) return SF_EARG;
            p.B[e] = boosters[q].B[e];
        }
        p.out = out[q];
        SfSliceSizes sz;
        sf_slice_sizes(D, &sz);
        double wmax = D.n_i[0], tot = 0;
        for (int e = 0; e < 4; ++e) wmax *= D.k_max[e] > D.n_i[e + 1] ? D.k_max[e] : D.n_i[e + 1];
        for (int w = 0; w < 5; ++w) tot += (double)sz.n[w];
        int nbw = 0;
        for (int e = 0; e < 4; ++e) {
            p.k_cap[e] = D.k_max[e];
            nbw += D.n_i[e + 1] * D.k_max[e];
        }
        p.nbw = nbw;
        const double need = 8.0 * (tot + SB_WARPS * (2.0 * wmax + (double)D.n_out + nbw));
        bool empty = false;
        for (int e = 0; e < 4; ++e) empty |= D.k_max[e] == 0;
        if (need > (double)smem_cap || D.nl > 16 || wmax > 500000.0) {
            p.large = 1;
        } else {
            p.n_out = (int)D.n_out;
            p.wmax = empty ? 0 : (int)wmax;
            long off = 0;
            for (int w = 0; w < 5; ++w) {
                p.s_off[w] = (int)off;
                off += sz.n[w];
            }
            p.s_off[5] = (int)off;
            const size_t bytes = 8 * (size_t)(off + SB_WARPS * (2L * p.wmax + p.n_out + p.nbw));
            if (bytes > smem_max) smem_max = bytes;
            ++n_small;
        }
    }
    if (n_small > 0) {
        static SfPerContext<size_t> attr_c(48 * 1024);
        size_t& attr = attr_c.get();
        if (smem_max > attr) {
            SF_CUDA_OK(cudaFuncSetAttribute(k_vertex_batch, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_max));
            attr = smem_max;
        }
        SfBatchProb* dprobs = nullptr;
        if (cudaMallocAsync((void**)&dprobs, sizeof(SfBatchProb) * (size_t)n, st) != cudaSuccess) {
            cudaGetLastError();
            return SF_ENOMEM;
        }
        // pageable source: the copy is staged before the call returns, so `probs` may go out of scope
        SF_CUDA_OK(cudaMemcpyAsync(dprobs, probs.data(), sizeof(SfBatchProb) * (size_t)n, cudaMemcpyHostToDevice, st));
        k_vertex_batch<<<(unsigned)n, SB_THREADS, smem_max, st>>>(dprobs, sf_sixj_table_get(), F);
        sf_count_launch(1);
        SF_CUDA_OK(cudaFreeAsync(dprobs, st));
        if (cudaGetLastError() != cudaSuccess) return SF_ECUDA;
    }
    for (int q = 0; q < n; ++q)                          // tensors too large for one SM: the single-tensor path, in order
        if (probs[q].large) {
            const int rc = sf_vertex_single(two_j + 10 * q, two_dl[q], &boosters[q], out[q], st);
            if (rc != SF_OK) return rc;
        }
    return SF_OK;
}
