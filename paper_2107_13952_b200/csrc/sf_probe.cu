// sf_probe.cu -- measurement helpers of the C ABI: the FP64 roofline denominators measured in the
// same process as the benchmark, and the exact count of {15j} summands (terms of eq. (5)) that the
// algorithmic assembly work F_asm = 6 * n_terms is defined from.
#include "sf_internal.h"

// ---- FP64 peak: dependent chains of DFMA / DMMA.8x8x4, enough independent chains per thread to fill the pipe ----
template <int NCHAIN>
__global__ void __launch_bounds__(256) k_peak_dfma(double* out, int iters, double a, double b)
{
    double acc[NCHAIN];
#pragma unroll
    for (int i = 0; i < NCHAIN; ++i) acc[i] = threadIdx.x * 1e-3 + i;
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int i = 0; i < NCHAIN; ++i) acc[i] = fma(acc[i], a, b);
    }
    double s = 0;
#pragma unroll
    for (int i = 0; i < NCHAIN; ++i) s += acc[i];
    out[blockIdx.x * blockDim.x + threadIdx.x] = s;
}

template <int NCHAIN>
__global__ void __launch_bounds__(256) k_peak_dmma(double* out, int iters, double a, double b)
{
    double c0[NCHAIN], c1[NCHAIN];
#pragma unroll
    for (int i = 0; i < NCHAIN; ++i) {
        c0[i] = threadIdx.x * 1e-3 + i;
        c1[i] = i;
    }
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int i = 0; i < NCHAIN; ++i)
            asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1},{%2},{%3},{%0,%1};\n"
                         : "+d"(c0[i]), "+d"(c1[i])
                         : "d"(a), "d"(b));
    }
    double s = 0;
#pragma unroll
    for (int i = 0; i < NCHAIN; ++i) s += c0[i] + c1[i];
    out[blockIdx.x * blockDim.x + threadIdx.x] = s;
}

// kind 2: the inner loop of a shared-memory-fed GEMM on the FP64 tensor cores, nothing else: per k-step a warp loads 2 A and 8 B
// fragments (conflict-free LDS.64, row strides = 4 mod 16 doubles, as k_fz_gemm<FzMapR>) and issues 16 DMMA; 8 warps per CTA, two
// CTAs per SM, no global traffic, no barrier.  What this reaches is the ceiling of such a loop, below the register-only chains
// of kind 1: the MMA operands come through the shared-memory pipe.
__global__ void __launch_bounds__(256, 2) k_peak_dmma_smem(double* out, int iters)
{
    extern __shared__ __align__(16) double probe_smem[];
    double *As = probe_smem, *Bs = probe_smem + 32 * 132;
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31, g = lane >> 2, q = lane & 3;
    for (int i = tid; i < 32 * 132; i += 256) As[i] = 1.0 + 1e-9 * i;
    for (int i = tid; i < 32 * 68; i += 256) Bs[i] = 1e-9 * (i & 7);
    __syncthreads();
    double acc[2][8][2];
#pragma unroll
    for (int i = 0; i < 2; ++i)
#pragma unroll
        for (int j = 0; j < 8; ++j) acc[i][j][0] = acc[i][j][1] = 0.0;
    const double* as = As + q * 132 + warp * 16 + g;
    const double* bs = Bs + q * 68 + g;
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int ks = 0; ks < 8; ++ks) {
            double a[2], b[8];
#pragma unroll
            for (int i = 0; i < 2; ++i) a[i] = as[ks * 4 * 132 + 8 * i];
#pragma unroll
            for (int j = 0; j < 8; ++j) b[j] = bs[ks * 4 * 68 + 8 * j];
#pragma unroll
            for (int i = 0; i < 2; ++i)
#pragma unroll
                for (int j = 0; j < 8; ++j)
                    asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1},{%2},{%3},{%0,%1};\n"
                                 : "+d"(acc[i][j][0]), "+d"(acc[i][j][1])
                                 : "d"(a[i]), "d"(b[j]));
        }
    }
    double s = 0;
#pragma unroll
    for (int i = 0; i < 2; ++i)
#pragma unroll
        for (int j = 0; j < 8; ++j) s += acc[i][j][0] + acc[i][j][1];
    out[blockIdx.x * blockDim.x + threadIdx.x] = s;
}

// kind 0: DFMA (vector FP64 FMA), kind 1: DMMA (mma.sync m8n8k4 f64), kind 2: DMMA fed from shared memory.  Best of 5 launches.
extern "C" int sf_fp64_peak(int kind, double* tflops)
{
    if (!tflops || kind < 0 || kind > 2) return SF_EARG;
    int dev = 0, n_sm = 0;
    SF_CUDA_OK(cudaGetDevice(&dev));
    SF_CUDA_OK(cudaDeviceGetAttribute(&n_sm, cudaDevAttrMultiProcessorCount, dev));
    const int grid = n_sm * 4, iters = 40000;
    double* out = (double*)sf_scratch(19, sizeof(double) * grid * 256);
    if (!out) return SF_ENOMEM;
    cudaEvent_t e0, e1;
    SF_CUDA_OK(cudaEventCreate(&e0));
    SF_CUDA_OK(cudaEventCreate(&e1));
    if (kind == 2 &&
        cudaFuncSetAttribute(k_peak_dmma_smem, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)(sizeof(double) * 32 * (132 + 68))) != cudaSuccess)
        return SF_ECUDA;
    float best = 1e30f;
    for (int rep = 0; rep < 6; ++rep) {
        cudaEventRecord(e0, 0);
        if (kind == 0)
            k_peak_dfma<16><<<grid, 256>>>(out, iters, 1.0000001, 1e-9);
        else if (kind == 1)
            k_peak_dmma<8><<<grid, 256>>>(out, iters, 1.0000001, 1e-9);
        else
            k_peak_dmma_smem<<<grid, 256, sizeof(double) * 32 * (132 + 68)>>>(out, iters / 16);
        cudaEventRecord(e1, 0);
        if (cudaEventSynchronize(e1) != cudaSuccess) return SF_ECUDA;
        float ms = 0;
        cudaEventElapsedTime(&ms, e0, e1);
        if (rep > 0 && ms < best) best = ms;
    }
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    const double flop = kind == 0   ? 2.0 * 16 * iters * 256.0 * grid
                        : kind == 1 ? 2.0 * 256 * 8 * iters * 8.0 * grid
                                    : 512.0 * 128 * (iters / 16) * 8.0 * grid;   // 128 DMMA per warp and iteration, 512 flop each
    *tflops = flop / (best * 1e-3) / 1e12;
    return SF_OK;
}

// ---- number of (entry, x) summands of eq. (5) over shells [lo, hi): sum over W entries of the size of the
//      intersection of the five triads that contain x ----
__global__ void __launch_bounds__(256) k_count_terms(SfProblem P, long shell_lo, long shell_hi, unsigned long long* total)
{
    __shared__ unsigned long long s_sum;
    if (threadIdx.x == 0) s_sum = 0;
    __syncthreads();
    unsigned long long mine = 0;
    for (long shell = shell_lo + blockIdx.x; shell < shell_hi; shell += gridDim.x) {
        int o[6], t[4], kmin[4], K[4];
        sf_shell_offsets(shell, P.nl, o);
        sf_triples(o, P.nl, t);
        bool empty = false;
        for (int e = 0; e < 4; ++e) {
            const SfKRange r = P.kr[e][t[e]];
            kmin[e] = r.two_k_min;
            K[e] = r.n_k;
            if (r.n_k == 0) empty = true;
        }
        if (empty) continue;
        const int l24 = P.two_j[J24] + 2 * o[1], l25 = P.two_j[J25] + 2 * o[2], l35 = P.two_j[J35] + 2 * o[4];
        const int j13 = P.two_j[J13], j14 = P.two_j[J14];
        const int rows = P.n_i[0] * K[0] * K[1] * K[2];
        for (int r = threadIdx.x; r < rows; r += blockDim.x) {
            int z = r;
            const int c4 = z % K[2]; z /= K[2];
            const int c3 = z % K[1]; z /= K[1];
            const int c2 = z % K[0]; z /= K[0];
            const int i1 = P.two_i_min[0] + 2 * z;
            const int k2 = kmin[0] + 2 * c2, k3 = kmin[1] + 2 * c3, k4 = kmin[2] + 2 * c4;
            int lo = abs(i1 - l25), hi = i1 + l25;
            lo = max(lo, abs(k4 - l35)); hi = min(hi, k4 + l35);
            lo = max(lo, abs(k3 - l24)); hi = min(hi, k3 + l24);
            lo = max(lo, abs(k2 - j13)); hi = min(hi, k2 + j13);
            for (int c5 = 0; c5 < K[3]; ++c5) {
                const int k5 = kmin[3] + 2 * c5;
                const int l2 = max(lo, abs(k5 - j14)), h2 = min(hi, k5 + j14);
                if (h2 >= l2) mine += (unsigned long long)((h2 - l2) / 2 + 1);
            }
        }
    }
    atomicAdd(&s_sum, mine);
    __syncthreads();
    if (threadIdx.x == 0) atomicAdd(total, s_sum);
}

void sf_launch_count_terms(const SfProblem& P, long shell_lo, long shell_hi, unsigned long long* total, cudaStream_t st)
{
    long nb = shell_hi - shell_lo;
    if (nb > 148 * 64) nb = 148 * 64;
    if (nb < 1) nb = 1;
    k_count_terms<<<(unsigned)nb, 256, 0, st>>>(P, shell_lo, shell_hi, total);
}
