// sf_contract.cu -- downstream contractions of vertex tensors (Fig. 3, Listing 7; SURVEY.md K-e):
//
//   sf_contract_vertices:  sum_{i1..i5} A[i1..i5] B[i1..i5]                                   (two vertices, all five edges glued)
//   sf_contract_vectors:   sum_{i1..i5} A[i1..i5] psi1[i1] psi2[i2] psi3[i3] psi4[i4] psi5[i5] (one vertex with five complex
//                          vectors: the paper's contract(v, cs5, cs4, cs3, cs2, cs1) with coherent-state coefficients)
//
// The paper sends these to cuBLAS through CUDA.jl.  Both read every tensor entry exactly once and do
// O(1) flop per entry: they are HBM-bound, so each is one streaming pass with a fixed-order reduction (per thread in
// index order, then a shared-memory tree, then the per-CTA partial sums in CTA order): bitwise reproducible, no atomics.
#include "sf_internal.h"

#define KE_THREADS 256
#define KE_MAX_CTAS 1184   /* 8 per SM on 148 SMs: the grid depends on the size only, so the summation order is fixed */

__device__ __forceinline__ void ke_block_sum(double& re, double& im, double* sh)
{
    const int tid = threadIdx.x;
    sh[tid] = re;
    sh[KE_THREADS + tid] = im;
    __syncthreads();
    for (int s = KE_THREADS / 2; s > 0; s >>= 1) {
        if (tid < s) {
            sh[tid] += sh[tid + s];
            sh[KE_THREADS + tid] += sh[KE_THREADS + tid + s];
        }
        __syncthreads();
    }
    re = sh[0];
    im = sh[KE_THREADS];
}

// partial[cta] = sum over this CTA's entries of a[z] b[z]; entries are dealt to threads with stride gridDim * blockDim
__global__ void __launch_bounds__(KE_THREADS) k_ke_dot(const double* __restrict__ a, const double* __restrict__ b, long n,
                                                       double* __restrict__ partial, unsigned* __restrict__ ticket,
                                                       double* __restrict__ result)
{
    __shared__ double sh[2 * KE_THREADS];
    __shared__ bool last;
    double s = 0.0, unused = 0.0;
    const long stride = (long)gridDim.x * KE_THREADS;
    for (long z = (long)blockIdx.x * KE_THREADS + threadIdx.x; z < n; z += stride) s = fma(a[z], b[z], s);
    ke_block_sum(s, unused, sh);
    if (threadIdx.x == 0) {
        partial[blockIdx.x] = s;
        __threadfence();
        last = atomicAdd(ticket, 1u) == gridDim.x - 1;       // integer ticket: who finishes last is free, what it adds is not
    }
    __syncthreads();
    if (last && threadIdx.x == 0) {                           // the per-CTA partial sums in CTA order
        __threadfence();
        double t = 0.0;
        for (unsigned c = 0; c < gridDim.x; ++c) t += __ldcg(partial + c);
        result[0] = t;
        *ticket = 0;                                          // ready for the next call on this stream
    }
}

// A tile = TR consecutive rows (i1 i2 i3 i4) = TR * n5 consecutive entries: loaded coalesced into shared memory by
// cp.async one tile ahead (two buffers), then four lanes sum each row: sum_i5 A[row][i5] psi5[i5], times
// psi4[i4] psi3[i3] psi2[i2] psi1[i1].  Row stride n5 in shared memory: conflict-free for odd n5 (2j+1 values of an
// integer-spin intertwiner), at worst a few-way conflict otherwise.
#define KE_TILE 2688   /* doubles of shared memory per tile: 64 rows of up to 42 entries; two buffers, 5 CTAs per SM */
__global__ void __launch_bounds__(KE_THREADS) k_ke_vectors(const double* __restrict__ A, long rows, int n2, int n3, int n4,
                                                           int n5, int TR, const double2* __restrict__ p1,
                                                           const double2* __restrict__ p2, const double2* __restrict__ p3,
                                                           const double2* __restrict__ p4, const double2* __restrict__ p5,
                                                           double* __restrict__ partial)
{
    __shared__ __align__(16) double tiles[2][KE_TILE];
    __shared__ double2 s5[64];                       // psi5 when it has at most 64 entries; longer vectors are read from global
    const bool p5s = n5 <= 64;
    if (p5s)
        for (int e = threadIdx.x; e < n5; e += KE_THREADS) s5[e] = p5[e];
    __shared__ double sh[2 * KE_THREADS];
    double sre = 0.0, sim = 0.0;
    const long n_tiles = (rows + TR - 1) / TR;
    auto stage = [&](long t, int buf) {              // asynchronous copy of tile t (nothing if t is past the end)
        if (t < n_tiles) {
            const long r0 = t * TR;
            const int cnt = (int)min((long)TR, rows - r0) * n5;
            const double* src = A + r0 * n5;
            const unsigned dst = (unsigned)__cvta_generic_to_shared(&tiles[buf][0]);
            if ((TR & 1) == 0) {                     // an even number of rows per tile: every tile starts 16-byte aligned
                for (int e = 2 * threadIdx.x; e < cnt; e += 2 * KE_THREADS)
                    asm volatile("cp.async.cg.shared.global [%0], [%1], 16, %2;" ::"r"(dst + 8u * e), "l"(src + e),
                                 "r"(e + 1 < cnt ? 16 : 8)
                                 : "memory");
            } else {
                for (int e = threadIdx.x; e < cnt; e += KE_THREADS)
                    asm volatile("cp.async.ca.shared.global [%0], [%1], 8;" ::"r"(dst + 8u * e), "l"(src + e) : "memory");
            }
        }
        asm volatile("cp.async.commit_group;" ::: "memory");
    };
    int buf = 0;
    stage(blockIdx.x, 0);
    for (long t = blockIdx.x; t < n_tiles; t += gridDim.x, buf ^= 1) {
        const long r0 = t * TR;
        const int nr = (int)min((long)TR, rows - r0);
        stage(t + gridDim.x, buf ^ 1);               // the next tile streams in while this one is summed
        asm volatile("cp.async.wait_group 1;" ::: "memory");
        __syncthreads();
        const double* tile = tiles[buf];
        // four lanes per row, each a quarter of its entries (interleaved), combined by two shuffles in a fixed order
        const int rr = threadIdx.x >> 2, part = threadIdx.x & 3;
        double tre = 0.0, tim = 0.0;
        if (rr < nr) {
            const double* row = tile + rr * n5;
            for (int i5 = part; i5 < n5; i5 += 4) {
                const double a = row[i5];
                const double2 w = p5s ? s5[i5] : p5[i5];
                tre = fma(a, w.x, tre);
                tim = fma(a, w.y, tim);
            }
        }
        tre += __shfl_xor_sync(0xffffffffu, tre, 1);
        tim += __shfl_xor_sync(0xffffffffu, tim, 1);
        tre += __shfl_xor_sync(0xffffffffu, tre, 2);
        tim += __shfl_xor_sync(0xffffffffu, tim, 2);
        if (rr < nr && part == 0) {
            unsigned q = (unsigned)(r0 + rr);        // rows < 2^31 (checked by the caller): 32-bit divisions
            const int i4 = (int)(q % (unsigned)n4); q /= (unsigned)n4;
            const int i3 = (int)(q % (unsigned)n3); q /= (unsigned)n3;
            const int i2 = (int)(q % (unsigned)n2);
            const int i1 = (int)(q / (unsigned)n2);
            // (tre + i tim) * psi4 * psi3 * psi2 * psi1, complex products in this order
            const double2 ws[4] = {p4[i4], p3[i3], p2[i2], p1[i1]};
#pragma unroll
            for (int k = 0; k < 4; ++k) {
                const double nre = tre * ws[k].x - tim * ws[k].y, nim = tre * ws[k].y + tim * ws[k].x;
                tre = nre;
                tim = nim;
            }
            sre += tre;
            sim += tim;
        }
        __syncthreads();                             // this buffer is free for the tile after next
    }
    ke_block_sum(sre, sim, sh);
    if (threadIdx.x == 0) {
        partial[2 * blockIdx.x] = sre;
        partial[2 * blockIdx.x + 1] = sim;
    }
}


// Second kernel for vertex x five vectors (n5 <= 48, 16-byte aligned tensor): every WARP streams its own tiles of 32 rows
// (i1 i2 i3 i4) through a private double buffer filled by ONE bulk copy per tile (cp.async.bulk = SASS UBLKCP, completion on
// the buffer's mbarrier), so there is no CTA-wide barrier in the loop and a whole tile is in flight per warp while the
// previous one is summed.  Each lane owns one row: sum_i5 A[row][i5] psi5[i5] (row stride n5: conflict-free for odd n5),
// times psi4 psi3 psi2 psi1.  Fixed order: lanes in row order by shuffles, tiles in sequence per warp, warps and CTAs in
// index order; the last CTA to finish (an integer ticket) adds the per-CTA partial sums in CTA order.
#define KE2_WARPS 8
#define KE2_ROWS 32
__global__ void __launch_bounds__(32 * KE2_WARPS) k_ke_vectors2(const double* __restrict__ A, long rows, int n2, int n3, int n4,
                                                               int n5, const double2* __restrict__ p1,
                                                               const double2* __restrict__ p2, const double2* __restrict__ p3,
                                                               const double2* __restrict__ p4, const double2* __restrict__ p5,
                                                               double* __restrict__ partial, unsigned* __restrict__ ticket,
                                                               double* __restrict__ result)
{
    extern __shared__ __align__(16) double ke2_smem[];
    __shared__ __align__(8) unsigned long long bars[KE2_WARPS][2];
    __shared__ double2 s5[48];
    __shared__ double wsum[KE2_WARPS][2];
    __shared__ bool last;
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int tile_d = KE2_ROWS * n5;                         // doubles per tile
    double* buf = ke2_smem + (long)warp * 2 * tile_d;
    for (int e = threadIdx.x; e < n5; e += blockDim.x) s5[e] = p5[e];
    if (lane == 0) {
        for (int b = 0; b < 2; ++b)
            asm volatile("mbarrier.init.shared::cta.b64 [%0], 1;" ::"r"((unsigned)__cvta_generic_to_shared(&bars[warp][b])));
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();
    const long n_tiles = (rows + KE2_ROWS - 1) / KE2_ROWS;
    const long first = (long)blockIdx.x * KE2_WARPS + warp, stride = (long)gridDim.x * KE2_WARPS;
    auto stage = [&](long t, int b) {                        // lane 0: one bulk copy of tile t into buffer b
        if (t >= n_tiles) return;
        const long r0 = t * KE2_ROWS;
        const int cnt = (int)min((long)KE2_ROWS, rows - r0) * n5;
        const unsigned bar = (unsigned)__cvta_generic_to_shared(&bars[warp][b]);
        if (cnt & 1) {                                       // a short last tile that is no multiple of 16 bytes: plain copies
            double* dst = buf + (long)b * tile_d;
            for (int e = lane; e < cnt; e += 32) dst[e] = __ldg(A + r0 * n5 + e);
            __syncwarp();
            if (lane == 0) asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(bar) : "memory");
        } else if (lane == 0) {
            const unsigned bytes = 8u * (unsigned)cnt;
            asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
            asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(
                             (unsigned)__cvta_generic_to_shared(buf + (long)b * tile_d)),
                         "l"(A + r0 * n5), "r"(bytes), "r"(bar)
                         : "memory");
        }
    };
    double sre = 0.0, sim = 0.0;
    stage(first, 0);
    int it = 0;
    for (long t = first; t < n_tiles; t += stride, ++it) {
        const int b = it & 1;
        stage(t + stride, b ^ 1);                            // the next tile streams in while this one is summed
        {
            const unsigned bar = (unsigned)__cvta_generic_to_shared(&bars[warp][b]), parity = (unsigned)((it >> 1) & 1);
            unsigned done = 0;
            while (!done)
                asm volatile("{\n.reg .pred p;\nmbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\nselp.u32 %0, 1, 0, p;\n}"
                             : "=r"(done)
                             : "r"(bar), "r"(parity)
                             : "memory");
        }
        const long r0 = t * KE2_ROWS;
        const int nr = (int)min((long)KE2_ROWS, rows - r0);
        double tre = 0.0, tim = 0.0;
        if (lane < nr) {
            const double* row = buf + (long)b * tile_d + lane * n5;
            double tre2 = 0.0, tim2 = 0.0;                   // two chains per component: even and odd i5
            int i5 = 0;
            for (; i5 + 1 < n5; i5 += 2) {
                const double a0 = row[i5], a1 = row[i5 + 1];
                const double2 w0 = s5[i5], w1 = s5[i5 + 1];
                tre = fma(a0, w0.x, tre);
                tim = fma(a0, w0.y, tim);
                tre2 = fma(a1, w1.x, tre2);
                tim2 = fma(a1, w1.y, tim2);
            }
            if (i5 < n5) {
                const double a0 = row[i5];
                const double2 w0 = s5[i5];
                tre = fma(a0, w0.x, tre);
                tim = fma(a0, w0.y, tim);
            }
            tre += tre2;
            tim += tim2;
            unsigned q = (unsigned)(r0 + lane);              // rows < 2^31 (checked by the caller): 32-bit divisions
            const int i4 = (int)(q % (unsigned)n4); q /= (unsigned)n4;
            const int i3 = (int)(q % (unsigned)n3); q /= (unsigned)n3;
            const int i2 = (int)(q % (unsigned)n2);
            const int i1 = (int)(q / (unsigned)n2);
            const double2 ws[4] = {p4[i4], p3[i3], p2[i2], p1[i1]};
#pragma unroll
            for (int k = 0; k < 4; ++k) {
                const double nre = tre * ws[k].x - tim * ws[k].y, nim = tre * ws[k].y + tim * ws[k].x;
                tre = nre;
                tim = nim;
            }
        }
        __syncwarp();                                        // every lane has read the buffer before it is refilled
        // the 32 rows of the tile in a fixed (butterfly) order
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) {
            tre += __shfl_xor_sync(0xffffffffu, tre, o);
            tim += __shfl_xor_sync(0xffffffffu, tim, o);
        }
        sre += tre;
        sim += tim;
    }
    if (lane == 0) {
        wsum[warp][0] = sre;
        wsum[warp][1] = sim;
    }
    __syncthreads();
    if (threadIdx.x == 0) {
        double a = 0.0, b = 0.0;
        for (int w = 0; w < KE2_WARPS; ++w) {
            a += wsum[w][0];
            b += wsum[w][1];
        }
        partial[2 * blockIdx.x] = a;
        partial[2 * blockIdx.x + 1] = b;
        __threadfence();
        last = atomicAdd(ticket, 1u) == gridDim.x - 1;       // integer ticket: who finishes last is free, what it adds is not
    }
    __syncthreads();
    if (last && threadIdx.x < 2) {
        __threadfence();
        double s = 0.0;
        for (unsigned c = 0; c < gridDim.x; ++c) s += __ldcg(partial + 2 * c + threadIdx.x);
        result[threadIdx.x] = s;
        if (threadIdx.x == 0) *ticket = 0;                   // ready for the next call on this stream
    }
}

// result[c] = sum of partial[cta * nc + c] in CTA order
__global__ void k_ke_final(const double* __restrict__ partial, int n_ctas, int nc, double* __restrict__ result)
{
    const int c = threadIdx.x;
    if (c >= nc) return;
    double s = 0.0;
    for (int b = 0; b < n_ctas; ++b) s += partial[b * nc + c];
    result[c] = s;
}

static int ke_grid(long work)
{
    long g = (work + KE_THREADS * 4L - 1) / (KE_THREADS * 4L);
    if (g < 1) g = 1;
    if (g > KE_MAX_CTAS) g = KE_MAX_CTAS;
    return (int)g;
}

enum { KE_SLOT_TICKET = 20, KE_SLOT_PART = 21 };
// the ticket block that has been zeroed (tickets return to 0 at the end of every call); per context: the block of a new context
// may come back at the old address with other contents
static SfPerContext<unsigned*> g_ke_ticket_zeroed(nullptr);

extern "C" int sf_contract_vertices(const double* a, const double* b, long n, double* result, sf_stream_t stream)
{
    if (!a || !b || !result || n < 0) return SF_EARG;
    cudaStream_t st = (cudaStream_t)stream;
    if (sf_stream_is_captured(st)) return SF_ECAPTURE;
    SfCallGuard guard(st);
    const int grid = ke_grid(n);
    double* partial = (double*)sf_scratch(KE_SLOT_PART, sizeof(double) * 2 * KE_MAX_CTAS);
    unsigned* ticket = (unsigned*)sf_scratch(KE_SLOT_TICKET, 64);
    if (!partial || !ticket) return SF_ENOMEM;
    unsigned*& zeroed = g_ke_ticket_zeroed.get();
    if (zeroed != ticket) {
        SF_CUDA_OK(cudaMemsetAsync(ticket, 0, 64, st));
        zeroed = ticket;
    }
    k_ke_dot<<<grid, KE_THREADS, 0, st>>>(a, b, n, partial, ticket + 1, result);
    sf_count_launch(1);
    return cudaGetLastError() == cudaSuccess ? SF_OK : SF_ECUDA;
}

extern "C" int sf_contract_vectors(const double* A, const int n_i[5], const double* const psi[5], double* result,
                                   sf_stream_t stream)
{
    if (!A || !n_i || !psi || !result) return SF_EARG;
    for (int e = 0; e < 5; ++e)
        if (n_i[e] < 1 || !psi[e]) return SF_EARG;
    cudaStream_t st = (cudaStream_t)stream;
    if (sf_stream_is_captured(st)) return SF_ECAPTURE;
    SfCallGuard guard(st);
    const long rows = (long)n_i[0] * n_i[1] * n_i[2] * n_i[3];
    if (n_i[4] > KE_TILE || rows > 2147483647L) return SF_EARG;
    // warp-private bulk-copy pipeline: tiles of 32 rows are 16-byte sized and aligned (a shorter last tile is copied by hand)
    if (n_i[4] <= 48 && ((size_t)A & 15) == 0) {
        static SfPerContext<int> n_sm_c(0);
        int& n_sm = n_sm_c.get();
        if (!n_sm) {
            int dev = 0;
            SF_CUDA_OK(cudaGetDevice(&dev));
            SF_CUDA_OK(cudaDeviceGetAttribute(&n_sm, cudaDevAttrMultiProcessorCount, dev));
        }
        const size_t smem = sizeof(double) * 2 * KE2_WARPS * KE2_ROWS * (size_t)n_i[4];
        static SfPerContext<size_t> attr_c(48 * 1024);
        size_t& attr = attr_c.get();
        if (smem > attr) {
            SF_CUDA_OK(cudaFuncSetAttribute(k_ke_vectors2, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
            attr = smem;
        }
        unsigned* ticket = (unsigned*)sf_scratch(KE_SLOT_TICKET, 64);
        double* part2 = (double*)sf_scratch(KE_SLOT_PART, sizeof(double) * 2 * KE_MAX_CTAS);
        if (!ticket || !part2) return SF_ENOMEM;
        unsigned*& zeroed = g_ke_ticket_zeroed.get();
        if (zeroed != ticket) {
            SF_CUDA_OK(cudaMemsetAsync(ticket, 0, 64, st));
            zeroed = ticket;
        }
        const long nt = (rows + KE2_ROWS - 1) / KE2_ROWS;
        const int per_sm = smem <= 100 * 1024 ? 2 : 1;
        long g = (nt + KE2_WARPS - 1) / KE2_WARPS;
        if (g > (long)per_sm * n_sm) g = (long)per_sm * n_sm;
        k_ke_vectors2<<<(unsigned)g, 32 * KE2_WARPS, smem, st>>>(A, rows, n_i[1], n_i[2], n_i[3], n_i[4], (const double2*)psi[0],
                                                                  (const double2*)psi[1], (const double2*)psi[2],
                                                                  (const double2*)psi[3], (const double2*)psi[4], part2, ticket, result);
        sf_count_launch(1);
        return cudaGetLastError() == cudaSuccess ? SF_OK : SF_ECUDA;
    }
    int TR = KE_TILE / n_i[4];
    if (TR > KE_THREADS / 4) TR = KE_THREADS / 4;    // four lanes per row
    if (TR > 1) TR &= ~1;                            // even: tiles start 16-byte aligned
    const long n_tiles = (rows + TR - 1) / TR;
    const int grid = (int)(n_tiles < 740 ? n_tiles : 740);      // 5 CTAs of 47 KB per SM: one wave
    double* partial = (double*)sf_scratch(KE_SLOT_PART, sizeof(double) * 2 * KE_MAX_CTAS);
    if (!partial) return SF_ENOMEM;
    k_ke_vectors<<<grid, KE_THREADS, 0, st>>>(A, rows, n_i[1], n_i[2], n_i[3], n_i[4], TR, (const double2*)psi[0],
                                              (const double2*)psi[1], (const double2*)psi[2], (const double2*)psi[3],
                                              (const double2*)psi[4], partial);
    k_ke_final<<<1, 32, 0, st>>>(partial, grid, 2, result);
    sf_count_launch(2);
    return cudaGetLastError() == cudaSuccess ? SF_OK : SF_ECUDA;
}
