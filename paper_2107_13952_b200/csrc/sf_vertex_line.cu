// sf_vertex_line.cu -- the on-chip path of steps 5-7 of the vertex-tensor algorithm: kernels (b) {15j}
// assembly, (c) mode-product contraction and (d) fixed-order shell accumulation of north_star in one persistent kernel.
//
// Work unit = (block of shells with the same (l23 l24 l25), boundary intertwiner i1, batch of SLOTS values of k2
// [, sub-range of the block's lines]).  The canonical shell order (eq. (9)) has l45 fastest, so a "line" =
// the nl consecutive shells that differ only in l45, and a block = nl^2 consecutive lines.  Rows r = (s, c3): k2 slot s
// of the batch and the compact index c3 of k3; c4 = compact index of k4 inside the shell's own range.
//
//   prep Z[l25 i1 l35 l45][k4][i5][x] = (-1)^(..) sum_k5 S2 S1 (2k5+1) B5[i5,k5]      two {6j} of eq. (5)
//        contracted with the edge-5 booster (step 6(iii)).  S1, S2 and B5 depend on (l25 l35 l45, i1) only,
//        so this product is formed once per (triple, i1) by k_line_prep_z -- a precomputation like the paper's steps 3-4.
//   P1   T4[r,c4][i5] = sum_x (U[r][x] S3[c3,c4][x]) Z[c4][x][i5]     the sum over the recoupling spin x of eq. (5) with the
//        other three {6j} (U = (2x+1) S5 S4 is unit constant, S3 line constant): the {15j} of the shell, already
//        contracted over k5.  One GEMM over x per c4.
//   P2   T3[(r,i5)][i4] += sum_c4 T4 . (2k4+1) B4[i4,c4]              accumulated in registers over the shells of a line
//   G3   T2[(s,i4,i5)][i3] += sum_c3 T3 . (2k3+1) B3[i3,c3]           once per line (B3 does not depend on l45: linearity)
//   G4   A[i2][(i3,i4,i5)]  = sum_s  T2 . (2k2+1) B2[i2,k2(s)]        once per unit (B2 depends on (l23 l24 l25) only)
//
// Every product is an FP64 tensor-core MMA (mma.sync m8n8k4 f64 = SASS DMMA.8x8x4; tcgen05 has no FP64 kind).  The CTA
// is warp specialised: 15 consumer warps run P1/P2/G3/G4, one producer warp streams each shell's Z block and weighted
// B4 block from global memory into a two-stage shared-memory ring with bulk asynchronous copies (cp.async.bulk, SASS
// UBLKCP) signalled through mbarriers.  T4 lives in shared memory in MMA-fragment order (one 32-lane fragment per
// (tile, k-step), tile bases skewed) so that both the C-fragment stores of P1 and the A-fragment loads of P2 are
// bank-conflict free and need no index arithmetic.
//
// Step 6(iv), the accumulation over shells, happens on T3 / T2 / A in a fixed order (shells ascending inside a unit,
// units ascending in k_reduce_units), so the result is bitwise reproducible.  No float atomics.
#include <stdio.h>

#include "sf_internal.h"

#define LINE_CONSUMERS 480
#define LINE_WARPS 15
#define LINE_THREADS (LINE_CONSUMERS + 32)

struct LineParams {
    SfProblem P;
    long shell_lo, shell_hi;
    long blk0;                  // first block (shell_lo / nl^3)
    int n_blocks, n_batches, n_sub, n_units;
    int slots;                  // k2 values per batch
    int NXF;                    // x stride (doubles) of U, S3s, Z rows: 4 * k-steps of x, = 4 mod 8
    int KS3, KS4, LDK3, LDK4;   // k-steps of the c3 / c4 contractions (call maxima) and the booster row strides 4*KS
    int TS4, TS3;               // tile strides (doubles) of T4 (32 KS4 + 4) and of the G3 operand A3 (32 KS3)
    int mt_max;                 // row tiles of 8 a unit can have
    int jsum;                   // sum of the ten boundary spins (2j units)
    int zslab;                  // doubles of one (slab, k4) block of Z: NT8 * NXF
    int offX2, offU, offS3, offZ, offBw4, offBw3, offBw2, offRow, offSh, offBar, n_smem;   // shared-memory offsets (doubles)
    const double* Zg;           // [l25][i1][l35][l45][q4][NT8][NXF]
    const double* Bw4g;         // [t4][NT8][LDK4] weighted, compact in c4, zero padded
    double* partial;            // [n_units][n2][n3*n4*n5]
};

__device__ __forceinline__ void line_dmma(double& c0, double& c1, double a, double b)
{
    asm("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1},{%2},{%3},{%0,%1};\n"
        : "+d"(c0), "+d"(c1)
        : "d"(a), "d"(b));
}

// ---- mbarrier / bulk-copy primitives (PTX ISA: mbarrier, cp.async.bulk) ----
__device__ __forceinline__ unsigned smem_u32(const void* p) { return (unsigned)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(unsigned bar, unsigned count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count));
}
__device__ __forceinline__ void mbar_arrive(unsigned bar)
{
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(bar) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(unsigned bar, unsigned bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(unsigned bar, unsigned parity)
{
    unsigned done = 0;
    for (unsigned spin = 0; !done; ++spin) {
        asm volatile(
            "{\n.reg .pred p;\n"
            "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n"
            "selp.u32 %0, 1, 0, p;\n}"
            : "=r"(done)
            : "r"(bar), "r"(parity)
            : "memory");
        if (spin > (1u << 28)) __trap();   // a lost signal must fail the launch, never hang the device
    }
}
__device__ __forceinline__ void bulk_g2s(unsigned dst, const void* src, unsigned bytes, unsigned bar)
{
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(dst),
                 "l"(src), "r"(bytes), "r"(bar)
                 : "memory");
}
__device__ __forceinline__ void consumer_bar() { asm volatile("bar.sync 1, %0;" ::"n"(LINE_CONSUMERS) : "memory"); }

// ---------------------------------------------------------------------------------------------------------
// precomputation: Z and the weighted edge-4 booster blocks
// ---------------------------------------------------------------------------------------------------------
// Z[slab][q4][n][v], slab = ((o25 n1 + a1) nl + o35) nl + o45, x = |i1 - l25| + 2v:
//   (-1)^(o25+o35+o45+q4) sum_{k5 valid} (-1)^q5 {j14 k5 x; l35 k4 l45} {i1 l25 x; k5 j14 j15} (2k5+1) B5[t5][n][q5]
// one CTA per (slab, q4), one thread per (n, v).
__global__ void k_line_prep_z(SfProblem P, int NT8, int NXF, double* __restrict__ Z)
{
    const int nl = P.nl, n1 = P.n_i[0], n5 = P.n_i[4], P4 = P.n_k_pad[2], P5 = P.n_k_pad[3], NX = P.n_x_pad;
    long b = blockIdx.x;
    const int q4 = (int)(b % P4);
    b /= P4;
    const long slab = b;
    const int o45 = (int)(b % nl);
    b /= nl;
    const int o35 = (int)(b % nl);
    b /= nl;
    const int a1 = (int)(b % n1);
    const int o25 = (int)(b / n1);
    const int v = threadIdx.x % NXF, n = threadIdx.x / NXF;
    const int i1 = P.two_i_min[0] + 2 * a1, l25 = P.two_j[J25] + 2 * o25;
    const int x0 = abs(i1 - l25), nxs = ((i1 + l25 - x0) >> 1) + 1;
    const int xg = ((x0 - P.two_x_base) >> 1) + v;
    const int t5 = (o25 * nl + o35) * nl + o45;
    const SfKRange r5 = P.kr[3][t5];
    double val = 0.0;
    if (n < n5 && v < nxs && r5.n_k > 0) {
        const int q5b = (r5.two_k_min - P.two_k_base[3]) >> 1;
        const double* s2 = P.S[1] + ((((long)(o35 * nl + o45) * P4 + q4) * P5 + q5b) * NX) + xg;
        const double* s1 = P.S[0] + (((long)(o25 * n1 + a1) * P5 + q5b) * NX) + xg;
        const double* b5 = sf_brow(P, 3, t5, n) + q5b;
        for (int c = 0; c < r5.n_k; ++c) {
            double term = s2[(long)c * NX] * s1[(long)c * NX] * ((double)(r5.two_k_min + 2 * c + 1) * b5[c]);
            if ((q5b + c) & 1) term = -term;
            val += term;
        }
        if ((o25 + o35 + o45 + q4) & 1) val = -val;
    }
    Z[(slab * P4 + q4) * (long)(NT8 * NXF) + threadIdx.x] = val;
}

// Bw4[t4][n][c] = (2k4+1) B4[t4][n][q4b + c] for c < K4(t4), n < n4; zero elsewhere.  One CTA per triple.
__global__ void k_line_prep_b4(SfProblem P, int NT8, int LDK4, double* __restrict__ Bw4)
{
    const int t4 = blockIdx.x, n4 = P.n_i[3], P4 = P.n_k_pad[2];
    const SfKRange r4 = P.kr[2][t4];
    const int q4b = (r4.two_k_min - P.two_k_base[2]) >> 1;
    for (int e = threadIdx.x; e < NT8 * LDK4; e += blockDim.x) {
        const int n = e / LDK4, c = e - n * LDK4;
        double val = 0.0;
        if (n < n4 && c < r4.n_k) val = (double)(r4.two_k_min + 2 * c + 1) * sf_brow(P, 2, t4, n)[q4b + c];
        Bw4[(long)t4 * NT8 * LDK4 + e] = val;
    }
}

// ---------------------------------------------------------------------------------------------------------
// the persistent kernel
// ---------------------------------------------------------------------------------------------------------
struct LineUnit {
    long blk, s_begin, s_end;
    int a1, o23, o24, o25, cb, nslots, q2b, k2min, i1, l25, x0, nxs, ksx, xg0;
    bool empty;
};

__device__ __forceinline__ void line_unit(const LineParams& lp, int unit, LineUnit& u)
{
    const SfProblem& P = lp.P;
    const int nl = P.nl, n1 = P.n_i[0];
    int r_ = unit;
    const int sub = r_ % lp.n_sub; r_ /= lp.n_sub;
    const int batch = r_ % lp.n_batches; r_ /= lp.n_batches;
    u.a1 = r_ % n1;
    u.blk = lp.blk0 + r_ / n1;
    u.o25 = (int)(u.blk % nl);
    u.o24 = (int)((u.blk / nl) % nl);
    u.o23 = (int)(u.blk / ((long)nl * nl));
    const SfKRange r2 = P.kr[0][u.blk];
    u.cb = batch * lp.slots;
    u.nslots = min(lp.slots, r2.n_k - u.cb);
    u.k2min = r2.two_k_min;
    u.q2b = (r2.two_k_min - P.two_k_base[0]) >> 1;
    const int nl2 = nl * nl;
    const long nl3 = (long)nl2 * nl;
    u.s_begin = max(u.blk * nl3 + (long)(sub * nl2 / lp.n_sub) * nl, lp.shell_lo);
    u.s_end = min(u.blk * nl3 + (long)((sub + 1) * nl2 / lp.n_sub) * nl, lp.shell_hi);
    u.i1 = P.two_i_min[0] + 2 * u.a1;
    u.l25 = P.two_j[J25] + 2 * u.o25;
    u.x0 = abs(u.i1 - u.l25);                        // the triad (i1 l25 x) of eq. (5)
    u.nxs = ((u.i1 + u.l25 - u.x0) >> 1) + 1;
    u.ksx = (u.nxs + 3) >> 2;
    u.xg0 = (u.x0 - P.two_x_base) >> 1;
    u.empty = u.nslots <= 0 || u.s_begin >= u.s_end;
}

template <int NT, int TPW>
__global__ void __launch_bounds__(LINE_THREADS, 1) k_vertex_line(const LineParams lp)
{
    extern __shared__ __align__(16) double smem[];
    const SfProblem& P = lp.P;
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31, g = lane >> 2, q = lane & 3;
    constexpr int NT8 = NT * 8;
    const int NXF = lp.NXF, SLOTS = lp.slots, TS4 = lp.TS4, TS3 = lp.TS3, LDK3 = lp.LDK3, LDK4 = lp.LDK4;
    double* T4 = smem;                               // fragment-major [tile (mt,i5)][k-step][lane]; at a line's end A3
    double* X2 = smem + lp.offX2;                    // T2 sums [SLOTS][n3][n4*n5]
    double* U = smem + lp.offU;                      // [SLOTS*P3 + 1][NXF], last row zero
    double* S3s = smem + lp.offS3;                   // [K3][P4][NXF]
    double* Zs = smem + lp.offZ;                     // [2][K4max][NT8][NXF]
    double* Bw4s = smem + lp.offBw4;                 // [2][NT8][LDK4]
    double* Bw3 = smem + lp.offBw3;                  // [NT8][LDK3]
    double* Bw2 = smem + lp.offBw2;                  // [n2][SLOTS]
    int2* rowtab = (int2*)(smem + lp.offRow);        // per row: offsets of its U row and S3s row
    int2* rowsc = rowtab + lp.mt_max * 8;            // per row: (s, c3), s = -1 beyond the line's rows
    int2* shtab = (int2*)(smem + lp.offSh);          // [2][nl + 1]: per shell of the line (K4 or 0, q4b); [nl].x = count
    const unsigned bar0 = smem_u32(smem + lp.offBar);   // full[0], full[1], empty[0], empty[1]
    const int nl = P.nl, n1 = P.n_i[0], n2 = P.n_i[1], n3 = P.n_i[2], n4 = P.n_i[3], n5 = P.n_i[4];
    const int n45 = n4 * n5, R = n3 * n45, NX = P.n_x_pad;
    const int P2 = P.n_k_pad[0], P3 = P.n_k_pad[1], P4 = P.n_k_pad[2];
    const long nl3 = (long)nl * nl * nl;
    const int zstage = P.k_max[2] * lp.zslab, bstage = NT8 * LDK4;

    for (int z = tid; z < lp.n_smem; z += LINE_THREADS) smem[z] = 0.0;   // padding must hold finite values
    __syncthreads();
    if (tid == 0) {
        mbar_init(bar0, 1);
        mbar_init(bar0 + 8, 1);
        mbar_init(bar0 + 16, LINE_WARPS);
        mbar_init(bar0 + 24, LINE_WARPS);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();

    // =====================================================================================================
    // producer warp: for every non-empty shell of this CTA's units, in order, one Z block and one B4 block
    // =====================================================================================================
    if (warp == LINE_WARPS) {
        int st = 0;
        unsigned pe0 = 1, pe1 = 1;                   // a fresh barrier passes a wait on parity 1
        for (int unit = blockIdx.x; unit < lp.n_units; unit += gridDim.x) {
            LineUnit u;
            line_unit(lp, unit, u);
            if (u.empty) continue;
            const long slab0 = (long)(u.o25 * n1 + u.a1) * nl;
            for (long base = u.s_begin; base < u.s_end; base += 32) {
                const long shell = base + lane;
                bool ne = false;
                long zoff = 0;
                int zbytes = 0, boff = 0;
                if (shell < u.s_end) {
                    const int r = (int)(shell % nl3);
                    const int o45 = r % nl, o35 = (r / nl) % nl, o34 = r / (nl * nl);
                    const int t3 = (o34 * nl + o35) * nl + u.o23, t4 = (o45 * nl + u.o24) * nl + o34;
                    const int t5 = (u.o25 * nl + o35) * nl + o45;
                    const SfKRange r3 = P.kr[1][t3], r4 = P.kr[2][t4], r5 = P.kr[3][t5];
                    ne = r3.n_k > 0 && r4.n_k > 0 && r5.n_k > 0;
                    const int q4b = (r4.two_k_min - P.two_k_base[2]) >> 1;
                    zoff = (((slab0 + o35) * nl + o45) * P4 + q4b) * (long)lp.zslab;
                    zbytes = r4.n_k * lp.zslab * 8;
                    boff = t4 * bstage;
                }
                unsigned mask = __ballot_sync(0xffffffffu, ne);
                while (mask) {
                    const int l = __ffs(mask) - 1;
                    mask &= mask - 1;
                    const long zo = __shfl_sync(0xffffffffu, zoff, l);
                    const int zb = __shfl_sync(0xffffffffu, zbytes, l), bo = __shfl_sync(0xffffffffu, boff, l);
                    if (lane == 0) {
                        const unsigned full = bar0 + 8 * st, empty = bar0 + 16 + 8 * st;
                        mbar_wait(empty, st ? pe1 : pe0);
                        mbar_expect_tx(full, (unsigned)zb + (unsigned)bstage * 8u);
                        bulk_g2s(smem_u32(Zs + st * zstage), lp.Zg + zo, (unsigned)zb, full);
                        bulk_g2s(smem_u32(Bw4s + st * bstage), lp.Bw4g + bo, (unsigned)bstage * 8u, full);
                    }
                    if (st) pe1 ^= 1; else pe0 ^= 1;
                    st ^= 1;
                }
            }
        }
        return;
    }

    // =====================================================================================================
    // consumer warps
    // =====================================================================================================
    int st = 0;
    unsigned pf0 = 0, pf1 = 0;
    int lbuf = 0;                                    // shell-table buffer of the current line
    int tbase[TPW];                                  // fragment address of this warp's T4 tiles (tile = warp + 16 j)
#pragma unroll
    for (int j = 0; j < TPW; ++j) {
        const int tl = warp + LINE_WARPS * j;
        tbase[j] = tl * TS4 + (((tl % n5) >> 1) & 3) + lane;
    }
    const int st_thread = 2 * q * TS4 + q + 4 * g;   // C-fragment store offset of this lane inside a row tile group

    for (int unit = blockIdx.x; unit < lp.n_units; unit += gridDim.x) {
        LineUnit u;
        line_unit(lp, unit, u);
        double* dst = lp.partial + (long)unit * n2 * R;
        if (u.empty) {                               // uniform over the CTA
            for (int z = tid; z < n2 * R; z += LINE_CONSUMERS) dst[z] = 0.0;
            continue;
        }
        const int nslots = u.nslots, nxs = u.nxs, KSX = u.ksx, xg0 = u.xg0;
        // (-1)^R, 2R = sum of all fifteen labels (reading G1) = jsum + i1 + sum_a base_a + 2 (sum o + sum q_a)
        const int h0 = (lp.jsum + u.i1 + P.two_k_base[0] + P.two_k_base[1] + P.two_k_base[2] + P.two_k_base[3]) >> 1;
        consumer_bar();                              // the previous unit's G4 has read X2 and Bw2

        // ---- unit constants: U = (-1)^(h0+o23+o24+q2+q3) (2x+1) S5 S4, weighted B2, zeroed T2 sums ----
        {
            const int cq2 = u.q2b + u.cb;
            const double* s5 = P.S[4] + (((long)u.o25 * n1 + u.a1) * P2 + cq2) * NX + xg0;
            const double* s4 = P.S[3] + ((((long)u.o23 * nl + u.o24) * P2 + cq2) * P3) * NX + xg0;
            const int par = h0 + u.o23 + u.o24 + cq2;
            for (int e = tid; e < SLOTS * P3 * NXF; e += LINE_CONSUMERS) {
                const int v = e % NXF, r = e / NXF, q3 = r % P3, s = r / P3;
                double val = 0.0;
                if (s < nslots && v < nxs) {
                    val = (double)(u.x0 + 2 * v + 1) * s5[(long)s * NX + v] * s4[((long)s * P3 + q3) * NX + v];
                    if ((par + s + q3) & 1) val = -val;
                }
                U[e] = val;
            }
            for (int e = tid; e < n2 * SLOTS; e += LINE_CONSUMERS) {
                const int s = e % SLOTS, i2 = e / SLOTS;
                Bw2[e] = s < nslots ? (double)(u.k2min + 2 * (u.cb + s) + 1) * sf_brow(P, 0, u.blk, i2)[u.q2b + u.cb + s] : 0.0;
            }
            for (int e = tid; e < SLOTS * R; e += LINE_CONSUMERS) X2[e] = 0.0;
        }

        double acc3[TPW][NT][2];
#pragma unroll
        for (int j = 0; j < TPW; ++j)
#pragma unroll
            for (int nt = 0; nt < NT; ++nt) acc3[j][nt][0] = acc3[j][nt][1] = 0.0;

        for (long line = u.s_begin / nl; line * nl < u.s_end; ++line) {
            // ---- line constants (step 2 ranges of the line, S3, weighted B3, row tables) ----
            const int rl = (int)((line * nl) % nl3);
            const int o35 = (rl / nl) % nl, o34 = rl / (nl * nl);
            const int t3 = (o34 * nl + o35) * nl + u.o23;
            const SfKRange r3 = P.kr[1][t3];
            const int K3 = r3.n_k;
            if (K3 == 0) continue;                   // uniform
            const int q3b = (r3.two_k_min - P.two_k_base[1]) >> 1;
            const int rows1 = nslots * K3, MT1 = (rows1 + 7) >> 3;
            lbuf ^= 1;
            int2* sh = shtab + lbuf * (nl + 1);
            if (warp == 0) {
                const long shell = line * nl + lane;
                int K4 = 0, q4b = 0;
                if (lane < nl && shell >= u.s_begin && shell < u.s_end) {
                    const int t4 = (lane * nl + u.o24) * nl + o34, t5 = (u.o25 * nl + o35) * nl + lane;
                    const SfKRange r4 = P.kr[2][t4], r5 = P.kr[3][t5];
                    if (r4.n_k > 0 && r5.n_k > 0) {
                        K4 = r4.n_k;
                        q4b = (r4.two_k_min - P.two_k_base[2]) >> 1;
                    }
                }
                const unsigned any = __ballot_sync(0xffffffffu, K4 > 0);
                if (lane < nl) sh[lane] = make_int2(K4, q4b);
                if (lane == 0) sh[nl] = make_int2(__popc(any), 0);
            }
            {
                const double* s3 = P.S[2] + (((((long)u.o24 * nl + o34) * nl + o35) * P3 + q3b) * P4) * NX + xg0;
                const bool neg = o34 & 1;
                for (int e = tid; e < K3 * P4 * NXF; e += LINE_CONSUMERS) {
                    const int v = e % NXF, r = e / NXF;
                    double val = v < nxs ? s3[(long)r * NX + v] : 0.0;
                    S3s[e] = neg ? -val : val;
                }
                for (int e = tid; e < NT8 * LDK3; e += LINE_CONSUMERS) {
                    const int ii = e / LDK3, c = e - ii * LDK3;
                    Bw3[e] = (ii < n3 && c < K3)
                                 ? (double)(r3.two_k_min + 2 * c + 1) * sf_brow(P, 1, t3, ii)[q3b + c]
                                 : 0.0;
                }
                for (int row = tid; row < lp.mt_max * 8; row += LINE_CONSUMERS) {
                    if (row < rows1) {
                        const int s = row / K3, c3 = row - s * K3;
                        rowtab[row] = make_int2((s * P3 + q3b + c3) * NXF, c3 * P4 * NXF);
                        rowsc[row] = make_int2(s, c3);
                    } else {
                        rowtab[row] = make_int2(SLOTS * P3 * NXF, 0);
                        rowsc[row] = make_int2(-1, 0);
                    }
                }
            }
            consumer_bar();
            if (sh[nl].x == 0) continue;             // no shell of this line is in range and non-empty (uniform)

            const int mt0 = warp % MT1, c40 = warp / MT1, dm = LINE_WARPS % MT1, dc = LINE_WARPS / MT1;
            const int ntiles2 = MT1 * n5;

            for (int o45 = 0; o45 < nl; ++o45) {
                const int2 shd = sh[o45];
                const int K4 = shd.x, q4b = shd.y;
                if (K4 == 0) continue;               // uniform
                mbar_wait(bar0 + 8 * st, st ? pf1 : pf0);
                if (st) pf1 ^= 1; else pf0 ^= 1;
                const double* Zc = Zs + st * zstage;

                // ---- P1: T4[r,c4][i5] = sum_x (U S3) Z, C fragments stored in fragment order ----
                for (int mt = mt0, c4 = c40; c4 < K4;) {
                    const int2 ro = rowtab[mt * 8 + g];
                    const double* up = U + ro.x + q;
                    const double* sp = S3s + ro.y + (q4b + c4) * NXF + q;
                    const double* zp = Zc + (c4 * NT8 + g) * NXF + q;
                    double c[NT][2];
#pragma unroll
                    for (int nt = 0; nt < NT; ++nt) c[nt][0] = c[nt][1] = 0.0;
                    for (int ks = 0; ks < KSX; ++ks) {
                        const double av = up[4 * ks] * sp[4 * ks];
#pragma unroll
                        for (int nt = 0; nt < NT; ++nt) line_dmma(c[nt][0], c[nt][1], av, zp[nt * 8 * NXF + 4 * ks]);
                    }
                    double* t4 = T4 + mt * n5 * TS4 + st_thread + ((c4 >> 2) << 5) + (c4 & 3);
#pragma unroll
                    for (int nt = 0; nt < NT; ++nt) {
                        const int i5 = nt * 8 + 2 * q;
                        if (i5 < n5) t4[(nt * 8) * TS4] = c[nt][0];
                        if (i5 + 1 < n5) t4[(nt * 8 + 1) * TS4] = c[nt][1];
                    }
                    mt += dm;
                    c4 += dc;
                    if (mt >= MT1) {
                        mt -= MT1;
                        ++c4;
                    }
                }
                consumer_bar();

                // ---- P2: T3 += sum_c4 T4 . (2k4+1) B4, accumulated in registers over the line ----
                {
                    const double* bw = Bw4s + st * bstage + g * LDK4 + q;
                    const int ks4 = (K4 + 3) >> 2;
                    for (int ks = 0; ks < ks4; ++ks) {
                        double bq[NT];
#pragma unroll
                        for (int nt = 0; nt < NT; ++nt) bq[nt] = bw[nt * 8 * LDK4 + 4 * ks];
#pragma unroll
                        for (int j = 0; j < TPW; ++j) {
                            if (warp + LINE_WARPS * j < ntiles2) {
                                const double av = T4[tbase[j] + (ks << 5)];
#pragma unroll
                                for (int nt = 0; nt < NT; ++nt) line_dmma(acc3[j][nt][0], acc3[j][nt][1], av, bq[nt]);
                            }
                        }
                    }
                }
                __syncwarp();
                if (lane == 0) mbar_arrive(bar0 + 16 + 8 * st);      // this warp is done with the stage
                st ^= 1;
                consumer_bar();
            }

            // ---- G3 (once per line): T2 sums += sum_c3 T3 . (2k3+1) B3 ----
            {
#pragma unroll
                for (int j = 0; j < TPW; ++j) {
                    const int tl = warp + LINE_WARPS * j;
                    if (tl < ntiles2) {
                        const int mt = tl / n5, i5 = tl - mt * n5;
                        const int2 sc = rowsc[mt * 8 + g];
                        if (sc.x >= 0) {
                            const int kof = ((sc.y >> 2) << 5) + (sc.y & 3);
#pragma unroll
                            for (int nt = 0; nt < NT; ++nt)
#pragma unroll
                                for (int b = 0; b < 2; ++b) {
                                    const int i4 = nt * 8 + 2 * q + b;
                                    if (i4 < n4) {
                                        const int m3 = (sc.x * n4 + i4) * n5 + i5;
                                        T4[(m3 >> 3) * TS3 + kof + ((m3 & 7) << 2)] = acc3[j][nt][b];
                                    }
                                }
                        }
                    }
#pragma unroll
                    for (int nt = 0; nt < NT; ++nt) acc3[j][nt][0] = acc3[j][nt][1] = 0.0;
                }
                consumer_bar();
                const int rows3 = nslots * n45, ntiles3 = (rows3 + 7) >> 3, ks3 = (K3 + 3) >> 2;
#pragma unroll
                for (int j = 0; j < TPW; ++j) {
                    const int tile = warp + LINE_WARPS * j;
                    if (tile < ntiles3) {
                        double c[NT][2];
#pragma unroll
                        for (int nt = 0; nt < NT; ++nt) c[nt][0] = c[nt][1] = 0.0;
                        for (int ks = 0; ks < ks3; ++ks) {
                            const double av = T4[tile * TS3 + (ks << 5) + lane];
#pragma unroll
                            for (int nt = 0; nt < NT; ++nt)
                                line_dmma(c[nt][0], c[nt][1], av, Bw3[(nt * 8 + g) * LDK3 + 4 * ks + q]);
                        }
                        const int r = tile * 8 + g;
                        if (r < rows3) {
                            const int s = r / n45, m = r - s * n45;
                            double* x2 = X2 + (long)s * R + m;
#pragma unroll
                            for (int nt = 0; nt < NT; ++nt) {
                                const int i3 = nt * 8 + 2 * q;
                                if (i3 < n3) x2[(long)i3 * n45] += c[nt][0];
                                if (i3 + 1 < n3) x2[(long)(i3 + 1) * n45] += c[nt][1];
                            }
                        }
                    }
                }
                consumer_bar();
            }
        }

        // ---- G4 (once per unit): contract k2; the unit's tensor goes to partial[unit] ----
        for (int z = tid; z < n2 * R; z += LINE_CONSUMERS) {
            const int i2 = z / R, r = z - i2 * R;
            double sum = 0.0;
            for (int s = 0; s < nslots; ++s) sum = fma(Bw2[i2 * SLOTS + s], X2[(long)s * R + r], sum);
            dst[z] = sum;
        }
    }
}

// kernel (d): out[a1][i2][r] = prod_e sqrt(2 i_e + 1) * sum over the units of a1, in unit order, of partial[unit][i2][r]
// (step 6(iv) + the normalisation of eq. (3))
__global__ void __launch_bounds__(256) k_reduce_units(SfProblem P, int n_blocks, int per_block, long n_out,
                                                      const double* __restrict__ partial, double* __restrict__ out)
{
    const long z = blockIdx.x * (long)blockDim.x + threadIdx.x;
    if (z >= n_out) return;
    const int n1 = P.n_i[0];
    const long slice = n_out / n1;
    const long a1 = z / slice, rest = z - a1 * slice;
    double s = 0.0;
    for (int b = 0; b < n_blocks; ++b) {
        const double* p = partial + (((long)b * n1 + a1) * per_block) * slice + rest;
        for (int u = 0; u < per_block; ++u) s += p[(long)u * slice];
    }
    long r = z;
    double d = 1.0;
    for (int n = 4; n >= 0; --n) {
        d *= (double)(P.two_i_min[n] + 2 * (int)(r % P.n_i[n]) + 1);
        r /= P.n_i[n];
    }
    out[z] = s * sqrt(d);
}

// ---------------------------------------------------------------------------------------------------------
// host side
// ---------------------------------------------------------------------------------------------------------
struct LinePlan {
    bool ok;
    int NT, TPW;
    LineParams lp;
    size_t smem;
    long z_doubles, b4_doubles;
};

static int line_max_nxs(const SfDims& D)
{
    int m = 0;
    for (int a = 0; a < D.n_i[0]; ++a)
        for (int o = 0; o < D.nl; ++o) {
            const int i1 = D.two_i_min[0] + 2 * a, l25 = D.two_j[J25] + 2 * o;
            const int n = (i1 + l25 - abs(i1 - l25)) / 2 + 1;
            if (n > m) m = n;
        }
    return m;
}

static LinePlan line_plan(const SfDims& D)
{
    LinePlan pl;
    memset(&pl, 0, sizeof pl);
    int nmax = 0, kmax = 0;
    for (int e = 0; e < 4; ++e) {
        if (D.n_i[e + 1] > nmax) nmax = D.n_i[e + 1];
        if (D.k_max[e] > kmax) kmax = D.k_max[e];
        if (D.k_max[e] == 0) return pl;
    }
    if (nmax > 16 || kmax > 16 || D.nl > 32) return pl;
    const int nxs = line_max_nxs(D);
    if (nxs > 28) return pl;
    LineParams& lp = pl.lp;
    pl.NT = nmax <= 8 ? 1 : 2;
    const int NT8 = pl.NT * 8;
    lp.NXF = nxs <= 4 ? 4 : nxs <= 12 ? 12 : nxs <= 20 ? 20 : 28;
    lp.KS3 = (D.k_max[1] + 3) / 4;
    lp.KS4 = (D.k_max[2] + 3) / 4;
    lp.LDK3 = 4 * lp.KS3;
    lp.LDK4 = 4 * lp.KS4;
    lp.TS4 = 32 * lp.KS4 + 4;
    lp.TS3 = 32 * lp.KS3;
    lp.zslab = NT8 * lp.NXF;
    lp.jsum = 0;
    for (int s = 0; s < 10; ++s) lp.jsum += D.two_j[s];
    const int n2 = D.n_i[1], n3 = D.n_i[2], n4 = D.n_i[3], n5 = D.n_i[4];
    const int P3 = D.n_k_pad[1], P4 = D.n_k_pad[2];
    const long slabs = (long)D.nl * D.n_i[0] * D.nl * D.nl;
    pl.z_doubles = slabs * P4 * lp.zslab;
    pl.b4_doubles = (long)D.nl * D.nl * D.nl * NT8 * lp.LDK4;
    if (pl.z_doubles * 8 > (16L << 30)) return pl;
    for (int nb = 1; nb <= D.k_max[0]; ++nb) {
        const int slots = (D.k_max[0] + nb - 1) / nb;
        const int mt_max = (slots * D.k_max[1] + 7) / 8;
        const int tiles2 = mt_max * n5, tiles3 = (slots * n4 * n5 + 7) / 8;
        const int tiles = tiles2 > tiles3 ? tiles2 : tiles3;
        const int TPW = (tiles + LINE_WARPS - 1) / LINE_WARPS;
        if (TPW > 8) continue;
        int off = tiles2 * lp.TS4 + 8;
        if (tiles3 * lp.TS3 > off) off = tiles3 * lp.TS3;
        off = (off + 1) & ~1;
        lp.offX2 = off;
        off += slots * n3 * n4 * n5;
        off = (off + 1) & ~1;
        lp.offU = off;
        off += (slots * P3 + 1) * lp.NXF;
        lp.offS3 = off;
        off += D.k_max[1] * P4 * lp.NXF;
        off = (off + 1) & ~1;
        lp.offZ = off;
        off += 2 * D.k_max[2] * lp.zslab;
        lp.offBw4 = off;
        off += 2 * NT8 * lp.LDK4;
        lp.offBw3 = off;
        off += NT8 * lp.LDK3;
        lp.offBw2 = off;
        off += n2 * slots;
        off = (off + 1) & ~1;
        lp.offRow = off;
        off += 2 * mt_max * 8;
        lp.offSh = off;
        off += 2 * (D.nl + 1);
        lp.offBar = off;
        off += 4;
        lp.n_smem = off;
        if (sizeof(double) * (size_t)off > 226 * 1024) continue;
        pl.TPW = TPW;
        lp.slots = slots;
        lp.mt_max = mt_max;
        lp.n_batches = nb;
        pl.smem = sizeof(double) * (size_t)off;
        pl.ok = true;
        return pl;
    }
    return pl;
}

bool sf_vertex_line_supported(const SfDims& D) { return line_plan(D).ok; }

template <int NT, int TPW>
static int launch_line(const LinePlan& pl, int grid, cudaStream_t st)
{
    static SfPerContext<bool> attr_set_c(false);
    bool& attr_set = attr_set_c.get();
    if (!attr_set) {
        if (cudaFuncSetAttribute(k_vertex_line<NT, TPW>, cudaFuncAttributeMaxDynamicSharedMemorySize, 226 * 1024) != cudaSuccess)
            return SF_ECUDA;
        attr_set = true;
    }
    k_vertex_line<NT, TPW><<<grid, LINE_THREADS, pl.smem, st>>>(pl.lp);
    return SF_OK;
}

int sf_vertex_line(const SfDims& D, const SfProblem& P, long shell_lo, long shell_hi, double* out, cudaStream_t st)
{
    LinePlan pl = line_plan(D);
    if (!pl.ok) return SF_EARG;
    static SfPerContext<int> n_sm_c(0);
    int& n_sm = n_sm_c.get();
    if (!n_sm) {
        int dev = 0;
        SF_CUDA_OK(cudaGetDevice(&dev));
        SF_CUDA_OK(cudaDeviceGetAttribute(&n_sm, cudaDevAttrMultiProcessorCount, dev));
    }
    LineParams& lp = pl.lp;
    lp.P = P;
    lp.shell_lo = shell_lo;
    lp.shell_hi = shell_hi;
    const long nl3 = (long)D.nl * D.nl * D.nl;
    const int n1 = D.n_i[0], NT8 = pl.NT * 8;
    if (shell_hi > shell_lo) {
        lp.blk0 = shell_lo / nl3;
        lp.n_blocks = (int)((shell_hi - 1) / nl3 - lp.blk0 + 1);
    } else {
        lp.blk0 = 0;
        lp.n_blocks = 0;
    }
    // few units: split every block into sub-ranges of whole lines so that all SMs have work
    const long base_units = (long)lp.n_blocks * n1 * lp.n_batches;
    lp.n_sub = 1;
    if (base_units > 0 && base_units < 4L * n_sm) {
        long want = (4L * n_sm + base_units - 1) / base_units;
        const long nl2 = (long)D.nl * D.nl;
        lp.n_sub = (int)(want < nl2 ? want : nl2);
    }
    lp.n_units = (int)(base_units * lp.n_sub);
    const long slice = D.n_out / n1;
    double* partial = (double*)sf_scratch(17, sizeof(double) * (size_t)(lp.n_units > 0 ? lp.n_units : 1) * slice);
    double* Zg = (double*)sf_scratch(19, sizeof(double) * (size_t)pl.z_doubles);
    double* Bw4g = (double*)sf_scratch(20, sizeof(double) * (size_t)pl.b4_doubles);
    if (!partial || !Zg || !Bw4g) return SF_ENOMEM;
    // a unit without work writes no slice, and k_reduce_units adds every slice: start from zeros (recycled device memory is not)
    SF_CUDA_OK(cudaMemsetAsync(partial, 0, sizeof(double) * (size_t)(lp.n_units > 0 ? lp.n_units : 1) * slice, st));
    lp.partial = partial;
    lp.Zg = Zg;
    lp.Bw4g = Bw4g;
    if (lp.n_units > 0) {
        const long slabs = (long)D.nl * n1 * D.nl * D.nl;
        k_line_prep_z<<<(unsigned)(slabs * D.n_k_pad[2]), lp.zslab, 0, st>>>(P, NT8, lp.NXF, Zg);
        k_line_prep_b4<<<(unsigned)nl3, 128, 0, st>>>(P, NT8, lp.LDK4, Bw4g);
        sf_count_launch(2);
        const int grid = lp.n_units < n_sm ? lp.n_units : n_sm;
        int rc = SF_EARG;
#define SF_SHAPE(a, b) \
    if (pl.NT == a && pl.TPW == b) rc = launch_line<a, b>(pl, grid, st);
        SF_SHAPE(1, 1) SF_SHAPE(1, 2) SF_SHAPE(1, 3) SF_SHAPE(1, 4) SF_SHAPE(1, 5) SF_SHAPE(1, 6) SF_SHAPE(1, 7) SF_SHAPE(1, 8)
        SF_SHAPE(2, 1) SF_SHAPE(2, 2) SF_SHAPE(2, 3) SF_SHAPE(2, 4) SF_SHAPE(2, 5) SF_SHAPE(2, 6) SF_SHAPE(2, 7) SF_SHAPE(2, 8)
#undef SF_SHAPE
        if (rc != SF_OK) return rc;
        sf_count_launch(1);
    }
    sf_timing_mark(2, st);
    k_reduce_units<<<(unsigned)((D.n_out + 255) / 256), 256, 0, st>>>(P, lp.n_blocks, lp.n_batches * lp.n_sub, D.n_out, partial, out);
    sf_count_launch(1);
    return cudaGetLastError() == cudaSuccess ? SF_OK : SF_ECUDA;
}
