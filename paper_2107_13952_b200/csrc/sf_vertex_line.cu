// sf_vertex_line.cu -- the on-chip path of steps 5-7 of the vertex-tensor algorithm: kernels (b) {15j}
// assembly, (c) mode-product contraction and (d) fixed-order shell accumulation of north_star in one persistent kernel.
//
// Work unit = (block of shells with the same (l23 l24 l25), boundary intertwiner i1, batch of SLOTS values of k2
// [, sub-range of the block's lines]).  The canonical shell order (eq. (9)) has l45 fastest, so a "line" =
// the nl consecutive shells that differ only in l45, and a block = nl^2 consecutive lines.  For every shell of the unit
// the CTA (16 warps) computes, with FP64 tensor-core MMAs (mma.sync m8n8k4 f64 = SASS DMMA.8x8x4; tcgen05 has no FP64
// kind) whose operands are staged in shared memory:
//
//   asm  W[(s,c3),c4][c5] = (-1)^R sum_x U[(s,c3)][x] S3[c3,c4][x] Y[c4][x][c5]                  eq. (5)
//        per c4 one GEMM over the recoupling spin x (K = x), U = (2x+1) S5 S4 (unit constant), S3 (line constant),
//        Y = S2 S1 (per shell): the five {6j} of eq. (5); the per-shell {15j} tensor W lives in MMA C fragments
//   G1   T4[(s,c3),c4][i5] = sum_c5 W . (2k5+1) B5[i5,c5]      step 6(iii): the C fragments of W ARE the A
//        fragments of this product under a permuted order of the contracted index (no data movement)
//   G2   T3[(s,c3,i5)][i4] += sum_c4 T4 . (2k4+1) B4[i4,c4]    accumulated in registers over the shells of the line
//   G3   T2[(s,i4,i5)][i3] += sum_c3 T3 . (2k3+1) B3[i3,c3]    once per line: B3 depends on (l34 l35 l23) only, so by
//        linearity the product is applied to the line's sum (the contracted index is extended by the shell offset)
//   G4   A[i2][(i3,i4,i5)]  = sum_s  T2 . (2k2+1) B2[i2,k2(s)] once per unit: B2 depends on (l23 l24 l25) only
//
// Every shell's W is assembled and contracted with its own four booster sub-matrices (step 6(i)-(iii)); step 6(iv),
// the accumulation over shells, happens on T3 / T2 / A in a fixed order (shells ascending inside a unit, units
// ascending in k_reduce_units), so the result is bitwise reproducible.  No float atomics.
#include <stdio.h>

#include "sf_internal.h"

#define LINE_THREADS 512
#define LINE_WARPS 16
#define LINE_PFY 8              // prefetch registers (doubles) per thread for the next shell's Y operand

struct LineParams {
    SfProblem P;
    long shell_lo, shell_hi;
    long blk0;                  // first block (shell_lo / nl^3)
    int n_blocks, n_batches, n_sub, n_units;
    int slots;                  // k2 values per batch
    int LDK, NXF;               // row strides (doubles) of [rows][contracted k] and [rows][x] operands; both = 4 mod 8
    int g1_shfl;                // 1: k ranges <= 12, the third k-step of G1 is built with one quad shuffle
    int jsum;                   // sum of the ten boundary spins (2j units)
    int offX2, offU, offS3, offY, offS1, offBw, offB2, n_smem;   // shared-memory offsets / total (doubles)
    double* partial;            // [n_units][n2][n3*n4*n5]
    unsigned int* counter;
};

__device__ __forceinline__ void line_dmma(double& c0, double& c1, double a, double b)
{
    asm("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1},{%2},{%3},{%0,%1};\n"
        : "+d"(c0), "+d"(c1)
        : "d"(a), "d"(b));
}

struct LineShell {              // per-shell quantities (steps 2 and 6(ii): ranges of k3 k4 k5 and the selected sub-matrices)
    int o34, o35, o45;
    int t3, t4, t5;
    int K3, K4, K5, q3b, q4b, q5b, kmin3, kmin4, kmin5;
    int osum;
};

__device__ __forceinline__ bool line_shell(const SfProblem& P, long shell, int o23, int o24, int o25, LineShell& S)
{
    const int nl = P.nl;
    const int r = (int)(shell % ((long)nl * nl * nl));
    S.o45 = r % nl;
    S.o35 = (r / nl) % nl;
    S.o34 = r / (nl * nl);
    S.t3 = (S.o34 * nl + S.o35) * nl + o23;
    S.t4 = (S.o45 * nl + o24) * nl + S.o34;
    S.t5 = (o25 * nl + S.o35) * nl + S.o45;
    const SfKRange r3 = P.kr[1][S.t3], r4 = P.kr[2][S.t4], r5 = P.kr[3][S.t5];
    S.K3 = r3.n_k; S.K4 = r4.n_k; S.K5 = r5.n_k;
    S.kmin3 = r3.two_k_min; S.kmin4 = r4.two_k_min; S.kmin5 = r5.two_k_min;
    S.q3b = (r3.two_k_min - P.two_k_base[1]) >> 1;
    S.q4b = (r4.two_k_min - P.two_k_base[2]) >> 1;
    S.q5b = (r5.two_k_min - P.two_k_base[3]) >> 1;
    S.osum = o23 + o24 + o25 + S.o34 + S.o35 + S.o45;
    return S.K3 > 0 && S.K4 > 0 && S.K5 > 0;
}

struct LinePF {                 // operands of the next shell, in flight while the current shell's G2 runs
    double y[LINE_PFY];
    double b[2];
};

// loads of the per-shell operands: Y[c4][k5][x] = (-1)^(..) S2 S1 (eq. (5)) and the weighted booster sub-matrices of
// edges 5 and 4 (step 6(ii)).  Element e of thread tid is e = tid + 512 i.
template <int NT>
__device__ __forceinline__ void line_pf_load(const LineParams& lp, const LineShell& S, int tid, int h0, int nxs, int xg0,
                                             const double* __restrict__ S1s, LinePF& pf)
{
    const SfProblem& P = lp.P;
    const int NT8 = NT * 8, NXF = lp.NXF, LDK = lp.LDK, nl = P.nl, NX = P.n_x_pad;
    const int P4 = P.n_k_pad[2], P5 = P.n_k_pad[3];
    const int n_y = S.K4 * NT8 * NXF;
    const double* s2 = P.S[1] + (((long)(S.o35 * nl + S.o45) * P4 + S.q4b) * P5 + S.q5b) * NX + xg0;
    const int par0 = h0 + S.osum + S.q4b + S.q5b;
#pragma unroll
    for (int i = 0; i < LINE_PFY; ++i) {
        const int e = tid + LINE_THREADS * i;
        double val = 0.0;
        if (e < n_y) {
            const int v = e % NXF, r = e / NXF, k5c = r % NT8, c4 = r / NT8;
            if (k5c < S.K5 && v < nxs) {
                val = s2[((long)c4 * P5 + k5c) * NX + v] * S1s[(S.q5b + k5c) * NXF + v];
                if ((par0 + c4 + k5c) & 1) val = -val;
            }
        }
        pf.y[i] = val;
    }
    const int nb = NT8 * LDK;
#pragma unroll
    for (int i = 0; i < 2; ++i) {
        const int e = tid + LINE_THREADS * i;
        double val = 0.0;
        if (e < 2 * nb) {
            const int which = e / nb, rem = e - which * nb, ii = rem / LDK, c = rem - ii * LDK;
            if (which == 0) {
                if (ii < P.n_i[4] && c < S.K5)
                    val = (double)(S.kmin5 + 2 * c + 1) * P.B[3][((long)S.t5 * P.n_i[4] + ii) * P5 + S.q5b + c];
            } else {
                if (ii < P.n_i[3] && c < S.K4)
                    val = (double)(S.kmin4 + 2 * c + 1) * P.B[2][((long)S.t4 * P.n_i[3] + ii) * P4 + S.q4b + c];
            }
        }
        pf.b[i] = val;
    }
}

template <int NT>
__device__ __forceinline__ void line_pf_store(const LineParams& lp, const LineShell& S, int tid, double* __restrict__ Ys,
                                              double* __restrict__ Bw5, double* __restrict__ Bw4, const LinePF& pf)
{
    const int NT8 = NT * 8, nb = NT8 * lp.LDK;
    const int n_y = S.K4 * NT8 * lp.NXF;
#pragma unroll
    for (int i = 0; i < LINE_PFY; ++i) {
        const int e = tid + LINE_THREADS * i;
        if (e < n_y) Ys[e] = pf.y[i];
    }
#pragma unroll
    for (int i = 0; i < 2; ++i) {
        const int e = tid + LINE_THREADS * i;
        if (e < nb)
            Bw5[e] = pf.b[i];
        else if (e < 2 * nb)
            Bw4[e - nb] = pf.b[i];
    }
}

template <int NT, int TPW>
__global__ void __launch_bounds__(LINE_THREADS, 1) k_vertex_line(const LineParams lp)
{
    extern __shared__ __align__(16) double smem[];
    __shared__ unsigned int s_unit;
    const SfProblem& P = lp.P;
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31, g = lane >> 2, q = lane & 3;
    constexpr int NT8 = NT * 8;
    constexpr int NKS1 = NT == 1 ? 2 : 4;           // k-steps of G1 (NT == 2: 3 of them when lp.g1_shfl)
    const int LDK = lp.LDK, NXF = lp.NXF, SLOTS = lp.slots;
    double* T4 = smem;                               // [rows (s,c3,i5)][LDK]; at a line's end A3 [rows (s,i4,i5)][LDK]
    double* X2 = smem + lp.offX2;                    // T2 sums [SLOTS][n3][n4*n5]
    double* U = smem + lp.offU;                      // [SLOTS][P3][NXF]
    double* S3s = smem + lp.offS3;                   // [K3][P4][NXF]
    double* Ys = smem + lp.offY;                     // [K4][NT8][NXF]
    double* S1s = smem + lp.offS1;                   // [P5][NXF]
    double* Bw5 = smem + lp.offBw;                   // [NT8][LDK] weighted boosters (2k+1) B[i][c], zero padded
    double* Bw4 = Bw5 + NT8 * LDK;                   // [2][NT8][LDK]
    double* Bw3 = Bw4 + 2 * NT8 * LDK;               // [NT8][LDK]
    double* Bw2 = smem + lp.offB2;                   // [n2][SLOTS]
    const int nl = P.nl, n1 = P.n_i[0], n2 = P.n_i[1], n3 = P.n_i[2], n4 = P.n_i[3], n5 = P.n_i[4];
    const int n45 = n4 * n5, R = n3 * n45, NX = P.n_x_pad;
    const int P2 = P.n_k_pad[0], P3 = P.n_k_pad[1], P4 = P.n_k_pad[2], P5 = P.n_k_pad[3];
    const long nl3 = (long)nl * nl * nl;

    for (int z = tid; z < lp.n_smem; z += LINE_THREADS) smem[z] = 0.0;   // padding must hold finite values

    for (;;) {
        __syncthreads();
        if (tid == 0) s_unit = atomicAdd(lp.counter, 1u);
        __syncthreads();
        const int unit = (int)s_unit;
        if (unit >= lp.n_units) break;
        int r_ = unit;
        const int sub = r_ % lp.n_sub; r_ /= lp.n_sub;
        const int batch = r_ % lp.n_batches; r_ /= lp.n_batches;
        const int a1 = r_ % n1;
        const long blk = lp.blk0 + r_ / n1;
        const int o25 = (int)(blk % nl), o24 = (int)((blk / nl) % nl), o23 = (int)(blk / ((long)nl * nl));
        const SfKRange r2 = P.kr[0][blk];
        const int cb = batch * SLOTS, nslots = min(SLOTS, r2.n_k - cb);
        const int q2b = (r2.two_k_min - P.two_k_base[0]) >> 1;
        const int nl2 = nl * nl;
        long s_begin = blk * nl3 + (long)(sub * nl2 / lp.n_sub) * nl, s_end = blk * nl3 + (long)((sub + 1) * nl2 / lp.n_sub) * nl;
        s_begin = max(s_begin, lp.shell_lo);
        s_end = min(s_end, lp.shell_hi);
        double* dst = lp.partial + (long)unit * n2 * R;
        const int i1 = P.two_i_min[0] + 2 * a1, l25 = P.two_j[J25] + 2 * o25, j13 = P.two_j[J13];
        // x-range of the unit: the triad (i1 l25 x) of eq. (5) cut by the triads (k2 j13 x) of the batch's k2 values
        const int k2f = r2.two_k_min + 2 * cb, k2l = k2f + 2 * (nslots - 1);
        int x0 = abs(i1 - l25), x1 = i1 + l25;
        {
            const int lo2 = (k2f <= j13 && j13 <= k2l) ? ((j13 - k2f) & 1) : min(abs(k2f - j13), abs(k2l - j13));
            const int hi2 = k2l + j13;
            if (lo2 > x0) x0 += ((lo2 - x0 + 1) >> 1) << 1;
            if (hi2 < x1) x1 -= ((x1 - hi2 + 1) >> 1) << 1;
        }
        const int nxs = x1 >= x0 ? ((x1 - x0) >> 1) + 1 : 0;
        if (nslots <= 0 || s_begin >= s_end || nxs <= 0) {       // uniform over the CTA
            for (int z = tid; z < n2 * R; z += LINE_THREADS) dst[z] = 0.0;
            continue;
        }
        const int xg0 = (x0 - P.two_x_base) >> 1;
        // (-1)^R, 2R = sum of all fifteen labels (reading G1) = jsum + i1 + sum_a base_a + 2 (sum o + sum q_a)
        const int h0 = (lp.jsum + i1 + P.two_k_base[0] + P.two_k_base[1] + P.two_k_base[2] + P.two_k_base[3]) >> 1;

        // ---- unit constants: U = (-1)^(q2+q3) (2x+1) S5 S4, S1, weighted B2, zeroed T2 sums ----
        {
            const double* s5 = P.S[4] + (((long)o25 * n1 + a1) * P2 + q2b + cb) * NX + xg0;
            const double* s4 = P.S[3] + ((((long)o23 * nl + o24) * P2 + q2b + cb) * P3) * NX + xg0;
            for (int e = tid; e < SLOTS * P3 * NXF; e += LINE_THREADS) {
                const int v = e % NXF, r = e / NXF, q3 = r % P3, s = r / P3;
                double val = 0.0;
                if (s < nslots && v < nxs) {
                    val = (double)(x0 + 2 * v + 1) * s5[(long)s * NX + v] * s4[((long)s * P3 + q3) * NX + v];
                    if ((q2b + cb + s + q3) & 1) val = -val;
                }
                U[e] = val;
            }
            const double* s1 = P.S[0] + (((long)o25 * n1 + a1) * P5) * NX + xg0;
            for (int e = tid; e < P5 * NXF; e += LINE_THREADS) {
                const int v = e % NXF, q5 = e / NXF;
                S1s[e] = v < nxs ? s1[(long)q5 * NX + v] : 0.0;
            }
            for (int e = tid; e < n2 * SLOTS; e += LINE_THREADS) {
                const int s = e % SLOTS, i2 = e / SLOTS;
                Bw2[e] = s < nslots ? (double)(r2.two_k_min + 2 * (cb + s) + 1) * P.B[0][((long)blk * n2 + i2) * P2 + q2b + cb + s] : 0.0;
            }
            for (int e = tid; e < SLOTS * R; e += LINE_THREADS) X2[e] = 0.0;
        }
        __syncthreads();                             // S1s is read by the operand loads below

        double acc3[TPW][NT][2];
#pragma unroll
        for (int j = 0; j < TPW; ++j)
#pragma unroll
            for (int nt = 0; nt < NT; ++nt) acc3[j][nt][0] = acc3[j][nt][1] = 0.0;

        // ---- G3 (once per line): T2 sums += sum_c3 T3 . (2k3+1) B3 ----
        auto flush_line = [&](int K3) {
            const int rows2 = nslots * K3 * n5, rows3 = nslots * n45;
#pragma unroll
            for (int j = 0; j < TPW; ++j) {
                const int r = (warp + LINE_WARPS * j) * 8 + g;
                if (r < rows2) {
                    const int s = r / (K3 * n5), rem = r - s * K3 * n5, c3 = rem / n5, i5 = rem - c3 * n5;
                    double* a3 = T4 + ((long)(s * n4) * n5 + i5) * LDK + c3;
#pragma unroll
                    for (int nt = 0; nt < NT; ++nt) {
                        const int i4 = nt * 8 + 2 * q;
                        if (i4 < n4) a3[(long)i4 * n5 * LDK] = acc3[j][nt][0];
                        if (i4 + 1 < n4) a3[(long)(i4 + 1) * n5 * LDK] = acc3[j][nt][1];
                    }
                }
#pragma unroll
                for (int nt = 0; nt < NT; ++nt) acc3[j][nt][0] = acc3[j][nt][1] = 0.0;
            }
            __syncthreads();
            double bq3[NT][4];
#pragma unroll
            for (int nt = 0; nt < NT; ++nt)
#pragma unroll
                for (int ks = 0; ks < 4; ++ks) bq3[nt][ks] = (4 * ks < LDK) ? Bw3[(nt * 8 + g) * LDK + 4 * ks + q] : 0.0;
            const int ks3 = (K3 + 3) >> 2, ntiles3 = (rows3 + 7) >> 3;
#pragma unroll
            for (int j = 0; j < TPW; ++j) {
                const int tile = warp + LINE_WARPS * j;
                if (tile < ntiles3) {
                    const double* a = T4 + (long)(tile * 8 + g) * LDK + q;
                    double c[NT][2];
#pragma unroll
                    for (int nt = 0; nt < NT; ++nt) c[nt][0] = c[nt][1] = 0.0;
#pragma unroll
                    for (int ks = 0; ks < 4; ++ks)
                        if (ks < ks3) {
                            const double av = a[4 * ks];
#pragma unroll
                            for (int nt = 0; nt < NT; ++nt) line_dmma(c[nt][0], c[nt][1], av, bq3[nt][ks]);
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
            __syncthreads();
        };

        // ---- first non-empty shell of the unit: stage its operands directly ----
        LineShell S;
        long shell = s_begin;
        while (shell < s_end && !line_shell(P, shell, o23, o24, o25, S)) ++shell;
        int pb = 0;                                  // Bw4 buffer of the current shell
        if (shell < s_end) {
            LinePF pf;
            line_pf_load<NT>(lp, S, tid, h0, nxs, xg0, S1s, pf);
            line_pf_store<NT>(lp, S, tid, Ys, Bw5, Bw4, pf);
        }
        long cur_line = -1;
        int K3 = 0, q3b = 0;

        while (shell < s_end) {
            const long line = shell / nl;
            if (line != cur_line) {
                if (cur_line >= 0) flush_line(K3);
                // ---- line constants: S3[c3][q4][x] and the weighted B3 ----
                K3 = S.K3;
                q3b = S.q3b;
                const double* s3 = P.S[2] + (((((long)o24 * nl + S.o34) * nl + S.o35) * P3 + q3b) * P4) * NX + xg0;
                for (int e = tid; e < K3 * P4 * NXF; e += LINE_THREADS) {
                    const int v = e % NXF, r = e / NXF;
                    S3s[e] = v < nxs ? s3[(long)r * NX + v] : 0.0;
                }
                for (int e = tid; e < NT8 * LDK; e += LINE_THREADS) {
                    const int ii = e / LDK, c = e - ii * LDK;
                    Bw3[e] = (ii < n3 && c < K3)
                                 ? (double)(S.kmin3 + 2 * c + 1) * P.B[1][((long)S.t3 * n3 + ii) * P3 + q3b + c]
                                 : 0.0;
                }
                cur_line = line;
                __syncthreads();
            }
            const int K4 = S.K4, K5 = S.K5, q4b = S.q4b, l35 = P.two_j[J35] + 2 * S.o35;

            // ---- P1: assembly of W (eq. (5)) chained into G1 (contract k5); T4 -> shared memory ----
            {
                double bq5[NT][NKS1];
#pragma unroll
                for (int nt = 0; nt < NT; ++nt) {
                    const double* b = Bw5 + (nt * 8 + g) * LDK;
                    bq5[nt][0] = b[2 * q];
                    bq5[nt][1] = b[2 * q + 1];
                    if (NT == 2) {
                        if (lp.g1_shfl) {            // contracted index of k-step 2 in the order 8 10 9 11
                            bq5[nt][2] = b[8 + ((q & 1) << 1) + (q >> 1)];
                            bq5[nt][NKS1 - 1] = 0.0;
                        } else {
                            bq5[nt][2] = b[8 + 2 * q];
                            bq5[nt][NKS1 - 1] = b[9 + 2 * q];
                        }
                    }
                }
                const int rows1 = nslots * K3, MT1 = (rows1 + 7) >> 3, ntasks = MT1 * K4;
                for (int task = warp; task < ntasks; task += LINE_WARPS) {
                    const int c4 = task / MT1, mt = task - c4 * MT1;
                    const bool valid = mt * 8 + g < rows1;
                    const int row = valid ? mt * 8 + g : 0;
                    const int s = row / K3, c3 = row - s * K3;
                    const double* up = U + ((long)(s * P3 + q3b + c3)) * NXF + q;
                    const double* sp = S3s + ((long)(c3 * P4 + q4b + c4)) * NXF + q;
                    const double* yp = Ys + ((long)(c4 * NT8 + g)) * NXF + q;
                    double c[NT][2];
#pragma unroll
                    for (int nt = 0; nt < NT; ++nt) c[nt][0] = c[nt][1] = 0.0;
                    // k-steps of x that the triads (k2 j13 x) of the tile's rows and (k4 l35 x) leave (warp uniform)
                    int ks_lo, ks_hi;
                    {
                        const int sf = (mt * 8) / K3, sl = min(mt * 8 + 7, rows1 - 1) / K3;
                        const int ka = k2f + 2 * sf, kb = k2f + 2 * sl;
                        int tlo = (ka <= j13 && j13 <= kb) ? 0 : min(abs(ka - j13), abs(kb - j13)), thi = kb + j13;
                        const int k4 = S.kmin4 + 2 * c4;
                        tlo = max(tlo, abs(k4 - l35));
                        thi = min(thi, k4 + l35);
                        const int vlo = tlo > x0 ? (tlo - x0 + 1) >> 1 : 0;
                        const int vhi = thi >= x0 ? min(nxs - 1, (thi - x0) >> 1) : -1;
                        ks_lo = vlo >> 2;
                        ks_hi = vhi >= vlo ? vhi >> 2 : ks_lo - 1;
                    }
                    for (int ks = ks_lo; ks <= ks_hi; ++ks) {
                        const double av = valid ? up[4 * ks] * sp[4 * ks] : 0.0;
#pragma unroll
                        for (int nt = 0; nt < NT; ++nt) line_dmma(c[nt][0], c[nt][1], av, yp[(long)nt * 8 * NXF + 4 * ks]);
                    }
                    // G1: the C fragment (row g; columns 2q, 2q+1 of each n-tile) is the A fragment of k-steps whose
                    // contracted index runs 2q | 2q+1 | 8+2q (or 8 10 9 11) | 9+2q
                    double d[NT][2];
#pragma unroll
                    for (int nt = 0; nt < NT; ++nt) d[nt][0] = d[nt][1] = 0.0;
#pragma unroll
                    for (int nt = 0; nt < NT; ++nt) line_dmma(d[nt][0], d[nt][1], c[0][0], bq5[nt][0]);
#pragma unroll
                    for (int nt = 0; nt < NT; ++nt) line_dmma(d[nt][0], d[nt][1], c[0][1], bq5[nt][1]);
                    if (NT == 2 && K5 > 8) {
                        if (lp.g1_shfl) {
                            const double t = __shfl_sync(0xffffffffu, c[NT - 1][1], (lane & ~3) + (q & 1));
                            const double av = q < 2 ? c[NT - 1][0] : t;
#pragma unroll
                            for (int nt = 0; nt < NT; ++nt) line_dmma(d[nt][0], d[nt][1], av, bq5[nt][2]);
                        } else {
#pragma unroll
                            for (int nt = 0; nt < NT; ++nt) line_dmma(d[nt][0], d[nt][1], c[NT - 1][0], bq5[nt][2]);
#pragma unroll
                            for (int nt = 0; nt < NT; ++nt) line_dmma(d[nt][0], d[nt][1], c[NT - 1][1], bq5[nt][NKS1 - 1]);
                        }
                    }
                    if (valid) {
                        double* t4 = T4 + ((long)(s * K3 + c3) * n5) * LDK + c4;
#pragma unroll
                        for (int nt = 0; nt < NT; ++nt) {
                            const int i5 = nt * 8 + 2 * q;
                            if (i5 < n5) t4[(long)i5 * LDK] = d[nt][0];
                            if (i5 + 1 < n5) t4[(long)(i5 + 1) * LDK] = d[nt][1];
                        }
                    }
                }
            }
            __syncthreads();

            // ---- P2: G2 (contract k4) accumulated in registers over the line; the next shell's operands are fetched
            //      meanwhile ----
            LineShell Sn;
            long next = shell + 1;
            while (next < s_end && !line_shell(P, next, o23, o24, o25, Sn)) ++next;
            LinePF pf;
            if (next < s_end) line_pf_load<NT>(lp, Sn, tid, h0, nxs, xg0, S1s, pf);
            {
                double bq4[NT][4];
                const double* bw = Bw4 + pb * NT8 * LDK;
#pragma unroll
                for (int nt = 0; nt < NT; ++nt)
#pragma unroll
                    for (int ks = 0; ks < 4; ++ks) bq4[nt][ks] = (4 * ks < LDK) ? bw[(nt * 8 + g) * LDK + 4 * ks + q] : 0.0;
                const int ks4 = (K4 + 3) >> 2, ntiles2 = (nslots * K3 * n5 + 7) >> 3;
#pragma unroll
                for (int ks = 0; ks < 4; ++ks)
                    if (ks < ks4) {
#pragma unroll
                        for (int j = 0; j < TPW; ++j) {
                            const int tile = warp + LINE_WARPS * j;
                            if (tile < ntiles2) {
                                const double av = T4[(long)(tile * 8 + g) * LDK + q + 4 * ks];
#pragma unroll
                                for (int nt = 0; nt < NT; ++nt) line_dmma(acc3[j][nt][0], acc3[j][nt][1], av, bq4[nt][ks]);
                            }
                        }
                    }
            }
            if (next < s_end) line_pf_store<NT>(lp, Sn, tid, Ys, Bw5, Bw4 + (pb ^ 1) * NT8 * LDK, pf);
            pb ^= 1;
            __syncthreads();
            shell = next;
            S = Sn;
        }
        if (cur_line >= 0) flush_line(K3);

        // ---- G4 (once per unit): contract k2; the unit's tensor goes to partial[unit] ----
        for (int z = tid; z < n2 * R; z += LINE_THREADS) {
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
    if (nmax > 16 || kmax > 16) return pl;
    const int nxs_all = line_max_nxs(D);
    LineParams& lp = pl.lp;
    pl.NT = (nmax <= 8 && kmax <= 8) ? 1 : 2;
    const int NT8 = pl.NT * 8;
    lp.LDK = kmax <= 12 ? 12 : 20;
    lp.g1_shfl = (pl.NT == 2 && kmax <= 12) ? 1 : 0;
    lp.jsum = 0;
    for (int s = 0; s < 10; ++s) lp.jsum += D.two_j[s];
    const int n2 = D.n_i[1], n3 = D.n_i[2], n4 = D.n_i[3], n5 = D.n_i[4];
    const int P3 = D.n_k_pad[1], P4 = D.n_k_pad[2], P5 = D.n_k_pad[3];
    static const int tpws[] = {1, 2, 4, 6, 8};
    for (int nb = 1; nb <= D.k_max[0]; ++nb) {
        const int slots = (D.k_max[0] + nb - 1) / nb;
        // x values a unit can see: the triad (i1 l25 x) cut by the triads (k2 j13 x) of `slots` consecutive k2
        int nxs = D.two_j[J13] + slots;
        if (nxs_all < nxs) nxs = nxs_all;
        if (nxs > 28) continue;
        lp.NXF = nxs <= 4 ? 4 : nxs <= 12 ? 12 : nxs <= 20 ? 20 : 28;
        if (D.k_max[2] * NT8 * lp.NXF > LINE_PFY * LINE_THREADS) continue;
        int rows = D.k_max[1] * n5 > n4 * n5 ? D.k_max[1] * n5 : n4 * n5;
        rows *= slots;
        const int tiles = (rows + 7) / 8, tpw = (tiles + LINE_WARPS - 1) / LINE_WARPS;
        int TPW = 0;
        for (int t : tpws)
            if (t >= tpw) {
                TPW = t;
                break;
            }
        if (!TPW) continue;
        int off = (tiles * 8 + 8) * lp.LDK;
        lp.offX2 = off;
        off += slots * n3 * n4 * n5;
        off = (off + 1) & ~1;
        lp.offU = off;
        off += (slots * P3 + 8) * lp.NXF;
        lp.offS3 = off;
        off += (D.k_max[1] * P4 + 8) * lp.NXF;
        lp.offY = off;
        off += (D.k_max[2] * NT8 + 8) * lp.NXF;
        lp.offS1 = off;
        off += P5 * lp.NXF;
        lp.offBw = off;
        off += 4 * NT8 * lp.LDK;
        lp.offB2 = off;
        off += n2 * slots;
        off = (off + 1) & ~1;
        lp.n_smem = off;
        if (sizeof(double) * (size_t)off > 224 * 1024) continue;
        pl.TPW = TPW;
        lp.slots = slots;
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
    static bool attr_set = false;
    if (!attr_set) {
        if (cudaFuncSetAttribute(k_vertex_line<NT, TPW>, cudaFuncAttributeMaxDynamicSharedMemorySize, 224 * 1024) != cudaSuccess)
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
    static int n_sm = 0;
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
    const int n1 = D.n_i[0];
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
    unsigned int* counter = (unsigned int*)sf_scratch(18, 256);
    if (!partial || !counter) return SF_ENOMEM;
    lp.partial = partial;
    lp.counter = counter;
    if (lp.n_units > 0) {
        SF_CUDA_OK(cudaMemsetAsync(counter, 0, sizeof(unsigned int), st));
        const int grid = lp.n_units < n_sm ? lp.n_units : n_sm;
        int rc = SF_EARG;
#define SF_SHAPE(a, b) \
    if (pl.NT == a && pl.TPW == b) rc = launch_line<a, b>(pl, grid, st);
        SF_SHAPE(1, 1) SF_SHAPE(1, 2) SF_SHAPE(1, 4) SF_SHAPE(1, 6) SF_SHAPE(1, 8)
        SF_SHAPE(2, 1) SF_SHAPE(2, 2) SF_SHAPE(2, 4) SF_SHAPE(2, 6) SF_SHAPE(2, 8)
#undef SF_SHAPE
        if (rc != SF_OK) return rc;
        sf_count_launch(1);
    }
    sf_timing_mark(2, st);
    k_reduce_units<<<(unsigned)((D.n_out + 255) / 256), 256, 0, st>>>(P, lp.n_blocks, lp.n_batches * lp.n_sub, D.n_out, partial, out);
    sf_count_launch(1);
    return cudaGetLastError() == cudaSuccess ? SF_OK : SF_ECUDA;
}
