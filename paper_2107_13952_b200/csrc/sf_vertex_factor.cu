// sf_vertex_factor.cu -- the factorised path of steps 5-7 of the vertex-tensor algorithm.
//
// Eq. (3) with the {15j} of eq. (5) written out is one big multilinear sum
//
//   A[i1..i5] = N(i) sum_{l23..l45} sum_{k2..k5} sum_x  (-1)^R (2x+1) S1 S2 S3 S4 S5  Bw2 Bw3 Bw4 Bw5 ,   Bw_a = (2k_a+1) B_a
//
// in which every booster depends on three of the six virtual spins only and every {6j} tensor S_n
// of step 4 on at most three.  The paper's loop (steps 5-6) builds the {15j} of
// one shell and contracts it with that shell's four boosters; by linearity the same sum can be taken one virtual spin
// at a time, keeping the recoupling spin x open.  The order used here, all FP64:
//
//   Z [l25 i1 l35 l45; k4 x i5]        = sum_k5   S2 S1 Bw5                      (k_fz_pre, task Z: two {6j} of eq. (5) and the edge-5 product)
//   Q [.. l24 l34; k4 x i5 i4]         = sum_l45  Z Bw4                          (k_fz_qp4, Q phase: the shells of a line l45 = j..j+Dl)
//   P [l24 l25 i1; k3 x; l34 l35; i5 i4] = sum_k4 S3 Q                           (k_fz_qp4, P phase: third {6j}, edge-4 mode product)
//   R [l24 l25 i1; k3 x; l23 i3; i5 i4]  = sum_{l34 l35} Bw3 P                   (k_fz_gemm<FzMapR>: edge-3 mode product + shell sum)
//   G [l23 l24 l25 i1; k3 x; i2]       = sum_k2   Bw2 (-1)^.. (2x+1) S5 S4       (k_fz_pre, task G: last two {6j}, edge-2 booster)
//   A'[l24 l25; i1 i2 i3 i4 i5]        = sum_{k3 x l23} G R                      (k_fz_gemm<FzMapA>: sum over x of eq. (5), edge-2 product)
//   A [i1..i5]                         = N(i) sum_{l24 l25} A'                   (k_fz_reduce: fixed order, step 6(iv) + eq. (3))
//
// Every term of the paper's sum is still there, exactly once; only the order of the additions differs, so the result
// agrees with the per-shell paths (sf_vertex_line.cu) to rounding.  The {6j} tensors are exactly 0 where a triad
// fails (sf_slices.cu) and the weighted boosters are masked to each triple's own k-range (reading G9), so the dense
// index ranges used below add only exact zeros.  All sums run in a fixed order: bitwise reproducible.
//
// Every product is an FP64 tensor-core MMA (mma.sync m8n8k4 f64, SASS DMMA.8x8x4).  The two big contractions (R, A')
// are gather-GEMMs: C[m][n] = sum_k A[k][m] B[k][n] with per-index offset tables built from the spin ranges, so the
// irregular ranges of the spin-foam sum (step 2) turn into plain index lists.
//
// A sub-range of the canonical shell order (sf_vertex_amplitude_range) is split into at most 11 boxes of virtual-spin
// offsets (digit decomposition in base Dl+1); the factorisation applies to each box.
#include <stdio.h>
#include <string.h>

#include "sf_factor.cuh"

// ---------------------------------------------------------------------------------------------------------
// small precomputations (step 2 windows, weighted / transposed operands)
// ---------------------------------------------------------------------------------------------------------
__device__ __forceinline__ void fz_windows_entry(const SfProblem& P, int2* w3A, int2* w3B, int2* w4A, int2* w4B, int t)
{
    const int nl = P.nl;
    const int* j = P.two_j;
    if (t < nl * nl) {
        const int u = t / nl, v = t % nl;
        w3A[t] = fz_window(j[J34] + 2 * u, j[J35] + 2 * v, P.two_k_base[1], P.n_k_pad[1]);
        w4A[t] = fz_window(j[J24] + 2 * u, j[J34] + 2 * v, P.two_k_base[2], P.n_k_pad[2]);
    }
    if (t < nl) {
        w3B[t] = fz_window(j[J13], j[J23] + 2 * t, P.two_k_base[1], P.n_k_pad[1]);
        w4B[t] = fz_window(j[J45] + 2 * t, j[J14], P.two_k_base[2], P.n_k_pad[2]);
    }
}

// Z[b25][a1][b35][b45][q4][v][i5] = (-1)^(o25+o35+o45+q4) sum_{k5 valid} (-1)^q5 {j14 k5 x; l35 k4 l45} {i1 l25 x; k5 j14 j15} (2k5+1) B5[t5][i5][q5]
// one CTA per (b25, a1, b35, b45) and k4 (grid.y): single-shell problems (Delta_l = 0, large spins) have few (l25 l35 l45)
__device__ __forceinline__ void fz_z_block(const FzParams& p, double* __restrict__ Z, long bx, int by, int gy)
{
    const SfProblem& P = p.P;
    const int nl = P.nl, n1 = P.n_i[0], n5 = P.n_i[4], P4 = P.n_k_pad[2], P5 = P.n_k_pad[3], NX = P.n_x_pad, V = p.V;
    const int c35 = p.box.cnt[4], c45 = p.box.cnt[5];
    long b = bx;
    const int b45 = (int)(b % c45); b /= c45;
    const int b35 = (int)(b % c35); b /= c35;
    const int a1 = (int)(b % n1);
    const int b25 = (int)(b / n1);
    const int o25 = p.box.lo[2] + b25, o35 = p.box.lo[4] + b35, o45 = p.box.lo[5] + b45;
    int x0, nxs, xg0;
    fz_xrange(P.two_i_min[0], P.two_j[J25], P.two_x_base, a1, o25, x0, nxs, xg0);
    const int t5 = (o25 * nl + o35) * nl + o45;
    const SfKRange r5 = P.kr[3][t5];
    const int q5b = (r5.two_k_min - P.two_k_base[3]) >> 1;
    double* z = Z + bx * P4 * V * n5;
    const int nq4 = (P4 - by + gy - 1) / gy;      // the k4 of this block: by + gy * n
    const double* s1b = P.S[0] + (((long)(o25 * n1 + a1) * P5 + q5b) * NX) + xg0;
    for (int e = threadIdx.x; e < nq4 * nxs * n5; e += blockDim.x) {
        const int i5 = e % n5, r = e / n5, v = r % nxs, q4 = by + gy * (r / nxs);
        const double* s2 = P.S[1] + ((((long)(o35 * nl + o45) * P4 + q4) * P5 + q5b) * NX) + xg0 + v;
        const double* s1 = s1b + v;
        const double* b5 = sf_brow(P, 3, t5, i5) + q5b;
        double val = 0.0;
        // {j14 k5 x; l35 k4 l45} vanishes unless the triads (j14 k4 l45) and (l35 k4 x) hold: such entries are exact zeros
        const int k4 = P.two_k_base[2] + 2 * q4, x = x0 + 2 * v;
        const int l35 = P.two_j[J35] + 2 * o35, l45 = P.two_j[J45] + 2 * o45, j14 = P.two_j[J14];
        const bool live = k4 >= abs(j14 - l45) && k4 <= j14 + l45 && !((j14 + l45 + k4) & 1) && k4 >= abs(l35 - x) && k4 <= l35 + x &&
                          !((l35 + x + k4) & 1);
        for (int c = 0; live && c < r5.n_k; ++c) {
            double term = s2[(long)c * NX] * s1[(long)c * NX] * ((double)(r5.two_k_min + 2 * c + 1) * b5[c]);
            if ((q5b + c) & 1) term = -term;
            val += term;
        }
        if ((o25 + o35 + o45 + q4) & 1) val = -val;
        z[(q4 * V + v) * n5 + i5] = val;
    }
}

// Bw4T[q4][b45][b24][b34][i4] = (2k4+1) B4[(o45 o24 o34)][i4][q4] inside the triple's k-range, 0 outside
__device__ __forceinline__ void fz_b4t_entry(const FzParams& p, long n, double* __restrict__ out, long e)
{
    const SfProblem& P = p.P;
    if (e >= n) return;
    const int nl = P.nl, n4 = P.n_i[3], P4 = P.n_k_pad[2];
    const int c24 = p.box.cnt[1], c34 = p.box.cnt[3], c45 = p.box.cnt[5];
    long r = e;
    const int i4 = (int)(r % n4); r /= n4;
    const int b34 = (int)(r % c34); r /= c34;
    const int b24 = (int)(r % c24); r /= c24;
    const int b45 = (int)(r % c45);
    const int q4 = (int)(r / c45);
    const int t4 = ((p.box.lo[5] + b45) * nl + p.box.lo[1] + b24) * nl + p.box.lo[3] + b34;
    const SfKRange r4 = P.kr[2][t4];
    const int c = q4 - ((r4.two_k_min - P.two_k_base[2]) >> 1);
    double val = 0.0;
    if (c >= 0 && c < r4.n_k) val = (double)(r4.two_k_min + 2 * c + 1) * sf_brow(P, 2, t4, i4)[q4];
    out[e] = val;
}

// Bw3T[q3][b34][b35][b23][i3] = (2k3+1) B3[(o34 o35 o23)][i3][q3] inside the triple's k-range, 0 outside
__device__ __forceinline__ void fz_b3t_entry(const FzParams& p, long n, double* __restrict__ out, long e)
{
    const SfProblem& P = p.P;
    if (e >= n) return;
    const int nl = P.nl, n3 = P.n_i[2], P3 = P.n_k_pad[1];
    const int c23 = p.box.cnt[0], c34 = p.box.cnt[3], c35 = p.box.cnt[4];
    long r = e;
    const int i3 = (int)(r % n3); r /= n3;
    const int b23 = (int)(r % c23); r /= c23;
    const int b35 = (int)(r % c35); r /= c35;
    const int b34 = (int)(r % c34);
    const int q3 = (int)(r / c34);
    const int t3 = ((p.box.lo[3] + b34) * nl + p.box.lo[4] + b35) * nl + p.box.lo[0] + b23;
    const SfKRange r3 = P.kr[1][t3];
    const int c = q3 - ((r3.two_k_min - P.two_k_base[1]) >> 1);
    double val = 0.0;
    if (c >= 0 && c < r3.n_k) val = (double)(r3.two_k_min + 2 * c + 1) * sf_brow(P, 1, t3, i3)[q3];
    out[e] = val;
}

// S3T[b24][b34][b35][xx][q3][q4] = (-1)^o34 {k4 l35 x; k3 l24 l34}
__device__ __forceinline__ void fz_s3t_entry(const FzParams& p, long n, double* __restrict__ out, long e)
{
    const SfProblem& P = p.P;
    if (e >= n) return;
    const int nl = P.nl, P3 = P.n_k_pad[1], P4 = P.n_k_pad[2], NX = P.n_x_pad;
    const int c34 = p.box.cnt[3], c35 = p.box.cnt[4];
    long r = e;
    const int q4 = (int)(r % P4); r /= P4;
    const int q3 = (int)(r % P3); r /= P3;
    const int xx = (int)(r % NX); r /= NX;
    const int b35 = (int)(r % c35); r /= c35;
    const int b34 = (int)(r % c34);
    const int b24 = (int)(r / c34);
    const int o24 = p.box.lo[1] + b24, o34 = p.box.lo[3] + b34, o35 = p.box.lo[4] + b35;
    const double val = P.S[2][(((((long)o24 * nl + o34) * nl + o35) * P3 + q3) * P4 + q4) * NX + xx];
    out[e] = (o34 & 1) ? -val : val;
}

// G[b24][b25][a1][q3][v][b23][i2] = sum_{k2 valid} (2k2+1) B2[(o23 o24 o25)][i2][q2] (-1)^(h0+o23+o24+q2+q3) (2x+1)
//                                   {k2 j13 x; i1 l25 j12} {l24 k3 x; j13 k2 l23}
// h0 = (sum of boundary spins + i1 + sum of the k bases) / 2: with the signs folded into Z and S3T this is the
// (-1)^R of eq. (5), 2R = sum of all fifteen labels (reading G1)
// One block per (b24 b25 a1 q3): only the x of the triad (k3 l24 x) and the l23 of the pair (j13 l23) that allow this k3 are
// visited (three quarters of the dense index space (v, l23) are excluded by them: a thread per dense entry spent its time
// on early exits), entries (v, b23, i2) in memory order.
__device__ __forceinline__ void fz_g_block(const FzParams& p, double* __restrict__ out, long blk_id)
{
    const SfProblem& P = p.P;
    const int nl = P.nl, n1 = P.n_i[0], n2 = P.n_i[1], P2 = P.n_k_pad[0], P3 = P.n_k_pad[1], NX = P.n_x_pad, V = p.V;
    const int c23 = p.box.cnt[0], c25 = p.box.cnt[2];
    long r = blk_id;
    const int q3 = (int)(r % P3); r /= P3;
    const int a1 = (int)(r % n1); r /= n1;
    const int b25 = (int)(r % c25);
    const int b24 = (int)(r / c25);
    const int o24 = p.box.lo[1] + b24, o25 = p.box.lo[2] + b25;
    int x0, nxs, xg0;
    fz_xrange(P.two_i_min[0], P.two_j[J25], P.two_x_base, a1, o25, x0, nxs, xg0);
    // only the entries k_fz_gemm<FzMapA> reads: x of this (i1 l25) with the triad (k3 l24 x), k3 allowed by (j13 l23)
    const int2 vr = fz_vrange(P.two_j[J24] + 2 * o24, P.two_k_base[1] + 2 * q3, x0, nxs);
    if (vr.y == 0) return;
    int blo = 0, bcnt = 0;                                    // the l23 of the box whose pair (j13 l23) allows k3: contiguous
    for (int b = 0; b < c23; ++b) {
        const int2 wb = fz_window(P.two_j[J13], P.two_j[J23] + 2 * (p.box.lo[0] + b), P.two_k_base[1], P3);
        if (q3 >= wb.x && q3 < wb.x + wb.y) {
            if (!bcnt) blo = b;
            ++bcnt;
        }
    }
    if (bcnt == 0) return;
    const int i1 = P.two_i_min[0] + 2 * a1;
    const int h0 = (p.jsum + i1 + P.two_k_base[0] + P.two_k_base[1] + P.two_k_base[2] + P.two_k_base[3]) >> 1;
    double* ob = out + ((((long)b24 * c25 + b25) * n1 + a1) * P3 + q3) * ((long)V * c23 * n2);
    const int per_v = bcnt * n2, total = vr.y * per_v;
    for (int e = threadIdx.x; e < total; e += blockDim.x) {
        const int vi = e / per_v, r2i = e - vi * per_v, bi = r2i / n2, i2 = r2i - bi * n2;
        const int v = vr.x + vi, b23 = blo + bi, o23 = p.box.lo[0] + b23;
        const int blk = (o23 * nl + o24) * nl + o25;
        const SfKRange r2 = P.kr[0][blk];
        const int q2b = (r2.two_k_min - P.two_k_base[0]) >> 1;
        const double* s5 = P.S[4] + (((long)o25 * n1 + a1) * P2 + q2b) * NX + xg0 + v;
        const double* s4 = P.S[3] + ((((long)o23 * nl + o24) * P2 + q2b) * P3 + q3) * NX + xg0 + v;
        const double* b2 = sf_brow(P, 0, blk, i2) + q2b;
        double val = 0.0;
        for (int c = 0; c < r2.n_k; ++c) {
            double term = (double)(r2.two_k_min + 2 * c + 1) * b2[c] * s5[(long)c * NX] * s4[(long)c * P3 * NX];
            if ((q2b + c) & 1) term = -term;
            val += term;
        }
        val *= (double)(x0 + 2 * v + 1);
        if ((h0 + o23 + o24 + q3) & 1) val = -val;
        ob[((long)v * c23 + b23) * n2 + i2] = val;
    }
}

// per k3: the l23 of the box that allow it (contiguous: |k3 - j13| <= l23 <= k3 + j13) and the (l34 l35) pairs that do
__device__ __forceinline__ void fz_lists_warp(const FzParams& p, int2* __restrict__ win23, int* __restrict__ kl3, int q3, int lane)
{
    const SfProblem& P = p.P;
    const int P3 = P.n_k_pad[1];
    const int c23 = p.box.cnt[0], c34 = p.box.cnt[3], c35 = p.box.cnt[4];
    if (lane == 0) {
        int blo = -1, bcnt = 0;
        for (int b = 0; b < c23; ++b) {
            const int2 w = fz_window(P.two_j[J13], P.two_j[J23] + 2 * (p.box.lo[0] + b), P.two_k_base[1], P3);
            if (q3 >= w.x && q3 < w.x + w.y) {
                if (blo < 0) blo = b;
                ++bcnt;
            }
        }
        win23[q3] = make_int2(blo < 0 ? 0 : blo, bcnt);
    }
    int* list = kl3 + (long)q3 * (1 + c34 * c35);
    int cnt = 0;
    for (int base = 0; base < c34 * c35; base += 32) {
        const int c = base + lane;
        bool ok = false;
        if (c < c34 * c35) {
            const int2 w = fz_window(P.two_j[J34] + 2 * (p.box.lo[3] + c / c35), P.two_j[J35] + 2 * (p.box.lo[4] + c % c35), P.two_k_base[1], P3);
            ok = q3 >= w.x && q3 < w.x + w.y;
        }
        const unsigned mask = __ballot_sync(0xffffffffu, ok);
        if (ok) list[1 + cnt + __popc(mask & ((1u << lane) - 1u))] = c;
        cnt += __popc(mask);
    }
    if (lane == 0) list[0] = cnt;
}

// ONE launch for all the precomputations of a box: small problems are bound by the number of dependent launches, not by their
// work (config 0: 3.4e6 flop per tensor).  Blocks [first[t], first[t + 1]) run task t; the tasks are independent of one another
// (the windows the lists and G need are recomputed in place: a handful of integer operations).
struct FzPreArgs {
    long first[9];              // 0 G, 1 Z, 2 Bw4P / Bw4T, 3 Bw3T, 4 S3T, 5 windows, 6 lists, 7 scheduler counters; first[8] = all blocks
    long nB4, padB4, nB3, nS3, padS3;         // elements (pad: zeros behind the array, for whole-fragment reads)
    int gy, b4p;                // k4 split of the Z blocks; booster layout: Bw4P (1, k_fz_qp2 / k_fz_qp4) or Bw4T (0, k_fz_qp)
    int n_sched;
    double *Z, *B4, *B3, *S3, *G;
    int2 *w3A, *w3B, *w4A, *w4B, *win23;
    int *kl3, *sched;
};
__global__ void __launch_bounds__(256) k_fz_pre(const __grid_constant__ FzParams p, const __grid_constant__ FzPreArgs a)
{
    const long b = blockIdx.x;
    const int tid = threadIdx.x;
    if (b < a.first[1]) {                                     // the heavy tasks first: their blocks must not start last
        fz_g_block(p, a.G, b - a.first[0]);
    } else if (b < a.first[2]) {
        const long bz = b - a.first[1];
        fz_z_block(p, a.Z, bz / a.gy, (int)(bz % a.gy), a.gy);
    } else if (b < a.first[3]) {
        const long e = (b - a.first[2]) * 256 + tid;
        if (e >= a.nB4) {
            if (e < a.nB4 + a.padB4) a.B4[e] = 0.0;
        } else if (a.b4p) {
            fz_b4p_entry(p, a.nB4, a.B4, e);
        } else {
            fz_b4t_entry(p, a.nB4, a.B4, e);
        }
    } else if (b < a.first[4]) {
        fz_b3t_entry(p, a.nB3, a.B3, (b - a.first[3]) * 256 + tid);
    } else if (b < a.first[5]) {
        const long e = (b - a.first[4]) * 256 + tid;
        if (e >= a.nS3) {
            if (e < a.nS3 + a.padS3) a.S3[e] = 0.0;
        } else {
            fz_s3t_entry(p, a.nS3, a.S3, e);
        }
    } else if (b < a.first[6]) {
        fz_windows_entry(p.P, a.w3A, a.w3B, a.w4A, a.w4B, (int)(b - a.first[5]) * 256 + tid);
    } else if (b < a.first[7]) {
        const int q3 = (int)(b - a.first[6]) * 8 + (tid >> 5);
        if (q3 < p.P.n_k_pad[1]) fz_lists_warp(p, a.win23, a.kl3, q3, tid & 31);
    } else {
        for (int i = tid; i < a.n_sched; i += 256) a.sched[i] = 0;
    }
}

// ---------------------------------------------------------------------------------------------------------
// k_fz_qp: Q = sum_l45 Z Bw4 and P = sum_k4 S3 Q for one (i1, l25, l35, l24, l34), a few x at a time
// ---------------------------------------------------------------------------------------------------------
// Q phase, per k4:  C[(v i5)][i4] = sum_l45 Z[l45][k4][(v i5)] Bw4T[k4][l45][i4]        (A and B fragments straight from L1/L2)
// P phase, per v:   P[k3][(i5 i4)] = sum_k4 S3[k3][k4] Q[k4][(i5 i4)]                   (S3 from L1/L2, Q from shared memory)
// Persistent: a CTA walks the items with stride gridDim.x; its fragment offsets are computed once.
// The triads of eq. (5) that contain x, (k4 l35 x) and (k3 l24 x), bound k4 and k3 for every x: only those k4 are
// computed and only those rows k3 of P are written (k_fz_gemm reads exactly the same set, fz_vrange).
#define FZ_QP_THREADS 256
#define FZ_QKS 3      /* fast Q phase: c45 <= 12, (v, i5) rows of a pass <= 40; i4 in groups of FZ_QNT column tiles */
#define FZ_QNT 2
#define FZ_QMT 5
#define FZ_PKS 6      /* P phase: S3 fragments of 6 k-steps (24 values of k4) are loaded together */
__global__ void __launch_bounds__(FZ_QP_THREADS, 2) k_fz_qp(const FzParams p, long n_items)
{
    extern __shared__ __align__(16) double smem[];
    constexpr int NW = FZ_QP_THREADS / 32;
    const SfProblem& P = p.P;
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31, g = lane >> 2, q = lane & 3;
    const int nl = P.nl, n1 = P.n_i[0], n4 = P.n_i[3], n5 = P.n_i[4], n54 = n4 * n5;
    const int P3 = P.n_k_pad[1], P4 = P.n_k_pad[2], NX = P.n_x_pad, V = p.V, NP = p.NP;
    const int c24 = p.box.cnt[1], c25 = p.box.cnt[2], c34 = p.box.cnt[3], c35 = p.box.cnt[4], c45 = p.box.cnt[5];
    const int W4p = p.W4p, LDQ = p.LDQ, VG = p.VG;
    const int NT = (n54 + 7) >> 3, NT4 = (n4 + 7) >> 3, KS45 = (c45 + 3) >> 2, NTQ = (NT + 3) >> 2;
    const int sZ = P4 * V * n5, c2434n4 = c24 * c34 * n4;
    const long prow = (long)c34 * c35 * NP;          // stride of v in P
    const float inv_ntq = 1.0f / (float)NTQ;
    const bool fastq = KS45 <= FZ_QKS && ((VG * n5 + 7) >> 3) <= FZ_QMT;
    double* Qs = smem;                               // [VG][W4p][LDQ]
    for (int z = tid; z < VG * W4p * LDQ; z += FZ_QP_THREADS) Qs[z] = 0.0;   // rows never written must stay finite
    // constants of the CTA: this lane's fragment offsets inside one k4 block of Bw4T / of Z, its C rows in Qs (-1: none)
    int bofs[FZ_QKS], zofs[FZ_QMT][FZ_QKS], qrow[FZ_QMT];
#pragma unroll
    for (int ks = 0; ks < FZ_QKS; ++ks) {
        const int b45 = 4 * ks + q;
        const bool kin = ks < KS45 && b45 < c45;
        bofs[ks] = kin ? b45 * c2434n4 + g : -1;
#pragma unroll
        for (int mt = 0; mt < FZ_QMT; ++mt) zofs[mt][ks] = kin ? b45 * sZ + mt * 8 + g : -1;
    }
#pragma unroll
    for (int mt = 0; mt < FZ_QMT; ++mt) {
        const int m = mt * 8 + g, vv = m / n5, i5 = m - vv * n5;
        qrow[mt] = vv * W4p * LDQ + i5 * n4 + 2 * q;
    }
    unsigned ndm = 0;                                // DMMA instructions of this warp (reported when p.cnt is set)

    for (long item = blockIdx.x; item < n_items; item += gridDim.x) {
        long it = item;
        const int b34 = (int)(it % c34); it /= c34;
        const int b24 = (int)(it % c24); it /= c24;
        const int b35 = (int)(it % c35); it /= c35;
        const int b25 = (int)(it % c25);
        const int ac = (int)(it / c25);
        const int a1 = p.a_lo + ac;
        const int o24 = p.box.lo[1] + b24, o25 = p.box.lo[2] + b25, o34 = p.box.lo[3] + b34, o35 = p.box.lo[4] + b35;
        const int l24 = P.two_j[J24] + 2 * o24, l35 = P.two_j[J35] + 2 * o35;
        int x0, nxs, xg0;
        fz_xrange(P.two_i_min[0], P.two_j[J25], P.two_x_base, a1, o25, x0, nxs, xg0);
        const int2 w3 = p.w3A[o34 * nl + o35];       // the k3 the pair (l34 l35) allows
        if (w3.y == 0) continue;
        const int2 w4a = p.w4A[o24 * nl + o34];
        const int lo4 = max(w4a.x, p.hull4B.x);
        const int w4 = max(0, min(w4a.x + w4a.y, p.hull4B.y) - lo4);
        const int MT3 = (w3.y + 7) >> 3;
        const float inv_mt3 = 1.0f / (float)MT3;
        const double* Zb = p.Z + ((((long)b25 * n1 + a1) * c35 + b35) * c45) * (long)sZ;
        const double* S3b = p.S3T + ((((long)b24 * c34 + b34) * c35 + b35) * NX + xg0) * (long)(P3 * P4) + (long)w3.x * P4 + lo4;
        const double* B4b = p.Bw4T + ((long)b24 * c34 + b34) * n4;
        double* Pb = p.Pq + ((((long)ac * c24 + b24) * c25 + b25) * P3) * V * prow + ((long)b34 * c35 + b35) * NP;

        for (int v0 = 0; v0 < nxs; v0 += VG) {
            const int nv = min(VG, nxs - v0), rows = nv * n5, MT = (rows + 7) >> 3;
            // k4 of this pass: union over its x of the triad (k4 l35 x), inside the item's window
            int g4lo = w4, g4hi = 0;
            for (int vv = 0; vv < nv; ++vv) {
                const int2 w = fz_window(l35, x0 + 2 * (v0 + vv), P.two_k_base[2], P4);
                const int lo = max(w.x, lo4) - lo4, hi = min(w.x + w.y, lo4 + w4) - lo4;
                if (w.y > 0 && hi > lo) {
                    g4lo = min(g4lo, lo);
                    g4hi = max(g4hi, hi);
                }
            }
            if (g4hi <= g4lo) g4lo = g4hi = 0;
            const int k4a = g4lo & ~3, k4b = (g4hi + 3) & ~3;
            __syncthreads();                         // the previous P phase has read Qs
            // ---- Q phase ----
            if (fastq) {
                // common sizes: every fragment of a k4 is requested before the first MMA: one round of latency per k4
                for (int r4 = g4lo + warp; r4 < g4hi; r4 += NW) {
                    const int q4 = lo4 + r4;
                    const double* zq = Zb + ((long)q4 * V + v0) * n5;
                    const double* bq = B4b + (long)q4 * c45 * c2434n4;
                    ndm += MT * NT4 * KS45;
                    double a[FZ_QMT][FZ_QKS];
#pragma unroll
                    for (int ks = 0; ks < FZ_QKS; ++ks)
#pragma unroll
                        for (int mt = 0; mt < FZ_QMT; ++mt)
                            a[mt][ks] = (zofs[mt][ks] >= 0 && mt * 8 + g < rows) ? __ldg(zq + zofs[mt][ks]) : 0.0;
                    for (int ntc = 0; ntc < NT4; ntc += FZ_QNT) {           // FZ_QNT column tiles of i4 at a time
                        double b[FZ_QNT][FZ_QKS];
#pragma unroll
                        for (int ks = 0; ks < FZ_QKS; ++ks)
#pragma unroll
                            for (int nt = 0; nt < FZ_QNT; ++nt)
                                b[nt][ks] = (bofs[ks] >= 0 && (ntc + nt) * 8 + g < n4) ? __ldg(bq + bofs[ks] + (ntc + nt) * 8) : 0.0;
#pragma unroll
                        for (int mt = 0; mt < FZ_QMT; ++mt) {
                            if (mt >= MT) break;
                            double* dst = Qs + qrow[mt] + r4 * LDQ + ntc * 8;
                            const bool okm = mt * 8 + g < rows;
#pragma unroll
                            for (int nt = 0; nt < FZ_QNT; ++nt) {
                                if (ntc + nt >= NT4) break;
                                double c0 = 0.0, c1 = 0.0;
#pragma unroll
                                for (int ks = 0; ks < FZ_QKS; ++ks)
                                    if (ks < KS45) fz_dmma(c0, c1, a[mt][ks], b[nt][ks]);
                                const int j4 = (ntc + nt) * 8 + 2 * q;
                                if (okm && j4 < n4) dst[nt * 8] = c0;
                                if (okm && j4 + 1 < n4) dst[nt * 8 + 1] = c1;
                            }
                        }
                    }
                }
            } else {
                for (int r4 = g4lo + warp; r4 < g4hi; r4 += NW) {
                    const int q4 = lo4 + r4;
                    const double* zq = Zb + ((long)q4 * V + v0) * n5;
                    ndm += MT * NT4 * KS45;
                    for (int nt = 0; nt < NT4; ++nt) {
                        const int i4 = nt * 8 + g;
                        double bf[8];
#pragma unroll
                        for (int ks = 0; ks < 8; ++ks) {
                            const int b45 = 4 * ks + q;
                            bf[ks] = (ks < KS45 && b45 < c45 && i4 < n4) ? __ldg(B4b + ((long)q4 * c45 + b45) * c2434n4 + i4) : 0.0;
                        }
                        for (int mt = 0; mt < MT; ++mt) {
                            const int m = mt * 8 + g;
                            double c0 = 0.0, c1 = 0.0;
#pragma unroll
                            for (int ks = 0; ks < 8; ++ks) {
                                if (ks < KS45) {
                                    const int b45 = 4 * ks + q;
                                    const double av = (m < rows && b45 < c45) ? __ldg(zq + (long)b45 * sZ + m) : 0.0;
                                    fz_dmma(c0, c1, av, bf[ks]);
                                }
                            }
                            if (m < rows) {
                                const int vv = m / n5, i5 = m - vv * n5, j4 = nt * 8 + 2 * q;
                                double* dst = Qs + (vv * W4p + r4) * LDQ + i5 * n4 + j4;
                                if (j4 < n4) dst[0] = c0;
                                if (j4 + 1 < n4) dst[1] = c1;
                            }
                        }
                    }
                }
            }
            __syncthreads();                         // Qs of this pass is complete
            if (v0 + VG < nxs) {                     // the next pass's rows of Z and S3: into L1 under this pass's P phase
                const int nv2 = min(VG, nxs - v0 - VG), rows2 = nv2 * n5;
                for (int pr = tid; pr < c45 * w4; pr += FZ_QP_THREADS) {
                    const int b45 = pr / w4, r4 = pr - b45 * w4;
                    const double* row = Zb + (long)b45 * sZ + ((long)(lo4 + r4) * V + v0 + VG) * n5;
                    for (int off = 0; off < rows2; off += 16) fz_prefetch_l1(row + off);
                    fz_prefetch_l1(row + rows2 - 1);
                }
                for (int pr = tid; pr < nv2 * w3.y; pr += FZ_QP_THREADS) {
                    const int vv = pr / w3.y, r3 = pr - vv * w3.y;
                    const double* row = S3b + ((long)(v0 + VG + vv) * P3 + r3) * P4;
                    for (int off = 0; off < w4; off += 16) fz_prefetch_l1(row + off);
                    if (w4 > 0) fz_prefetch_l1(row + w4 - 1);
                }
            }
            // ---- P phase: one A fragment (S3, straight from L1/L2) feeds four column tiles of Q ----
            for (int task = warp; task < nv * MT3 * NTQ; task += NW) {
                // task = (vv MT3 + mt3) NTQ + ntq; quotients of small integers through one float multiply (exact: the
                // fractional part of (t + 0.5) / d is at least 0.5 / d, far above the rounding error)
                const int t2 = __float2int_rz(((float)task + 0.5f) * inv_ntq), ntq = task - t2 * NTQ;
                const int vv = __float2int_rz(((float)t2 + 0.5f) * inv_mt3), mt3 = t2 - vv * MT3;
                // rows k3 the triad (k3 l24 x) allows for this x
                const int2 wx = fz_window(l24, x0 + 2 * (v0 + vv), P.two_k_base[1], P3);
                const int rlo = max(wx.x, w3.x) - w3.x, rhi = wx.y > 0 ? min(wx.x + wx.y, w3.x + w3.y) - w3.x : 0;
                if (mt3 * 8 >= rhi || mt3 * 8 + 8 <= rlo) continue;
                const int r3 = mt3 * 8 + g;
                const bool rok = r3 < w3.y;
                const double* ap = S3b + ((long)(v0 + vv) * P3 + r3) * P4 + q;
                const double* bp = Qs + (vv * W4p + q) * LDQ + ntq * 32 + g;
                const int ntl = min(4, NT - ntq * 4);
                ndm += ((k4b - k4a) >> 2) * ntl;
                double c[4][2];
#pragma unroll
                for (int j = 0; j < 4; ++j) c[j][0] = c[j][1] = 0.0;
                for (int kc = k4a; kc < k4b; kc += 4 * FZ_PKS) {          // FZ_PKS k-steps at a time: their S3 fragments are
                    double av[FZ_PKS];                                     // requested together, before the first MMA
#pragma unroll
                    for (int i = 0; i < FZ_PKS; ++i) {
                        const int ks = kc + 4 * i;
                        av[i] = (ks < k4b && rok && ks + q < w4) ? __ldg(ap + ks) : 0.0;
                    }
#pragma unroll
                    for (int i = 0; i < FZ_PKS; ++i) {
                        const int ks = kc + 4 * i;
                        if (ks < k4b) {
#pragma unroll
                            for (int j = 0; j < 4; ++j)
                                if (j < ntl) fz_dmma(c[j][0], c[j][1], av[i], bp[ks * LDQ + 8 * j]);
                        }
                    }
                }
                if (r3 >= rlo && r3 < rhi) {
                    double* dst = Pb + ((long)(w3.x + r3) * V + v0 + vv) * prow + ntq * 32 + 2 * q;
#pragma unroll
                    for (int j = 0; j < 4; ++j)     // NP is even: n + 1 < NP whenever n < n54, and rows are 16-byte aligned
                        if (ntq * 32 + 8 * j + 2 * q < n54) *reinterpret_cast<double2*>(dst + 8 * j) = make_double2(c[j][0], c[j][1]);
                }
            }
        }
    }
    if (p.cnt && lane == 0) atomicAdd(p.cnt, (unsigned long long)ndm);
}

// ---------------------------------------------------------------------------------------------------------
// k_fz_gemm: gather-GEMM  C[offCm[m] + offCn[n]] = sum_kk A[kA kix[kk] + offAm[m]] B[kB kix[kk] + offBn[n]]
// ---------------------------------------------------------------------------------------------------------
struct FzGemmHdr {
    int M, N, K;
    int nsub;                   // products that share the index tables: A, B and C advance by sA, sB, sC
    long baseA, baseB, baseC, sA, sB, sC;
    int kA, kB;                 // strides of the k list: entry kk of the list sits at kA * kix[kk] in A, kB * kix[kk] in B
};

// R[l24 l25 i1; k3 x; l23 i3; (i5 i4)] = sum over the pairs (l34 l35) that allow k3 of P[..][(l34 l35)][(i5 i4)] Bw3T[k3][(l34 l35)][(l23 i3)]
// rows m = (i5 i4), columns n = (l23 i3) over the l23 whose pair (j13 l23) allows k3; one item = (i1, l24, l25, k3, tile),
// every x of (i1 l25) in turn
struct FzMapR {
    static constexpr bool A16 = true, B16 = false;
    static constexpr bool ABULK = true;  // the m-tile of a row of P is one contiguous, 16-byte aligned run: one bulk copy per k row
    static constexpr int CNT = 1, KC = 32, ST = 2;    // rows of P start 16-byte aligned (NP even) and m runs contiguously: copy pairs
    static __device__ const double* srcA(const FzParams& p) { return p.Pq; }
    static __device__ const double* srcB(const FzParams& p) { return p.Bw3T; }
    static __device__ double* dstC(const FzParams& p) { return p.Rq; }
    static __host__ __device__ long items(const FzParams& p, int BM, int BN)
    {
        const long ntm = (p.P.n_i[3] * p.P.n_i[4] + BM - 1) / BM, ntn = (p.box.cnt[0] * p.P.n_i[2] + BN - 1) / BN;
        return ntn * ntm * p.P.n_k_pad[1] * p.box.cnt[2] * p.box.cnt[1] * p.a_cnt;
    }
    static __device__ void setup(const FzParams& p, long item, int BM, int BN, FzGemmHdr* h, int* offAm, int* offCm,
                                 int* offBn, int* offCn, int* kix, int* tmp)
    {
        const SfProblem& P = p.P;
        const int n3 = P.n_i[2], n54 = P.n_i[3] * P.n_i[4], P3 = P.n_k_pad[1], V = p.V, NP = p.NP;
        const int c23 = p.box.cnt[0], c24 = p.box.cnt[1], c25 = p.box.cnt[2], c34 = p.box.cnt[3], c35 = p.box.cnt[4];
        const int ntm = (n54 + BM - 1) / BM, ntn = (c23 * n3 + BN - 1) / BN;
        const int nt = (int)(item % ntn); item /= ntn;
        const int mt = (int)(item % ntm); item /= ntm;
        const int q3 = (int)(item % P3); item /= P3;
        const int b25 = (int)(item % c25); item /= c25;
        const int b24 = (int)(item % c24);
        const int ac = (int)(item / c24);
        int x0, nxs, xg0;
        fz_xrange(P.two_i_min[0], P.two_j[J25], P.two_x_base, p.a_lo + ac, p.box.lo[2] + b25, x0, nxs, xg0);
        const int2 win = p.win23[q3];
        const int* list = p.kl3 + (long)q3 * (1 + c34 * c35);
        // the x for which the triad (k3 l24 x) of eq. (5) holds: the only rows of P that k_fz_qp wrote
        const int2 vr = fz_vrange(P.two_j[J24] + 2 * (p.box.lo[1] + b24), P.two_k_base[1] + 2 * q3, x0, nxs);
        const int m0 = mt * BM, n0 = nt * BN, N = min(BN, win.y * n3 - n0), K = list[0];
        const int M = (N > 0 && vr.y > 0) ? min(BM, n54 - m0) : 0;
        if (threadIdx.x == 0) {
            h->M = M;
            h->N = N;
            h->K = K;
            h->nsub = vr.y;
            const long slab = ((((long)ac * c24 + b24) * c25 + b25) * P3 + q3) * V + vr.x;
            h->baseA = slab * c34 * c35 * NP + m0;
            h->baseB = (long)q3 * c34 * c35 * c23 * n3 + (long)win.x * n3 + n0;
            h->baseC = ((slab * c23 + win.x) * n3 + n0) * NP + m0;
            h->sA = (long)c34 * c35 * NP;
            h->sB = 0;
            h->sC = (long)c23 * n3 * NP;
            h->kA = NP;
            h->kB = c23 * n3;
        }
        if (M <= 0) return;
        for (int m = threadIdx.x; m < BM; m += blockDim.x) offAm[m] = offCm[m] = m;
        for (int n = threadIdx.x; n < BN; n += blockDim.x) {
            offBn[n] = n;
            offCn[n] = n * NP;
        }
        for (int kk = threadIdx.x; kk < K; kk += blockDim.x) {
            const int c = list[1 + kk];
            kix[kk] = c;
        }
    }
};

// A'[l24 l25; i1; i2; (i3 i4 i5)] = sum over (k3, x, l23) with k3 allowed by (j13 l23) of G[..][(k3 x l23)][i2] R[..][(k3 x l23)][(i3, i5 i4)]
struct FzMapA {
    static constexpr bool A16 = false, ABULK = false;
    static constexpr bool B16 = true;    // columns run over the padded rows of R (i3, NP): contiguous and 16-byte aligned pairs
    static constexpr int CNT = 2, KC = 16, ST = 2;
    static __device__ const double* srcA(const FzParams& p) { return p.G; }
    static __device__ const double* srcB(const FzParams& p) { return p.Rq; }
    static __device__ double* dstC(const FzParams& p) { return p.Apart; }
    static __host__ __device__ long items(const FzParams& p, int BM, int BN)
    {
        const long ntn = ((long)p.P.n_i[2] * p.NP + BN - 1) / BN, ntm = (p.P.n_i[1] + BM - 1) / BM;
        return ntn * ntm * p.box.cnt[2] * p.box.cnt[1] * p.a_cnt;
    }
    static __device__ void setup(const FzParams& p, long item, int BM, int BN, FzGemmHdr* h, int* offAm, int* offCm,
                                 int* offBn, int* offCn, int* kix, int* tmp)
    {
        const SfProblem& P = p.P;
        const int n1 = P.n_i[0], n2 = P.n_i[1], n3 = P.n_i[2], n4 = P.n_i[3], n5 = P.n_i[4], n54 = n4 * n5, n345 = n3 * n54;
        const int P3 = P.n_k_pad[1], V = p.V, NP = p.NP;
        const int c23 = p.box.cnt[0], c24 = p.box.cnt[1], c25 = p.box.cnt[2];
        const int NN = n3 * NP;                      // columns (i3, r) over the padded rows of R; r >= n5 n4 is padding
        const int ntn = (NN + BN - 1) / BN, ntm = (n2 + BM - 1) / BM;
        const int nt = (int)(item % ntn); item /= ntn;
        const int mt = (int)(item % ntm); item /= ntm;
        const int b25 = (int)(item % c25); item /= c25;
        const int b24 = (int)(item % c24);
        const int ac = (int)(item / c24);
        const int a1 = p.a_lo + ac;
        int x0, nxs, xg0;
        fz_xrange(P.two_i_min[0], P.two_j[J25], P.two_x_base, a1, p.box.lo[2] + b25, x0, nxs, xg0);
        const int m0 = mt * BM, n0 = nt * BN, M = min(BM, n2 - m0), N = min(BN, NN - n0);
        // k list in the order (k3, x, l23): the x of each k3 (triad (k3 l24 x)), then prefix sums of (x count) * (l23 count)
        const int l24 = P.two_j[J24] + 2 * (p.box.lo[1] + b24);
        for (int q3 = threadIdx.x; q3 < P3; q3 += blockDim.x) {
            const int2 vr = fz_vrange(l24, P.two_k_base[1] + 2 * q3, x0, nxs);
            tmp[80 + q3] = vr.x;
            tmp[160 + q3] = vr.y;
        }
        __syncthreads();
        if (threadIdx.x == 0) {
            int run = 0;
            for (int q3 = 0; q3 < P3; ++q3) {
                tmp[q3] = run;
                run += p.win23[q3].y * tmp[160 + q3];
            }
            tmp[P3] = run;
            h->M = M;
            h->N = N;
            h->K = run;
            h->nsub = 1;
            h->baseA = ((((long)b24 * c25 + b25) * n1 + a1) * P3 * V * c23) * n2;
            h->baseB = (((long)ac * c24 + b24) * c25 + b25) * ((long)P3 * V * c23 * n3 * NP);
            h->baseC = ((p.part0 + (long)b24 * c25 + b25) * n1 + a1) * ((long)n2 * n345);
            h->sA = h->sB = h->sC = 0;
            h->kA = n2;
            h->kB = n3 * NP;
        }
        for (int m = threadIdx.x; m < BM; m += blockDim.x) {
            offAm[m] = m0 + m;
            offCm[m] = (m0 + m) * n345;
        }
        for (int n = threadIdx.x; n < BN; n += blockDim.x) {
            const int ng = n0 + n, i3 = ng / NP, r = ng - i3 * NP, i5 = r / n4, i4 = r - i5 * n4;
            offBn[n] = ng;
            offCn[n] = r < n54 ? (i3 * n4 + i4) * n5 + i5 : -1;      // -1: a padding column, never stored
        }
        __syncthreads();
        for (int e = threadIdx.x; e < P3 * nxs; e += blockDim.x) {
            const int q3 = e / nxs, vi = e - q3 * nxs;
            if (vi >= tmp[160 + q3]) continue;
            const int v = tmp[80 + q3] + vi;
            const int2 win = p.win23[q3];
            const int at = tmp[q3] + vi * win.y;
            for (int b = 0; b < win.y; ++b) {
                const int row = (q3 * V + v) * c23 + win.x + b;
                kix[at + b] = row;
            }
        }
    }
};

// one k-chunk of a warp tile with TNA live column tiles (tiles beyond N are skipped, not multiplied by zeros)
template <int TM, int TN, int TNA, int KC>
__device__ __forceinline__ void fz_chunk(double (&acc)[TM][TN][2], const double* as, const double* bs, int LDA, int LDB,
                                         int ksn, int tma)
{
#pragma unroll
    for (int ks = 0; ks < KC / 4; ++ks) {
        if (ks < ksn) {
            double a[TM], b[TNA];
#pragma unroll
            for (int i = 0; i < TM; ++i) a[i] = as[ks * 4 * LDA + 8 * i];
#pragma unroll
            for (int j = 0; j < TNA; ++j) b[j] = bs[ks * 4 * LDB + 8 * j];
#pragma unroll
            for (int i = 0; i < TM; ++i) {
                if (i < tma) {
#pragma unroll
                    for (int j = 0; j < TNA; ++j) fz_dmma(acc[i][j][0], acc[i][j][1], a[i], b[j]);
                }
            }
        }
    }
}
template <int TM, int TN, int TNA, int KC>
struct FzChunk {
    static __device__ __forceinline__ void run(double (&acc)[TM][TN][2], const double* as, const double* bs, int LDA,
                                               int LDB, int ksn, int tma, int tna)
    {
        if (tna == TNA)
            fz_chunk<TM, TN, TNA, KC>(acc, as, bs, LDA, LDB, ksn, tma);
        else
            FzChunk<TM, TN, TNA - 1, KC>::run(acc, as, bs, LDA, LDB, ksn, tma, tna);
    }
};
template <int TM, int TN, int KC>
struct FzChunk<TM, TN, 0, KC> {
    static __device__ __forceinline__ void run(double (&)[TM][TN][2], const double*, const double*, int, int, int, int, int) {}
};
template <class Map, int WGM, int WGN, int TM, int TN>
__global__ void __launch_bounds__(WGM* WGN * 32) k_fz_gemm(const FzParams p, int kcap)
{
    constexpr int BM = WGM * TM * 8, BN = WGN * TN * 8, NTH = WGM * WGN * 32, LDA = BM + 4, LDB = BN + 4;   // = 4 mod 16: half-warp fragment loads hit 16 different banks
    constexpr int KC = Map::KC, ST = Map::ST;        // k-chunk depth and ring stages
    extern __shared__ __align__(16) double smem[];
    __shared__ FzGemmHdr hdr;
    __shared__ __align__(8) unsigned long long abar[4];      // ABULK: one mbarrier per stage (ST <= 4)
    double* As = smem;                               // [ST][KC][LDA], [k][m]
    double* Bs = As + ST * KC * LDA;       // [ST][KC][LDB], [k][n]
    int* offAm = (int*)(Bs + ST * KC * LDB);
    int* offCm = offAm + BM;
    int* offBn = offCm + BM;
    int* offCn = offBn + BN;
    int* tmp = offCn + BN;                           // 240 ints of scratch for the setup
    int* kix = tmp + 240;                            // the k list (kcap entries)
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31, g = lane >> 2, q = lane & 3;
    const int wm = warp / WGN, wn = warp % WGN;
    if (Map::ABULK && tid == 0) {
        for (int s = 0; s < ST; ++s) fz_mbar_init(fz_smem_u32(&abar[s]), 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    Map::setup(p, blockIdx.x, BM, BN, &hdr, offAm, offCm, offBn, offCn, kix, tmp);
    __syncthreads();
    const int M = hdr.M, N = hdr.N, K = hdr.K, nsub = hdr.nsub;
    if (M <= 0) return;
    const double* A0 = Map::srcA(p);
    const double* B0 = Map::srcB(p);
    const double* A = A0 + hdr.baseA;
    const double* B = B0 + hdr.baseB;
    double* C = Map::dstC(p) + hdr.baseC;
    const long sA = hdr.sA, sB = hdr.sB, sC = hdr.sC;
    const long kA = hdr.kA, kB = hdr.kB;
    const int nchunks = (K + KC - 1) / KC, total = nsub * nchunks;
    int tma = 0, tna = 0;                            // live 8-row / 8-column tiles of this warp
#pragma unroll
    for (int i = 0; i < TM; ++i) tma += (wm * TM + i) * 8 < M;
#pragma unroll
    for (int j = 0; j < TN; ++j) tna += (wn * TN + j) * 8 < N;
    const bool active = tma > 0 && tna > 0;

    double acc[TM][TN][2];
#pragma unroll
    for (int i = 0; i < TM; ++i)
#pragma unroll
        for (int j = 0; j < TN; ++j) acc[i][j][0] = acc[i][j][1] = 0.0;
    auto store = [&](int sub) {                      // C fragments of one product to its rows of the destination
        if (!active) return;
        double* cs = C + sub * sC;
#pragma unroll
        for (int i = 0; i < TM; ++i) {
            const int m = wm * TM * 8 + 8 * i + g;
            if (m < M) {
                double* cm = cs + offCm[m];
#pragma unroll
                for (int j = 0; j < TN; ++j) {
                    const int n = wn * TN * 8 + 8 * j + 2 * q;
                    // maps whose columns include padding (B16) mark it with a negative offset
                    if (n < N && (!Map::B16 || offCn[n] >= 0)) cm[offCn[n]] = acc[i][j][0];
                    if (n + 1 < N && (!Map::B16 || offCn[n + 1] >= 0)) cm[offCn[n + 1]] = acc[i][j][1];
                }
            }
#pragma unroll
            for (int j = 0; j < TN; ++j) acc[i][j][0] = acc[i][j][1] = 0.0;
        }
    };
    if (nchunks == 0) {                              // nothing to sum: the destination rows are exact zeros
        for (int sub = 0; sub < nsub; ++sub) store(sub);
        return;
    }
    int l_sub = 0, l_c = 0;                          // next chunk to request: product l_sub, chunk l_c of it
    // every thread copies the same m (pair of m) and n of each k-row it serves: offsets and bounds are fixed per item
    constexpr int AW = Map::A16 ? 2 : 1, ATPR = BM / AW, ARPP = NTH / ATPR, APASS = KC / ARPP;
    constexpr int BW = Map::B16 ? 2 : 1, BTPR = BN / BW, BRPP = NTH / BTPR, BPASS = KC / BRPP;
    static_assert(NTH % ATPR == 0 && KC % ARPP == 0 && NTH % BTPR == 0 && KC % BRPP == 0, "loader shape");
    const int am = (tid % ATPR) * AW, akr = tid / ATPR, bn = (tid % BTPR) * BW, bkr = tid / BTPR;
    const int a_bytes = 8 * max(0, min(AW, M - am)), b_bytes = 8 * max(0, min(BW, N - bn));
    const int a_off = a_bytes ? offAm[am] : 0, b_off = b_bytes ? offBn[bn] : 0;
    const unsigned a_dst = fz_smem_u32(As + akr * LDA + am), b_dst = fz_smem_u32(Bs + bkr * LDB + bn);
    auto load_chunk = [&](int gc) {
        if (gc < total) {
            const int s = gc % ST, k0 = l_c * KC;
            const double* Aq = A + l_sub * sA + a_off;
            const double* Bq = B + l_sub * sB + b_off;
            if (Map::ABULK) {
                // warp 0: one bulk copy per k row (the row's M entries, rounded up to 16 bytes), completion on the stage's
                // mbarrier; rows past K of the last chunk are zeroed by hand (they are summed over)
                const int kv = min(KC, K - k0);
                const unsigned rowb = (unsigned)(((M + 1) & ~1) * 8);
                if (warp == 0) {
                    const unsigned bar = fz_smem_u32(&abar[s]);
                    // rows of this stage were zero-filled with generic stores two chunks ago (ordered by the CTA barrier):
                    // make them visible to the asynchronous proxy before the bulk copies overwrite the stage
                    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
                    if (lane == 0) fz_mbar_expect_tx(bar, rowb * (unsigned)kv);
                    __syncwarp();
                    for (int kr = lane; kr < kv; kr += 32)
                        fz_bulk_g2s(fz_smem_u32(As + (s * KC + kr) * LDA), A + l_sub * sA + kA * kix[k0 + kr], rowb, bar);
                }
                for (int e = tid; e < (KC - kv) * BM; e += NTH) As[(s * KC + kv + e / BM) * LDA + e % BM] = 0.0;
            } else {
#pragma unroll
                for (int it = 0; it < APASS; ++it) {
                    const int kr = akr + it * ARPP, k = k0 + kr;
                    const bool ok = a_bytes && k < K;
                    const unsigned dst = a_dst + 8u * (unsigned)((s * KC + it * ARPP) * LDA);
                    if (Map::A16)
                        fz_cp_async16(dst, ok ? Aq + kA * kix[k] : A0, ok ? a_bytes : 0);
                    else
                        fz_cp_async8(dst, ok ? Aq + kA * kix[k] : A0, ok ? 8 : 0);
                }
            }
#pragma unroll
            for (int it = 0; it < BPASS; ++it) {
                const int kr = bkr + it * BRPP, k = k0 + kr;
                const bool ok = b_bytes && k < K;
                const unsigned dst = b_dst + 8u * (unsigned)((s * KC + it * BRPP) * LDB);
                if (Map::B16)
                    fz_cp_async16(dst, ok ? Bq + kB * kix[k] : B0, ok ? b_bytes : 0);
                else
                    fz_cp_async8(dst, ok ? Bq + kB * kix[k] : B0, ok ? 8 : 0);
            }
            if (++l_c == nchunks) {
                l_c = 0;
                ++l_sub;
            }
        }
        fz_cp_commit();
    };
#pragma unroll
    for (int c = 0; c < ST - 1; ++c) load_chunk(c);
    int c_in = 0, sub = 0;
    unsigned ndm = 0;                                // DMMA instructions of this warp (reported when p.cnt is set)
    for (int gc = 0; gc < total; ++gc) {
        fz_cp_wait<ST - 2>();
        if (Map::ABULK) fz_mbar_wait(fz_smem_u32(&abar[gc % ST]), (unsigned)((gc / ST) & 1));
        __syncthreads();                             // chunk gc has landed; every warp is done with chunk gc - 1
        load_chunk(gc + ST - 1);              // refills the stage chunk gc - 1 used
        if (active) {
            const double* as = As + (gc % ST) * KC * LDA + q * LDA + wm * TM * 8 + g;
            const double* bs = Bs + (gc % ST) * KC * LDB + q * LDB + wn * TN * 8 + g;
            const int ksn = min(KC / 4, (K - c_in * KC + 3) >> 2);
            FzChunk<TM, TN, TN, KC>::run(acc, as, bs, LDA, LDB, ksn, tma, tna);
            ndm += tma * tna * ksn;
        }
        if (++c_in == nchunks) {
            store(sub);
            c_in = 0;
            ++sub;
        }
    }
    fz_cp_wait<0>();
    if (p.cnt && lane == 0) atomicAdd(p.cnt + Map::CNT, (unsigned long long)ndm);
}

// kernel (d): out[a1][i2][r] = prod_e sqrt(2 i_e + 1) * sum over the partial tensors, in order, of Apart[part][a1][i2][r]
// (step 6(iv) + the normalisation of eq. (3))
__global__ void __launch_bounds__(256) k_fz_reduce(SfProblem P, long n_parts, long n_out, const double* __restrict__ partial,
                                                   double* __restrict__ out)
{
    const long z = blockIdx.x * (long)blockDim.x + threadIdx.x;
    if (z >= n_out) return;
    double s = 0.0;
    for (long b = 0; b < n_parts; ++b) s += partial[b * n_out + z];
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
// [lo, hi) of the canonical shell order (o45 fastest, eq. (9)) as a disjoint union of boxes, in order
static void fz_boxes(int nl, long lo, long hi, int digit, FzBox prefix, FzBox* out, int* n)
{
    if (lo >= hi) return;
    long w = 1;
    for (int d = digit + 1; d < 6; ++d) w *= nl;      // shells per value of this digit
    if (lo == 0 && hi == w * nl) {
        for (int d = digit; d < 6; ++d) {
            prefix.lo[d] = 0;
            prefix.cnt[d] = nl;
        }
        out[(*n)++] = prefix;
        return;
    }
    const int a = (int)(lo / w), b = (int)((hi - 1) / w);
    if (digit == 5) {
        prefix.lo[5] = a;
        prefix.cnt[5] = b - a + 1;
        out[(*n)++] = prefix;
        return;
    }
    if (a == b) {
        prefix.lo[digit] = a;
        prefix.cnt[digit] = 1;
        fz_boxes(nl, lo - a * w, hi - a * w, digit + 1, prefix, out, n);
        return;
    }
    int first_full = a, last_full = b;               // digits whose whole sub-range is inside [lo, hi)
    if (lo != a * w) {
        prefix.lo[digit] = a;
        prefix.cnt[digit] = 1;
        fz_boxes(nl, lo - a * w, w, digit + 1, prefix, out, n);
        first_full = a + 1;
    }
    if (hi != (b + 1) * w) last_full = b - 1;
    if (last_full >= first_full) {
        FzBox m = prefix;
        m.lo[digit] = first_full;
        m.cnt[digit] = last_full - first_full + 1;
        for (int d = digit + 1; d < 6; ++d) {
            m.lo[d] = 0;
            m.cnt[d] = nl;
        }
        out[(*n)++] = m;
    }
    if (hi != (b + 1) * w) {
        prefix.lo[digit] = b;
        prefix.cnt[digit] = 1;
        fz_boxes(nl, 0, hi - b * w, digit + 1, prefix, out, n);
    }
}

/* Host helper behind the C ABI (include/sfoam.h): the boxes the factorised path splits [shell_lo, shell_hi) into. */
extern "C" int sf_shell_boxes(int two_dl, long shell_lo, long shell_hi, int boxes[16][12], int* n_boxes)
{
    if (!boxes || !n_boxes || two_dl < 0 || (two_dl & 1)) return SF_EARG;
    const int nl = two_dl / 2 + 1;
    long n_shells = 1;
    for (int d = 0; d < 6; ++d) n_shells *= nl;
    if (shell_lo < 0 || shell_hi > n_shells || shell_lo > shell_hi) return SF_EARG;
    FzBox b[16], none;
    memset(&none, 0, sizeof none);
    int n = 0;
    fz_boxes(nl, shell_lo, shell_hi, 0, none, b, &n);
    for (int k = 0; k < n; ++k)
        for (int d = 0; d < 6; ++d) {
            boxes[k][d] = b[k].lo[d];
            boxes[k][6 + d] = b[k].cnt[d];
        }
    *n_boxes = n;
    return SF_OK;
}

struct FzShape {
    bool ok;
    int V, NP, W4p, LDQ, VG;
    size_t qp_smem;
};

static FzShape fz_shape(const SfDims& D)
{
    FzShape s;
    memset(&s, 0, sizeof s);
    for (int e = 0; e < 4; ++e)
        if (D.k_max[e] == 0) return s;
    if (D.nl > 32 || D.n_k_pad[1] > 78) return s;     // k_fz_gemm keeps P3 + 1 prefix sums in 80 ints
    for (int a = 0; a < D.n_i[0]; ++a)
        for (int o = 0; o < D.nl; ++o) {
            int x0, nxs, xg0;
            fz_xrange(D.two_i_min[0], D.two_j[J25], D.two_x_base, a, o, x0, nxs, xg0);
            if (nxs > s.V) s.V = nxs;
        }
    const int n54 = D.n_i[3] * D.n_i[4];
    s.NP = (n54 + 1) & ~1;
    int w3 = 0, w4 = 0;
    for (int u = 0; u < D.nl; ++u)
        for (int v = 0; v < D.nl; ++v) {
            const int2 a = fz_window(D.two_j[J34] + 2 * u, D.two_j[J35] + 2 * v, D.two_k_base[1], D.n_k_pad[1]);
            const int2 b = fz_window(D.two_j[J24] + 2 * u, D.two_j[J34] + 2 * v, D.two_k_base[2], D.n_k_pad[2]);
            if (a.y > w3) w3 = a.y;
            if (b.y > w4) w4 = b.y;
        }
    s.W4p = (w4 + 3) & ~3;
    if (w3 == 0 || s.W4p == 0) return s;
    s.LDQ = ((n54 + 15) & ~15) + 4;                   // = 4 mod 16: conflict-free B fragments (lanes q * LDQ + g of a half warp)
    // x values per pass.  Every pass costs two CTA barriers and a fixed amount of index work, so more x per pass is better
    // as long as the 8-row tiles of (v, i5) stay well filled, the rows fit the fast Q phase (8 FZ_QMT) and two CTAs keep
    // ~100 KB of the SM for L1: the largest vg inside 80 KB with fill >= 0.8, else the best-filled one; a single x may take up
    // to 200 KB (one CTA per SM) before the path gives up.
    int best = 0, best_any = 0;
    double best_fill = 0.0;
    for (int vg = 1; vg <= s.V; ++vg) {
        const size_t bytes = sizeof(double) * (size_t)vg * s.W4p * s.LDQ;
        if (bytes > (vg == 1 ? 200 : 80) * 1024) break;
        const int rows = vg * D.n_i[4];
        const double fill = (double)rows / (((rows + 7) / 8) * 8);
        if (fill > best_fill + 1e-9) {
            best_fill = fill;
            best_any = vg;
        }
        if (fill >= 0.8 && (rows <= 8 * FZ_QMT || best == 0)) best = vg;
    }
    if (best == 0) best = best_any;
    if (best == 0) return s;
    s.VG = best;
    s.qp_smem = sizeof(double) * (size_t)s.VG * s.W4p * s.LDQ;
    // int offsets inside one gather-GEMM item
    const double slab = (double)D.n_k_pad[1] * s.V * D.nl * D.n_i[2] * s.NP;
    if (slab > 2.0e9 || (double)D.n_out / D.n_i[0] > 2.0e9) return s;
    // the k list of A' (one entry per (k3, x, l23)) lives in shared memory beside the operand ring of k_fz_gemm<FzMapA>
    if ((long)D.n_k_pad[1] * s.V * D.nl > 26000) return s;    // 226 KB - 116.7 KB ring - 3.4 KB tables = 4 B x 27 100 entries
    s.ok = true;
    return s;
}

bool sf_vertex_factor_supported(const SfDims& D) { return fz_shape(D).ok; }

static int g_fz_last_qp = 0;                         // Q/P kernel of the last call: 1 k_fz_qp, 2 k_fz_qp2, 4 k_fz_qp4 (sf_last_qp_kernel)
extern "C" int sf_last_qp_kernel(void) { return g_fz_last_qp; }
static int g_fz_variant = 0;                         // sf_set_factor_variant: bit 0 = R through the booster-stationary kernel
extern "C" void sf_set_factor_variant(int bits)
{
    SfHostLock lock;
    g_fz_variant = bits;
    sf_bump_generation();
}
static size_t g_fz_budget = 0;                       // sf_set_factor_budget: bytes for P and R of one pass (0 = a third of the device)
// Smallest P + R request (bytes of one pass) the device has refused so far (0 = none): later calls start below it instead of
// repeating, on every call, a cudaDeviceSynchronize, a cudaFree and a cudaMalloc that fails -- and a generation bump that keeps
// the call from ever being recorded.  Forgotten when the budget is set and by sf_finalize (the other tenant may be gone).
static size_t g_fz_refused = 0;
void sf_vertex_factor_forget(void) { g_fz_refused = 0; }
extern "C" void sf_set_factor_budget(unsigned long bytes)
{
    SfHostLock lock;
    g_fz_budget = bytes;
    g_fz_refused = 0;
    sf_bump_generation();
}

template <class Map, int WGM, int WGN, int TM, int TN>
static int fz_launch_gemm(const FzParams& p, int kcap, cudaStream_t st)
{
    constexpr int BM = WGM * TM * 8, BN = WGN * TN * 8;
    const size_t smem = sizeof(double) * Map::ST * Map::KC * (BM + 4 + BN + 4) + sizeof(int) * (2 * BM + 2 * BN + 240 + (size_t)kcap);
    if (smem > 226 * 1024) return SF_EARG;
    static SfPerContext<size_t> attr_c(0);
    size_t& attr = attr_c.get();
    if (smem > attr) {
        if (cudaFuncSetAttribute(k_fz_gemm<Map, WGM, WGN, TM, TN>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem) != cudaSuccess)
            return SF_ECUDA;
        attr = smem;
    }
    const long items = Map::items(p, BM, BN);
    if (items <= 0) return SF_OK;
    if (items > 2147483647L) return SF_EARG;
    k_fz_gemm<Map, WGM, WGN, TM, TN><<<(unsigned)items, WGM * WGN * 32, smem, st>>>(p, kcap);
    sf_count_launch(1);
    return SF_OK;
}

// ---- measurement: per-kernel CUDA-event times (sf_set_timing) and issued DMMA instructions (sf_set_counting) ----
#define FZ_MAX_EV 256
static cudaEvent_t g_fz_ev[FZ_MAX_EV];
static int g_fz_ev_made = 0, g_fz_ev_used = 0, g_fz_ev_class[FZ_MAX_EV / 2];
static double g_fz_ms[4], g_fz_dmma[3];

static void fz_ev_begin(int cls, cudaStream_t st)
{
    if (!sf_timing_on() || g_fz_ev_used + 2 > FZ_MAX_EV) return;
    while (g_fz_ev_made < g_fz_ev_used + 2) cudaEventCreate(&g_fz_ev[g_fz_ev_made++]);
    g_fz_ev_class[g_fz_ev_used / 2] = cls;
    cudaEventRecord(g_fz_ev[g_fz_ev_used], st);
}
static void fz_ev_end(cudaStream_t st)
{
    if (!sf_timing_on() || g_fz_ev_used + 2 > FZ_MAX_EV) return;
    cudaEventRecord(g_fz_ev[g_fz_ev_used + 1], st);
    g_fz_ev_used += 2;
}
/* ms[0..3] = k_fz_qp, k_fz_gemm<FzMapR>, k_fz_gemm<FzMapA>, the precomputations: summed over the launches of the last
 * factorised vertex call made with sf_set_timing(1) */
extern "C" int sf_last_kernel_ms(double ms[4])
{
    if (!ms) return SF_EARG;
    memcpy(ms, g_fz_ms, sizeof g_fz_ms);
    return SF_OK;
}
/* n[0..2] = DMMA.8x8x4 warp instructions issued by k_fz_qp, k_fz_gemm<FzMapR>, k_fz_gemm<FzMapA> in the last factorised
 * vertex call made with sf_set_counting(1) (512 flop each) */
extern "C" int sf_last_dmma(double n[3])
{
    if (!n) return SF_EARG;
    memcpy(n, g_fz_dmma, sizeof g_fz_dmma);
    return SF_OK;
}

int fz_launch_r2(const FzParams& p, const SfDims& D, int* sched, int n_sm, cudaStream_t st);   // sf_factor_r.cu
long fz_r3_b3w_elems(const FzParams& p, const SfDims& D, int* kcap);
int fz_launch_r3(const FzParams& p, const SfDims& D, double* Bw3W, bool build, cudaStream_t st);
bool fz_qp2_supported(const FzParams& p, const SfDims& D);                                     // sf_factor_qp.cu
long fz_qp2_b4p_elems(const FzParams& p, const SfDims& D);
int fz_launch_qp2(const FzParams& p, const SfDims& D, const double* Bw4P, int* sched, int n_sm, cudaStream_t st);
bool fz_qp4_supported(const FzParams& p, const SfDims& D);                                     // sf_factor_qp4.cu
int fz_launch_qp4(const FzParams& p, const SfDims& D, const double* Bw4P, int* sched, int n_sm, cudaStream_t st);

enum { FZ_SLOT_SCHED = 22, FZ_SLOT_CNT = 23, FZ_SLOT_WIN = 24, FZ_SLOT_LIST, FZ_SLOT_Z, FZ_SLOT_B4, FZ_SLOT_B3, FZ_SLOT_S3, FZ_SLOT_G, FZ_SLOT_P, FZ_SLOT_R, FZ_SLOT_PART, FZ_SLOT_B3W };

int sf_vertex_factor(const SfDims& D, const SfProblem& P, long shell_lo, long shell_hi, double* out, cudaStream_t st)
{
    const FzShape sh = fz_shape(D);
    if (!sh.ok) return SF_EARG;
    const int nl = D.nl, n1 = D.n_i[0], n2 = D.n_i[1], n3 = D.n_i[2], n4 = D.n_i[3], n5 = D.n_i[4];
    const int P3 = D.n_k_pad[1], P4 = D.n_k_pad[2];
    FzBox boxes[16];
    int nbox = 0;
    FzBox none;
    memset(&none, 0, sizeof none);
    fz_boxes(nl, shell_lo, shell_hi, 0, none, boxes, &nbox);
    long parts = 0;
    for (int b = 0; b < nbox; ++b) parts += (long)boxes[b].cnt[1] * boxes[b].cnt[2];

    FzParams p;
    memset(&p, 0, sizeof p);
    p.P = P;
    p.V = sh.V;
    p.NP = sh.NP;
    p.W4p = sh.W4p;
    p.LDQ = sh.LDQ;
    p.VG = sh.VG;
    for (int s = 0; s < 10; ++s) p.jsum += D.two_j[s];

    int* sched = (int*)sf_scratch(FZ_SLOT_SCHED, sizeof(int) * 1024);   // work counters: [pass] Q/P kernel, [512 + pass] R kernel
    if (!sched) return SF_ENOMEM;
    int2* win = (int2*)sf_scratch(FZ_SLOT_WIN, sizeof(int2) * (2 * (size_t)nl * nl + 2 * nl));
    double* Apart = (double*)sf_scratch(FZ_SLOT_PART, sizeof(double) * (size_t)(parts > 0 ? parts : 1) * D.n_out);
    if (!win || !Apart) return SF_ENOMEM;
    int2 *w3A = win, *w4A = win + nl * nl, *w3B = win + 2 * nl * nl, *w4B = w3B + nl;
    p.w3A = w3A;
    p.w3B = w3B;
    p.w4A = w4A;
    p.w4B = w4B;
    p.Apart = Apart;
    static SfPerContext<bool> qp_attr_c(false);
    bool& qp_attr = qp_attr_c.get();
    if (!qp_attr) {
        if (cudaFuncSetAttribute(k_fz_qp, cudaFuncAttributeMaxDynamicSharedMemorySize, 201 * 1024) != cudaSuccess) return SF_ECUDA;
        qp_attr = true;
    }
    static SfPerContext<int> n_sm_c(0);
    int& n_sm = n_sm_c.get();
    if (!n_sm) {
        int dev = 0;
        SF_CUDA_OK(cudaGetDevice(&dev));
        SF_CUDA_OK(cudaDeviceGetAttribute(&n_sm, cudaDevAttrMultiProcessorCount, dev));
    }
    static SfPerContext<size_t> total_b_c(0);        // device memory size: asked once per context (cudaMemGetInfo costs milliseconds)
    size_t& total_b = total_b_c.get();
    if (!total_b) {
        size_t free_b = 0;
        if (cudaMemGetInfo(&free_b, &total_b) != cudaSuccess) return SF_ECUDA;
    }

    g_fz_ev_used = 0;
    if (sf_counting_on()) {
        p.cnt = (unsigned long long*)sf_scratch(FZ_SLOT_CNT, 3 * sizeof(unsigned long long));
        if (!p.cnt) return SF_ENOMEM;
        SF_CUDA_OK(cudaMemsetAsync(p.cnt, 0, 3 * sizeof(unsigned long long), st));
    }
    long part0 = 0;
    for (int bi = 0; bi < nbox; ++bi) {
        const FzBox& bx = boxes[bi];
        p.box = bx;
        p.part0 = part0;
        const long c23 = bx.cnt[0], c24 = bx.cnt[1], c25 = bx.cnt[2], c34 = bx.cnt[3], c35 = bx.cnt[4], c45 = bx.cnt[5];
        int lo = 1 << 30, hi = 0;
        for (int o = bx.lo[5]; o < bx.lo[5] + bx.cnt[5]; ++o) {
            const int2 w = fz_window(D.two_j[J45] + 2 * o, D.two_j[J14], D.two_k_base[2], P4);
            if (w.y > 0) {
                if (w.x < lo) lo = w.x;
                if (w.x + w.y > hi) hi = w.x + w.y;
            }
        }
        p.hull4B = make_int2(lo < hi ? lo : 0, lo < hi ? hi : 0);

        const long nZ = c25 * n1 * c35 * c45 * ((long)P4 * sh.V * n5);
        const bool qp4 = !(g_fz_variant & 6) && fz_qp4_supported(p, D);      // warp-autonomous Q/P kernel (one warp per unit)
        const bool qp2 = qp4 || (!(g_fz_variant & 2) && fz_qp2_supported(p, D));   // second generation; both use the booster layout Bw4P
        g_fz_last_qp = qp4 ? 4 : qp2 ? 2 : 1;
        const long nB4 = qp2 ? fz_qp2_b4p_elems(p, D) : (long)P4 * c45 * c24 * c34 * n4, nB3 = (long)P3 * c34 * c35 * c23 * n3;
        const long nS3 = c24 * c34 * c35 * D.n_x_pad * P3 * P4;
        const long nG = c24 * c25 * n1 * P3 * sh.V * c23 * n2;
        const long pP = c24 * c25 * P3 * sh.V * c34 * c35 * sh.NP;     // per i1
        const long pR = c24 * c25 * P3 * sh.V * c23 * n3 * sh.NP;
        // i1 values per pass: P and R of a pass inside ~1/3 of the device memory
        const double budget = g_fz_budget ? (double)g_fz_budget : (double)total_b / 3.0;
        long na = (long)(budget / (8.0 * (double)(pP + pR)));
        if (na < 1) {
            if (!g_fz_budget) return SF_ENOMEM;
            na = 1;                                  // a test budget below one i1 still runs, one i1 per pass
        }
        if (na > n1) na = n1;
        na = (n1 + (n1 + na - 1) / na - 1) / ((n1 + na - 1) / na);   // the same number of passes, of equal size (config 3: 4 + 4 + 3, not 5 + 5 + 1)
        double* Z = (double*)sf_scratch(FZ_SLOT_Z, sizeof(double) * (size_t)nZ);
        const long padB4 = 4L * 12 * 16;             // k_fz_qp4 copies whole k-steps (4 k4) of Bw4P: the last one may end past the array
        double* B4 = (double*)sf_scratch(FZ_SLOT_B4, sizeof(double) * (size_t)(nB4 + padB4));
        double* B3 = (double*)sf_scratch(FZ_SLOT_B3, sizeof(double) * (size_t)nB3);
        const long padS3 = 24L * P4 + 8;             // k_fz_qp2 reads fragment rows / columns just past a block: keep them finite
        double* S3 = (double*)sf_scratch(FZ_SLOT_S3, sizeof(double) * (size_t)(nS3 + padS3));
        double* G = (double*)sf_scratch(FZ_SLOT_G, sizeof(double) * (size_t)nG);
        double *Pq = nullptr, *Rq = nullptr;
        while (na > 1 && g_fz_refused && sizeof(double) * (size_t)((pP + pR) * na) >= g_fz_refused) na = (na + 1) / 2;
        for (;;) {                                   // other tenants of the device may hold memory: shrink the pass until it fits
            Pq = (double*)sf_scratch(FZ_SLOT_P, sizeof(double) * (size_t)(pP * na));
            Rq = Pq ? (double*)sf_scratch(FZ_SLOT_R, sizeof(double) * (size_t)(pR * na)) : nullptr;
            if ((Pq && Rq) || na == 1) break;
            const size_t asked = sizeof(double) * (size_t)((pP + pR) * na);
            if (!g_fz_refused || asked < g_fz_refused) g_fz_refused = asked;
            if (Pq) sf_scratch_release(FZ_SLOT_P);   // P fitted, R did not: P's block of this size would starve the smaller R as well
            na = (na + 1) / 2;
        }
        int* lists = (int*)sf_scratch(FZ_SLOT_LIST, sizeof(int2) * P3 + sizeof(int) * (size_t)P3 * (1 + c34 * c35));
        int ldw = 0;
        const bool r3 = !(g_fz_variant & 9);             // R through the producer-warp kernel (bit 0: k_fz_r2, bit 3: the gather-GEMM)
        double* B3W = r3 ? (double*)sf_scratch(FZ_SLOT_B3W, sizeof(double) * (size_t)fz_r3_b3w_elems(p, D, &ldw)) : nullptr;
        if (!Z || !B4 || !B3 || !S3 || !G || !Pq || !Rq || !lists || (r3 && !B3W)) return SF_ENOMEM;
        p.win23 = (const int2*)lists;
        p.kl3 = lists + 2 * P3;
        p.Z = Z;
        p.Bw4T = B4;
        p.Bw3T = B3;
        p.S3T = S3;
        p.G = G;
        p.Pq = Pq;
        p.Rq = Rq;
        p.a_lo = 0;
        p.a_cnt = n1;
        if (sf_poison_on()) {                        // debug: an entry read without having been written becomes a NaN
            SF_CUDA_OK(cudaMemsetAsync(Z, 0xFF, sizeof(double) * (size_t)nZ, st));
            SF_CUDA_OK(cudaMemsetAsync(G, 0xFF, sizeof(double) * (size_t)nG, st));
        }
        fz_ev_begin(3, st);
        {   // every precomputation of the box in one launch (k_fz_pre)
            FzPreArgs a;
            memset(&a, 0, sizeof a);
            const long nz = c25 * n1 * c35 * c45;            // few (l25 i1 l35 l45): spread the k4 over more blocks as well
            a.gy = nz >= 592 ? 1 : (int)((592 + nz - 1) / nz < P4 ? (592 + nz - 1) / nz : P4);
            a.b4p = qp2;
            a.nB4 = nB4;
            a.padB4 = qp2 ? padB4 : 0;
            a.nB3 = nB3;
            a.nS3 = nS3;
            a.padS3 = padS3;
            a.n_sched = 1024;
            a.Z = Z;
            a.B4 = B4;
            a.B3 = B3;
            a.S3 = S3;
            a.G = G;
            a.w3A = w3A;
            a.w3B = w3B;
            a.w4A = w4A;
            a.w4B = w4B;
            a.win23 = (int2*)lists;
            a.kl3 = lists + 2 * P3;
            a.sched = sched;
            const long nb[8] = {c24 * c25 * n1 * P3, nz * a.gy, (a.nB4 + a.padB4 + 255) / 256, (nB3 + 255) / 256,
                                (nS3 + padS3 + 255) / 256, (nl * nl + 255) / 256, (P3 + 7) / 8, 1};
            a.first[0] = 0;
            for (int t = 0; t < 8; ++t) a.first[t + 1] = a.first[t] + nb[t];
            if (a.first[8] > 2147483647L) return SF_EARG;
            if (n1 > 512) return SF_EARG;                    // one counter per pass over i1
            k_fz_pre<<<(unsigned)a.first[8], 256, 0, st>>>(p, a);
        }
        sf_count_launch(1);
        fz_ev_end(st);
        int pass = 0;
        for (int a_lo = 0; a_lo < n1; a_lo += (int)na, ++pass) {
            p.a_lo = a_lo;
            p.a_cnt = (int)(a_lo + na <= n1 ? na : n1 - a_lo);
            if (sf_poison_on()) {
                SF_CUDA_OK(cudaMemsetAsync(Pq, 0xFF, sizeof(double) * (size_t)(pP * na), st));
                SF_CUDA_OK(cudaMemsetAsync(Rq, 0xFF, sizeof(double) * (size_t)(pR * na), st));
            }
            fz_ev_begin(0, st);
            if (qp2) {
                const int rcq = qp4 ? fz_launch_qp4(p, D, B4, sched + pass, n_sm, st) : fz_launch_qp2(p, D, B4, sched + pass, n_sm, st);
                if (rcq != SF_OK) return rcq;
            } else {                                  // shapes the newer kernels do not hold
                const long n_items = (long)p.a_cnt * c25 * c35 * c24 * c34;
                const long grid = n_items < 2L * n_sm ? n_items : 2L * n_sm;
                k_fz_qp<<<(unsigned)grid, FZ_QP_THREADS, sh.qp_smem, st>>>(p, n_items);
                sf_count_launch(1);
            }
            fz_ev_end(st);
            fz_ev_begin(1, st);
            int rc = r3 ? fz_launch_r3(p, D, B3W, pass == 0, st)                                          // producer warp, bulk copies for both operands
                        : g_fz_variant & 1 ? fz_launch_r2(p, D, sched + 512 + pass, n_sm, st) : SF_EARG;      // booster block stationary
            if (rc == SF_EARG) rc = fz_launch_gemm<FzMapR, 8, 1, 2, 8>(p, (int)(c34 * c35), st);   // shapes it does not hold
            fz_ev_end(st);
            if (rc != SF_OK) return rc;
            fz_ev_begin(2, st);
            rc = n2 <= 16 ? fz_launch_gemm<FzMapA, 1, 8, 2, 4>(p, (int)(P3 * sh.V * c23), st)      // rows i2: one tile of 16
                          : fz_launch_gemm<FzMapA, 1, 8, 4, 4>(p, (int)(P3 * sh.V * c23), st);     // or of 32: R is read once
            fz_ev_end(st);
            if (rc != SF_OK) return rc;
        }
        part0 += c24 * c25;
    }
    sf_timing_mark(2, st);
    k_fz_reduce<<<(unsigned)((D.n_out + 255) / 256), 256, 0, st>>>(P, parts, D.n_out, Apart, out);
    sf_count_launch(1);
    if (cudaGetLastError() != cudaSuccess) return SF_ECUDA;
    if (sf_timing_on() || sf_counting_on()) {        // measurement modes make the call synchronous
        SF_CUDA_OK(cudaStreamSynchronize(st));
        memset(g_fz_ms, 0, sizeof g_fz_ms);
        for (int e = 0; e + 1 < g_fz_ev_used; e += 2) {
            float ms = 0.f;
            cudaEventElapsedTime(&ms, g_fz_ev[e], g_fz_ev[e + 1]);
            g_fz_ms[g_fz_ev_class[e / 2]] += ms;
        }
        if (p.cnt) {
            unsigned long long h[3];
            SF_CUDA_OK(cudaMemcpy(h, p.cnt, sizeof h, cudaMemcpyDeviceToHost));
            for (int k = 0; k < 3; ++k) g_fz_dmma[k] = (double)h[k];
        }
    }
    return SF_OK;
}
