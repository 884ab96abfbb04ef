// sf_factor.cuh -- declarations shared by the kernels of the factorised path (sf_vertex_factor.cu and the sf_factor_*.cu
// files): the parameter block, the range predicates of step 2 that writer and reader of every intermediate
// share, and the PTX wrappers (FP64 tensor-core MMA, asynchronous copies, mbarriers).
#pragma once
#include "sf_internal.h"

// a box of shell offsets, order (o23 o24 o25 o34 o35 o45); o = lo .. lo + cnt - 1
struct FzBox {
    int lo[6], cnt[6];
};

struct FzParams {
    SfProblem P;
    FzBox box;
    int a_lo, a_cnt;            // the boundary intertwiners i1 of this pass (a1 = a_lo .. a_lo + a_cnt - 1)
    int V;                      // largest number of x values of any (i1, l25): triad (i1 l25 x) of eq. (5)
    int NP;                     // n5 * n4 rounded up to even: row length of P and R
    int jsum;                   // sum of the ten boundary spins (2j units)
    int W4p, LDQ, VG;           // k_fz_qp shared-memory shape: Qs[VG][W4p][LDQ]
    const int2* w3A;            // [o34][o35] window (lo, cnt) of q3 allowed by the pair (l34 l35)
    const int2* w3B;            // [o23]      window of q3 allowed by the pair (j13 l23)
    const int2* w4A;            // [o24][o34] window of q4 allowed by the pair (l24 l34)
    const int2* w4B;            // [o45]      window of q4 allowed by the pair (l45 j14)
    int2 hull4B;                // union of w4B over the box: (lo, hi exclusive)
    const int2* win23;          // [q3] (first b23, count) of the box's l23 whose pair (j13 l23) allows k3
    const int* kl3;             // [q3][1 + c34 c35]: count, then the box's pairs (b34 c35 + b35) whose (l34 l35) allow k3, ascending
    const double* Z;            // [b25][a1][b35][b45][q4][v][i5]
    const double* Bw4T;         // [q4][b45][b24][b34][i4]
    const double* Bw3T;         // [q3][b34][b35][b23][i3]
    const double* S3T;          // [b24][b34][b35][xx][q3][q4], sign (-1)^o34 folded in
    const double* G;            // [b24][b25][a1][q3][v][b23][i2]
    double* Pq;                 // [ac][b24][b25][q3][v][b34][b35][NP]
    double* Rq;                 // [ac][b24][b25][q3][v][b23][i3][NP]
    double* Apart;              // [part][a1][i2][i3][i4][i5]
    long part0;                 // first partial tensor of this box
    unsigned long long* cnt;    // measurement only (sf_set_counting): DMMA instructions issued by k_fz_qp, R, A'; else null
};

// window (lo, cnt) of q = (k - k_base) / 2 inside [0, n_pad) allowed by the triangle |a - b| <= k <= a + b
__host__ __device__ inline int2 fz_window(int a, int b, int two_k_base, int n_pad)
{
    int lo_k = a > b ? a - b : b - a;
    const int hi_k = a + b;
    int2 w;
    w.x = 0;
    w.y = 0;
    if ((lo_k - two_k_base) & 1) return w;
    int qlo = (lo_k - two_k_base) / 2, qhi = (hi_k - two_k_base) / 2;
    if (qlo < 0) qlo = 0;
    if (qhi > n_pad - 1) qhi = n_pad - 1;
    if (qhi < qlo) return w;
    w.x = qlo;
    w.y = qhi - qlo + 1;
    return w;
}

// x values of the triad (i1 l25 x): first x, count, index of the first in the S arrays' x layout
__host__ __device__ inline void fz_xrange(const int two_i1_min, int two_j25, int two_x_base, int a1, int o25, int& x0,
                                          int& nxs, int& xg0)
{
    const int i1 = two_i1_min + 2 * a1, l25 = two_j25 + 2 * o25;
    x0 = i1 > l25 ? i1 - l25 : l25 - i1;
    nxs = ((i1 + l25 - x0) >> 1) + 1;
    xg0 = (x0 - two_x_base) >> 1;
}

// the x indices v (x = x0 + 2v, v < nxs) for which the triad (k l x) holds: a contiguous run (first, count).  Same
// predicate as fz_window(l, x, ..) evaluated at k, so the rows k_fz_qp writes are the rows k_fz_gemm reads.
__host__ __device__ inline int2 fz_vrange(int two_l, int two_k, int x0, int nxs)
{
    int first = -1, cnt = 0;
    for (int v = 0; v < nxs; ++v) {
        const int x = x0 + 2 * v, d = two_l > x ? two_l - x : x - two_l;
        if (two_k >= d && two_k <= two_l + x && !((two_l + x + two_k) & 1)) {
            if (first < 0) first = v;
            ++cnt;
        }
    }
    int2 r;
    r.x = first < 0 ? 0 : first;
    r.y = cnt;
    return r;
}

// the booster operand of the Q phase in fragment order (k_fz_qp2, k_fz_qp4), 12 rows l45 per k4:
// Bw4P[b24][b34][q4][ks][lane][j] = (2k4+1) B4[(o45 o24 o34)][i4][q4], l45 = 4 ks + lane % 4, i4 = 8 j + lane / 4, inside the triple's
// k-range, 0 elsewhere: one 16-byte load per lane and k-step, 512 contiguous bytes per warp
__device__ __forceinline__ void fz_b4p_entry(const FzParams& p, long n, double* __restrict__ out, long e)
{
    const SfProblem& P = p.P;
    if (e >= n) return;
    const int nl = P.nl, n4 = P.n_i[3], P4 = P.n_k_pad[2];
    const int c34 = p.box.cnt[3], c45 = p.box.cnt[5];
    long r = e;
    const int jj = (int)(r % 2); r /= 2;
    const int ln = (int)(r % 32); r /= 32;
    const int ks = (int)(r % 3); r /= 3;
    const int i4 = 8 * jj + (ln >> 2), b45 = 4 * ks + (ln & 3);
    const int q4 = (int)(r % P4); r /= P4;
    const int b34 = (int)(r % c34);
    const int b24 = (int)(r / c34);
    double val = 0.0;
    if (i4 < n4 && b45 < c45) {
        const int t4 = ((p.box.lo[5] + b45) * nl + p.box.lo[1] + b24) * nl + p.box.lo[3] + b34;
        const SfKRange r4 = P.kr[2][t4];
        const int c = q4 - ((r4.two_k_min - P.two_k_base[2]) >> 1);
        if (c >= 0 && c < r4.n_k) val = (double)(r4.two_k_min + 2 * c + 1) * sf_brow(P, 2, t4, i4)[q4];
    }
    out[e] = val;
}


__device__ __forceinline__ void fz_dmma(double& c0, double& c1, double a, double b)
{
    asm("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1},{%2},{%3},{%0,%1};\n"
        : "+d"(c0), "+d"(c1)
        : "d"(a), "d"(b));
}

// the first MMA of a sum: C = A B (no accumulator to clear)
__device__ __forceinline__ void fz_dmma0(double& c0, double& c1, double a, double b)
{
    asm("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1},{%2},{%3},{%4,%4};\n"
        : "=d"(c0), "=d"(c1)
        : "d"(a), "d"(b), "d"(0.0));
}

__device__ __forceinline__ unsigned fz_smem_u32(const void* p) { return (unsigned)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void fz_cp_async8(unsigned dst, const void* src, int bytes)
{
    asm volatile("cp.async.ca.shared.global [%0], [%1], 8, %2;" ::"r"(dst), "l"(src), "r"(bytes) : "memory");
}
__device__ __forceinline__ void fz_cp_async16(unsigned dst, const void* src, int bytes)
{
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16, %2;" ::"r"(dst), "l"(src), "r"(bytes) : "memory");
}
__device__ __forceinline__ void fz_cp_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
template <int N>
__device__ __forceinline__ void fz_cp_wait()
{
    asm volatile("cp.async.wait_group %0;" ::"n"(N) : "memory");
}

// mbarrier / bulk-copy primitives (PTX ISA: mbarrier, cp.async.bulk; SASS UBLKCP)
__device__ __forceinline__ void fz_mbar_init(unsigned bar, unsigned count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count));
}
__device__ __forceinline__ void fz_mbar_expect_tx(unsigned bar, unsigned bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void fz_mbar_wait(unsigned bar, unsigned parity)
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
__device__ __forceinline__ void fz_bulk_g2s(unsigned dst, const void* src, unsigned bytes, unsigned bar)
{
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(dst),
                 "l"(src), "r"(bytes), "r"(bar)
                 : "memory");
}
__device__ __forceinline__ void fz_prefetch_l1(const void* p) { asm volatile("prefetch.global.L1 [%0];" ::"l"(p)); }

