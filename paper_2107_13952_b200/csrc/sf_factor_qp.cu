// sf_factor_qp.cu -- the edge-4 contraction of the factorised path (sf_vertex_factor.cu, DESIGN.md 5 K-f), second generation:
//
//   Q[k4; i5 i4]            = sum_l45 Z[l25 i1 l35 l45; k4 x i5] Bw4P[l24 l34; k4; l45; i4]      (the shells of a line l45)
//   P[k3; (i5 i4)]          = sum_k4  S3T[l24 l34 l35; x; k3 k4] Q[k4; i5 i4]                    (third {6j} of eq. (5), edge-4 product)
//
// for every (i1 l25 l35 | l24 l34 | x): steps 6(i)-(iii) of the algorithm for the factors of eq. (3) that
// carry l45 and k4.  Q never leaves the chip; the rows of P the triads allow go to HBM for the edge-3 contraction.
//
// Work decomposition (what differs from the first kernel, k_fz_qp):
//   * a CTA (16 warps, one per SM) takes items (i1, l25, l35, chunk of <= 4 x) from an atomic counter (execution order only:
//     every row of P has one writer) and keeps the item's slab of Z in shared memory (8-byte cp.async), where all the
//     121 x 4 units (l24, l34, x) of the item read it;
//   * the 16 warps form 4 independent GROUPS of 4 warps (one warp per SM sub-partition); a group takes units (l24 l34 x)
//     and walks the k4 of the unit 4 at a time.  For each such k-step: every warp computes Q for one k4 (2 x 2 tiles, K =
//     l45) into the group's private double-buffered Q tile, one named barrier among the group's 128 threads, then every
//     warp accumulates its quarter of the columns (i5 i4) of P over the k-step from that tile.  No CTA-wide barrier inside
//     an item, and the index windows (k3 by (l34 l35) and (l24 x); k4 by (l24 l34), (l45 j14) and (l35 x)) are exact per unit;
//   * operands are laid out so that the inner loop needs no predicates and one address addition per fragment group: the
//     weighted booster Bw4P[l24 l34; k4; 12; 16] is zero-padded in global memory, the Q tile keeps (i5, i4) in a 16 x 16
//     grid per k4 (the column (i5 i4) of P a lane needs is a per-lane constant offset), the {6j} array is exactly zero where
//     a triad fails, and a k4 beyond the unit's window gets a zero row of Q;
//   * all fragment loads from shared memory are conflict-free (row strides = 4 mod 16 doubles).
//
// Shapes it holds: n5 <= 16, n4 <= 16, n5 n4 <= 128, at most 12 values of l45 in the box, k3 windows of at most 24 values,
// at most 24 values of k4 in the layout.  sf_vertex_factor falls back to k_fz_qp otherwise.
#include "sf_factor.cuh"

#define FQ_THREADS 512
#define FQ_XC 4                   // x values per item
#define FQ_QI5 24                 // stride of i5 inside a Q tile row: 16 i4 + 8 pad, so that the 16-byte stores of a quarter warp
                                  // (two i5, four column pairs) fall into different banks
#define FQ_LDQ 388                // row stride of the Q tiles: 16 x FQ_QI5 entries (i5, i4) per k4, + 4 (= 4 mod 16)
#define FQ_GRP (2 * 4 * FQ_LDQ + 2 * 3 * 32)   // doubles of shared memory per group: two Q tiles, two S3 fragment tiles
#define FQ_L45 12                 // l45 rows per k4 in the Z slab and in Bw4P (3 k-steps)

struct FzQp2Args {
    int ldz;                      // row stride of the Z slab (= 4 mod 16, >= 3 n5 + 16)
    int vc;                       // chunks of FQ_XC x per (i1 l25)
    int n_items;
    int* sched;
    const double* Bw4P;           // [b24][b34][q4][k-step 3][lane 32][column tile 2]: the B fragments of Q in the order the lanes
                                  // read them (l45 = 4 ks + lane % 4, i4 = 8 j + lane / 4), zero outside the triple's k-range
                                  // and beyond (c45, n4)
};

__device__ __forceinline__ void fq_group_sync(int grp)
{
    asm volatile("bar.sync %0, 128;" ::"r"(grp + 1) : "memory");
}
__device__ __forceinline__ double fq_lds(unsigned addr)
{
    double v;
    asm volatile("ld.shared.f64 %0, [%1];" : "=d"(v) : "r"(addr));
    return v;
}
__device__ __forceinline__ void fq_sts2(unsigned addr, double a, double b)
{
    asm volatile("st.shared.v2.f64 [%0], {%1, %2};" ::"r"(addr), "d"(a), "d"(b) : "memory");
}

__global__ void __launch_bounds__(FQ_THREADS, 1) k_fz_qp2(const __grid_constant__ FzParams p, const __grid_constant__ FzQp2Args a)
{
    extern __shared__ __align__(16) double smem[];
    __shared__ int s_item;
    __shared__ int2 s_wx[32 * FQ_XC];                         // [b24][x of the item]: window of k3 allowed by the triad (k3 l24 x)
    __shared__ int2 s_w4x[FQ_XC];                             // [x of the item]: window of k4 allowed by the triad (k4 l35 x)
    const SfProblem& P = p.P;
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31, g = lane >> 2, q = lane & 3;
    const int grp = warp >> 2, wq = warp & 3;                 // group of 4 warps; this warp's k4 of a k-step / column quarter
    const int nl = P.nl, n1 = P.n_i[0], n4 = P.n_i[3], n5 = P.n_i[4], n54 = n4 * n5;
    const int P3 = P.n_k_pad[1], P4 = P.n_k_pad[2], NX = P.n_x_pad, V = p.V, NP = p.NP;
    const int c24 = p.box.cnt[1], c25 = p.box.cnt[2], c34 = p.box.cnt[3], c35 = p.box.cnt[4], c45 = p.box.cnt[5];
    const int ldz = a.ldz, KS45 = (c45 + 3) >> 2, NT = (n54 + 7) >> 3;
    const int sZ = P4 * V * n5;
    const long prow = (long)c34 * c35 * NP;                   // stride of v in P
    const int nzs = P4 * FQ_L45 * ldz;
    double* Zs = smem;                                        // [P4][FQ_L45][ldz]
    for (int z = tid; z < nzs + 4 * FQ_GRP; z += FQ_THREADS) smem[z] = 0.0;   // pad rows stay finite
    const unsigned zs_u32 = fz_smem_u32(Zs);
    const unsigned qs_u32 = zs_u32 + 8u * (unsigned)(nzs + grp * FQ_GRP);                 // this group's Q tiles [2][4][FQ_LDQ]
    const unsigned s3s_u32 = qs_u32 + 8u * (unsigned)(2 * 4 * FQ_LDQ + lane);             // and S3 fragment tiles [2][3][32], this lane's entry
    // per-lane constants of the fragment addresses (bytes)
    const unsigned z_lane = 8u * (unsigned)(q * ldz + g);                             // A of Q: row l45 = 4 ks + q, column + g
    const unsigned z_ks = 8u * (unsigned)(4 * ldz), z_k4 = 8u * (unsigned)(FQ_L45 * ldz);
    const unsigned qst_lane = 8u * (unsigned)(wq * FQ_LDQ + g * FQ_QI5 + 2 * q);          // C of Q: row i5 = 8 i + g, columns 8 j + 2 q, + 1
    unsigned qld_lane[4];                                                             // B of P: k4 row q, column (i5 i4) = 8 (4 wq + j) + g
#pragma unroll
    for (int j = 0; j < 4; ++j) {
        const int col = min(8 * (4 * wq + j) + g, n54 - 1), i5 = col / n4, i4 = col - i5 * n4;
        qld_lane[j] = 8u * (unsigned)(q * FQ_LDQ + i5 * FQ_QI5 + i4);
    }
    const int njt = min(4, max(0, NT - 4 * wq));              // live column tiles of this warp
    const int b4_lane = 2 * lane;                             // B of Q: fragment-major, (column tile 0, 1) adjacent
    unsigned ndm = 0;

    for (;;) {
        __syncthreads();                                      // everybody is done with the previous slab of Z and the tables
        if (tid == 0) s_item = atomicAdd(a.sched, 1);
        __syncthreads();
        int it = s_item;
        if (it >= a.n_items) break;
        const int b35 = it % c35; it /= c35;
        const int b25 = it % c25; it /= c25;
        const int ac = it % p.a_cnt;
        const int vc = it / p.a_cnt;
        const int a1 = p.a_lo + ac, o25 = p.box.lo[2] + b25, o35 = p.box.lo[4] + b35;
        int x0, nxs, xg0;
        fz_xrange(P.two_i_min[0], P.two_j[J25], P.two_x_base, a1, o25, x0, nxs, xg0);
        const int v0 = vc * FQ_XC, nv = min(FQ_XC, nxs - v0);
        if (nv <= 0) continue;
        const int l35 = P.two_j[J35] + 2 * o35;
        // k4 of the item: the union over its x of the triad (k4 l35 x), inside the l45 the box holds
        int h4lo = P4, h4hi = 0;
        for (int vv = 0; vv < nv; ++vv) {
            const int2 w = fz_window(l35, x0 + 2 * (v0 + vv), P.two_k_base[2], P4);
            if (w.y > 0) {
                h4lo = min(h4lo, w.x);
                h4hi = max(h4hi, w.x + w.y);
            }
        }
        h4lo = max(h4lo, p.hull4B.x);
        h4hi = min(h4hi, p.hull4B.y);
        if (tid < c24 * nv) {
            const int b24 = tid / nv, vv = tid - b24 * nv;
            s_wx[b24 * FQ_XC + vv] = fz_window(P.two_j[J24] + 2 * (p.box.lo[1] + b24), x0 + 2 * (v0 + vv), P.two_k_base[1], P3);
        }
        if (tid >= 480 && tid - 480 < nv) s_w4x[tid - 480] = fz_window(l35, x0 + 2 * (v0 + tid - 480), P.two_k_base[2], P4);
        // the slab of Z: rows (k4, l45), nv * n5 entries (x i5) each
        {
            const double* Zb = p.Z + ((((long)b25 * n1 + a1) * c35 + b35) * c45) * (long)sZ + (long)v0 * n5;
            const int rowlen = nv * n5, nrow = max(0, h4hi - h4lo) * c45;
            for (int r = warp; r < nrow; r += FQ_THREADS / 32) {
                const int r4 = r / c45, b45 = r - r4 * c45;
                const double* src = Zb + ((long)b45 * P4 + h4lo + r4) * (V * n5);
                const unsigned dst = zs_u32 + 8u * (unsigned)((r4 * FQ_L45 + b45) * ldz);
                for (int c = lane; c < rowlen; c += 32) fz_cp_async8(dst + 8u * c, src + c, 8);
            }
            fz_cp_commit();
            fz_cp_wait<0>();
        }
        __syncthreads();

        // units (b24, b34, x of the item), x fastest, round robin over the 4 groups
        int xloc = grp, b34 = 0, b24 = 0;
        for (;;) {
            while (xloc >= nv) {
                xloc -= nv;
                if (++b34 == c34) {
                    b34 = 0;
                    ++b24;
                }
            }
            if (b24 >= c24) break;
            const int xl = xloc;
            xloc += 4;
            const int o24 = p.box.lo[1] + b24, o34 = p.box.lo[3] + b34;
            const int2 w3 = p.w3A[o34 * nl + o35];            // the k3 the pair (l34 l35) allows
            if (w3.y == 0) continue;
            // rows k3 of this unit: (k3 l34 l35) and the triad (k3 l24 x)
            const int2 wx = s_wx[b24 * FQ_XC + xl];
            const int q3lo = max(wx.x, w3.x), q3hi = wx.y > 0 ? min(wx.x + wx.y, w3.x + w3.y) : 0;
            if (q3hi <= q3lo) continue;
            // k4 of this unit: (k4 l24 l34), the triad (k4 l35 x) and the l45 of the box
            const int2 w4a = p.w4A[o24 * nl + o34], w4x = s_w4x[xl];
            const int k4lo = max(max(w4a.x, w4x.x), h4lo);
            const int k4hi = (w4a.y > 0 && w4x.y > 0) ? min(min(w4a.x + w4a.y, w4x.x + w4x.y), h4hi) : 0;
            const int ng = k4hi > k4lo ? (k4hi - k4lo + 3) >> 2 : 0;
            const int MT3 = (q3hi - q3lo + 7) >> 3;           // <= 3
            // this lane's operand pointers at the first k-step
            const double* s3p = p.S3T + ((((long)b24 * c34 + b34) * c35 + b35) * NX + xg0 + v0 + xl) * (long)(P3 * P4) +
                                (long)(q3lo + 8 * wq + g) * P4 + k4lo + q;              // A of P, row tile wq: row k3 = q3lo + 8 wq + g, column k4
            const double* b4p = a.Bw4P + (((long)b24 * c34 + b34) * P4 + k4lo + wq) * (FQ_L45 * 16) + b4_lane;
            unsigned zq = zs_u32 + z_lane + 8u * (unsigned)(xl * n5) + (unsigned)(k4lo + wq - h4lo) * z_k4;

            double acc[3][4][2];
#pragma unroll
            for (int i = 0; i < 3; ++i)
#pragma unroll
                for (int j = 0; j < 4; ++j) acc[i][j][0] = acc[i][j][1] = 0.0;

            // Q of one k-step: this warp's k4 = k4lo + 4 gi + wq, into buffer gi & 1 (a zero row beyond the window); its booster
            // fragments bq are requested before the barrier that precedes it (b4_fetch)
            double bq[3][2];
            auto b4_fetch = [&](int gi) {
                const bool ok = k4lo + 4 * gi + wq < k4hi;
#pragma unroll
                for (int ks = 0; ks < 3; ++ks) {
                    const double2 v = (ok && ks < KS45) ? __ldg(reinterpret_cast<const double2*>(b4p + ks * 64)) : make_double2(0.0, 0.0);
                    bq[ks][0] = v.x;
                    bq[ks][1] = v.y;
                }
                b4p += 4 * FQ_L45 * 16;
            };
            auto q_phase = [&](int gi) {
                const unsigned dst = qs_u32 + qst_lane + 8u * (unsigned)((gi & 1) * 4 * FQ_LDQ);
                double c[2][2][2];
#pragma unroll
                for (int i = 0; i < 2; ++i)
#pragma unroll
                    for (int j = 0; j < 2; ++j) c[i][j][0] = c[i][j][1] = 0.0;
                if (k4lo + 4 * gi + wq < k4hi) {
#pragma unroll
                    for (int ks = 0; ks < 3; ++ks) {
                        if (ks < KS45) {
                            const double a0 = fq_lds(zq + ks * z_ks), a1v = fq_lds(zq + ks * z_ks + 64);
                            fz_dmma(c[0][0][0], c[0][0][1], a0, bq[ks][0]);
                            fz_dmma(c[0][1][0], c[0][1][1], a0, bq[ks][1]);
                            fz_dmma(c[1][0][0], c[1][0][1], a1v, bq[ks][0]);
                            fz_dmma(c[1][1][0], c[1][1][1], a1v, bq[ks][1]);
                        }
                    }
                    ndm += 4 * KS45;
                }
                zq += 4 * z_k4;
#pragma unroll
                for (int i = 0; i < 2; ++i)
#pragma unroll
                    for (int j = 0; j < 2; ++j) fq_sts2(dst + 8u * (unsigned)(i * 8 * FQ_QI5 + j * 8), c[i][j][0], c[i][j][1]);
            };
            // S3 fragments of a k-step: warp i < MT3 of the group fetches the fragment of row tile i (straight from L1/L2; the
            // {6j} array is zero wherever a triad fails, so rows and columns beyond the unit's windows need no predicate: their
            // k4 meet zero rows of Q, their k3 are not stored) and leaves it in the group's fragment tile for the other three
            double s3v = 0.0;                                 // this lane's S3 entry of the next k-step to be staged, fetched one k-step ahead
            auto s3_fetch = [&]() {
                if (wq < MT3) s3v = __ldg(s3p);
                s3p += 4;
            };
            auto s3_stage = [&](int gi) {
                if (wq < MT3)
                    asm volatile("st.shared.f64 [%0], %1;" ::"r"(s3s_u32 + 8u * (unsigned)(((gi & 1) * 3 + wq) * 32)), "d"(s3v) : "memory");
            };

            if (ng > 0) {
                b4_fetch(0);
                s3_fetch();
            }
            fq_group_sync(grp);                               // the group is done with the previous unit's tiles
            if (ng > 0) {
                s3_stage(0);
                if (ng > 1) s3_fetch();
                q_phase(0);
            }
            for (int gi = 0; gi < ng; ++gi) {
                if (gi + 1 < ng) b4_fetch(gi + 1);
                fq_group_sync(grp);                           // Q and S3 of k-step gi are complete; everybody finished P of gi - 1
                if (gi + 1 < ng) {
                    s3_stage(gi + 1);
                    if (gi + 2 < ng) s3_fetch();
                    q_phase(gi + 1);
                }
                const unsigned bs = qs_u32 + 8u * (unsigned)((gi & 1) * 4 * FQ_LDQ);
                double av[3], bv[4];
#pragma unroll
                for (int i = 0; i < 3; ++i) av[i] = i < MT3 ? fq_lds(s3s_u32 + 8u * (unsigned)(((gi & 1) * 3 + i) * 32)) : 0.0;
#pragma unroll
                for (int j = 0; j < 4; ++j) bv[j] = fq_lds(bs + qld_lane[j]);
#pragma unroll
                for (int i = 0; i < 3; ++i) {
                    if (i < MT3) {
#pragma unroll
                        for (int j = 0; j < 4; ++j)
                            if (j < njt) fz_dmma(acc[i][j][0], acc[i][j][1], av[i], bv[j]);
                    }
                }
                ndm += MT3 * njt;
            }
            // the rows of P of this unit (zeros when no k4 survives: the readers expect every allowed row)
            {
                double* Pb = p.Pq + ((((long)ac * c24 + b24) * c25 + b25) * P3) * V * prow + ((long)b34 * c35 + b35) * NP +
                             (long)(v0 + xl) * prow + wq * 32 + 2 * q;
#pragma unroll
                for (int i = 0; i < 3; ++i) {
                    const int q3 = q3lo + 8 * i + g;
                    if (i < MT3 && q3 < q3hi) {
                        double* dst = Pb + (long)q3 * V * prow;
#pragma unroll
                        for (int j = 0; j < 4; ++j)           // NP is even and the row starts 16-byte aligned
                            if (wq * 32 + 8 * j + 2 * q < n54) *reinterpret_cast<double2*>(dst + 8 * j) = make_double2(acc[i][j][0], acc[i][j][1]);
                    }
                }
            }
        }
    }
    if (p.cnt && lane == 0 && ndm) atomicAdd(p.cnt, (unsigned long long)ndm);
}

/* True when k_fz_qp2 holds the shape of the box (the caller then builds Bw4P instead of Bw4T). */
bool fz_qp2_supported(const FzParams& p, const SfDims& D)
{
    const int n4 = D.n_i[3], n5 = D.n_i[4], P3 = D.n_k_pad[1], P4 = D.n_k_pad[2];
    if (n5 > 16 || n4 > 16 || n4 * n5 > 128 || p.box.cnt[5] > FQ_L45 || p.box.cnt[1] > 32 || P4 > 24 || P4 < 1 || P3 < 1) return false;
    // k3 rows of a unit: inside the window of a pair (l34 l35), at most 24
    for (int u = 0; u < p.box.cnt[3]; ++u)
        for (int v = 0; v < p.box.cnt[4]; ++v) {
            const int2 w = fz_window(D.two_j[J34] + 2 * (p.box.lo[3] + u), D.two_j[J35] + 2 * (p.box.lo[4] + v), D.two_k_base[1], P3);
            if (w.y > 24) return false;
        }
    const int need = (FQ_XC - 1) * n5 + 16;
    int ldz = ((need + 11) & ~15) + 4;
    if (ldz < need) ldz += 16;
    return sizeof(double) * ((size_t)P4 * FQ_L45 * ldz + 4 * FQ_GRP) <= 225 * 1024;
}

long fz_qp2_b4p_elems(const FzParams& p, const SfDims& D)
{
    return (long)p.box.cnt[1] * p.box.cnt[3] * D.n_k_pad[2] * FQ_L45 * 16;
}

/* Launches k_fz_qp2 for the pass described by p (fz_qp2_supported must hold; Bw4P built by fz_launch_b4p). */
int fz_launch_qp2(const FzParams& p, const SfDims& D, const double* Bw4P, int* sched, int n_sm, cudaStream_t st)
{
    const int n5 = D.n_i[4], P4 = D.n_k_pad[2];
    FzQp2Args a;
    memset(&a, 0, sizeof a);
    const int need = (FQ_XC - 1) * n5 + 16;                   // last x of a chunk reads 16 rows from its first i5
    a.ldz = ((need + 11) & ~15) + 4;
    if (a.ldz < need) a.ldz += 16;
    const size_t smem = sizeof(double) * ((size_t)P4 * FQ_L45 * a.ldz + 4 * FQ_GRP);
    a.vc = (p.V + FQ_XC - 1) / FQ_XC;
    const long n_items = (long)a.vc * p.a_cnt * p.box.cnt[2] * p.box.cnt[4];
    if (n_items > 2000000000L) return SF_EARG;
    a.n_items = (int)n_items;
    a.sched = sched;
    a.Bw4P = Bw4P;
    static SfPerContext<size_t> attr_c(0);
    size_t& attr = attr_c.get();
    if (smem > attr) {
        if (cudaFuncSetAttribute(k_fz_qp2, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem) != cudaSuccess) return SF_ECUDA;
        attr = smem;
    }
    const int grid = (int)(n_items < n_sm ? n_items : n_sm);
    k_fz_qp2<<<grid, FQ_THREADS, smem, st>>>(p, a);
    sf_count_launch(1);
    return SF_OK;
}
