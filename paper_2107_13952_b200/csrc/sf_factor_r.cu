// sf_factor_r.cu -- the edge-3 contraction of the factorised path (sf_vertex_factor.cu, DESIGN.md 5 K-f):
//
//   R[l24 l25 i1; k3 x; (l23 i3); (i5 i4)] = sum over the pairs (l34 l35) that allow k3 of
//                                            Bw3T[k3; (l34 l35); (l23 i3)] P[l24 l25 i1; k3 x; (l34 l35); (i5 i4)]
//
// i.e. the mode product with the edge-3 booster (step 6(iii)) taken together with the shell sums over l34 and
// l35 (eq. (3)).  For one k3 the booster block is the same for every (l24 l25 i1 x), so the kernel keeps it
// STATIONARY in shared memory and streams the rows of P past it exactly once:
//
//   * a CTA takes chunks (k3, m-tile, n-tile, a few (i1 l24 l25)) from an atomic counter (execution order only: every
//     output has one writer, so the result does not depend on it); the booster block Bs[k][n] of the chunk's k3 is
//     gathered once per chunk by the consumer warps (8-byte cp.async);
//   * one PRODUCER warp walks the chunk's products (one per x the triad (k3 l24 x) allows) and fills a ring of stages with
//     16 rows of P each: one cp.async.bulk (SASS UBLKCP) per row, completion on the stage's `full` mbarrier;
//   * sixteen CONSUMER warps (4 x 4, warp tile 32 rows (i5 i4) x up to 32 columns (l23 i3)) wait on `full`, run the FP64
//     tensor-core MMAs (mma.sync m8n8k4 f64 = DMMA.8x8x4) from shared memory with conflict-free fragment loads (row strides
//     = 4 mod 16 doubles), and release the stage through its `empty` mbarrier: no CTA-wide barrier inside a chunk.
//
// Rows beyond K in the last stage of a product hold finite stale values (the ring starts zeroed and only ever receives
// rows of P that k_fz_qp wrote) and meet zero rows of Bs, so they add exact zeros.
#include "sf_factor.cuh"

#define FZR_KC 16                 // rows of P per stage
#define FZR_NWC 16                // consumer warps: 4 x 4, warp tile 32 rows (i5 i4) x up to 32 columns (l23 i3)
#define FZR_THREADS (32 * (FZR_NWC + 1))
#define FZR_BM 128
#define FZR_BN 128
#define FZR_LDA 132               // = 4 mod 16: the 16 lanes of a half warp (fragment row g = 0..3 or 4..7, k index q = 0..3) read
                                  // 16 different 8-byte banks (q * 4 + g); 1056 B per row keeps bulk copies 16-byte aligned

struct FzR2Args {
    int ldb;                      // row stride of Bs (= 4 mod 16)
    int kcap;                     // rows of Bs: the largest K of any k3, rounded up to 4
    int ns;                       // ring stages
    int spc, nsc;                 // slabs (i1 l24 l25) per chunk, chunks per (k3, m-tile, n-tile)
    int ntm, ntn;                 // tiles over (i5 i4) and over (l23 i3)
    int n_chunks;
    int* sched;                   // chunk counter (zeroed before the launch)
    unsigned char q3ord[80];      // k3 in order of decreasing work
};

__device__ __forceinline__ void fzr_mbar_arrive(unsigned bar)
{
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(bar) : "memory");
}

// the MMAs of one stage for a warp with TNA live column tiles
template <int TNA>
__device__ __forceinline__ void fzr_stage(double (&acc)[4][4][2], const double* as, const double* bs, int ldb, int ksn, int tma)
{
#pragma unroll
    for (int ks = 0; ks < FZR_KC / 4; ++ks) {
        if (ks < ksn) {
            double a[4], b[TNA];
#pragma unroll
            for (int i = 0; i < 4; ++i) a[i] = as[ks * 4 * FZR_LDA + 8 * i];
#pragma unroll
            for (int j = 0; j < TNA; ++j) b[j] = bs[ks * 4 * ldb + 8 * j];
#pragma unroll
            for (int i = 0; i < 4; ++i) {
                if (i < tma) {
#pragma unroll
                    for (int j = 0; j < TNA; ++j) fz_dmma(acc[i][j][0], acc[i][j][1], a[i], b[j]);
                }
            }
        }
    }
}

__global__ void __launch_bounds__(FZR_THREADS, 1) k_fz_r2(const __grid_constant__ FzParams p, const __grid_constant__ FzR2Args a)
{
    extern __shared__ __align__(16) double smem[];
    __shared__ __align__(8) unsigned long long bars[16];     // full[ns], empty[ns]
    __shared__ int s_chunk;
    const SfProblem& P = p.P;
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31, g = lane >> 2, q = lane & 3;
    const int ns = a.ns, ldb = a.ldb;
    double* As = smem;                                        // [ns][KC][LDA]
    double* Bs = As + ns * FZR_KC * FZR_LDA;                  // [kcap][ldb]
    const unsigned full0 = fz_smem_u32(&bars[0]), empty0 = fz_smem_u32(&bars[8]);

    const int n3 = P.n_i[2], n54 = P.n_i[3] * P.n_i[4], P3 = P.n_k_pad[1], V = p.V, NP = p.NP;
    const int c23 = p.box.cnt[0], c24 = p.box.cnt[1], c25 = p.box.cnt[2], c34 = p.box.cnt[3], c35 = p.box.cnt[4];
    const int npair = c34 * c35, S = p.a_cnt * c24 * c25;

    for (int z = tid; z < ns * FZR_KC * FZR_LDA; z += FZR_THREADS) As[z] = 0.0;
    if (tid == 0) {
        for (int s = 0; s < ns; ++s) {
            fz_mbar_init(full0 + 8 * s, 1);
            fz_mbar_init(empty0 + 8 * s, FZR_NWC);
        }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");   // the zeroed ring is next written by bulk copies
    int it = 0;                                               // stages used so far: slot it % ns, phase (it / ns) & 1
    int have_q3 = -1, have_nt = -1;
    unsigned ndm = 0;
    const int wm = (warp >> 2) & 3, wn = warp & 3;

    for (;;) {
        __syncthreads();                                      // everybody is done with the previous chunk (and with Bs)
        if (tid == 0) s_chunk = atomicAdd(a.sched, 1);
        __syncthreads();
        int ch = s_chunk;
        if (ch >= a.n_chunks) break;
        // k3 runs fastest: at any moment the SMs work on light (HBM-bound: few columns per row of P) and heavy
        // (tensor-pipe-bound) k3 alike, heavy ones first inside every group of slabs
        const int P3c = P.n_k_pad[1];
        const int q3 = a.q3ord[ch % P3c]; ch /= P3c;
        const int nt = ch % a.ntn; ch /= a.ntn;
        const int mt = ch % a.ntm;
        const int sc = ch / a.ntm;
        const int2 win = p.win23[q3];
        const int* list = p.kl3 + (long)q3 * (1 + npair);
        const int K = list[0];
        const int n0 = nt * FZR_BN, N = min(FZR_BN, win.y * n3 - n0);
        const int m0 = mt * FZR_BM, M = min(FZR_BM, n54 - m0);
        if (N <= 0) continue;
        if (warp < FZR_NWC) {
            if (have_q3 != q3 || have_nt != nt) {             // gather the booster block of this k3 (rows = allowed pairs):
                const int Kp = (K + 3) & ~3, ncol = (N + 7) & ~7;    // asynchronous 8-byte copies, zero-filled outside K x N
                const double* Bg = p.Bw3T + (long)q3 * npair * c23 * n3 + (long)win.x * n3 + n0;
                for (int kk = warp; kk < Kp; kk += FZR_NWC) {
                    const double* row = Bg + (kk < K ? (long)__ldg(list + 1 + kk) * (c23 * n3) : 0);
                    const unsigned dst = fz_smem_u32(Bs + kk * ldb);
                    for (int n = lane; n < ncol; n += 32) {
                        const bool ok = kk < K && n < N;
                        fz_cp_async8(dst + 8u * n, ok ? row + n : Bg, ok ? 8 : 0);
                    }
                }
                fz_cp_commit();
                fz_cp_wait<0>();
                have_q3 = q3;
                have_nt = nt;
                asm volatile("bar.sync 1, %0;" ::"n"(FZR_NWC * 32) : "memory");   // consumers only: the producer is already loading
            }
        }
        const int nchunks = (K + FZR_KC - 1) / FZR_KC;
        const int two_k3 = P.two_k_base[1] + 2 * q3;
        const int s_lo = sc * a.spc, s_hi = min(S, s_lo + a.spc);

        if (warp == FZR_NWC) {
            // ---------------- producer ----------------
            const unsigned rowb = (unsigned)(((M + 1) & ~1) * 8);
            for (int slab = s_lo; slab < s_hi; ++slab) {
                const int b25 = slab % c25, b24 = (slab / c25) % c24, ac = slab / (c25 * c24);
                int x0, nxs, xg0;
                fz_xrange(P.two_i_min[0], P.two_j[J25], P.two_x_base, p.a_lo + ac, p.box.lo[2] + b25, x0, nxs, xg0);
                const int2 vr = fz_vrange(P.two_j[J24] + 2 * (p.box.lo[1] + b24), two_k3, x0, nxs);
                for (int vi = 0; vi < vr.y; ++vi) {
                    const double* Ap = p.Pq + (((long)slab * P3 + q3) * V + vr.x + vi) * ((long)npair * NP) + m0;
                    for (int c = 0; c < nchunks; ++c, ++it) {
                        const int s = it % ns, k0 = c * FZR_KC, kv = min(FZR_KC, K - k0);
                        fz_mbar_wait(empty0 + 8 * s, (unsigned)(((it / ns) & 1) ^ 1));
                        if (lane == 0) fz_mbar_expect_tx(full0 + 8 * s, rowb * (unsigned)kv);
                        __syncwarp();
                        if (lane < kv)
                            fz_bulk_g2s(fz_smem_u32(As + (s * FZR_KC + lane) * FZR_LDA), Ap + (long)NP * __ldg(list + 1 + k0 + lane), rowb,
                                        full0 + 8 * s);
                    }
                }
            }
        } else {
            // ---------------- consumers ----------------
            const int NT = (N + 7) >> 3;
            const int ntb = NT >> 2, ntr = NT & 3;            // column tiles over the four warp columns
            const int nt0 = wn * ntb + min(wn, ntr), tna = ntb + (wn < ntr ? 1 : 0);
            int tma = 0;
#pragma unroll
            for (int i = 0; i < 4; ++i) tma += (wm * 32 + 8 * i) < M;
            const bool active = tma > 0 && tna > 0;
            double acc[4][4][2];
#pragma unroll
            for (int i = 0; i < 4; ++i)
#pragma unroll
                for (int j = 0; j < 4; ++j) acc[i][j][0] = acc[i][j][1] = 0.0;
            const double* as0 = As + q * FZR_LDA + wm * 32 + g;
            const double* bs0 = Bs + q * ldb + nt0 * 8 + g;
            for (int slab = s_lo; slab < s_hi; ++slab) {
                const int b25 = slab % c25, b24 = (slab / c25) % c24, ac = slab / (c25 * c24);
                int x0, nxs, xg0;
                fz_xrange(P.two_i_min[0], P.two_j[J25], P.two_x_base, p.a_lo + ac, p.box.lo[2] + b25, x0, nxs, xg0);
                const int2 vr = fz_vrange(P.two_j[J24] + 2 * (p.box.lo[1] + b24), two_k3, x0, nxs);
                for (int vi = 0; vi < vr.y; ++vi) {
                    for (int c = 0; c < nchunks; ++c, ++it) {
                        const int s = it % ns;
                        fz_mbar_wait(full0 + 8 * s, (unsigned)((it / ns) & 1));
                        if (active) {
                            const int ksn = min(FZR_KC / 4, (K - c * FZR_KC + 3) >> 2);
                            const double* as = as0 + s * FZR_KC * FZR_LDA;
                            const double* bs = bs0 + (long)c * FZR_KC * ldb;
                            switch (tna) {
                                case 4: fzr_stage<4>(acc, as, bs, ldb, ksn, tma); break;
                                case 3: fzr_stage<3>(acc, as, bs, ldb, ksn, tma); break;
                                case 2: fzr_stage<2>(acc, as, bs, ldb, ksn, tma); break;
                                default: fzr_stage<1>(acc, as, bs, ldb, ksn, tma); break;
                            }
                            ndm += tma * tna * ksn;
                        }
                        __syncwarp();
                        if (lane == 0) fzr_mbar_arrive(empty0 + 8 * s);
                    }
                    // the product of this x: rows (l23 i3) of R, NP entries (i5 i4) each
                    if (active) {
                        double* C = p.Rq + (((((long)slab * P3 + q3) * V + vr.x + vi) * c23 + win.x) * n3 + n0) * (long)NP + m0;
#pragma unroll
                        for (int i = 0; i < 4; ++i) {
                            const int m = wm * 32 + 8 * i + g;
#pragma unroll
                            for (int j = 0; j < 4; ++j) {
                                const int n = (nt0 + j) * 8 + 2 * q;
                                if (i < tma && j < tna && m < M) {
                                    if (n < N) C[(long)n * NP + m] = acc[i][j][0];
                                    if (n + 1 < N) C[(long)(n + 1) * NP + m] = acc[i][j][1];
                                }
                                acc[i][j][0] = acc[i][j][1] = 0.0;
                            }
                        }
                    }
                }
            }
        }
    }
    if (p.cnt && lane == 0 && ndm) atomicAdd(p.cnt + 1, (unsigned long long)ndm);
}

/* Launches k_fz_r2 for the pass described by p.  SF_EARG when the shape does not fit its shared-memory plan (the caller
 * then uses the general gather-GEMM). */
int fz_launch_r2(const FzParams& p, const SfDims& D, int* sched, int n_sm, cudaStream_t st)
{
    const int n3 = D.n_i[2], n54 = D.n_i[3] * D.n_i[4], P3 = D.n_k_pad[1];
    const int c23 = p.box.cnt[0], c24 = p.box.cnt[1], c25 = p.box.cnt[2], c34 = p.box.cnt[3], c35 = p.box.cnt[4];
    if (P3 > 80 || P3 < 1) return SF_EARG;
    FzR2Args a;
    memset(&a, 0, sizeof a);
    // work per k3 from the windows of step 2 (the same predicates the device lists use)
    double work[80];
    int kmax = 0;
    for (int q3 = 0; q3 < P3; ++q3) {
        int K = 0, nb = 0;
        for (int u = 0; u < c34; ++u)
            for (int v = 0; v < c35; ++v) {
                const int2 w = fz_window(D.two_j[J34] + 2 * (p.box.lo[3] + u), D.two_j[J35] + 2 * (p.box.lo[4] + v), D.two_k_base[1], P3);
                K += q3 >= w.x && q3 < w.x + w.y;
            }
        for (int b = 0; b < c23; ++b) {
            const int2 w = fz_window(D.two_j[J13], D.two_j[J23] + 2 * (p.box.lo[0] + b), D.two_k_base[1], P3);
            nb += q3 >= w.x && q3 < w.x + w.y;
        }
        work[q3] = (double)K * nb;
        if (K > kmax) kmax = K;
        a.q3ord[q3] = (unsigned char)q3;
    }
    for (int i = 1; i < P3; ++i)                               // insertion sort, descending work
        for (int j = i; j > 0 && work[a.q3ord[j]] > work[a.q3ord[j - 1]]; --j) {
            const unsigned char t = a.q3ord[j];
            a.q3ord[j] = a.q3ord[j - 1];
            a.q3ord[j - 1] = t;
        }
    const int nmax = c23 * n3 < FZR_BN ? c23 * n3 : FZR_BN;
    a.ldb = ((nmax + 7) & ~15) + 4;                            // >= N rounded up to 8, = 4 mod 16
    if (a.ldb < ((nmax + 7) & ~7)) a.ldb += 16;
    a.kcap = (kmax + 3) & ~3;
    if (a.kcap < 4) a.kcap = 4;
    const size_t fixed = sizeof(double) * (size_t)a.kcap * a.ldb;
    const size_t stage = sizeof(double) * FZR_KC * FZR_LDA;
    const size_t cap = 225 * 1024;
    if (fixed + 3 * stage > cap) return SF_EARG;
    a.ns = (int)((cap - fixed) / stage);
    if (a.ns > 8) a.ns = 8;
    const size_t smem = fixed + a.ns * stage;
    a.ntm = (n54 + FZR_BM - 1) / FZR_BM;
    a.ntn = (c23 * n3 + FZR_BN - 1) / FZR_BN;
    const long S = (long)p.a_cnt * c24 * c25;
    long spc = S * P3 * a.ntm * a.ntn / (24L * n_sm);
    if (spc < 1) spc = 1;
    if (spc > 16) spc = 16;
    a.spc = (int)spc;
    a.nsc = (int)((S + spc - 1) / spc);
    const long n_chunks = (long)P3 * a.ntm * a.ntn * a.nsc;
    if (n_chunks > 2000000000L) return SF_EARG;
    a.n_chunks = (int)n_chunks;
    a.sched = sched;
    static SfPerContext<size_t> attr_c(0);
    size_t& attr = attr_c.get();
    if (smem > attr) {
        if (cudaFuncSetAttribute(k_fz_r2, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem) != cudaSuccess) return SF_ECUDA;
        attr = smem;
    }
    const int grid = (int)(n_chunks < n_sm ? n_chunks : n_sm);
    k_fz_r2<<<grid, FZR_THREADS, smem, st>>>(p, a);
    sf_count_launch(1);
    return SF_OK;
}

// ---------------------------------------------------------------------------------------------------------------------------
// k_fz_r3: the same contraction, tile and occupancy as k_fz_gemm<FzMapR> (128 x 64, ring of two 32-row stages, two CTAs per SM), with
// the loader taken out of the compute warps.  A microbenchmark of the bare inner loop (sf_fp64_peak kind 2: 10 conflict-free
// LDS.64 per 16 DMMA, 16 warps per SM) reaches the full DMMA peak, so whatever k_fz_gemm<FzMapR> loses (0.67 pipe) it loses to
// its loader code (~250 instructions per chunk and warp, 8-byte cp.async for the booster rows), its CTA barrier per chunk and
// its epilogue.  Here
//   * a ninth PRODUCER warp fills the ring: one bulk copy per row of P and one per booster row (the booster is stored windowed
//     and padded, Bw3W[q3][pair][ldw], columns from the first l23 that allows k3: every tile row starts 16-byte aligned), rows
//     between K and the next k-step boundary come from a zero row, completion on the stage's `full` mbarrier;
//   * the eight CONSUMER warps run the inner loop, wait on `full` and release the stage through `empty`: no CTA barrier, no
//     loader instruction, between the first and the last chunk of an item.
// ---------------------------------------------------------------------------------------------------------------------------
#define FZ3_BM 128
#define FZ3_BN 64
#define FZ3_LDB 68
#define FZ3_NWC 8
#define FZ3_THREADS (32 * (FZ3_NWC + 1))

struct FzR3Args {
    const double* Bw;             // Bw3W[q3][n-tile][kcap][FZ3_LDB]: the booster tile of every (k3, n-tile) as it sits in shared memory
    int kcap;                     // rows per tile: the pairs (l34 l35) of the box rounded up to a multiple of 96 (rows beyond the list: zeros)
    int ntm, ntn;
};

// Bw3W[q3][nt][kk][c] = Bw3T[q3][pair kk of the list of k3][(first l23 that allows k3) n3 + 64 nt + c], 0 beyond the list, the window
// and in the 4 padding columns: a 32-row chunk of a tile is ONE contiguous, 16-byte aligned block with the pitch of the ring
__global__ void __launch_bounds__(256) k_fz_b3w(FzParams p, int kcap, int ntn, long n, double* __restrict__ out)   // kcap: multiple of the stage depth
{
    const long e = blockIdx.x * (long)blockDim.x + threadIdx.x;
    if (e >= n) return;
    const SfProblem& P = p.P;
    const int n3 = P.n_i[2], c23 = p.box.cnt[0], c34 = p.box.cnt[3], c35 = p.box.cnt[4], npair = c34 * c35;
    const int c = (int)(e % FZ3_LDB);
    long r = e / FZ3_LDB;
    const int kk = (int)(r % kcap); r /= kcap;
    const int nt = (int)(r % ntn);
    const int q3 = (int)(r / ntn);
    const int2 win = p.win23[q3];
    const int* list = p.kl3 + (long)q3 * (1 + npair);
    const int col = nt * FZ3_BN + c;
    double val = 0.0;
    if (c < FZ3_BN && kk < list[0] && col < win.y * n3) val = p.Bw3T[((long)q3 * npair + list[1 + kk]) * (c23 * n3) + (long)win.x * n3 + col];
    out[e] = val;
}

struct Fz3Job {
    const double *as0, *bs0;      // this lane's fragment bases in stage 0 of the ring
    unsigned full0, empty0;
    double* C;                    // this lane's first entry of the first product (row warp 16 + g, column 0)
    long sC;                      // products are sC apart
    int NP, nsub, nchunks, K, N, lane, q;
    bool mok0, mok1;              // rows g and 8 + g of the warp tile exist
};

// all chunks of all products of an item for a warp with TNA live column tiles and TMA row tiles
template <int TNA, int TMA, int KC, int ST, int LDA>
__device__ __forceinline__ unsigned fz3_consume(const Fz3Job& J)
{
    double acc[TMA > 0 ? TMA : 1][TNA > 0 ? TNA : 1][2];
#pragma unroll
    for (int i = 0; i < (TMA > 0 ? TMA : 1); ++i)
#pragma unroll
        for (int j = 0; j < (TNA > 0 ? TNA : 1); ++j) acc[i][j][0] = acc[i][j][1] = 0.0;
    unsigned ndm = 0;
    int it = 0;
    for (int sub = 0; sub < J.nsub; ++sub) {
        for (int c = 0; c < J.nchunks; ++c, ++it) {
            const int s = it % ST;
            fz_mbar_wait(J.full0 + 8 * s, (unsigned)((it / ST) & 1));
            if (TMA > 0) {
                const int ksn = min(KC / 4, (J.K - c * KC + 3) >> 2);
                const double* as = J.as0 + s * KC * LDA;
                const double* bs = J.bs0 + s * KC * FZ3_LDB;
#pragma unroll
                for (int ks = 0; ks < KC / 4; ++ks) {
                    if (ks < ksn) {
                        double av[TMA > 0 ? TMA : 1], bv[TNA > 0 ? TNA : 1];
#pragma unroll
                        for (int i = 0; i < TMA; ++i) av[i] = as[ks * 4 * LDA + 8 * i];
#pragma unroll
                        for (int j = 0; j < TNA; ++j) bv[j] = bs[ks * 4 * FZ3_LDB + 8 * j];
#pragma unroll
                        for (int i = 0; i < TMA; ++i)
#pragma unroll
                            for (int j = 0; j < TNA; ++j) fz_dmma(acc[i][j][0], acc[i][j][1], av[i], bv[j]);
                    }
                }
                ndm += (unsigned)(TMA * TNA * ksn);
            }
            __syncwarp();
            if (J.lane == 0) fzr_mbar_arrive(J.empty0 + 8 * s);
        }
        // the product of this x: rows (l23 i3) of R, NP entries (i5 i4) each
        if (TMA > 0) {
            double* Cs = J.C + (long)sub * J.sC;
#pragma unroll
            for (int i = 0; i < TMA; ++i) {
                const bool mok = i ? J.mok1 : J.mok0;
#pragma unroll
                for (int j = 0; j < TNA; ++j) {
                    const int n = 8 * j + 2 * J.q;
                    if (mok) {
                        if (n < J.N) Cs[(long)n * J.NP + 8 * i] = acc[i][j][0];
                        if (n + 1 < J.N) Cs[(long)(n + 1) * J.NP + 8 * i] = acc[i][j][1];
                    }
                    acc[i][j][0] = acc[i][j][1] = 0.0;
                }
            }
        }
    }
    return ndm;
}

// KC rows per stage, ST stages, LDA = row pitch of the P rows in the ring (= 4 or 12 mod 16: conflict-free fragment loads).  Two
// shapes: 3 x 24 rows at pitch 124 when a row of P (n5 n4 <= 122 entries) fits it, else 2 x 32 at pitch 132.  Chosen by
// measurement (config 3, bench.py, three runs): 15.3 ms against 16.1-16.2 ms.  The pitch is not the cause (2 x 32 at 124: 16.1;
// 4 x 16 at 124 / 132: 16.4 / 16.5), and the mechanism is NOT identified: under ncu the share of mbarrier waits (11.5 %) and
// the first-pass time are the same for both shapes (profiles/r2_hot_kernels.md).
template <int KC, int ST, int LDA>
__global__ void __maxnreg__(112) k_fz_r3(const __grid_constant__ FzParams p, const __grid_constant__ FzR3Args a)
{
    extern __shared__ __align__(16) double smem[];
    __shared__ __align__(8) unsigned long long bars[2 * ST];     // full[ST], empty[ST]
    const SfProblem& P = p.P;
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31, g = lane >> 2, q = lane & 3;
    double* As = smem;                                        // [ST][KC][LDA]
    double* Bs = As + ST * KC * LDA;              // [ST][KC][LDB]
    const unsigned full0 = fz_smem_u32(&bars[0]), empty0 = fz_smem_u32(&bars[ST]);
    const int n3 = P.n_i[2], n54 = P.n_i[3] * P.n_i[4], P3 = P.n_k_pad[1], V = p.V, NP = p.NP;
    const int c23 = p.box.cnt[0], c24 = p.box.cnt[1], c25 = p.box.cnt[2], c34 = p.box.cnt[3], c35 = p.box.cnt[4];
    const int npair = c34 * c35;
    // the item: (i1, l24, l25, k3, tile), every x of the triad (k3 l24 x) in turn
    long item = blockIdx.x;
    const int nt = (int)(item % a.ntn); item /= a.ntn;
    const int mt = (int)(item % a.ntm); item /= a.ntm;
    const int q3 = (int)(item % P3); item /= P3;
    const int b25 = (int)(item % c25); item /= c25;
    const int b24 = (int)(item % c24);
    const int ac = (int)(item / c24);
    int x0, nxs, xg0;
    fz_xrange(P.two_i_min[0], P.two_j[J25], P.two_x_base, p.a_lo + ac, p.box.lo[2] + b25, x0, nxs, xg0);
    const int2 win = p.win23[q3];
    const int* list = p.kl3 + (long)q3 * (1 + npair);
    const int2 vr = fz_vrange(P.two_j[J24] + 2 * (p.box.lo[1] + b24), P.two_k_base[1] + 2 * q3, x0, nxs);
    const int m0 = mt * FZ3_BM, n0 = nt * FZ3_BN, N = min(FZ3_BN, win.y * n3 - n0), K = list[0];
    const int M = (N > 0 && vr.y > 0) ? min(FZ3_BM, n54 - m0) : 0;
    if (M <= 0) return;
    const int nsub = vr.y, nchunks = (K + KC - 1) / KC;
    const long slab = ((((long)ac * c24 + b24) * c25 + b25) * P3 + q3) * V + vr.x;
    const double* A = p.Pq + slab * npair * NP + m0;          // product sub: + sub * npair * NP; row kk: + NP * list[1 + kk]
    double* C = p.Rq + ((slab * c23 + win.x) * n3 + n0) * NP + m0;   // product sub: + sub * c23 n3 NP; entry (m, n): + n NP + m

    for (int z = tid; z < ST * KC * (LDA + FZ3_LDB); z += FZ3_THREADS) smem[z] = 0.0;   // rows never copied stay finite
    if (tid == 0) {
        for (int s = 0; s < ST; ++s) {
            fz_mbar_init(full0 + 8 * s, 1);
            fz_mbar_init(empty0 + 8 * s, FZ3_NWC);
        }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");   // the zeroed ring is next written by bulk copies
    __syncthreads();
    if (nchunks == 0) {                                       // nothing to sum: the destination rows are exact zeros
        for (int sub = 0; sub < nsub; ++sub)
            for (int e = tid; e < M * N; e += FZ3_THREADS) C[(long)sub * c23 * n3 * NP + (long)(e / M) * NP + e % M] = 0.0;
        return;
    }
    if (warp == FZ3_NWC) {
        // ---------------- producer ----------------
        const unsigned rowa = (unsigned)(((M + 1) & ~1) * 8);
        const double* Bq = a.Bw + ((long)q3 * a.ntn + nt) * a.kcap * FZ3_LDB;       // the tile of this (k3, n-tile), chunk c at + c KC LDB
        int it = 0;
        for (int sub = 0; sub < nsub; ++sub) {
            const double* Ap = A + (long)sub * npair * NP;
            for (int c = 0; c < nchunks; ++c, ++it) {
                const int s = it % ST, k0 = c * KC, kv = min(KC, K - k0);
                fz_mbar_wait(empty0 + 8 * s, (unsigned)(((it / ST) & 1) ^ 1));
                if (lane == 0) {
                    fz_mbar_expect_tx(full0 + 8 * s, rowa * (unsigned)kv + 8u * KC * FZ3_LDB);
                    fz_bulk_g2s(fz_smem_u32(Bs + s * KC * FZ3_LDB), Bq + (long)k0 * FZ3_LDB, 8u * KC * FZ3_LDB, full0 + 8 * s);
                }
                __syncwarp();
                if (lane < kv)
                    fz_bulk_g2s(fz_smem_u32(As + (s * KC + lane) * LDA), Ap + (long)NP * __ldg(list + 1 + k0 + lane), rowa, full0 + 8 * s);
            }
        }
        return;
    }
    // ---------------- consumers: warp tile 16 rows (i5 i4) x up to 64 columns (l23 i3) ----------------
    const int NT = (N + 7) >> 3;
    const int tma = (warp * 16 < M ? 1 : 0) + (warp * 16 + 8 < M ? 1 : 0);
    Fz3Job job;
    job.as0 = As + q * LDA + warp * 16 + g;
    job.bs0 = Bs + q * FZ3_LDB + g;
    job.full0 = full0;
    job.empty0 = empty0;
    job.C = C + warp * 16 + g;
    job.sC = (long)c23 * n3 * NP;
    job.NP = NP;
    job.nsub = nsub;
    job.nchunks = nchunks;
    job.K = K;
    job.N = N;
    job.mok0 = warp * 16 + g < M;
    job.mok1 = warp * 16 + 8 + g < M;
    job.lane = lane;
    job.q = q;
    unsigned ndm = 0;
    // the whole loop exists once per shape of the warp tile (live column tiles 1..8, one or two row tiles): straight-line MMA code
    if (tma == 2) {
        switch (NT) {
            case 8: ndm = fz3_consume<8, 2, KC, ST, LDA>(job); break;
            case 7: ndm = fz3_consume<7, 2, KC, ST, LDA>(job); break;
            case 6: ndm = fz3_consume<6, 2, KC, ST, LDA>(job); break;
            case 5: ndm = fz3_consume<5, 2, KC, ST, LDA>(job); break;
            case 4: ndm = fz3_consume<4, 2, KC, ST, LDA>(job); break;
            case 3: ndm = fz3_consume<3, 2, KC, ST, LDA>(job); break;
            case 2: ndm = fz3_consume<2, 2, KC, ST, LDA>(job); break;
            default: ndm = fz3_consume<1, 2, KC, ST, LDA>(job); break;
        }
    } else if (tma == 1) {
        switch (NT) {
            case 8: ndm = fz3_consume<8, 1, KC, ST, LDA>(job); break;
            case 7: ndm = fz3_consume<7, 1, KC, ST, LDA>(job); break;
            case 6: ndm = fz3_consume<6, 1, KC, ST, LDA>(job); break;
            case 5: ndm = fz3_consume<5, 1, KC, ST, LDA>(job); break;
            case 4: ndm = fz3_consume<4, 1, KC, ST, LDA>(job); break;
            case 3: ndm = fz3_consume<3, 1, KC, ST, LDA>(job); break;
            case 2: ndm = fz3_consume<2, 1, KC, ST, LDA>(job); break;
            default: ndm = fz3_consume<1, 1, KC, ST, LDA>(job); break;
        }
    } else {
        ndm = fz3_consume<0, 0, KC, ST, LDA>(job);                         // no rows of the tile: keeps the barriers moving
    }
    if (p.cnt && lane == 0 && ndm) atomicAdd(p.cnt + 1, (unsigned long long)ndm);
}

/* Elements of the tile-major booster copy Bw3W for the box of p. */
long fz_r3_b3w_elems(const FzParams& p, const SfDims& D, int* kcap)
{
    const int npair = p.box.cnt[3] * p.box.cnt[4], ntn = (p.box.cnt[0] * D.n_i[2] + FZ3_BN - 1) / FZ3_BN;
    *kcap = (npair + 95) / 96 * 96;                          // a multiple of both stage depths (24 and 32)
    return (long)D.n_k_pad[1] * ntn * *kcap * FZ3_LDB;
}

/* Builds Bw3W (after k_fz_pre: it reads Bw3T, win23 and the lists) and launches k_fz_r3 for the pass described by p. */
int fz_launch_r3(const FzParams& p, const SfDims& D, double* Bw3W, bool build, cudaStream_t st)
{
    FzR3Args a;
    memset(&a, 0, sizeof a);
    const long nW = fz_r3_b3w_elems(p, D, &a.kcap);
    const int ntn_b = (p.box.cnt[0] * D.n_i[2] + FZ3_BN - 1) / FZ3_BN;
    if (build) {
        k_fz_b3w<<<(unsigned)((nW + 255) / 256), 256, 0, st>>>(p, a.kcap, ntn_b, nW, Bw3W);
        sf_count_launch(1);
    }
    a.Bw = Bw3W;
    const int n3 = D.n_i[2], n54 = D.n_i[3] * D.n_i[4];
    a.ntm = (n54 + FZ3_BM - 1) / FZ3_BM;
    a.ntn = (p.box.cnt[0] * n3 + FZ3_BN - 1) / FZ3_BN;
    const long items = (long)a.ntn * a.ntm * D.n_k_pad[1] * p.box.cnt[2] * p.box.cnt[1] * p.a_cnt;
    if (items <= 0) return SF_OK;
    if (items > 2147483647L) return SF_EARG;
    const bool deep = n54 <= 122;                             // a row of P fits the pitch of the 3 x 24 ring
    const size_t smem = deep ? sizeof(double) * 3 * 24 * (124 + FZ3_LDB) : sizeof(double) * 2 * 32 * (132 + FZ3_LDB);
    static SfPerContext<bool> attr_c[2] = {SfPerContext<bool>(false), SfPerContext<bool>(false)};
    bool& attr_set = attr_c[deep].get();
    if (!attr_set) {
        const cudaError_t e = deep ? cudaFuncSetAttribute(k_fz_r3<24, 3, 124>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem)
                                   : cudaFuncSetAttribute(k_fz_r3<32, 2, 132>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e != cudaSuccess) return SF_ECUDA;
        attr_set = true;
    }
    if (deep)
        k_fz_r3<24, 3, 124><<<(unsigned)items, FZ3_THREADS, smem, st>>>(p, a);
    else
        k_fz_r3<32, 2, 132><<<(unsigned)items, FZ3_THREADS, smem, st>>>(p, a);
    sf_count_launch(1);
    return SF_OK;
}
