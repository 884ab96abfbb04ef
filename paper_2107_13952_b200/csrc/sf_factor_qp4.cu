// sf_factor_qp4.cu -- the edge-4 contraction of the factorised path (sf_vertex_factor.cu, DESIGN.md 5 K-f), warp-autonomous kernel:
//
//   Q[k4; i5 i4]            = sum_l45 Z[l25 i1 l35 l45; k4 x i5] Bw4P[l24 l34; k4; l45; i4]      (the shells of a line l45)
//   P[k3; (i5 i4)]          = sum_k4  S3T[l24 l34 l35; x; k3 k4] Q[k4; i5 i4]                    (third {6j} of eq. (5), edge-4 product)
//
// for every (i1 l25 l35 | l24 l34 | x): steps 6(i)-(iii) of the algorithm for the factors of eq. (3) that
// carry l45 and k4.  Q never leaves the chip; the rows of P the triads allow go to HBM for the edge-3 contraction.
//
// k_fz_qp2 (sf_factor_qp.cu) shares a unit (l24 l34 x) among four warps: ~60 MMA per warp between two named barriers, 15
// issued instructions per MMA, the FP64 tensor pipe 40 % busy.  Here ONE warp owns a unit from its first k4 to its rows of P:
//   * a CTA (8 warps, one per SM) takes items (i1, l25, l35, chunk of <= 4 x) from an atomic counter (execution order only:
//     every row of P has one writer) and keeps the item's slab of Z in shared memory, as k_fz_qp2 does;
//   * the windows of every unit of the item are computed once, cooperatively, into a descriptor table in shared memory (units
//     with more than 16 rows k3 are split in two, so that a warp holds two row tiles x 16 column tiles = 128 accumulator
//     registers); the warps draw units from a shared-memory counter;
//   * per k-step of 4 k4 the warp computes Q for the four k4 (2 x 2 tiles each, only over the k-steps of l45 that the triad
//     (k4 l45 j14) allows: both operands are exactly zero elsewhere) into its PRIVATE tile [4][n5 n4] (compact, row stride = 4
//     mod 16: conflict-free B fragments), __syncwarp, then accumulates all 16 column tiles of P from that tile: 50-64
//     independent MMA per k-step and no barrier other than the warp's own;
//   * the booster fragments of a k-step (4 k4 x 1536 contiguous bytes of Bw4P) arrive by ONE bulk asynchronous copy
//     (cp.async.bulk = SASS UBLKCP, completion on the warp's own mbarrier) into the warp's slot, issued as soon as the Q phase
//     has read the slot, so that the copy runs under the P phase; S3 fragments come straight from L1/L2 into registers, one
//     k-step ahead, their lines sent for into L1 a whole unit earlier.
//
// Shapes it holds: those of k_fz_qp2 with c24 c34 <= 256.  sf_vertex_factor falls back to k_fz_qp2 / k_fz_qp otherwise.
#include "sf_factor.cuh"

#define F4_THREADS 256
#define F4_WARPS 8
#define F4_XC 4                   // x values per item
#define F4_L45 12                 // l45 rows per k4 in the Z slab and in Bw4P (3 k-steps)
#define F4_LDQ 132                // row stride of a Q tile: >= 128 columns, = 4 mod 16
#define F4_BSLOT (4 * F4_L45 * 16) // doubles of booster fragments per k-step
#define F4_MAXU 1024              // units (l24 l34 x) per item; as many overflow units (rows k3 beyond the first 16)

struct FzQp4Args {
    int ldz;                      // row stride of the Z slab (= 4 mod 16)
    int vc;                       // chunks of F4_XC x per (i1 l25)
    int n_items;
    int* sched;
    const double* Bw4P;           // [b24][b34][q4][k-step 3][lane 32][column tile 2], see k_fz_b4p (sf_factor_qp.cu)
};

struct FzTrue { static constexpr bool value = true; };
struct FzFalse { static constexpr bool value = false; };

__device__ __forceinline__ double f4_lds(unsigned addr)
{
    double v;
    asm volatile("ld.shared.f64 %0, [%1];" : "=d"(v) : "r"(addr));
    return v;
}
__device__ __forceinline__ void f4_sts(unsigned addr, double a)
{
    asm volatile("st.shared.f64 [%0], %1;" ::"r"(addr), "d"(a) : "memory");
}

// LDZ = row stride of the Z slab: 52 for n5 <= 12, else 68 (= 4 mod 16, >= 3 n5 + 16)
// N5T, N4T = tiles of 8 over i5 and over i4 in the Q phase (1 or 2): compile-time, so that the k-step body is straight-line code
template <int LDZ, int N5T, int N4T>
__global__ void __launch_bounds__(F4_THREADS, 1) k_fz_qp4(const __grid_constant__ FzParams p, const __grid_constant__ FzQp4Args a)
{
    extern __shared__ __align__(16) double smem[];
    __shared__ int s_item, s_next;
    __shared__ int2 s_unit[2 * F4_MAXU];                      // per (b24, b34, x) and its overflow: packed windows, see below
    __shared__ __align__(8) unsigned long long s_bar[F4_WARPS];   // per warp: completion of the bulk copy into its booster slot
    const SfProblem& P = p.P;
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31, g = lane >> 2, q = lane & 3;
    const int nl = P.nl, n1 = P.n_i[0], n4 = P.n_i[3], n5 = P.n_i[4], n54 = n4 * n5;
    const int P3 = P.n_k_pad[1], P4 = P.n_k_pad[2], NX = P.n_x_pad, V = p.V, NP = p.NP;
    const int c24 = p.box.cnt[1], c25 = p.box.cnt[2], c34 = p.box.cnt[3], c35 = p.box.cnt[4], c45 = p.box.cnt[5];
    constexpr int ldz = LDZ, ldq = F4_LDQ;
    const int NT = (n54 + 7) >> 3;
    const int sZ = P4 * V * n5;
    const long prow = (long)c34 * c35 * NP;                   // stride of v in P
    const int nzs = P4 * F4_L45 * ldz;
    for (int z = tid; z < nzs + F4_WARPS * (4 * ldq + F4_BSLOT); z += F4_THREADS) smem[z] = 0.0;   // pad rows and columns stay finite
    if (lane == 0) fz_mbar_init(fz_smem_u32(&s_bar[warp]), 1);
    if (tid == 0) asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");   // the zeroed slots are next written by bulk copies
    const unsigned zs_u32 = fz_smem_u32(smem);                // Zs[P4][F4_L45][ldz]
    const unsigned qs_u32 = zs_u32 + 8u * (unsigned)(nzs + warp * (4 * ldq + F4_BSLOT));   // this warp's Q tile [4][ldq]
    const unsigned bs_u32 = qs_u32 + 8u * (unsigned)(4 * ldq);                           // and booster slot [4 k4][3 k-steps][32 lanes][2]
    const unsigned bar_u32 = fz_smem_u32(&s_bar[warp]);
    unsigned bphase = 0;                                      // parity of the next completion of the warp's mbarrier
    // per-lane constants of the fragment addresses (bytes)
    const unsigned z_lane = zs_u32 + 8u * (unsigned)(q * ldz + g);                    // A of Q: row l45 = 4 ks + q, column + g
    constexpr unsigned z_ks = 8u * (unsigned)(4 * ldz), z_k4 = 8u * (unsigned)(F4_L45 * ldz);
    // C of Q: rows i5 = g, 8 + g; columns i4 = 2 q, 2 q + 1, 8 + 2 q, 9 + 2 q; smask: which of the 2 x 4 entries exist
    const unsigned qst_lane = qs_u32 + 8u * (unsigned)(g * n4 + 2 * q);
    unsigned smask = 0;
#pragma unroll
    for (int t = 0; t < 2; ++t)
#pragma unroll
        for (int e = 0; e < 4; ++e)
            if (8 * t + g < n5 && 8 * (e >> 1) + 2 * q + (e & 1) < n4) smask |= 1u << (4 * t + e);
    // B of P: one 16-byte load gives this lane's entries of TWO column tiles: k4 row q, columns 16 jp + 2 g (tile 2 jp) and
    // 16 jp + 2 g + 1 (tile 2 jp + 1); the C fragments of the pair then hold four consecutive columns 16 jp + 4 q .. + 3
    const unsigned qld_lane = qs_u32 + 8u * (unsigned)(q * ldq + 2 * g);
    unsigned pmask = 0;                                       // column pairs 16 jp + 4 q (bit 2 jp) and 16 jp + 4 q + 2 (bit 2 jp + 1) this lane stores
#pragma unroll
    for (int jp = 0; jp < 8; ++jp) {
        if (16 * jp + 4 * q < n54) pmask |= 1u << (2 * jp);
        if (16 * jp + 4 * q + 2 < n54) pmask |= 2u << (2 * jp);
    }
    const unsigned b4_lane = bs_u32 + 16u * (unsigned)lane;   // B of Q: fragment-major, (column tile 0, 1) adjacent
    unsigned ndm = 0;

    for (;;) {
        __syncthreads();                                      // everybody is done with the previous slab of Z and the tables
        if (tid == 0) {
            s_item = atomicAdd(a.sched, 1);
            s_next = 0;
        }
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
        const int v0 = vc * F4_XC, nv = min(F4_XC, nxs - v0);
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
        // the slab of Z: rows (k4, l45), nv * n5 entries (x i5) each
        {
            const double* Zb = p.Z + ((((long)b25 * n1 + a1) * c35 + b35) * c45) * (long)sZ + (long)v0 * n5;
            const int rowlen = nv * n5, nrow = max(0, h4hi - h4lo) * c45;
            for (int r = warp; r < nrow; r += F4_WARPS) {
                const int r4 = r / c45, b45 = r - r4 * c45;
                const double* src = Zb + ((long)b45 * P4 + h4lo + r4) * (V * n5);
                const unsigned dst = zs_u32 + 8u * (unsigned)((r4 * F4_L45 + b45) * ldz);
                for (int c = lane; c < rowlen; c += 32) fz_cp_async8(dst + 8u * c, src + c, 8);
            }
            fz_cp_commit();
        }
        // the units (b24, b34, x) of the item: rows k3 = (k3 l34 l35) and the triad (k3 l24 x); k4 = (k4 l24 l34), the triad
        // (k4 l35 x), and the l45 of the box.  At most 16 rows per unit; rows beyond go to the overflow unit nun + u.
        //   .x = q3lo | n3 << 8 | k4lo << 16 | k4hi << 24        .y = b24 | b34 << 8 | x << 16 | valid << 24
        const int nun = c24 * c34 * nv;
        for (int u = tid; u < nun; u += F4_THREADS) {
            const int xl = u % nv, r = u / nv, b34 = r % c34, b24 = r / c34;
            const int o24 = p.box.lo[1] + b24, o34 = p.box.lo[3] + b34;
            const int x = x0 + 2 * (v0 + xl);
            const int2 w3 = p.w3A[o34 * nl + o35], w4a = p.w4A[o24 * nl + o34];
            const int2 wx = fz_window(P.two_j[J24] + 2 * o24, x, P.two_k_base[1], P3);
            const int2 w4x = fz_window(l35, x, P.two_k_base[2], P4);
            const int q3lo = max(wx.x, w3.x), q3hi = (wx.y > 0 && w3.y > 0) ? min(wx.x + wx.y, w3.x + w3.y) : 0;
            const int n3 = max(0, q3hi - q3lo);
            const int k4lo = max(max(w4a.x, w4x.x), h4lo);
            int k4hi = (w4a.y > 0 && w4x.y > 0) ? min(min(w4a.x + w4a.y, w4x.x + w4x.y), h4hi) : 0;
            if (k4hi < k4lo) k4hi = k4lo;
            const int k4w = (k4lo << 16) | (k4hi << 24), id = b24 | (b34 << 8) | (xl << 16);
            s_unit[u] = make_int2(q3lo | (min(n3, 16) << 8) | k4w, id | (n3 > 0 ? 1 << 24 : 0));
            s_unit[nun + u] = make_int2((q3lo + 16) | (max(n3 - 16, 0) << 8) | k4w, id | (n3 > 16 ? 1 << 24 : 0));
        }
        fz_cp_wait<0>();
        __syncthreads();

        // units from the item's counter, one per warp at a time; the next unit is drawn one unit ahead, so that the S3 rows
        // it will ask for can be sent for into L1 a whole unit earlier
        auto draw = [&]() {
            int u = 0;
            if (lane == 0) u = atomicAdd(&s_next, 1);
            return __shfl_sync(0xffffffffu, u, 0);
        };
        const long s3item = ((long)b35 * NX + xg0 + v0) * (long)(P3 * P4);
        for (int u = draw(), un; u < 2 * nun; u = un) {
            un = draw();
            if (un < 2 * nun) {
                const int2 dn = s_unit[un];
                if (dn.y >> 24) {
                    const int q3n = dn.x & 255, k4n0 = (dn.x >> 16) & 255, k4n1 = (dn.x >> 24) & 255;
                    const long pr = (long)(dn.y & 255) * c34 + ((dn.y >> 8) & 255);
                    const double* s3r = p.S3T + (pr * c35 * NX + ((dn.y >> 16) & 255)) * (long)(P3 * P4) + s3item + (long)(q3n + (lane & 15)) * P4;
                    fz_prefetch_l1(s3r + (lane < 16 ? k4n0 : max(k4n1 - 1, k4n0)));
                }
            }
            const int2 d = s_unit[u];
            if (!(d.y >> 24)) continue;                       // no rows of P
            const int q3lo = d.x & 255, n3 = (d.x >> 8) & 255, k4lo = (d.x >> 16) & 255, k4hi = (d.x >> 24) & 255;
            const int b24 = d.y & 255, b34 = (d.y >> 8) & 255, xl = (d.y >> 16) & 255;
            const int ng = (k4hi - k4lo + 3) >> 2;
            const bool two3 = n3 > 8;                         // a second row tile of k3
            // this lane's operand pointers at the first k4
            const double* s3p = p.S3T + ((((long)b24 * c34 + b34) * c35 + b35) * NX + xg0 + v0 + xl) * (long)(P3 * P4) + (long)(q3lo + g) * P4 +
                                k4lo + q;                     // A of P: row k3 = q3lo + 8 i + g, column k4
            const double* b4g = a.Bw4P + (((long)b24 * c34 + b34) * P4 + k4lo) * (F4_L45 * 16);   // the unit's first k-step of fragments
            unsigned zq = z_lane + 8u * (unsigned)(xl * n5) + (unsigned)(k4lo - h4lo) * z_k4;

            double acc[2][16][2];
#pragma unroll
            for (int i = 0; i < 2; ++i)
#pragma unroll
                for (int j = 0; j < 16; ++j) acc[i][j][0] = acc[i][j][1] = 0.0;

            // one bulk copy per k-step into the warp's slot (every lane has read the slot: __syncwarp before)
            auto b4_copy = [&]() {
                if (lane == 0) {
                    fz_mbar_expect_tx(bar_u32, 8u * F4_BSLOT);
                    fz_bulk_g2s(bs_u32, b4g, 8u * F4_BSLOT, bar_u32);
                }
                b4g += F4_BSLOT;
            };
            // the {6j} array is exactly zero wherever a triad fails, so rows and columns beyond the unit's windows need no predicate:
            // their k4 meet zero rows of Q or zero entries of S3, their k3 are not stored
            double s3n[2];
            auto s3_fetch = [&]() {
                s3n[0] = __ldg(s3p);
                s3n[1] = two3 ? __ldg(s3p + 8 * P4) : 0.0;
                s3p += 4;
            };
            if (ng > 0) {
                __syncwarp();                                 // the previous unit's last Q phase has read the slot
                b4_copy();
                s3_fetch();
            }
            for (int gi = 0; gi < ng; ++gi) {
                const double s30 = s3n[0], s31 = s3n[1];      // requested a whole k-step ago
                if (gi + 1 < ng) s3_fetch();                  // S3 of the next k-step: a Q phase, a P phase and a Q phase to arrive
                fz_mbar_wait(bar_u32, bphase);                // the booster fragments of this k-step have landed
                bphase ^= 1u;
                // ---- Q of the four k4 of this k-step into the warp's tile (the P phase of the previous k-step has read it: the
                // __syncwarp below, after that phase).  k4 beyond the window get a zero row: their booster fragments are not used ----
#pragma unroll
                for (int kk = 0; kk < 4; ++kk) {
                    double c[N5T][2][2];
                    if (k4lo + 4 * gi + kk < k4hi) {          // uniform.  All three k-steps of l45: where the triad (k4 l45 j14) fails or the
                        double af[3][N5T];                    // box has no l45, Z and the booster are exactly zero: nothing skipped, nothing tested
                        double2 bf[3];
#pragma unroll
                        for (int ks = 0; ks < 3; ++ks) {
#pragma unroll
                            for (int t = 0; t < N5T; ++t) af[ks][t] = f4_lds(zq + kk * z_k4 + ks * z_ks + 64 * t);
                            asm volatile("ld.shared.v2.f64 {%0, %1}, [%2];" : "=d"(bf[ks].x), "=d"(bf[ks].y) : "r"(b4_lane + 8u * (unsigned)((kk * 3 + ks) * 64)));
                        }
#pragma unroll
                        for (int t = 0; t < N5T; ++t) {
                            fz_dmma0(c[t][0][0], c[t][0][1], af[0][t], bf[0].x);
                            if (N4T > 1) fz_dmma0(c[t][1][0], c[t][1][1], af[0][t], bf[0].y);
                        }
#pragma unroll
                        for (int ks = 1; ks < 3; ++ks) {
#pragma unroll
                            for (int t = 0; t < N5T; ++t) {
                                fz_dmma(c[t][0][0], c[t][0][1], af[ks][t], bf[ks].x);
                                if (N4T > 1) fz_dmma(c[t][1][0], c[t][1][1], af[ks][t], bf[ks].y);
                            }
                        }
                        ndm += (unsigned)(3 * N5T * N4T);
                    } else {
#pragma unroll
                        for (int t = 0; t < N5T; ++t) c[t][0][0] = c[t][0][1] = c[t][1][0] = c[t][1][1] = 0.0;
                    }
                    const unsigned dst = qst_lane + 8u * (unsigned)(kk * ldq);
#pragma unroll
                    for (int t = 0; t < N5T; ++t) {
                        const unsigned rowa = dst + 8u * (unsigned)(8 * t * n4);
                        if (smask & (1u << (4 * t))) f4_sts(rowa, c[t][0][0]);
                        if (smask & (2u << (4 * t))) f4_sts(rowa + 8u, c[t][0][1]);
                        if (N4T > 1) {
                            if (smask & (4u << (4 * t))) f4_sts(rowa + 64u, c[t][1][0]);
                            if (smask & (8u << (4 * t))) f4_sts(rowa + 72u, c[t][1][1]);
                        }
                    }
                }
                zq += 4 * z_k4;
                __syncwarp();                                 // the tile is complete; every lane has read the booster slot
                if (gi + 1 < ng) b4_copy();                   // the next k-step's fragments arrive under this k-step's P phase
                // ---- P: all column tiles (i5 i4), K = the four k4 of the tile ----
                auto p_phase = [&](auto rt2, auto all) {      // rt2: a second row tile of k3; all: every one of the 16 column tiles exists
#pragma unroll
                    for (int jp = 0; jp < 8; ++jp) {
                        if (decltype(all)::value || 2 * jp < NT) {
                            double2 bv;
                            asm volatile("ld.shared.v2.f64 {%0, %1}, [%2];" : "=d"(bv.x), "=d"(bv.y) : "r"(qld_lane + 128u * jp));
                            fz_dmma(acc[0][2 * jp][0], acc[0][2 * jp][1], s30, bv.x);
                            fz_dmma(acc[0][2 * jp + 1][0], acc[0][2 * jp + 1][1], s30, bv.y);
                            if (decltype(rt2)::value) {
                                fz_dmma(acc[1][2 * jp][0], acc[1][2 * jp][1], s31, bv.x);
                                fz_dmma(acc[1][2 * jp + 1][0], acc[1][2 * jp + 1][1], s31, bv.y);
                            }
                        }
                    }
                };
                if (NT >= 15) {
                    if (two3) p_phase(FzTrue(), FzTrue()); else p_phase(FzFalse(), FzTrue());
                } else {
                    if (two3) p_phase(FzTrue(), FzFalse()); else p_phase(FzFalse(), FzFalse());
                }
                ndm += (unsigned)(((NT + 1) & ~1) * (two3 ? 2 : 1));
                __syncwarp();                                 // the P phase has read the tile
            }
            // the rows of P of this unit (zeros when no k4 survives: the readers expect every allowed row)
            {
                double* Pb = p.Pq + ((((long)ac * c24 + b24) * c25 + b25) * P3) * V * prow + ((long)b34 * c35 + b35) * NP +
                             (long)(v0 + xl) * prow + 4 * q;
#pragma unroll
                for (int i = 0; i < 2; ++i) {
                    const int r3 = 8 * i + g;
                    if (r3 < n3) {
                        double* dst = Pb + (long)(q3lo + r3) * V * prow;
#pragma unroll
                        for (int jp = 0; jp < 8; ++jp) {      // NP is even and the row starts 16-byte aligned
                            if (pmask & (1u << (2 * jp)))
                                *reinterpret_cast<double2*>(dst + 16 * jp) = make_double2(acc[i][2 * jp][0], acc[i][2 * jp + 1][0]);
                            if (pmask & (2u << (2 * jp)))
                                *reinterpret_cast<double2*>(dst + 16 * jp + 2) = make_double2(acc[i][2 * jp][1], acc[i][2 * jp + 1][1]);
                        }
                    }
                }
            }
        }
    }
    if (p.cnt && lane == 0 && ndm) atomicAdd(p.cnt, (unsigned long long)ndm);
}

static void f4_shape(const SfDims& D, int* ldz, size_t* smem)
{
    const int n5 = D.n_i[4], P4 = D.n_k_pad[2];
    *ldz = (F4_XC - 1) * n5 + 16 <= 52 ? 52 : 68;             // the last x of a chunk reads 16 rows from its first i5; = 4 mod 16
    *smem = sizeof(double) * ((size_t)P4 * F4_L45 * *ldz + (size_t)F4_WARPS * (4 * F4_LDQ + F4_BSLOT));
}

/* True when k_fz_qp4 holds the shape of the box (the caller then builds Bw4P, as for k_fz_qp2). */
bool fz_qp4_supported(const FzParams& p, const SfDims& D)
{
    const int n4 = D.n_i[3], n5 = D.n_i[4], P3 = D.n_k_pad[1], P4 = D.n_k_pad[2];
    if (n5 > 16 || n4 > 16 || n4 * n5 > 128 || p.box.cnt[5] > F4_L45 || P4 > 24 || P4 < 1 || P3 < 1 || P3 > 239) return false;
    if (p.box.cnt[1] > 255 || p.box.cnt[3] > 255 || p.box.cnt[1] * p.box.cnt[3] * F4_XC > F4_MAXU) return false;
    // k3 rows of a unit: inside the window of a pair (l34 l35), at most 32 (two units of 16)
    for (int u = 0; u < p.box.cnt[3]; ++u)
        for (int v = 0; v < p.box.cnt[4]; ++v) {
            const int2 w = fz_window(D.two_j[J34] + 2 * (p.box.lo[3] + u), D.two_j[J35] + 2 * (p.box.lo[4] + v), D.two_k_base[1], P3);
            if (w.y > 32) return false;
        }
    int ldz;
    size_t smem;
    f4_shape(D, &ldz, &smem);
    return smem + 18 * 1024 <= 227 * 1024;                    // + the static tables
}

/* Launches k_fz_qp4 for the pass described by p (fz_qp4_supported must hold; Bw4P built by fz_launch_b4p). */
int fz_launch_qp4(const FzParams& p, const SfDims& D, const double* Bw4P, int* sched, int n_sm, cudaStream_t st)
{
    FzQp4Args a;
    memset(&a, 0, sizeof a);
    size_t smem;
    f4_shape(D, &a.ldz, &smem);
    a.vc = (p.V + F4_XC - 1) / F4_XC;
    const long n_items = (long)a.vc * p.a_cnt * p.box.cnt[2] * p.box.cnt[4];
    if (n_items > 2000000000L) return SF_EARG;
    a.n_items = (int)n_items;
    a.sched = sched;
    a.Bw4P = Bw4P;
    const int n5t = D.n_i[4] > 8 ? 2 : 1, n4t = D.n_i[3] > 8 ? 2 : 1;
    void (*kern)(const FzParams, const FzQp4Args) =
        a.ldz == 68 ? (n4t == 2 ? k_fz_qp4<68, 2, 2> : k_fz_qp4<68, 2, 1>)
                    : n5t == 2 ? (n4t == 2 ? k_fz_qp4<52, 2, 2> : k_fz_qp4<52, 2, 1>) : (n4t == 2 ? k_fz_qp4<52, 1, 2> : k_fz_qp4<52, 1, 1>);
    if (cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem) != cudaSuccess) return SF_ECUDA;
    const int grid = (int)(n_items < n_sm ? n_items : n_sm);
    kern<<<grid, F4_THREADS, smem, st>>>(p, a);
    sf_count_launch(1);
    return SF_OK;
}
