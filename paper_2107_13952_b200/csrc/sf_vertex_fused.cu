// sf_vertex_fused.cu -- the on-chip path of steps 5-7 of the vertex-tensor algorithm for tensors
// whose i1-slice fits one SM: kernels (b) {15j} assembly, (c) mode-product contraction and (d) fixed-order shell
// accumulation of north_star, fused so that the per-shell {15j} tensor W never leaves the SM.
//
// Work unit = (chunk of consecutive shells, boundary intertwiner i1).  One persistent CTA (16 warps) per SM takes
// units from a counter; for each shell of the unit and each batch of four k2 values it runs, entirely in shared
// memory and registers,
//
//   asm  W2[s][(c3,c4)][c5] = (-1)^R sum_x U[c2][c3][x] S3[c3][c4][x] Y[c4][c5][x]           eq. (5)
//        with U = (2x+1) S5 S4 and Y = S2 S1 staged once per shell (the five {6j} of eq. (5); factors that fail a
//        triad are exactly 0, so the sum runs over the window of x allowed by the triads (i1 l25 x) and (k2 j13 x))
//   G1   T4[s][(c3,i5)][c4]  = sum_c5 W2 . (2k5+1) B5[i5,c5]          step 6(iii), "loop over GEMM"
//   G2   T3[s][(i4,i5)][c3]  = sum_c4 T4 . (2k4+1) B4[i4,c4]
//   G3   T2[(i3,i4,i5)][s]   = sum_c3 T3 . (2k3+1) B3[i3,c3]
//   G4   acc[(i3,i4,i5)][i2] += sum_s T2 . (2k2+1) B2[i2,c2(s)]       step 6(iv): accumulators stay in registers
//
// Every product is an FP64 tensor-core GEMM (mma.sync m8n8k4 f64 -> SASS DMMA.8x8x4; tcgen05 has no FP64 kind) whose
// A operand is read from shared memory with the contracted index fastest (row stride LDK = 4 mod 8: conflict-free
// fragment loads) and whose C fragments are scattered into the layout the next product needs.  A unit's accumulators
// are written once to partial[unit]; k_reduce_partials sums the chunks of each i1 in chunk order and applies
// prod sqrt(2i+1) (eq. (3)).  No float atomics anywhere: results are bitwise reproducible.
#include <stdio.h>

#include "sf_internal.h"

#define FUSED_THREADS 512
#define FUSED_WARPS 16
#define SLOTS 4                 // k2 values per batch = K of the G4 tensor-core step
#define KS_MAX 4                // k-steps of 4: virtual intertwiner ranges up to 16 values

struct FusedParams {
    SfProblem P;
    long shell_lo, shell_hi;
    int chunk, n_chunks, n_units;
    int LDK;                    // row stride (doubles) of every [rows][contracted] operand
    int R1, R2, R3, R, Rp;      // padded row counts: W2, T4, T3 buffers per slot; T2 rows and their padding
    int offB, offX2, offBw, offU, offY, offS3, y_stride;   // shared-memory offsets (doubles)
    int NXF;                    // x stride of U, Y, S3s: covers the x-range of the triad (i1 l25 x), even
    double* partial;            // [n_units][n2][R]
    unsigned int* counter;
};

__device__ __forceinline__ void dmma884(double& c0, double& c1, double a, double b)
{
    asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1},{%2},{%3},{%0,%1};\n"
                 : "+d"(c0), "+d"(c1)
                 : "d"(a), "d"(b));
}

struct ShellDesc {
    int o[6], t[4], kmin[4], K[4];
    bool empty;
};

// One [rows][K] x [K][N] product on the tensor cores: rows are taken in tiles of 8 by the warps in turn.
// A[(slot*rows_pad + m)*LDK + c]; B fragments bf[nt][ks] already in registers; the C fragment of row m, columns
// (n, n+1) is handed to `store(slot, m, n, c0, c1)`.
template <int NT, class Store>
__device__ __forceinline__ void gemm_rows(const double* __restrict__ A, int rows, int rows_pad, int nslots, int LDK,
                                          int ksteps, const double (&bf)[NT][KS_MAX], int warp, int lane, Store store)
{
    const int g = lane >> 2, q = lane & 3;
    const int tiles_per_slot = (rows + 7) >> 3;
    const int ntiles = nslots * tiles_per_slot;
    for (int tile = warp; tile < ntiles; tile += FUSED_WARPS) {
        const int slot = tile / tiles_per_slot, m0 = (tile - slot * tiles_per_slot) << 3;
        const double* a = A + ((long)(slot * rows_pad + m0 + g)) * LDK + q;
        double c[NT][2];
#pragma unroll
        for (int nt = 0; nt < NT; ++nt) c[nt][0] = c[nt][1] = 0.0;
#pragma unroll
        for (int ks = 0; ks < KS_MAX; ++ks)
            if (ks < ksteps) {
                const double av = a[4 * ks];
#pragma unroll
                for (int nt = 0; nt < NT; ++nt) dmma884(c[nt][0], c[nt][1], av, bf[nt][ks]);
            }
#pragma unroll
        for (int nt = 0; nt < NT; ++nt) store(slot, m0 + g, nt * 8 + 2 * q, c[nt][0], c[nt][1]);
    }
}

template <int NT>
__device__ __forceinline__ void load_bfrag(const double* __restrict__ Bw, int LDK, int lane, double (&bf)[NT][KS_MAX])
{
    const int g = lane >> 2, q = lane & 3;
#pragma unroll
    for (int nt = 0; nt < NT; ++nt)
#pragma unroll
        for (int ks = 0; ks < KS_MAX; ++ks) bf[nt][ks] = (4 * ks < LDK) ? Bw[(nt * 8 + g) * LDK + 4 * ks + q] : 0.0;
}

template <int NT, int TPM, int NXS>
__global__ void __launch_bounds__(FUSED_THREADS, 1) k_vertex_fused(const FusedParams fp)
{
    extern __shared__ __align__(16) double smem[];
    __shared__ unsigned int s_unit;
    const SfProblem& P = fp.P;
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31, g = lane >> 2, q = lane & 3;
    const int LDK = fp.LDK;
    double* bufA = smem;                    // W2 [SLOTS][R1][LDK], later T3 [SLOTS][R3][LDK]
    double* bufB = smem + fp.offB;          // T4 [SLOTS][R2][LDK]
    double* X2 = smem + fp.offX2;           // T2 [Rp][SLOTS]
    double* Bw = smem + fp.offBw;           // [4][NT*8][LDK] weighted boosters (2k+1) B_e[i][c], zero padded
    double* U = smem + fp.offU;             // [k_max2*k_max3][NXF]
    double* Y = smem + fp.offY;             // [k_max4][y_stride], y_stride = k_max5*NXF + 2
    double* S3s = smem + fp.offS3;          // [k_max3*k_max4][NXF]
    const int n1 = P.n_i[0], n2 = P.n_i[1], n3 = P.n_i[2], n4 = P.n_i[3], n5 = P.n_i[4];
    const int M3 = P.k_max[1], M4 = P.k_max[2];
    const int R = fp.R, n45 = n4 * n5;
    const int nl = P.nl, NX = P.n_x_pad, NXF = fp.NXF;

    // zero all dynamic shared memory once: padding rows / columns must hold finite values (they meet zero operands)
    for (int z = tid; z < fp.offS3 + M3 * M4 * NXF; z += FUSED_THREADS) smem[z] = 0.0;

    for (;;) {
        __syncthreads();
        if (tid == 0) s_unit = atomicAdd(fp.counter, 1u);
        __syncthreads();
        const int unit = (int)s_unit;
        if (unit >= fp.n_units) break;
        const int chunk_id = unit / n1, a1 = unit - chunk_id * n1;
        const int i1 = P.two_i_min[0] + 2 * a1;
        const long s_begin = fp.shell_lo + (long)chunk_id * fp.chunk;
        const long s_end = min(s_begin + fp.chunk, fp.shell_hi);

        double acc[TPM][NT][2];
#pragma unroll
        for (int j = 0; j < TPM; ++j)
#pragma unroll
            for (int nt = 0; nt < NT; ++nt) acc[j][nt][0] = acc[j][nt][1] = 0.0;

        for (long shell = s_begin; shell < s_end; ++shell) {
            ShellDesc sd;
            sf_shell_offsets(shell, nl, sd.o);
            sf_triples(sd.o, nl, sd.t);
            sd.empty = false;
#pragma unroll
            for (int e = 0; e < 4; ++e) {
                const SfKRange r = P.kr[e][sd.t[e]];
                sd.kmin[e] = r.two_k_min;
                sd.K[e] = r.n_k;
                if (r.n_k == 0) sd.empty = true;
            }
            if (sd.empty) continue;   // uniform over the CTA
            const int K2 = sd.K[0], K3 = sd.K[1], K4 = sd.K[2], K5 = sd.K[3];
            const int l25 = P.two_j[J25] + 2 * sd.o[2];
            const int x0 = abs(i1 - l25);
            const int nxs = ((i1 + l25 - x0) >> 1) + 1;            // x-range of the triad (i1 l25 x)
            const int xg0 = (x0 - P.two_x_base) >> 1;

            __syncthreads();   // previous shell has finished with U, Y, S3s, Bw
            // ---- per-shell staging: U, Y, S3s from the S arrays of step 4, weighted booster sub-matrices (step 6(ii))
            {
                const int q2b = (sd.kmin[0] - P.two_k_base[0]) >> 1, q3b = (sd.kmin[1] - P.two_k_base[1]) >> 1;
                const int q4b = (sd.kmin[2] - P.two_k_base[2]) >> 1, q5b = (sd.kmin[3] - P.two_k_base[3]) >> 1;
                const int P2 = P.n_k_pad[0], P3 = P.n_k_pad[1], P4 = P.n_k_pad[2], P5 = P.n_k_pad[3];
                const double* s1 = P.S[0] + ((long)sd.o[2] * n1 + a1) * P5 * NX + xg0;
                const double* s2 = P.S[1] + ((long)sd.o[4] * nl + sd.o[5]) * P4 * P5 * NX + xg0;
                const double* s3 = P.S[2] + (((long)sd.o[1] * nl + sd.o[3]) * nl + sd.o[4]) * P3 * P4 * NX + xg0;
                const double* s4 = P.S[3] + ((long)sd.o[0] * nl + sd.o[1]) * P2 * P3 * NX + xg0;
                const double* s5 = P.S[4] + ((long)sd.o[2] * n1 + a1) * P2 * NX + xg0;
                for (int z = tid; z < K4 * K5 * nxs; z += FUSED_THREADS) {
                    const int xx = z % nxs, r = z / nxs, c5 = r % K5, c4 = r / K5;
                    Y[c4 * fp.y_stride + c5 * NXF + xx] =
                        s2[((long)(q4b + c4) * P5 + q5b + c5) * NX + xx] * s1[(long)(q5b + c5) * NX + xx];
                }
                for (int z = tid; z < K2 * K3 * nxs; z += FUSED_THREADS) {
                    const int xx = z % nxs, r = z / nxs, c3 = r % K3, c2 = r / K3;
                    U[(c2 * M3 + c3) * NXF + xx] = (double)(x0 + 2 * xx + 1) * s5[(long)(q2b + c2) * NX + xx] *
                                                   s4[((long)(q2b + c2) * P3 + q3b + c3) * NX + xx];
                }
                for (int z = tid; z < K3 * K4 * nxs; z += FUSED_THREADS) {
                    const int xx = z % nxs, r = z / nxs, c4 = r % K4, c3 = r / K4;
                    S3s[(c3 * M4 + c4) * NXF + xx] = s3[((long)(q3b + c3) * P4 + q4b + c4) * NX + xx];
                }
                const int bw_rows = NT * 8;
                for (int z = tid; z < 4 * bw_rows * LDK; z += FUSED_THREADS) {
                    const int c = z % LDK, r = z / LDK, ii = r % bw_rows, e = r / bw_rows;
                    double v = 0.0;
                    if (ii < P.n_i[e + 1] && c < sd.K[e]) {
                        const int kk0 = (sd.kmin[e] - P.two_k_base[e]) >> 1;
                        v = (double)(sd.kmin[e] + 2 * c + 1) *
                            sf_brow(P, e, sd.t[e], ii)[kk0 + c];
                    }
                    Bw[z] = v;
                }
            }
            __syncthreads();

            // sign base: 2R = i1 + k2 + k3 + k4 + k5 + all ten spins  (reading G1)
            int two_l_sum = P.two_j[J12] + P.two_j[J13] + P.two_j[J14] + P.two_j[J15] + i1;
#pragma unroll
            for (int s = 0; s < 6; ++s) two_l_sum += P.two_j[J23 + s] + 2 * sd.o[s];

            const int ks5 = (K5 + 3) >> 2, ks4 = (K4 + 3) >> 2, ks3 = (K3 + 3) >> 2;
            const int rows1 = K3 * K4, rows2 = K3 * n5, rows3 = n45;

            for (int cb = 0; cb < K2; cb += SLOTS) {
                const int nslots = min(SLOTS, K2 - cb);
                // ---- asm: one thread per (slot, c3, c4) row of W2, all c5 ----
                if (tid < nslots * rows1) {
                    const int slot = tid / rows1, m = tid - slot * rows1, c3 = m / K4, c4 = m - c3 * K4;
                    const int c2 = cb + slot;
                    // window of x allowed by the triads (i1 l25 x) and (k2 j13 x): at most NXS - 1 values; it starts at
                    // an even offset w0e so that the operands can be read as aligned pairs
                    const int k2 = sd.kmin[0] + 2 * c2, j13 = P.two_j[J13];
                    const int xlo = max(x0, abs(k2 - j13)), xhi = min(x0 + 2 * (nxs - 1), k2 + j13);
                    const int w0 = (xlo - x0) >> 1, w1 = w0 + ((xhi - xlo) >> 1);      // first / last xx of the window
                    const int w0e = min(w0 & ~1, NXF - NXS);
                    const double* u = U + (c2 * M3 + c3) * NXF + w0e;
                    const double* s3v = S3s + (c3 * M4 + c4) * NXF + w0e;
                    double T[NXS];
#pragma unroll
                    for (int w = 0; w < NXS; ++w) T[w] = (xhi >= xlo && w0e + w >= w0 && w0e + w <= w1) ? u[w] * s3v[w] : 0.0;
                    const int sb = two_l_sum + k2 + sd.kmin[1] + 2 * c3 + sd.kmin[2] + 2 * c4 + sd.kmin[3];
                    double* wrow = bufA + ((long)(slot * fp.R1 + m)) * LDK;
                    const double* yrow = Y + c4 * fp.y_stride + w0e;
                    for (int c5 = 0; c5 < K5; ++c5) {
                        double w = 0.0;
#pragma unroll
                        for (int v = 0; v < NXS; ++v) w = fma(T[v], yrow[c5 * NXF + v], w);
                        wrow[c5] = (((sb + 2 * c5) >> 1) & 1) ? -w : w;
                    }
                }
                __syncthreads();
                // ---- G1: contract k5 ----
                {
                    double bf[NT][KS_MAX];
                    load_bfrag<NT>(Bw + 3 * NT * 8 * LDK, LDK, lane, bf);
                    gemm_rows<NT>(bufA, rows1, fp.R1, nslots, LDK, ks5, bf, warp, lane,
                                  [&](int slot, int m, int n, double c0, double c1) {
                                      if (m < rows1) {
                                          const int c3 = m / K4, c4 = m - c3 * K4;
                                          double* dst = bufB + ((long)(slot * fp.R2 + c3 * n5 + n)) * LDK + c4;
                                          if (n < n5) dst[0] = c0;
                                          if (n + 1 < n5) dst[LDK] = c1;
                                      }
                                  });
                }
                __syncthreads();
                // ---- G2: contract k4 ----
                {
                    double bf[NT][KS_MAX];
                    load_bfrag<NT>(Bw + 2 * NT * 8 * LDK, LDK, lane, bf);
                    gemm_rows<NT>(bufB, rows2, fp.R2, nslots, LDK, ks4, bf, warp, lane,
                                  [&](int slot, int m, int n, double c0, double c1) {
                                      if (m < rows2) {
                                          const int c3 = m / n5, i5 = m - c3 * n5;
                                          double* dst = bufA + ((long)(slot * fp.R3 + n * n5 + i5)) * LDK + c3;
                                          if (n < n4) dst[0] = c0;
                                          if (n + 1 < n4) dst[(long)n5 * LDK] = c1;
                                      }
                                  });
                }
                __syncthreads();
                // ---- G3: contract k3 ----
                {
                    double bf[NT][KS_MAX];
                    load_bfrag<NT>(Bw + 1 * NT * 8 * LDK, LDK, lane, bf);
                    gemm_rows<NT>(bufA, rows3, fp.R3, nslots, LDK, ks3, bf, warp, lane,
                                  [&](int slot, int m, int n, double c0, double c1) {
                                      if (m < rows3) {
                                          double* dst = X2 + ((long)(n * n45 + m)) * SLOTS + slot;
                                          if (n < n3) dst[0] = c0;
                                          if (n + 1 < n3) dst[(long)n45 * SLOTS] = c1;
                                      }
                                  });
                }
                __syncthreads();
                // ---- G4: contract k2 (the batch's slots are the K of one tensor-core step), accumulate in registers ----
                {
                    double b2[NT];
#pragma unroll
                    for (int nt = 0; nt < NT; ++nt)
                        b2[nt] = (q < nslots) ? Bw[(nt * 8 + g) * LDK + cb + q] : 0.0;
                    const int mtiles = fp.Rp >> 3;
#pragma unroll
                    for (int j = 0; j < TPM; ++j) {
                        const int mt = warp + FUSED_WARPS * j;
                        if (mt < mtiles) {
                            const double av = X2[(long)(mt * 8 + g) * SLOTS + q];
#pragma unroll
                            for (int nt = 0; nt < NT; ++nt) dmma884(acc[j][nt][0], acc[j][nt][1], av, b2[nt]);
                        }
                    }
                }
                // no barrier here: the next batch's asm writes bufA (last read by G3), its G3 writes X2 only after
                // three more barriers
            }
        }
        // ---- flush the unit's accumulators: partial[unit][i2][r] ----
        {
            double* dst = fp.partial + (long)unit * n2 * R;
#pragma unroll
            for (int j = 0; j < TPM; ++j) {
                const int r = (warp + FUSED_WARPS * j) * 8 + g;
                if (r < R) {
#pragma unroll
                    for (int nt = 0; nt < NT; ++nt) {
                        const int i2 = nt * 8 + 2 * q;
                        if (i2 < n2) dst[(long)i2 * R + r] = acc[j][nt][0];
                        if (i2 + 1 < n2) dst[(long)(i2 + 1) * R + r] = acc[j][nt][1];
                    }
                }
            }
        }
    }
}

// kernel (d): out[a1][i2][r] = prod sqrt(2i+1) * sum over chunks (in chunk order) of partial[chunk*n1 + a1][i2][r]
__global__ void __launch_bounds__(256) k_reduce_partials(SfProblem P, int n_chunks, long n_out, const double* __restrict__ partial,
                                                         double* __restrict__ out)
{
    const long z = blockIdx.x * (long)blockDim.x + threadIdx.x;
    if (z >= n_out) return;
    const long slice = n_out / P.n_i[0];
    const long a1 = z / slice, rest = z - a1 * slice;
    double s = 0.0;
    for (int c = 0; c < n_chunks; ++c) s += partial[((long)c * P.n_i[0] + a1) * slice + rest];
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
static inline int ceil8(int v) { return (v + 7) & ~7; }

struct FusedPlan {
    int NT, TPM, NXS;
    FusedParams fp;
    size_t smem;
    bool ok;
};

static int max_nxs(const SfDims& D)
{
    int m = 0;
    for (int a = 0; a < D.n_i[0]; ++a)
        for (int o = 0; o < D.nl; ++o) {
            int i1 = D.two_i_min[0] + 2 * a, l25 = D.two_j[J25] + 2 * o;
            int n = (i1 + l25 - abs(i1 - l25)) / 2 + 1;
            if (n > m) m = n;
        }
    return m;
}

static FusedPlan make_plan(const SfDims& D)
{
    FusedPlan pl;
    memset(&pl, 0, sizeof pl);
    pl.ok = false;
    int nmax = 0, kmax = 0;
    for (int e = 0; e < 4; ++e) {
        if (D.n_i[e + 1] > nmax) nmax = D.n_i[e + 1];
        if (D.k_max[e] > kmax) kmax = D.k_max[e];
        if (D.k_max[e] == 0) return pl;
    }
    if (nmax > 16 || kmax > 4 * KS_MAX) return pl;
    pl.NT = nmax <= 8 ? 1 : 2;
    const int nxs = max_nxs(D);
    // window of x per W2 row: the triads (i1 l25 x) and (k2 j13 x) leave at most min(nxs, 2 j13 + 1) values, +1 for the
    // even alignment of its start
    int win = D.two_j[J13] + 1;
    if (nxs < win) win = nxs;
    win += 1;
    if (win > 16) return pl;
    const int R = D.n_i[2] * D.n_i[3] * D.n_i[4], Rp = ceil8(R);
    const int tpm = (Rp / 8 + FUSED_WARPS - 1) / FUSED_WARPS;
    // instantiated shapes (NT, TPM, NXS)
    static const int shapes[][3] = {{1, 1, 4}, {1, 4, 8}, {1, 4, 16}, {2, 4, 16}, {2, 11, 12}, {2, 11, 16}};
    int pick = -1;
    for (int s = 0; s < 6; ++s)
        if (shapes[s][0] == pl.NT && shapes[s][1] >= tpm && shapes[s][2] >= win) {
            pick = s;
            break;
        }
    if (pick < 0) return pl;
    pl.TPM = shapes[pick][1];
    pl.NXS = shapes[pick][2];
    FusedParams& fp = pl.fp;
    const int ks = (kmax + 3) / 4;
    fp.NXF = ((nxs > pl.NXS ? nxs : pl.NXS) + 1) & ~1;
    fp.LDK = (ks & 1) ? 4 * ks : 4 * ks + 4;
    fp.R1 = ceil8(D.k_max[1] * D.k_max[2]);
    fp.R2 = ceil8(D.k_max[1] * D.n_i[4]);
    fp.R3 = ceil8(D.n_i[3] * D.n_i[4]);
    fp.R = R;
    fp.Rp = Rp;
    const int ra = fp.R1 > fp.R3 ? fp.R1 : fp.R3;
    int off = SLOTS * ra * fp.LDK;
    fp.offB = off;
    off += SLOTS * fp.R2 * fp.LDK;
    fp.offX2 = off;
    off += Rp * SLOTS;
    fp.offBw = off;
    off += 4 * pl.NT * 8 * fp.LDK;
    fp.offU = off;
    off += D.k_max[0] * D.k_max[1] * fp.NXF;
    fp.offY = off;
    fp.y_stride = D.k_max[3] * fp.NXF + 2;
    off += D.k_max[2] * fp.y_stride;
    off = (off + 1) & ~1;
    fp.offS3 = off;
    off += D.k_max[1] * D.k_max[2] * fp.NXF;
    pl.smem = sizeof(double) * (size_t)off;
    if (pl.smem > 220 * 1024) return pl;
    if (SLOTS * D.k_max[1] * D.k_max[2] > FUSED_THREADS) return pl;
    pl.ok = true;
    return pl;
}

bool sf_vertex_fused_supported(const SfDims& D) { return make_plan(D).ok; }

template <int NT, int TPM, int NXS>
static int launch_fused(const FusedPlan& pl, int grid, cudaStream_t st)
{
    static bool attr_set = false;
    if (!attr_set) {
        if (cudaFuncSetAttribute(k_vertex_fused<NT, TPM, NXS>, cudaFuncAttributeMaxDynamicSharedMemorySize, 220 * 1024) !=
            cudaSuccess)
            return SF_ECUDA;
        attr_set = true;
    }
    k_vertex_fused<NT, TPM, NXS><<<grid, FUSED_THREADS, pl.smem, st>>>(pl.fp);
    return SF_OK;
}

int sf_vertex_fused(const SfDims& D, const SfProblem& P, long shell_lo, long shell_hi, double* out, cudaStream_t st)
{
    FusedPlan pl = make_plan(D);
    if (!pl.ok) return SF_EARG;
    static int n_sm = 0;
    if (!n_sm) {
        int dev = 0;
        SF_CUDA_OK(cudaGetDevice(&dev));
        SF_CUDA_OK(cudaDeviceGetAttribute(&n_sm, cudaDevAttrMultiProcessorCount, dev));
    }
    FusedParams& fp = pl.fp;
    fp.P = P;
    fp.shell_lo = shell_lo;
    fp.shell_hi = shell_hi;
    const long nsh = shell_hi - shell_lo;
    const int n1 = D.n_i[0];
    // chunks: about 16 units per SM so that the dynamic schedule balances; partial[unit] stays small
    long chunk = (nsh * n1 + 16L * n_sm - 1) / (16L * n_sm);
    if (chunk < 1) chunk = 1;
    fp.chunk = (int)chunk;
    fp.n_chunks = (int)((nsh + chunk - 1) / chunk);
    fp.n_units = fp.n_chunks * n1;
    const long slice = D.n_out / n1;
    double* partial = (double*)sf_scratch(17, sizeof(double) * (size_t)(fp.n_units > 0 ? fp.n_units : 1) * slice);
    unsigned int* counter = (unsigned int*)sf_scratch(18, 256);
    if (!partial || !counter) return SF_ENOMEM;
    fp.partial = partial;
    fp.counter = counter;
    if (fp.n_units > 0) {
        SF_CUDA_OK(cudaMemsetAsync(counter, 0, sizeof(unsigned int), st));
        const int grid = fp.n_units < n_sm ? fp.n_units : n_sm;
        int rc = SF_EARG;
#define SF_SHAPE(a, b, c) \
    if (pl.NT == a && pl.TPM == b && pl.NXS == c) rc = launch_fused<a, b, c>(pl, grid, st);
        SF_SHAPE(1, 1, 4)
        SF_SHAPE(1, 4, 8)
        SF_SHAPE(1, 4, 16)
        SF_SHAPE(2, 4, 16)
        SF_SHAPE(2, 11, 12)
        SF_SHAPE(2, 11, 16)
#undef SF_SHAPE
        if (rc != SF_OK) return rc;
        sf_count_launch(1);
    }
    sf_timing_mark(2, st);
    k_reduce_partials<<<(unsigned)((D.n_out + 255) / 256), 256, 0, st>>>(P, fp.n_chunks, D.n_out, partial, out);
    sf_count_launch(1);
    return cudaGetLastError() == cudaSuccess ? SF_OK : SF_ECUDA;
}
