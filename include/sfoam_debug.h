/* sfoam_debug.h -- measurement and debugging entry points of libsfoam.  NOT part of the product contract (include/sfoam.h):
 * bench.py and the tests use them to time kernels, count work, probe the FP64 peak and force the size-dependent branches of
 * the paths on small inputs.  Same conventions as sfoam.h (extern "C", status codes, spins as 2j integers).
 */
#ifndef SFOAM_DEBUG_H
#define SFOAM_DEBUG_H

#include "sfoam.h"

#ifdef __cplusplus
extern "C" {
#endif

/* Number of (entry, x) summands of eq. (5) over shells [shell_lo, shell_hi): the sum over the entries
 * (i1 k2 k3 k4 k5) of every non-empty shell of the size of the intersection of the five triads that contain x.  The
 * algorithmic assembly work of the per-shell method is F_asm = 6 * n_terms (five multiplications by a
 * {6j} or by (2x+1), one addition).  Counted by a device kernel (integer work, exact); synchronises the default stream. */
int sf_vertex_terms(const int two_j[10], int two_dl, long shell_lo, long shell_hi, double *n_terms);

/* Useful work of the FACTORISED path (sf_set_path 4; DESIGN.md 5 K-f) for the full shell range: multiply-adds of each of its
 * six contractions counted on the index combinations the triangle inequalities of eqs. (3), (5) allow -- no tile padding,
 * no window rounding.  Pure host integer function (no device needed).
 *   mac[0] Z  = sum_k5 S2 S1 Bw5      mac[1] Q  = sum_l45 Z Bw4       mac[2] P  = sum_k4 S3 Q
 *   mac[3] R  = sum_{l34 l35} Bw3 P   mac[4] G  = sum_k2 Bw2 S5 S4    mac[5] A' = sum_{k3 x l23} G R
 *   elems[0..3] = structurally non-zero entries of Z, Q, P, R (8 bytes each: the intermediates' algorithmic size)
 * flop = 2 * mac.  SF_EARG / SF_ESPIN as sf_vertex_dims. */
int sf_factor_work(const int two_j[10], int two_dl, double mac[6], double elems[4]);

/* Entries of the five S arrays of step 4 in the library's dense layout = {6j} symbols gathered (or
 * evaluated) per vertex call: the unit count of the {6j}-gather bandwidth figure (16 B each: 8 read, 8 written).  -1 on bad
 * arguments.  Host integer function. */
long sf_slice_elems(const int two_j[10], int two_dl);

/* Number of vertex calls answered by replaying a recorded launch sequence (sf_set_graphs) since sf_init / the last reset:
 * lets a test see that repeated identical calls do reach the recording (they never do while every call changes the library
 * state, e.g. by re-growing a scratch block). */
long sf_graph_replays(int reset);

/* FP64 roofline denominators measured in this process: TFLOP/s of dependent-chain microbenchmarks,
 * kind 0 = DFMA (vector FP64 fused multiply-add), kind 1 = DMMA (mma.sync m8n8k4 f64 on the tensor cores), kind 2 = the inner
 * loop of a shared-memory-fed GEMM (10 conflict-free LDS.64 per 16 DMMA, 16 warps per SM, nothing else): the practical ceiling
 * of the gather-GEMM kernels, reported beside the peak, never used as the denominator.
 * Best of 5 launches of a few ms each; synchronises the default stream.  Requires sf_init. */
int sf_fp64_peak(int kind, double *tflops);

/* Milliseconds of device time (CUDA events on the call's stream) spent in each stage of the LAST vertex call,
 * recorded when sf_set_timing(1) is on: [0] S arrays (step 4), [1] assembly + contraction (steps 5-6(iii)),
 * [2] accumulation (step 6(iv) + normalisation).  Enabling timing makes the vertex calls synchronous. */
int sf_set_timing(int on);
int sf_last_stage_ms(double ms[3]);
/* Factorised path only: CUDA-event times of its kernels, summed over the launches of the last vertex call made with
 * sf_set_timing(1): ms[0] Q/P kernel (sums over l45 and k4), ms[1] R kernel (sum over l34 l35, edge-3 product),
 * ms[2] A' kernel (sum over x, k3, l23, edge-2 product), ms[3] the precomputations (Z, weighted boosters, G). */
int sf_last_kernel_ms(double ms[4]);
/* sf_set_counting(1): the factorised kernels count the FP64 MMA instructions (DMMA.8x8x4, 512 flop each) they issue, padding
 * included; sf_last_dmma returns the counts of the last vertex call, same order as ms[0..2] above.  Measurement only: the
 * call becomes synchronous and slightly slower; the result is unchanged. */
int sf_set_counting(int on);
int sf_last_dmma(double n[3]);
/* Debug aid of the factorised path: when on, its intermediate arrays (Z, G, P, R) are filled with NaN bit patterns before
 * they are produced, so that reading an entry nobody wrote shows up as a NaN in the tensor.  The result must not change. */
int sf_set_debug_poison(int on);

/* Bytes of global scratch the staged path may use for its two ping-pong buffers (default 6 GiB). */
void sf_set_staged_budget(unsigned long bytes);
/* Bytes of device memory the factorised path may use for its intermediates P and R of one pass over i1 (default 0 = a
 * third of the device).  A small budget forces several passes over i1 on a small problem: the test hook for the branches
 * that otherwise only the full-size workloads take. */
void sf_set_factor_budget(unsigned long bytes);

/* Kernel variants of the factorised path, for cross-checks and A/B timing: bit 0 = take the edge-3 contraction (R) through
 * the booster-stationary kernel (sf_factor_r.cu) instead of the general gather-GEMM; bit 1 = take Q/P through the first-generation kernel
 * (k_fz_qp); bit 2 = take Q/P through the second-generation kernel (k_fz_qp2) instead of the warp-autonomous one (k_fz_qp4).
 * bit 3 = take R through the general gather-GEMM (k_fz_gemm<FzMapR>) instead of the producer-warp kernel (k_fz_r3).
 * 0 = default (the fastest kernels that hold the shape).  All variants compute the same sums. */
void sf_set_factor_variant(int bits);
/* The Q/P kernel the last factorised call (its last box) took: 1 = k_fz_qp, 2 = k_fz_qp2, 4 = k_fz_qp4; 0 before any call. */
int sf_last_qp_kernel(void);

#ifdef __cplusplus
}
#endif
#endif /* SFOAM_DEBUG_H */
