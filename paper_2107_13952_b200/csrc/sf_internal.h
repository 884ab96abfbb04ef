// sf_internal.h -- internal declarations of libsfoam (CUDA path).  Not part of the C ABI (include/sfoam.h is).
//
// Notation follows the paper (arXiv 2107.13952): boundary spins j_ab, virtual spins l_ab, boundary intertwiners i_e,
// virtual intertwiners k_e, recoupling spin x of eq. (5).  All spins are integers two_* = 2*spin.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include "../../include/sfoam.h"
#include "../../include/sfoam_debug.h"

// spin order of two_j[10] (Listing 8)
enum { J12 = 0, J13, J14, J15, J23, J24, J25, J34, J35, J45 };

// -------------------------------------------------------------------------------------------------------------
// Host-side description of one vertex problem (steps 1-2 of the algorithm)
// -------------------------------------------------------------------------------------------------------------
struct SfDims {
    int two_j[10];
    int two_dl, nl;                 // nl = Delta_l + 1
    long n_shells;                  // nl^6
    int two_i_min[5], n_i[5];       // boundary intertwiner ranges, nodes 1..5
    int two_k_base[4], n_k_pad[4];  // booster k layout of edges 2..5 (union over triples)
    int k_max[4];                   // largest n_k over the triples of each edge
    int two_x_base, n_x_pad;        // union range of the recoupling spin x (triad (i1 l25 x))
    long n_out;                     // prod n_i
};

// per-triple k-range tables, kr[e][t] = (two_k_min, n_k), e = 0..3 for edges 2..5
struct SfKRange {
    int two_k_min, n_k;
};

int sf_host_pair_range(int a, int b, int c, int d, int* lo);           // count, *lo = minimum
int sf_host_dims(const int two_j[10], int two_dl, SfDims* D);          // SF_OK / SF_EARG / SF_ESPIN
void sf_host_kranges(const SfDims& D, int e, SfKRange* out);           // out[nl^3]
void sf_host_shell_offsets(const SfDims& D, long shell, int o[6]);

// -------------------------------------------------------------------------------------------------------------
// Device-side problem descriptor, passed by value to every vertex kernel
// -------------------------------------------------------------------------------------------------------------
struct SfProblem {
    int two_j[10];
    int nl;
    int two_i_min[5], n_i[5];
    int two_k_base[4], n_k_pad[4], k_max[4];
    int two_x_base, n_x_pad;
    const SfKRange* kr[4];        // device: per edge, nl^3 entries
    const double* S[5];           // device: S1..S5, layouts in sf_slices.cu
    const double* B[4];           // device: caller's boosters, edges 2..5
    int b_n[4], b_i0[4];          // rows per triple of the caller's booster, and the row of this problem's first intertwiner
                                  // (a restricted intertwiner range, keeps the caller's full layout)
};

// row (i, :) of the booster of edge e + 2 at triple t; ii counts from this problem's first intertwiner
__host__ __device__ inline const double* sf_brow(const SfProblem& P, int e, long t, int ii)
{
    return P.B[e] + (t * P.b_n[e] + P.b_i0[e] + ii) * P.n_k_pad[e];
}

// shell -> offsets (o23 o24 o25 o34 o35 o45), o45 fastest (eq. (9))
__host__ __device__ inline void sf_shell_offsets(long shell, int nl, int o[6])
{
    for (int q = 5; q >= 0; --q) {
        o[q] = (int)(shell % nl);
        shell /= nl;
    }
}
// booster triple indices in the paper's superscript order
__host__ __device__ inline void sf_triples(const int o[6], int nl, int t[4])
{
    t[0] = (o[0] * nl + o[1]) * nl + o[2];   // edge 2: (l23 l24 l25)
    t[1] = (o[3] * nl + o[4]) * nl + o[0];   // edge 3: (l34 l35 l23)
    t[2] = (o[5] * nl + o[1]) * nl + o[3];   // edge 4: (l45 l24 l34)
    t[3] = (o[2] * nl + o[4]) * nl + o[5];   // edge 5: (l25 l35 l45)
}

// -------------------------------------------------------------------------------------------------------------
// {6j} machinery (sf_sixj.cu)
// -------------------------------------------------------------------------------------------------------------
// Accuracy envelope of the double-double Racah sum (sf_sixj.cuh), measured against the exact oracle on the symbols whose sum
// cancels most (all six labels within 4 of 2j, every valid combination) and on random symbols (tests/test_gpu_sixj.py,
// test_large_label_envelope): bit-identical to the correctly rounded value up to 2j ~ 176, relative error <= 4e-15 up to 220,
// <= 2.5e-13 up to 244; from 2j = 248 on symbols close to a zero of the {6j} miss relative 1e-12 (2.7e-11 at 248, 8.7e-12
// at 256, absolute error <= 2.5e-17).  The bound is the largest label for which relative 1e-12 has been demonstrated; larger
// arguments are refused (SF_EARG) instead of returning cancelled digits.  Config 4 at lambda = 6 reaches 168.
#define SF_SIXJ_MAX_TWO_J 240

struct SfSixjTable {
    int two_jmax;            // -1 if absent
    long n_slots;
    const double* values;    // device
    const long* base4;       // device: prefix sums over (a,b,c,e) groups
};

int sf_sixj_module_init(void);                       // uploads the factorial table
void sf_sixj_module_free(void);
int sf_sixj_table_build(int two_jmax, cudaStream_t st);
SfSixjTable sf_sixj_table_get(void);

// -------------------------------------------------------------------------------------------------------------
// S arrays of step 4 (sf_slices.cu) and the two vertex paths
// -------------------------------------------------------------------------------------------------------------
struct SfSliceSizes {
    long n[5];    // elements of S1..S5
};
void sf_slice_sizes(const SfDims& D, SfSliceSizes* sz);
// one launch: the five S arrays and, when kr is given, the k-range tables kr[e * nl^3 + t] of the four edges (step 2)
int sf_build_slices(const SfDims& D, double* const S[5], const SfSixjTable& tab, SfKRange* kr, cudaStream_t st);
void sf_launch_kranges(const SfDims& D, SfKRange* out, cudaStream_t st);   // the k-range tables alone

struct SfScratch;   // owned by the context (sf_api.cu)
int sf_vertex_staged(const SfDims& D, const SfProblem& P, long shell_lo, long shell_hi, double* out, cudaStream_t st);
int sf_vertex_line(const SfDims& D, const SfProblem& P, long shell_lo, long shell_hi, double* out, cudaStream_t st);
bool sf_vertex_line_supported(const SfDims& D);
int sf_vertex_factor(const SfDims& D, const SfProblem& P, long shell_lo, long shell_hi, double* out, cudaStream_t st);
bool sf_vertex_factor_supported(const SfDims& D);
void sf_vertex_factor_forget(void);               // drops what the factorised path remembers about refused allocations (sf_finalize)

// scratch allocator owned by the context: grows on demand, freed by sf_finalize.  slot = small integer id.
void* sf_scratch(int slot, size_t bytes);
void sf_scratch_release(int slot);                // frees the slot's block (synchronises the device); no-op while recording
void sf_count_launch(int n);
// Guard of every compute entry point of the C ABI (the vertex calls, the contractions, sf_vertex_terms, sf_sixj_table and
// sf_sixj_batch / sf_sixj_get, the last three on the legacy stream): the library keeps ONE set of scratch buffers and one {6j}
// table, so calls are serialised -- host threads by a mutex, streams by an event (a call on another stream than the previous
// call's first waits for that call).  sf_contract_vertices_noalloc is outside it by design (sf_contract_noalloc.cu).
struct SfCallGuard {
    explicit SfCallGuard(cudaStream_t st);
    ~SfCallGuard();
    cudaStream_t st;
    bool events;
};
// Host-side part of the guard alone (the mutex): for the setters, sf_init and sf_finalize, which change the state the compute
// calls read (generation, graph cache, settings, table pointers) but launch nothing.
struct SfHostLock {
    SfHostLock();
    ~SfHostLock();
};
// What a function caches about the device (SM count, memory size, "shared-memory attribute already raised" flags) holds for one
// context only: sf_finalize + sf_init may continue on another device.  A cached value remembers the context it was filled in and
// starts again from `init` in the next one.   static SfPerContext<int> c(0); int& n_sm = c.get();
long sf_context_epoch(void);                      // number of contexts created so far (sf_init)
template <class T>
struct SfPerContext {
    T value, init;
    long epoch;
    explicit SfPerContext(T i) : value(i), init(i), epoch(-1) {}
    T& get()
    {
        const long e = sf_context_epoch();
        if (epoch != e) {
            value = init;
            epoch = e;
        }
        return value;
    }
};
bool sf_stream_is_captured(cudaStream_t st);      // the caller is capturing `st`: entry points that use the scratch return SF_ECAPTURE
void sf_bump_generation(void);                    // drops the recorded launch sequences (sf_api.cu): call when a setting they depend on changes
bool sf_timing_on(void);
bool sf_counting_on(void);
bool sf_poison_on(void);
void sf_timing_mark(int idx, cudaStream_t st);   // records event idx of the stage timing when it is enabled
void sf_launch_finalize(const SfProblem& P, long n_out, const double* acc, double* out, cudaStream_t st);

#define SF_CUDA_OK(call)                                   \
    do {                                                   \
        cudaError_t err__ = (call);                        \
        if (err__ != cudaSuccess) return SF_ECUDA;         \
    } while (0)
