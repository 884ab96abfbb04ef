// sf_contract_noalloc.cu -- sf_contract_vertices_noalloc: the two-vertex contraction  sum_z a[z] b[z]  (PAPER.md:327-365,
// Fig. 3: two vertex tensors glued along all five edges) for callers that must not, or cannot, allocate device memory.
//
// Who these callers are.  A spin-foam sum over bulk spins, or a Monte Carlo sampler over them, calls this contraction
// millions of times from inside a host program that has usually handed the whole GPU to an allocator of its own (the
// CUDA.jl pool the paper's Julia front end runs on, PyTorch's caching allocator, a fixed MIG / MPS memory slice).  In such a
// process a cudaMalloc coming out of a C library either fails outright (nothing is left outside the pool) or forces the
// pool to give memory back; and cudaMalloc / cudaFree synchronise the whole device, which a caller that keeps several
// streams busy, or that sits in a section where implicit synchronisation is not allowed, cannot accept at an arbitrary
// point of its loop.  sf_contract_vertices (sf_contract.cu) takes its per-CTA partial sums and its ticket from the library
// context's growable scratch (sf_scratch -> cudaMalloc on first use); this variant needs neither the context nor sf_init.
//
// How.  The scratch is the file-scope device array g_kn_scratch below: 8192 partial sums and one ticket, 65 792 bytes that
// every GPU on which this library's code is loaded keeps until the process exits.  The size of the array fixes the largest
// input: one partial sum per CTA, one CTA per 4096 entries, hence n <= 8192 * 4096 = 33 554 432 entries (32^5; the paper's
// largest vertex tensors, 21^5 = 4 084 101 entries, use 998 of the 8192 slots).  Larger n is refused with SF_ELIMIT before
// anything is launched.  No cudaMalloc, cudaFree, event / stream creation or other allocating routine is called.
//
// In host code the NAME g_kn_scratch is only the host-side handle of the symbol, not an address the GPU can use: the address
// has to be asked for, per device, with cudaGetSymbolAddress while that device is current.  The first call on each device
// does this (kn_scratch_for_current_device) and remembers the answer; because that query may make the CUDA runtime load this
// library's device code, make the first call on a device BEFORE any stream capture is begun in the process.
//
// Sharing.  All calls on one device use the same array, and it still holds what the previous call left in it.  The ticket
// must start at zero, so every call clears it on the caller's stream ahead of its kernel; the partial sums need no clearing
// (every slot that is read was written by the same launch).  Two calls whose kernels can be in flight on the same GPU at
// the same time (different streams without an ordering between them, or several host threads) RACE on the array and give
// wrong sums: order them, e.g. by issuing all of them on one stream.  Calls of sf_contract_vertices do not touch this array.
//
// Summation order: entry z belongs to CTA z / 4096, thread (z % 4096) % 256, in ascending z per thread; the 256 threads of
// a CTA by a shared-memory tree; the CTAs' partial sums by the CTA that finishes last (integer ticket -- which CTA that is
// does not matter, what it adds does not depend on it): thread t adds slots t, t + 256, ... in ascending order, then the same
// tree.  Fixed for a given n, so the result is bitwise reproducible; it differs from sf_contract_vertices (another grid,
// another order) by rounding only.
#include <mutex>

#include "sf_internal.h"

#define KN_THREADS 256
#define KN_PER_THREAD 16
#define KN_CHUNK (KN_THREADS * KN_PER_THREAD)          /* 4096 entries per CTA                                      */
#define KN_MAX_PARTIALS 8192                           /* slots of the static scratch = largest grid                */
#define KN_MAX_N ((long)KN_MAX_PARTIALS * KN_CHUNK)    /* 33 554 432 entries                                        */
#define KN_TICKET_DOUBLES 32                           /* the ticket has a 256-byte line of its own after the slots */
#define KN_MAX_DEVICES 64

// [0, KN_MAX_PARTIALS): per-CTA partial sums; then 256 bytes whose first word is the ticket
static __device__ __align__(256) double g_kn_scratch[KN_MAX_PARTIALS + KN_TICKET_DOUBLES];

// sum of v over the CTA in a fixed tree order; the value is returned to every thread
__device__ __forceinline__ double kn_block_sum(double v, double* sh)
{
    const int tid = threadIdx.x;
    sh[tid] = v;
    __syncthreads();
    for (int s = KN_THREADS / 2; s > 0; s >>= 1) {
        if (tid < s) sh[tid] += sh[tid + s];
        __syncthreads();
    }
    v = sh[0];
    __syncthreads();                                    // sh may be reused by the caller
    return v;
}

// One CTA per KN_CHUNK consecutive entries (no grid-stride loop: the number of partial sums is the number of chunks, which
// is what the fixed scratch bounds).  scratch = DEVICE address of g_kn_scratch, passed in by the host (it could be named
// directly here; passing it keeps the kernel usable with any buffer of that layout).
__global__ void __launch_bounds__(KN_THREADS) k_ke_dot_noalloc(const double* __restrict__ a, const double* __restrict__ b, long n,
                                                               double* __restrict__ scratch, double* __restrict__ result)
{
    __shared__ double sh[KN_THREADS];
    __shared__ bool last;
    double* partial = scratch;
    unsigned* ticket = reinterpret_cast<unsigned*>(scratch + KN_MAX_PARTIALS);
    const long base = (long)blockIdx.x * KN_CHUNK + threadIdx.x;
    double s = 0.0;
    if (base - threadIdx.x + KN_CHUNK <= n) {           // a full chunk: sixteen independent loads of a and of b in flight
        double av[KN_PER_THREAD], bv[KN_PER_THREAD];
#pragma unroll
        for (int k = 0; k < KN_PER_THREAD; ++k) {
            av[k] = __ldg(a + base + (long)k * KN_THREADS);
            bv[k] = __ldg(b + base + (long)k * KN_THREADS);
        }
#pragma unroll
        for (int k = 0; k < KN_PER_THREAD; ++k) s = fma(av[k], bv[k], s);
    } else {                                            // the ragged last chunk (or n = 0: nothing to add)
        for (int k = 0; k < KN_PER_THREAD; ++k) {
            const long z = base + (long)k * KN_THREADS;
            if (z < n) s = fma(a[z], b[z], s);
        }
    }
    s = kn_block_sum(s, sh);
    if (threadIdx.x == 0) {
        partial[blockIdx.x] = s;
        __threadfence();
        last = atomicAdd(ticket, 1u) == gridDim.x - 1;
    }
    __syncthreads();
    if (!last) return;
    __threadfence();
    double t = 0.0;
    for (unsigned c = threadIdx.x; c < gridDim.x; c += KN_THREADS) t += __ldcg(partial + c);
    t = kn_block_sum(t, sh);
    if (threadIdx.x == 0) result[0] = t;
}

// Device address of g_kn_scratch on the CURRENT device, asked for once per device (see the header of this file).
static std::mutex g_kn_mutex;
static double* g_kn_addr[KN_MAX_DEVICES];               // zero-initialised: not yet asked for

static int kn_scratch_for_current_device(double** out)
{
    int dev = -1;
    SF_CUDA_OK(cudaGetDevice(&dev));
    if (dev < 0 || dev >= KN_MAX_DEVICES) return SF_ELIMIT;
    std::lock_guard<std::mutex> lock(g_kn_mutex);
    if (!g_kn_addr[dev]) {
        double* p = nullptr;
        if (cudaGetSymbolAddress((void**)&p, g_kn_scratch) != cudaSuccess || !p) {
            cudaGetLastError();
            return SF_ECUDA;
        }
        g_kn_addr[dev] = p;
    }
    *out = g_kn_addr[dev];
    return SF_OK;
}

extern "C" long sf_contract_noalloc_max_n(void) { return KN_MAX_N; }

extern "C" int sf_contract_vertices_noalloc(const double* a, const double* b, long n, double* result, sf_stream_t stream)
{
    if (!a || !b || !result || n < 0) return SF_EARG;
    if (n > KN_MAX_N) return SF_ELIMIT;                  // more chunks than the static scratch has slots
    cudaStream_t st = (cudaStream_t)stream;
    double* scratch = nullptr;
    const int rc = kn_scratch_for_current_device(&scratch);
    if (rc != SF_OK) return rc;
    // the array keeps the previous call's contents: the ticket has to start at zero (the slots are written before they are read)
    SF_CUDA_OK(cudaMemsetAsync(scratch + KN_MAX_PARTIALS, 0, sizeof(double) * KN_TICKET_DOUBLES, st));
    const unsigned grid = n == 0 ? 1u : (unsigned)((n + KN_CHUNK - 1) / KN_CHUNK);
    k_ke_dot_noalloc<<<grid, KN_THREADS, 0, st>>>(a, b, n, scratch, result);
    return cudaGetLastError() == cudaSuccess ? SF_OK : SF_ECUDA;
}
