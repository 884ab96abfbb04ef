// sf_sixj.cu -- kernel (a): the {6j} table builder and the batch evaluation hooks.
// The paper precomputes its 3j/6j tables; here the table is built on the device, one slot
// per canonical tuple under the 24 tetrahedral symmetries (layout in sf_sixj.cuh).
#include <stdio.h>
#include <stdlib.h>

#include <vector>

#include "sf_sixj.cuh"

static SfFact* g_fact_dev = nullptr;
static double* g_tab_values = nullptr;
static long* g_tab_base4 = nullptr;
static long g_tab_slots = 0;
static int g_tab_two_jmax = -1;

const SfFact* sf_fact_table(void) { return g_fact_dev; }

int sf_sixj_module_init(void)
{
    if (g_fact_dev) return SF_OK;
    // n! as a double-double significand with a separate exponent; the factor n is exact, so each step costs one
    // dd*double rounding (~2^-104): 2047 steps stay below 2^-92 relative.
    std::vector<SfFact> F(SF_NFACT);
    dd_t m = dd_make(0.5, 0.0);
    int e = 1;
    for (int n = 0; n < SF_NFACT; ++n) {
        if (n > 0) {
            m = dd_mul_d(m, (double)n);
            int sh;
            double h = frexp(m.hi, &sh);
            m = dd_make(h, ldexp(m.lo, -sh));
            e += sh;
        }
        F[n].hi = m.hi;
        F[n].lo = m.lo;
        F[n].e = e;
        F[n].pad = 0;
    }
    SF_CUDA_OK(cudaMalloc(&g_fact_dev, sizeof(SfFact) * SF_NFACT));
    SF_CUDA_OK(cudaMemcpy(g_fact_dev, F.data(), sizeof(SfFact) * SF_NFACT, cudaMemcpyHostToDevice));
    return SF_OK;
}

static void table_free(void)
{
    if (g_tab_values) cudaFree(g_tab_values);
    if (g_tab_base4) cudaFree(g_tab_base4);
    g_tab_values = nullptr;
    g_tab_base4 = nullptr;
    g_tab_slots = 0;
    g_tab_two_jmax = -1;
}

void sf_sixj_module_free(void)
{
    table_free();
    if (g_fact_dev) cudaFree(g_fact_dev);
    g_fact_dev = nullptr;
}

SfSixjTable sf_sixj_table_get(void)
{
    SfSixjTable t;
    t.two_jmax = g_tab_two_jmax;
    t.n_slots = g_tab_slots;
    t.values = g_tab_values;
    t.base4 = g_tab_base4;
    return t;
}

// ---------------------------------------------------------------------------------------------------------
// table builder
// ---------------------------------------------------------------------------------------------------------
// rectangular enumeration of the (a, b, ci, ei) groups; returns false for combinations outside the canonical set
__device__ __forceinline__ bool group_decode(long r, int J, int& a, int& b, int& c, int& e)
{
    const int NC = J / 2 + 1, NE = J + 1;
    int ei = (int)(r % NE);
    r /= NE;
    int ci = (int)(r % NC);
    r /= NC;
    b = (int)(r % (J + 1));
    a = (int)(r / (J + 1));
    if (b > a) return false;
    c = a - b + 2 * ci;
    e = a - b + ei;
    return c <= b && e <= b;
}

__global__ void k_sixj_count(int J, long n_rect, long* __restrict__ counts)
{
    long r = blockIdx.x * (long)blockDim.x + threadIdx.x;
    if (r >= n_rect) return;
    int a, b, c, e;
    if (!group_decode(r, J, a, b, c, e)) return;
    long n = 0;
    int dlo;
    for (int f = a - e; f <= b; f += 2) n += sf_sixj_nd(a, b, c, e, f, &dlo);
    counts[sf_sixj_group(J, a, b, c, e)] = n;
}

// one warp per group: f sequential, lanes over d
__global__ void __launch_bounds__(128) k_sixj_fill(int J, long n_rect, const long* __restrict__ base4,
                                                   const SfFact* __restrict__ F, double* __restrict__ values)
{
    const long r = blockIdx.x * (long)(blockDim.x >> 5) + (threadIdx.x >> 5);
    const int lane = threadIdx.x & 31;
    if (r >= n_rect) return;
    int a, b, c, e;
    if (!group_decode(r, J, a, b, c, e)) return;
    long s = base4[sf_sixj_group(J, a, b, c, e)];
    for (int f = a - e; f <= b; f += 2) {
        int dlo;
        const int nd = sf_sixj_nd(a, b, c, e, f, &dlo);
        for (int q = lane; q < nd; q += 32) values[s + q] = sf_sixj_eval(F, a, b, c, dlo + 2 * q, e, f);
        s += nd;
    }
}

int sf_sixj_table_build(int two_jmax, cudaStream_t st)
{
    table_free();
    if (two_jmax < 0) return SF_OK;
    if (two_jmax > 100) return SF_EARG;
    if (!g_fact_dev) return SF_ENOTINIT;
    const int J = two_jmax;
    const long NC = J / 2 + 1, NE = J + 1;
    const long n_groups = (long)(J + 1) * (J + 2) / 2 * NC * NE;
    const long n_rect = (long)(J + 1) * (J + 1) * NC * NE;
    long* counts = nullptr;
    if (cudaMalloc(&counts, sizeof(long) * n_groups) != cudaSuccess) return SF_ENOMEM;
    cudaMemsetAsync(counts, 0, sizeof(long) * n_groups, st);
    k_sixj_count<<<(unsigned)((n_rect + 255) / 256), 256, 0, st>>>(J, n_rect, counts);
    sf_count_launch(1);
    std::vector<long> h(n_groups);
    if (cudaMemcpyAsync(h.data(), counts, sizeof(long) * n_groups, cudaMemcpyDeviceToHost, st) != cudaSuccess ||
        cudaStreamSynchronize(st) != cudaSuccess) {
        cudaFree(counts);
        return SF_ECUDA;
    }
    long total = 0;
    for (long g = 0; g < n_groups; ++g) {   // exclusive prefix sum
        long n = h[g];
        h[g] = total;
        total += n;
    }
    g_tab_base4 = counts;
    if (cudaMemcpyAsync(g_tab_base4, h.data(), sizeof(long) * n_groups, cudaMemcpyHostToDevice, st) != cudaSuccess) {
        table_free();
        return SF_ECUDA;
    }
    if (cudaMalloc(&g_tab_values, sizeof(double) * (total > 0 ? total : 1)) != cudaSuccess) {
        table_free();
        return SF_ENOMEM;
    }
    k_sixj_fill<<<(unsigned)((n_rect + 3) / 4), 128, 0, st>>>(J, n_rect, g_tab_base4, g_fact_dev, g_tab_values);
    sf_count_launch(1);
    if (cudaStreamSynchronize(st) != cudaSuccess) {   // h must outlive the upload
        table_free();
        return SF_ECUDA;
    }
    g_tab_slots = total;
    g_tab_two_jmax = J;
    return SF_OK;
}

// ---------------------------------------------------------------------------------------------------------
// batch evaluation (test hooks of the C ABI)
// ---------------------------------------------------------------------------------------------------------
__global__ void k_sixj_batch(const int* __restrict__ args, long n, int mode, SfSixjTable tab, const SfFact* __restrict__ F,
                             double* __restrict__ out)
{
    long q = blockIdx.x * (long)blockDim.x + threadIdx.x;
    if (q >= n) return;
    const int* p = args + 6 * q;
    out[q] = mode ? sf_sixj_lookup(tab, p[0], p[1], p[2], p[3], p[4], p[5])
                  : sf_sixj_eval(F, p[0], p[1], p[2], p[3], p[4], p[5]);
}

extern "C" int sf_sixj_batch(const int* two_j6, long n, int mode, double* host_out)
{
    if (!two_j6 || !host_out || n < 0 || (mode != 0 && mode != 1)) return SF_EARG;
    if (!g_fact_dev) return SF_ENOTINIT;
    if (n == 0) return SF_OK;
    int jmax = 0;
    for (long q = 0; q < 6 * n; ++q) {
        if (two_j6[q] < 0) return SF_EARG;
        if (two_j6[q] > jmax) jmax = two_j6[q];
    }
    SfCallGuard guard(0);                                        // reads the table another thread's sf_sixj_table may replace
    if (mode == 1 && (g_tab_two_jmax < 0 || jmax > g_tab_two_jmax)) return SF_ETABLE;
    if (mode == 0 && jmax > SF_SIXJ_MAX_TWO_J) return SF_EARG;   // beyond the validated accuracy envelope (sf_internal.h)
    int* dargs = nullptr;
    double* dout = nullptr;
    if (cudaMalloc(&dargs, sizeof(int) * 6 * n) != cudaSuccess) return SF_ENOMEM;
    if (cudaMalloc(&dout, sizeof(double) * n) != cudaSuccess) {
        cudaFree(dargs);
        return SF_ENOMEM;
    }
    int rc = SF_OK;
    if (cudaMemcpy(dargs, two_j6, sizeof(int) * 6 * n, cudaMemcpyHostToDevice) != cudaSuccess) rc = SF_ECUDA;
    if (rc == SF_OK) {
        k_sixj_batch<<<(unsigned)((n + 127) / 128), 128>>>(dargs, n, mode, sf_sixj_table_get(), g_fact_dev, dout);
        sf_count_launch(1);
        if (cudaMemcpy(host_out, dout, sizeof(double) * n, cudaMemcpyDeviceToHost) != cudaSuccess) rc = SF_ECUDA;
    }
    cudaFree(dargs);
    cudaFree(dout);
    return rc;
}

extern "C" int sf_sixj_get(const int two_j6[6], double* host_out) { return sf_sixj_batch(two_j6, 1, 0, host_out); }
extern "C" long sf_sixj_table_slots(void) { return g_tab_slots; }
extern "C" int sf_sixj_table_two_jmax(void) { return g_tab_two_jmax; }
