// sf_api.cu -- the C ABI of libsfoam (include/sfoam.h): context, scratch memory, and the vertex entry points that
// string the steps of the vertex-tensor algorithm together.
#include <stdio.h>
#include <stdlib.h>
#include <string.h>

#include "sf_internal.h"

#define SF_NSCRATCH 40
enum { SLOT_ACC = 0, SLOT_BUF0 = 1, SLOT_BUF1 = 2, SLOT_S = 3 /*..7*/, SLOT_KR = 8 /*..11*/, SLOT_HB = 12 /*..15*/,
       SLOT_HOUT = 16, SLOT_PART = 17, SLOT_MISC = 18 };

struct SfContext {
    bool init = false;
    double gamma = 0.0;
    void* scratch[SF_NSCRATCH] = {};
    size_t scratch_bytes[SF_NSCRATCH] = {};
    long launches = 0;
    int path = 0;          // sf_set_path: 0 automatic, 1 staged, 3 line, 4 factorised
    int last_path = 0;
    bool timing = false;
    bool counting = false;
    bool poison = false;
    cudaEvent_t ev[4] = {};
    double stage_ms[3] = {};
};
static SfContext g_ctx;

void sf_count_launch(int n) { g_ctx.launches += n; }

void* sf_scratch(int slot, size_t bytes)
{
    if (slot < 0 || slot >= SF_NSCRATCH) return nullptr;
    if (bytes == 0) bytes = 8;
    if (g_ctx.scratch_bytes[slot] >= bytes) return g_ctx.scratch[slot];
    if (g_ctx.scratch[slot]) {
        cudaDeviceSynchronize();   // the old block may still be in use on a stream
        cudaFree(g_ctx.scratch[slot]);
        g_ctx.scratch[slot] = nullptr;
        g_ctx.scratch_bytes[slot] = 0;
    }
    void* p = nullptr;
    if (cudaMalloc(&p, bytes) != cudaSuccess) {
        cudaGetLastError();
        return nullptr;
    }
    g_ctx.scratch[slot] = p;
    g_ctx.scratch_bytes[slot] = bytes;
    return p;
}

bool sf_timing_on(void) { return g_ctx.timing; }
bool sf_counting_on(void) { return g_ctx.counting; }
bool sf_poison_on(void) { return g_ctx.poison; }

void sf_timing_mark(int idx, cudaStream_t st)
{
    if (g_ctx.timing && idx >= 0 && idx < 4) cudaEventRecord(g_ctx.ev[idx], st);
}

extern "C" int sf_init(double gamma)
{
    if (g_ctx.init) {
        g_ctx.gamma = gamma;
        return SF_OK;
    }
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev == 0) {
        cudaGetLastError();
        return SF_ECUDA;   // no CPU fallback
    }
    int rc = sf_sixj_module_init();
    if (rc != SF_OK) return rc;
    for (int q = 0; q < 4; ++q)
        if (cudaEventCreate(&g_ctx.ev[q]) != cudaSuccess) return SF_ECUDA;
    g_ctx.gamma = gamma;
    g_ctx.init = true;
    g_ctx.launches = 0;
    return SF_OK;
}

extern "C" int sf_finalize(void)
{
    if (!g_ctx.init) return SF_OK;
    cudaDeviceSynchronize();
    for (int s = 0; s < SF_NSCRATCH; ++s) {
        if (g_ctx.scratch[s]) cudaFree(g_ctx.scratch[s]);
        g_ctx.scratch[s] = nullptr;
        g_ctx.scratch_bytes[s] = 0;
    }
    sf_sixj_module_free();
    for (int q = 0; q < 4; ++q) cudaEventDestroy(g_ctx.ev[q]);
    g_ctx.init = false;
    return SF_OK;
}

extern "C" double sf_gamma(void) { return g_ctx.gamma; }

extern "C" const char* sf_strerror(int status)
{
    switch (status) {
        case SF_OK: return "ok";
        case SF_ENOTINIT: return "sf_init has not been called";
        case SF_EARG: return "invalid argument";
        case SF_ESPIN: return "a boundary node has an odd spin sum or an empty intertwiner range";
        case SF_ETABLE: return "6j table absent or too small";
        case SF_ENOMEM: return "out of memory";
        case SF_ECUDA: return "CUDA error (no device or launch failure)";
        default: return "unknown status";
    }
}

extern "C" int sf_sixj_table(int two_jmax)
{
    if (!g_ctx.init) return SF_ENOTINIT;
    return sf_sixj_table_build(two_jmax, 0);
}

extern "C" long sf_launch_count(int reset)
{
    long n = g_ctx.launches;
    if (reset) g_ctx.launches = 0;
    return n;
}

extern "C" int sf_set_timing(int on)
{
    g_ctx.timing = on != 0;
    return SF_OK;
}
extern "C" int sf_set_counting(int on)
{
    g_ctx.counting = on != 0;
    return SF_OK;
}
extern "C" int sf_set_debug_poison(int on)
{
    g_ctx.poison = on != 0;
    return SF_OK;
}
extern "C" int sf_last_stage_ms(double ms[3])
{
    if (!ms) return SF_EARG;
    memcpy(ms, g_ctx.stage_ms, sizeof g_ctx.stage_ms);
    return SF_OK;
}
// 0 = automatic (factorised, else line, else staged), 1 = staged, 3 = line, 4 = factorised (include/sfoam.h)
extern "C" int sf_set_path(int path)
{
    if (path < 0 || path > 4 || path == 2) return SF_EARG;
    g_ctx.path = path;
    return SF_OK;
}
extern "C" int sf_last_path(void) { return g_ctx.last_path; }

// ranges of the virtual intertwiners k_a for every booster triple (step 2): the node's recoupling
// pairs with the edge's three virtual spins at l = j + offset (superscript order of PAPER.md:171)
__global__ void k_kranges(SfProblem P, int nt, SfKRange* __restrict__ out)
{
    const int q = blockIdx.x * blockDim.x + threadIdx.x;
    if (q >= 4 * nt) return;
    const int e = q / nt, t = q % nt, nl = P.nl;
    const int u = 2 * (t / (nl * nl)), v = 2 * ((t / nl) % nl), w = 2 * (t % nl);
    const int* j = P.two_j;
    int a, b, c, d;
    if (e == 0) {          // node 2 (l23 l24 | l25 j12), triple (l23 l24 l25)
        a = j[J23] + u; b = j[J24] + v; c = j[J25] + w; d = j[J12];
    } else if (e == 1) {   // node 3 (l34 l35 | j13 l23), triple (l34 l35 l23)
        a = j[J34] + u; b = j[J35] + v; c = j[J13]; d = j[J23] + w;
    } else if (e == 2) {   // node 4 (l45 j14 | l24 l34), triple (l45 l24 l34)
        a = j[J45] + u; b = j[J14]; c = j[J24] + v; d = j[J34] + w;
    } else {               // node 5 (j15 l25 | l35 l45), triple (l25 l35 l45)
        a = j[J15]; b = j[J25] + u; c = j[J35] + v; d = j[J45] + w;
    }
    const int lo = max(abs(a - b), abs(c - d)), hi = min(a + b, c + d);
    SfKRange r;
    r.two_k_min = lo;
    r.n_k = (((a + b) ^ (c + d)) & 1) || hi < lo ? 0 : (hi - lo) / 2 + 1;
    out[q] = r;
}

// steps 1-2 on the device side: the problem descriptor and the per-triple k-range tables (no host->device copy)
static int setup_problem(const SfDims& D, const sf_boosters* boosters, SfProblem& P, cudaStream_t st,
                         const int* b_rows = nullptr, const int* b_first = nullptr)
{
    memset(&P, 0, sizeof P);
    memcpy(P.two_j, D.two_j, sizeof P.two_j);
    P.nl = D.nl;
    memcpy(P.two_i_min, D.two_i_min, sizeof P.two_i_min);
    memcpy(P.n_i, D.n_i, sizeof P.n_i);
    memcpy(P.two_k_base, D.two_k_base, sizeof P.two_k_base);
    memcpy(P.n_k_pad, D.n_k_pad, sizeof P.n_k_pad);
    memcpy(P.k_max, D.k_max, sizeof P.k_max);
    P.two_x_base = D.two_x_base;
    P.n_x_pad = D.n_x_pad;
    for (int e = 0; e < 4; ++e) {
        P.B[e] = boosters ? boosters->B[e] : nullptr;
        P.b_n[e] = b_rows ? b_rows[e] : D.n_i[e + 1];
        P.b_i0[e] = b_first ? b_first[e] : 0;
    }
    const int nt = D.nl * D.nl * D.nl;
    SfKRange* d = (SfKRange*)sf_scratch(SLOT_KR, sizeof(SfKRange) * nt * 4);
    if (!d) return SF_ENOMEM;
    for (int e = 0; e < 4; ++e) P.kr[e] = d + (long)e * nt;
    k_kranges<<<(4 * nt + 127) / 128, 128, 0, st>>>(P, nt, d);
    sf_count_launch(1);
    return SF_OK;
}

static int vertex_range(const int two_j[10], int two_dl, const sf_boosters* boosters, long shell_lo, long shell_hi,
                        double* out, cudaStream_t st, bool full, const int* i_first = nullptr, const int* i_count = nullptr)
{
    if (!g_ctx.init) return SF_ENOTINIT;
    if (!two_j || !boosters || !out) return SF_EARG;
    for (int e = 0; e < 4; ++e)
        if (!boosters->B[e]) return SF_EARG;
    SfDims D;
    int rc = sf_host_dims(two_j, two_dl, &D);
    if (rc != SF_OK) return rc;
    if (full) {
        shell_lo = 0;
        shell_hi = D.n_shells;
    }
    // a restricted range of boundary intertwiners: the same problem with shifted range minima; only
    // the rows taken from the caller's boosters keep the full layout
    int b_rows[4], b_first[4];
    for (int e = 0; e < 4; ++e) {
        b_rows[e] = D.n_i[e + 1];
        b_first[e] = 0;
    }
    if (i_first && i_count) {
        long n_out = 1;
        for (int n = 0; n < 5; ++n) {
            if (i_first[n] < 0 || i_count[n] < 1 || i_first[n] + i_count[n] > D.n_i[n]) return SF_EARG;
            n_out *= i_count[n];
        }
        for (int n = 0; n < 5; ++n) {
            if (n > 0) b_first[n - 1] = i_first[n];
            D.two_i_min[n] += 2 * i_first[n];
            D.n_i[n] = i_count[n];
        }
        D.n_out = n_out;
    }
    if (shell_lo < 0 || shell_hi > D.n_shells || shell_lo > shell_hi) return SF_EARG;
    // every label of the {6j} of eq. (5) is a spin l <= j + Delta_l or a recoupling of two of them (k, x <= 2 (j + Delta_l)):
    // the largest one must stay inside the validated accuracy envelope of the {6j} evaluation
    {
        int m = 0;
        for (int s = 0; s < 10; ++s) m = two_j[s] > m ? two_j[s] : m;
        if (2 * (m + two_dl) > SF_SIXJ_MAX_TWO_J) return SF_EARG;
    }

    SfProblem P;
    rc = setup_problem(D, boosters, P, st, b_rows, b_first);
    if (rc != SF_OK) return rc;

    // step 4: the five S arrays
    SfSliceSizes sz;
    sf_slice_sizes(D, &sz);
    double* S[5];
    for (int w = 0; w < 5; ++w) {
        S[w] = (double*)sf_scratch(SLOT_S + w, sizeof(double) * sz.n[w]);
        if (!S[w]) return SF_ENOMEM;
        P.S[w] = S[w];
    }
    sf_timing_mark(0, st);
    rc = sf_build_slices(D, S, sf_sixj_table_get(), st);
    if (rc != SF_OK) return rc;
    sf_timing_mark(1, st);

    // steps 5-7
    const bool line_ok = sf_vertex_line_supported(D), factor_ok = sf_vertex_factor_supported(D);
    if ((g_ctx.path == 3 && !line_ok) || (g_ctx.path == 4 && !factor_ok)) return SF_EARG;
    // automatic: the fastest path that holds the problem; a path that runs out of device memory hands over to the next
    int path = g_ctx.path ? g_ctx.path : factor_ok ? 4 : line_ok ? 3 : 1;
    for (;;) {
        g_ctx.last_path = path;
        rc = path == 4   ? sf_vertex_factor(D, P, shell_lo, shell_hi, out, st)
             : path == 3 ? sf_vertex_line(D, P, shell_lo, shell_hi, out, st)
                         : sf_vertex_staged(D, P, shell_lo, shell_hi, out, st);
        if (rc != SF_ENOMEM || g_ctx.path != 0 || path == 1) break;
        path = (path == 4 && line_ok) ? 3 : 1;
    }
    if (rc != SF_OK) return rc;
    sf_timing_mark(3, st);
    if (g_ctx.timing) {
        SF_CUDA_OK(cudaEventSynchronize(g_ctx.ev[3]));
        float a = 0, b = 0, c = 0;
        cudaEventElapsedTime(&a, g_ctx.ev[0], g_ctx.ev[1]);
        cudaEventElapsedTime(&b, g_ctx.ev[1], g_ctx.ev[2]);
        cudaEventElapsedTime(&c, g_ctx.ev[2], g_ctx.ev[3]);
        g_ctx.stage_ms[0] = a;
        g_ctx.stage_ms[1] = b;
        g_ctx.stage_ms[2] = c;
    }
    return SF_OK;
}

extern "C" int sf_vertex_amplitude(const int two_j[10], int two_dl, const sf_boosters* boosters, double* out,
                                   sf_stream_t stream)
{
    return vertex_range(two_j, two_dl, boosters, 0, 0, out, (cudaStream_t)stream, true);
}

extern "C" int sf_vertex_amplitude_range(const int two_j[10], int two_dl, const sf_boosters* boosters, long shell_lo,
                                         long shell_hi, double* out, sf_stream_t stream)
{
    return vertex_range(two_j, two_dl, boosters, shell_lo, shell_hi, out, (cudaStream_t)stream, false);
}

extern "C" int sf_vertex_amplitude_intertwiners(const int two_j[10], int two_dl, const sf_boosters* boosters,
                                                const int i_first[5], const int i_count[5], double* out, sf_stream_t stream)
{
    if (!i_first || !i_count) return SF_EARG;
    return vertex_range(two_j, two_dl, boosters, 0, 0, out, (cudaStream_t)stream, true, i_first, i_count);
}

int sf_vertex_single(const int two_j[10], int two_dl, const sf_boosters* boosters, double* out, cudaStream_t st)
{
    return vertex_range(two_j, two_dl, boosters, 0, 0, out, st, true);
}

int sf_vertex_batch_run(int n, const int* two_j, const int* two_dl, const sf_boosters* boosters, double* const* out,
                        cudaStream_t st);   // sf_vertex_batch.cu

extern "C" int sf_vertex_amplitude_batch(int n, const int* two_j, const int* two_dl, const sf_boosters* boosters,
                                         double* const* out, sf_stream_t stream)
{
    if (!g_ctx.init) return SF_ENOTINIT;
    if (n < 0 || (n > 0 && (!two_j || !two_dl || !boosters || !out))) return SF_EARG;
    if (n == 0) return SF_OK;
    return sf_vertex_batch_run(n, two_j, two_dl, boosters, out, (cudaStream_t)stream);
}

extern "C" int sf_vertex_amplitude_host(const int two_j[10], int two_dl, const double* const host_boosters[4],
                                        double* host_out, sf_stream_t stream)
{
    if (!g_ctx.init) return SF_ENOTINIT;
    if (!two_j || !host_boosters || !host_out) return SF_EARG;
    cudaStream_t st = (cudaStream_t)stream;
    SfDims D;
    int rc = sf_host_dims(two_j, two_dl, &D);
    if (rc != SF_OK) return rc;
    const long nt = (long)D.nl * D.nl * D.nl;
    sf_boosters b;
    for (int e = 0; e < 4; ++e) {
        if (!host_boosters[e]) return SF_EARG;
        const size_t bytes = sizeof(double) * nt * D.n_i[e + 1] * D.n_k_pad[e];
        double* d = (double*)sf_scratch(SLOT_HB + e, bytes);
        if (!d) return SF_ENOMEM;
        SF_CUDA_OK(cudaMemcpyAsync(d, host_boosters[e], bytes, cudaMemcpyHostToDevice, st));
        b.B[e] = d;
    }
    double* dout = (double*)sf_scratch(SLOT_HOUT, sizeof(double) * D.n_out);
    if (!dout) return SF_ENOMEM;
    rc = vertex_range(two_j, two_dl, &b, 0, 0, dout, st, true);
    if (rc != SF_OK) return rc;
    SF_CUDA_OK(cudaMemcpyAsync(host_out, dout, sizeof(double) * D.n_out, cudaMemcpyDeviceToHost, st));
    SF_CUDA_OK(cudaStreamSynchronize(st));
    return SF_OK;
}

void sf_launch_count_terms(const SfProblem& P, long shell_lo, long shell_hi, unsigned long long* total, cudaStream_t st);

extern "C" int sf_vertex_terms(const int two_j[10], int two_dl, long shell_lo, long shell_hi, double* n_terms)
{
    if (!g_ctx.init) return SF_ENOTINIT;
    if (!two_j || !n_terms) return SF_EARG;
    SfDims D;
    int rc = sf_host_dims(two_j, two_dl, &D);
    if (rc != SF_OK) return rc;
    if (shell_lo < 0 || shell_hi > D.n_shells || shell_lo > shell_hi) return SF_EARG;
    SfProblem P;
    rc = setup_problem(D, nullptr, P, 0);
    if (rc != SF_OK) return rc;
    unsigned long long* d = (unsigned long long*)sf_scratch(SLOT_MISC, 256);
    if (!d) return SF_ENOMEM;
    SF_CUDA_OK(cudaMemsetAsync(d, 0, sizeof(unsigned long long), 0));
    if (shell_hi > shell_lo) {
        sf_launch_count_terms(P, shell_lo, shell_hi, d, 0);
        sf_count_launch(1);
    }
    unsigned long long h = 0;
    SF_CUDA_OK(cudaMemcpy(&h, d, sizeof h, cudaMemcpyDeviceToHost));
    *n_terms = (double)h;
    return SF_OK;
}
