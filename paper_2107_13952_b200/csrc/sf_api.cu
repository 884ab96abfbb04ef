// sf_api.cu -- the C ABI of libsfoam (include/sfoam.h): context, scratch memory, and the vertex entry points that
// string the steps of the vertex-tensor algorithm together.
#include <stdio.h>
#include <stdlib.h>
#include <string.h>

#include <mutex>

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
    long replays = 0;      // vertex calls answered by a recorded launch sequence (sf_graph_replays)
    int path = 0;          // sf_set_path: 0 automatic, 1 staged, 3 line, 4 factorised
    int last_path = 0;
    bool timing = false;
    bool counting = false;
    bool poison = false;
    cudaEvent_t ev[4] = {};
    double stage_ms[3] = {};
    long epoch = 0;        // contexts created so far (sf_context_epoch): per-device caches of the other files are refilled when it moves
    long gen = 0;          // bumped by everything a recorded launch sequence depends on (scratch blocks, settings, the {6j} table)
    bool capturing = false;
    bool graphs = true;    // sf_set_graphs
    cudaStream_t cap_stream = nullptr;
    cudaEvent_t done = nullptr;     // end of the last compute call (SfCallGuard)
    cudaStream_t last_stream = nullptr;
    bool have_last = false;
};
static SfContext g_ctx;
static std::recursive_mutex g_call_mutex;

SfCallGuard::SfCallGuard(cudaStream_t s) : st(s), events(false)
{
    g_call_mutex.lock();
    if (!g_ctx.init || !g_ctx.done) return;
    cudaStreamCaptureStatus cs = cudaStreamCaptureStatusNone;
    if (cudaStreamIsCapturing(st, &cs) != cudaSuccess || cs != cudaStreamCaptureStatusNone) {
        cudaGetLastError();
        return;                        // (a captured stream never gets here: the entry points refuse it with SF_ECAPTURE)
    }
    events = true;
    if (g_ctx.have_last && g_ctx.last_stream != st) cudaStreamWaitEvent(st, g_ctx.done, 0);   // the scratch buffers are shared
}
SfCallGuard::~SfCallGuard()
{
    if (events) {
        cudaEventRecord(g_ctx.done, st);
        g_ctx.last_stream = st;
        g_ctx.have_last = true;
    }
    g_call_mutex.unlock();
}

// True when `st` is inside a stream capture begun by the CALLER (the library's own recordings run on g_ctx.cap_stream and never
// come through the extern "C" entry points).  Every entry point that uses the context's scratch refuses such a call: the
// scratch blocks may be freed or regrown by a later call, a batch's descriptors are copied from host memory that is gone at
// replay, growing a block calls cudaDeviceSynchronize / cudaFree / cudaMalloc (which invalidate the capture), and the call guard
// orders nothing when the caller's graph replays.  The legacy stream queried while another stream captures in global mode
// (cudaErrorStreamCaptureImplicit) counts as captured; without a context (no sf_init, no device) the answer is no and the
// entry point reports its usual error.
bool sf_stream_is_captured(cudaStream_t st)
{
    if (!g_ctx.init) return false;
    cudaStreamCaptureStatus cs = cudaStreamCaptureStatusNone;
    const cudaError_t e = cudaStreamIsCapturing(st, &cs);
    if (e != cudaSuccess) {
        cudaGetLastError();
        return e == cudaErrorStreamCaptureImplicit;
    }
    return cs != cudaStreamCaptureStatusNone;
}

SfHostLock::SfHostLock() { g_call_mutex.lock(); }
SfHostLock::~SfHostLock() { g_call_mutex.unlock(); }

void sf_bump_generation(void) { ++g_ctx.gen; }
long sf_context_epoch(void) { return g_ctx.epoch; }

void sf_count_launch(int n) { g_ctx.launches += n; }

void* sf_scratch(int slot, size_t bytes)
{
    if (slot < 0 || slot >= SF_NSCRATCH) return nullptr;
    if (bytes == 0) bytes = 8;
    if (g_ctx.scratch_bytes[slot] >= bytes) return g_ctx.scratch[slot];
    if (g_ctx.capturing) return nullptr;   // a launch sequence being recorded must not allocate: the caller falls back to a plain run
    ++g_ctx.gen;                           // recorded launch sequences hold the old pointers
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

// Gives a block back before its size is known to be wrong for what comes next (the pass-size loop of the factorised path).
void sf_scratch_release(int slot)
{
    if (slot < 0 || slot >= SF_NSCRATCH || !g_ctx.scratch[slot] || g_ctx.capturing) return;
    ++g_ctx.gen;
    cudaDeviceSynchronize();
    cudaFree(g_ctx.scratch[slot]);
    g_ctx.scratch[slot] = nullptr;
    g_ctx.scratch_bytes[slot] = 0;
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
    SfHostLock lock;
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
    if (cudaStreamCreateWithFlags(&g_ctx.cap_stream, cudaStreamNonBlocking) != cudaSuccess) return SF_ECUDA;
    if (cudaEventCreateWithFlags(&g_ctx.done, cudaEventDisableTiming) != cudaSuccess) return SF_ECUDA;
    g_ctx.have_last = false;
    g_ctx.gamma = gamma;
    g_ctx.init = true;
    ++g_ctx.epoch;
    g_ctx.launches = 0;
    g_ctx.replays = 0;
    return SF_OK;
}

static void sf_graph_cache_clear(void);

extern "C" int sf_finalize(void)
{
    SfHostLock lock;
    if (!g_ctx.init) return SF_OK;
    cudaDeviceSynchronize();
    for (int s = 0; s < SF_NSCRATCH; ++s) {
        if (g_ctx.scratch[s]) cudaFree(g_ctx.scratch[s]);
        g_ctx.scratch[s] = nullptr;
        g_ctx.scratch_bytes[s] = 0;
    }
    sf_graph_cache_clear();
    sf_vertex_factor_forget();
    sf_sixj_module_free();
    for (int q = 0; q < 4; ++q) cudaEventDestroy(g_ctx.ev[q]);
    if (g_ctx.cap_stream) cudaStreamDestroy(g_ctx.cap_stream);
    g_ctx.cap_stream = nullptr;
    if (g_ctx.done) cudaEventDestroy(g_ctx.done);
    g_ctx.done = nullptr;
    g_ctx.have_last = false;
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
        case SF_ELIMIT: return "input exceeds the fixed built-in scratch of this allocation-free entry point";
        case SF_ECAPTURE: return "the stream is being captured: this entry point uses library-owned scratch and cannot be recorded into a caller's CUDA graph";
        default: return "unknown status";
    }
}

extern "C" int sf_sixj_table(int two_jmax)
{
    if (!g_ctx.init) return SF_ENOTINIT;
    SfCallGuard guard(0);                  // a vertex call in flight on another stream may still be gathering from the old table
    ++g_ctx.gen;
    return sf_sixj_table_build(two_jmax, 0);
}

extern "C" long sf_launch_count(int reset)
{
    long n = g_ctx.launches;
    if (reset) g_ctx.launches = 0;
    return n;
}

extern "C" long sf_graph_replays(int reset)
{
    SfHostLock lock;
    const long n = g_ctx.replays;
    if (reset) g_ctx.replays = 0;
    return n;
}

extern "C" int sf_set_timing(int on)
{
    SfHostLock lock;
    g_ctx.timing = on != 0;
    ++g_ctx.gen;
    return SF_OK;
}
extern "C" int sf_set_counting(int on)
{
    SfHostLock lock;
    g_ctx.counting = on != 0;
    ++g_ctx.gen;
    return SF_OK;
}
extern "C" int sf_set_debug_poison(int on)
{
    SfHostLock lock;
    g_ctx.poison = on != 0;
    ++g_ctx.gen;
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
    SfHostLock lock;
    g_ctx.path = path;
    ++g_ctx.gen;
    return SF_OK;
}
extern "C" int sf_last_path(void) { return g_ctx.last_path; }

// steps 1-2 on the device side: the problem descriptor and the per-triple k-range tables (no host->device copy)
// (launch_kr: fill the k-range tables now; otherwise sf_build_slices does it in its own launch)
static int setup_problem(const SfDims& D, const sf_boosters* boosters, SfProblem& P, cudaStream_t st,
                         const int* b_rows = nullptr, const int* b_first = nullptr, bool launch_kr = true)
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
    if (launch_kr) sf_launch_kranges(D, d, st);
    return SF_OK;
}

static int vertex_range_run(const int two_j[10], int two_dl, const sf_boosters* boosters, long shell_lo, long shell_hi,
                            double* out, cudaStream_t st, bool full, const int* i_first, const int* i_count)
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
    rc = setup_problem(D, boosters, P, st, b_rows, b_first, false);
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
    rc = sf_build_slices(D, S, sf_sixj_table_get(), const_cast<SfKRange*>(P.kr[0]), st);
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

// ---------------------------------------------------------------------------------------------------------------
// Recorded launch sequences.  A vertex call is 15-30 small launches (k-range tables, S arrays, the precomputations and the
// contractions of the factorised path); on small problems their launch latency is the whole cost (config 0: 0.1 ms for
// 3.4e6 flop).  A call that runs without changing the library state (no scratch block had to grow) is remembered; when it
// comes again with the same arguments (spins, Delta_l, ranges, booster and output POINTERS: the booster values are read when
// the kernels run, so they may change) and the same library state, its launches are recorded into a CUDA graph on a private
// stream and replayed; from then on the call is one graph launch on the caller's stream.  In a fresh context that makes the
// first call a plain run that allocates, the second a plain run that is remembered, the third the recording.
// Anything a recording depends on (a scratch block reallocated, a setting changed, the {6j} table rebuilt) bumps the
// generation and drops the recordings.  Measurement modes (timing, counting, poison) never use them.
// ---------------------------------------------------------------------------------------------------------------
struct SfGraphKey {
    int two_j[10], two_dl, full, has_i, i_first[5], i_count[5];
    long shell_lo, shell_hi;
    const void* ptr[5];
    long gen;
};
struct SfGraphEntry {
    bool used = false, no_record = false;
    SfGraphKey key;
    cudaGraphExec_t exec = nullptr;
    long launches = 0;
    int last_path = 0;
};
#define SF_NGRAPH 16
static SfGraphEntry g_graphs[SF_NGRAPH];
static int g_graph_next = 0;

static void sf_graph_cache_clear(void)
{
    for (int e = 0; e < SF_NGRAPH; ++e) {
        if (g_graphs[e].exec) cudaGraphExecDestroy(g_graphs[e].exec);
        g_graphs[e] = SfGraphEntry();
    }
}

/* 1 (default): repeated identical vertex calls replay a recorded launch sequence; 0: every call launches its kernels one by one. */
extern "C" int sf_set_graphs(int on)
{
    SfHostLock lock;
    g_ctx.graphs = on != 0;
    ++g_ctx.gen;
    return SF_OK;
}

static int vertex_range(const int two_j[10], int two_dl, const sf_boosters* boosters, long shell_lo, long shell_hi,
                        double* out, cudaStream_t st, bool full, const int* i_first = nullptr, const int* i_count = nullptr)
{
    if (!g_ctx.init) return SF_ENOTINIT;
    if (!two_j || !boosters || !out) return SF_EARG;
    cudaStreamCaptureStatus cs = cudaStreamCaptureStatusNone;
    if (!g_ctx.graphs || g_ctx.timing || g_ctx.counting || g_ctx.poison || (i_first && !i_count) ||
        cudaStreamIsCapturing(st, &cs) != cudaSuccess || cs != cudaStreamCaptureStatusNone) {
        cudaGetLastError();
        return vertex_range_run(two_j, two_dl, boosters, shell_lo, shell_hi, out, st, full, i_first, i_count);
    }
    SfGraphKey k;
    memset(&k, 0, sizeof k);
    memcpy(k.two_j, two_j, sizeof k.two_j);
    k.two_dl = two_dl;
    k.full = full;
    k.shell_lo = full ? 0 : shell_lo;
    k.shell_hi = full ? 0 : shell_hi;
    if (i_first && i_count) {
        k.has_i = 1;
        memcpy(k.i_first, i_first, sizeof k.i_first);
        memcpy(k.i_count, i_count, sizeof k.i_count);
    }
    for (int e = 0; e < 4; ++e) k.ptr[e] = boosters->B[e];
    k.ptr[4] = out;
    k.gen = g_ctx.gen;
    SfGraphEntry* hit = nullptr;
    for (int e = 0; e < SF_NGRAPH; ++e) {
        SfGraphEntry& g = g_graphs[e];
        if (!g.used) continue;
        if (g.key.gen != g_ctx.gen) {                         // stale: the library state has changed since
            if (g.exec) cudaGraphExecDestroy(g.exec);
            g = SfGraphEntry();
            continue;
        }
        if (!memcmp(&g.key, &k, sizeof k)) hit = &g;
    }
    if (hit && hit->exec) {
        if (cudaGraphLaunch(hit->exec, st) != cudaSuccess) return SF_ECUDA;
        ++g_ctx.replays;
        g_ctx.launches += hit->launches;
        g_ctx.last_path = hit->last_path;
        return SF_OK;
    }
    if (!hit) {                                               // first sight: run it, remember the arguments
        const long gen0 = g_ctx.gen;
        const int rc = vertex_range_run(two_j, two_dl, boosters, shell_lo, shell_hi, out, st, full, i_first, i_count);
        if (rc == SF_OK && gen0 == g_ctx.gen) {               // (a call that had to allocate is remembered at its next repetition)
            SfGraphEntry& g = g_graphs[g_graph_next];
            g_graph_next = (g_graph_next + 1) % SF_NGRAPH;
            if (g.exec) cudaGraphExecDestroy(g.exec);
            g = SfGraphEntry();
            g.used = true;
            memcpy(&g.key, &k, sizeof k);                     // byte copy: the key is compared with memcmp, padding included
        }
        return rc;
    }
    if (hit->no_record) return vertex_range_run(two_j, two_dl, boosters, shell_lo, shell_hi, out, st, full, i_first, i_count);
    // second sight: record the launches on the private stream, then replay them on the caller's
    const long before = g_ctx.launches;
    cudaGraph_t graph = nullptr;
    int rc = SF_ECUDA;
    if (cudaStreamBeginCapture(g_ctx.cap_stream, cudaStreamCaptureModeThreadLocal) == cudaSuccess) {
        g_ctx.capturing = true;
        rc = vertex_range_run(two_j, two_dl, boosters, shell_lo, shell_hi, out, g_ctx.cap_stream, full, i_first, i_count);
        g_ctx.capturing = false;
        if (cudaStreamEndCapture(g_ctx.cap_stream, &graph) != cudaSuccess) rc = SF_ECUDA;
    }
    const long recorded = g_ctx.launches - before;
    g_ctx.launches = before;
    if (rc == SF_OK && graph && cudaGraphInstantiate(&hit->exec, graph, 0) == cudaSuccess) {
        cudaGraphDestroy(graph);
        hit->launches = recorded;
        hit->last_path = g_ctx.last_path;
        if (cudaGraphLaunch(hit->exec, st) != cudaSuccess) return SF_ECUDA;
        ++g_ctx.replays;
        g_ctx.launches += recorded;
        return SF_OK;
    }
    if (graph) cudaGraphDestroy(graph);
    cudaGetLastError();
    hit->exec = nullptr;
    hit->no_record = true;                                    // this call cannot be recorded (it would allocate, or failed): plain runs
    return vertex_range_run(two_j, two_dl, boosters, shell_lo, shell_hi, out, st, full, i_first, i_count);
}

extern "C" int sf_vertex_amplitude(const int two_j[10], int two_dl, const sf_boosters* boosters, double* out,
                                   sf_stream_t stream)
{
    if (sf_stream_is_captured((cudaStream_t)stream)) return SF_ECAPTURE;
    SfCallGuard guard((cudaStream_t)stream);
    return vertex_range(two_j, two_dl, boosters, 0, 0, out, (cudaStream_t)stream, true);
}

extern "C" int sf_vertex_amplitude_range(const int two_j[10], int two_dl, const sf_boosters* boosters, long shell_lo,
                                         long shell_hi, double* out, sf_stream_t stream)
{
    if (sf_stream_is_captured((cudaStream_t)stream)) return SF_ECAPTURE;
    SfCallGuard guard((cudaStream_t)stream);
    return vertex_range(two_j, two_dl, boosters, shell_lo, shell_hi, out, (cudaStream_t)stream, false);
}

extern "C" int sf_vertex_amplitude_intertwiners(const int two_j[10], int two_dl, const sf_boosters* boosters,
                                                const int i_first[5], const int i_count[5], double* out, sf_stream_t stream)
{
    if (!i_first || !i_count) return SF_EARG;
    if (sf_stream_is_captured((cudaStream_t)stream)) return SF_ECAPTURE;
    SfCallGuard guard((cudaStream_t)stream);
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
    if (sf_stream_is_captured((cudaStream_t)stream)) return SF_ECAPTURE;   // (its descriptors are copied from host memory of this call)
    SfCallGuard guard((cudaStream_t)stream);
    return sf_vertex_batch_run(n, two_j, two_dl, boosters, out, (cudaStream_t)stream);
}

extern "C" int sf_vertex_amplitude_host(const int two_j[10], int two_dl, const double* const host_boosters[4],
                                        double* host_out, sf_stream_t stream)
{
    if (!g_ctx.init) return SF_ENOTINIT;
    if (!two_j || !host_boosters || !host_out) return SF_EARG;
    cudaStream_t st = (cudaStream_t)stream;
    if (sf_stream_is_captured(st)) return SF_ECAPTURE;
    SfCallGuard guard(st);
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
    SfCallGuard guard(0);                  // writes the shared k-range tables: ordered after a vertex call still reading them
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
