/* sfoam.h -- C ABI of libsfoam: the EPRL vertex-amplitude tensor of arXiv 2107.13952 on one B200 (sm_100a).
 *
 * What is computed (eq. (3)):
 *
 *   A[i1..i5] = prod_{e=1..5} sqrt(2 i_e+1) *
 *               sum_{shells l_f} sum_{k2..k5} prod_{a=2..5} (2 k_a+1) B_a[t_a(l)][i_a,k_a] * {15j}(l_f; i1,k2..k5)
 *
 * with the {15j} symbol of eq. (5) assembled from five {6j} symbols, the shells
 * j_f <= l_f <= j_f + Delta_l of the six virtual spins (l23 l24 l25 l34 l35 l45), l_1a = j_1a gauge-fixed, and the
 * four booster tensors B_a supplied by the caller (they are inputs: PAPER.md:169-171).  The steps are those of the
 * vertex-tensor algorithm.
 *
 * Conventions
 *   - Every spin is passed as the integer two_j = 2j.  two_dl = 2*Delta_l must be even (virtual spins step by 1).
 *   - Spin order  two_j[10] = (j12 j13 j14 j15 j23 j24 j25 j34 j35 j45)   (Listing 8).
 *   - Node spin orders (first pair | second pair); the node's intertwiner recouples the two pairs:
 *       node 1 (j12 j13 | j14 j15) -> i1        node 2 (j23 j24 | j25 j12) -> i2,k2     node 3 (j34 j35 | j13 j23) -> i3,k3
 *       node 4 (j45 j14 | j24 j34) -> i4,k4     node 5 (j15 j25 | j35 j45) -> i5,k5
 *   - Canonical shell order: lexicographic in the offsets (o23 o24 o25 o34 o35 o45), o = l - j in 0..Delta_l,
 *     o45 fastest (index order of eq. (9)).  shell = ((((o23*n+o24)*n+o25)*n+o34)*n+o35)*n+o45, n = Delta_l+1.
 *   - Booster layout (dense, C row-major, FP64, DEVICE memory):  B_a[t][ii][kk],  a = 2..5,
 *       t  = (u*n+v)*n+w with (u,v,w) the offsets of the edge's virtual spins in the paper's superscript order
 *            (PAPER.md:171): edge 2 (l23 l24 l25), edge 3 (l34 l35 l23), edge 4 (l45 l24 l34), edge 5 (l25 l35 l45);
 *       ii = (two_i - two_i_min_a)/2 in [0,n_i);  kk = (two_k - two_k_base_a)/2 in [0,n_k_pad), sizes from
 *            sf_booster_dims().  Entries outside the triple's valid k-range are ignored (treated as 0).
 *   - Output layout: out[(((a1*n2+a2)*n3+a3)*n4+a4)*n5+a5], a_e = (two_i_e - two_i_min_e)/2: the same bytes as the
 *     paper's column-major A^{i5 i4 i3 i2 i1}.
 *   - The result is bitwise reproducible run to run for identical inputs (fixed-order accumulation, no float atomics).
 *
 * Measurement and debugging entry points (timers, counters, peak probes, memory-budget hooks) are NOT part of this
 * contract: they live in include/sfoam_debug.h.
 *
 * Ownership: the caller owns booster and output buffers; the library owns the {6j} table and its scratch memory
 * (released by sf_finalize).  All functions return SF_OK (0) or a negative sf_status; none throws or aborts; `out` is
 * not written when an error is returned before launch.  There is NO CPU fallback: without a CUDA device every compute
 * entry point returns SF_ECUDA.
 *
 * Concurrency: one context per process, bound to the device that was current at sf_init; the library keeps its scratch
 * buffers and settings in that context.  Compute calls are therefore SERIALISED by the library: host threads by a mutex,
 * streams by an event -- a call on another stream than the previous call's first waits (on the device) for that call, so
 * two vertex calls on different streams are correct but do not overlap.  Calls are asynchronous on the stream they are
 * given.
 *
 * Stream capture: every compute entry point that works in the library's scratch -- the sf_vertex_amplitude* calls and
 * sf_contract_vertices / sf_contract_vectors -- REFUSES a `stream` that the caller is capturing into a CUDA graph and returns
 * SF_ECAPTURE before issuing any CUDA work (the capture stays valid and can be ended normally).  Reasons: the scratch blocks
 * a captured launch would point to are freed or regrown by later calls; growing one synchronises the device and allocates,
 * which invalidates a capture; the batch call copies its descriptors from host memory that is gone when the graph replays;
 * and the serialisation above cannot order a replay against other calls.  For repeated identical calls use the library's own
 * recordings (sf_set_graphs), which track all of that.
 */
#ifndef SFOAM_H
#define SFOAM_H

#ifdef __cplusplus
extern "C" {
#endif

typedef enum {
    SF_OK       = 0,
    SF_ENOTINIT = -1,   /* sf_init has not been called                                                   */
    SF_EARG     = -2,   /* null pointer, negative spin, two_dl negative or odd, bad edge / range           */
    SF_ESPIN    = -3,   /* a boundary node's four spins have an odd sum or an empty intertwiner range      */
    SF_ETABLE   = -4,   /* {6j} table requested but absent / too small                                     */
    SF_ENOMEM   = -5,   /* host or device allocation failed                                                */
    SF_ECUDA    = -6,   /* CUDA runtime error (no device, launch failure)                                  */
    SF_ELIMIT   = -7,   /* input larger than the fixed built-in scratch of an allocation-free entry point  */
    SF_ECAPTURE = -8    /* `stream` is being captured by the caller (see Concurrency)                      */
} sf_status;

/* CUDA stream handle (a cudaStream_t), passed as an opaque pointer so that this header needs no CUDA include. */
typedef void *sf_stream_t;

/* The four booster tensors of step 3: DEVICE pointers, edges 2,3,4,5 in B[0..3]. */
typedef struct {
    const double *B[4];
} sf_boosters;

/* Create the global context on the current CUDA device.  gamma is the Immirzi parameter the paper's cinit() takes
 * (PAPER.md:207-219); with caller-supplied boosters the path does not depend on it (it enters only through B4,
 * PAPER.md:61-65), so it is stored and reported back, nothing else.  Idempotent. */
int sf_init(double gamma);
int sf_finalize(void);
const char *sf_strerror(int status);
double sf_gamma(void);

/* Build (or replace) the device-resident table of all {6j} symbols with every 2j <= two_jmax, one slot per class
 * of the 24 tetrahedral symmetries (the paper precomputes 6j tables: PAPER.md:103, 207).  two_jmax < 0 frees it.
 * While a table is resident, the S arrays of step 4 are gathered from it when every argument fits, and evaluated
 * directly otherwise.  Returns SF_EARG for two_jmax > 100 (table would exceed 24 GB). */
int sf_sixj_table(int two_jmax);
/* Number of slots of the resident table (0 if none), and its two_jmax (-1 if none). */
long sf_sixj_table_slots(void);
int sf_sixj_table_two_jmax(void);

/* Test hooks for {6j} parity.  two_j6 = (a b c d e f) for {a b c; d e f}; HOST pointers.
 * sf_sixj_get evaluates one symbol on the device (direct Racah sum).  sf_sixj_batch evaluates n symbols;
 * mode 0 = direct evaluation, mode 1 = gather from the resident table (SF_ETABLE if absent or an argument exceeds it).
 * Accuracy of the direct evaluation (double-double Racah sum) against the exact value: relative 1e-12 for every label
 * 2j <= 240 -- measured: correctly rounded up to 2j ~ 176, <= 4e-15 up to 220, <= 2.5e-13 up to 244 on the symbols that cancel
 * most (six near-equal large labels); from 248 on, symbols near a zero of the {6j} miss 1e-12.  Arguments above 2j = 240 are
 * therefore refused (SF_EARG), and so is a vertex call whose largest {6j} label 2 * (max two_j + two_dl) exceeds 240: inside
 * that bound every {6j} entering a vertex tensor is good to 1e-12 and the tensor meets 1e-11 * sum|terms|. */
int sf_sixj_get(const int two_j6[6], double *host_out);
int sf_sixj_batch(const int *two_j6, long n, int mode, double *host_out);

/* Pure host integer helpers (step 2): boundary intertwiner ranges of nodes 1..5. */
int sf_vertex_dims(const int two_j[10], int two_i_min[5], int n_i[5]);
/* Booster tensor dims of edge a in 2..5: number of triples (Delta_l+1)^3, n_i, and the padded k layout. */
int sf_booster_dims(const int two_j[10], int two_dl, int edge, int *n_triples, int *n_i, int *two_k_base, int *n_k_pad);
/* Valid k-range of triple t of edge a (n_k = 0 if empty). */
int sf_booster_krange(const int two_j[10], int two_dl, int edge, int t, int *two_k_min, int *n_k);
/* The same for all (Delta_l+1)^3 triples of the edge at once: two_k_min[t], n_k[t]. */
int sf_booster_kranges(const int two_j[10], int two_dl, int edge, int *two_k_min, int *n_k);

/* Algorithmic work of shells [shell_lo, shell_hi) counted on valid ranges only:
 *   *f_con = sum over shells of 2*(n1 K2 K3 K4 K5 n5 + n1 K2 K3 K4 n4 n5 + n1 K2 K3 n3 n4 n5 + n1 K2 n2 n3 n4 n5)
 *   *n_nonempty = shells with all four k-ranges non-empty;  *n_w = sum over shells of n1 K2 K3 K4 K5.
 * Host integer function. */
int sf_vertex_work(const int two_j[10], int two_dl, long shell_lo, long shell_hi,
                   double *f_con, long *n_nonempty, double *n_w);

/* The vertex tensor (steps 4-7).  boosters / out: DEVICE pointers; out holds prod(n_i) doubles and
 * is overwritten.  Asynchronous w.r.t. the host, ordered on `stream`.  Requires sf_init. */
int sf_vertex_amplitude(const int two_j[10], int two_dl, const sf_boosters *boosters, double *out, sf_stream_t stream);
/* Same, restricted to shells [shell_lo, shell_hi) of the canonical order (the full call is [0,(Delta_l+1)^6)).
 * Ranges are additive: the sum of the outputs over a partition of the shells equals the full tensor up to rounding. */
int sf_vertex_amplitude_range(const int two_j[10], int two_dl, const sf_boosters *boosters,
                              long shell_lo, long shell_hi, double *out, sf_stream_t stream);
/* The vertex tensor for a reduced set of boundary intertwiners ("It is also possible to compute the vertex
 * tensor for a reduced set of intertwiner indices"; also the paper's way of splitting a tensor that does not
 * fit into batches over i1): node n = 1..5 keeps the i_count[n-1] values starting at index i_first[n-1] (0-based offset
 * from the range minimum of sf_vertex_dims, steps of 1 in spin).  boosters: the caller's full arrays, unchanged layout.
 * out: DEVICE pointer, prod(i_count) doubles, row-major out[i1][i2][i3][i4][i5] over the kept values, overwritten; equal to
 * the corresponding sub-block of the full tensor.  SF_EARG if a range leaves the node's range or a count is < 1. */
int sf_vertex_amplitude_intertwiners(const int two_j[10], int two_dl, const sf_boosters *boosters,
                                     const int i_first[5], const int i_count[5], double *out, sf_stream_t stream);
/* Many vertex tensors in one call (the paper's stated next step, "many vertex tensors with few shells"; graphs
 * with internal faces need one small tensor per value of the bulk spins).  Problem q = 0..n-1 has the boundary
 * spins two_j[10 q .. 10 q + 9], the shell count two_dl[q], the boosters boosters[q] and the output out[q], each exactly as in
 * sf_vertex_amplitude.  two_j, two_dl, boosters and out are HOST arrays (of spins, of device-pointer quadruples and of device
 * pointers); they may be freed when the call returns.  Every tensor whose {6j} arrays and per-shell intermediates fit one SM's
 * shared memory (small spins, few shells) is computed by ONE kernel launch, one CTA per tensor, everything on chip; larger ones
 * are computed afterwards by the single-tensor path.  Asynchronous on `stream`; bitwise reproducible.  Like every compute
 * call it is serialised with the calls before it (Concurrency above): a batch issued on another stream than the previous
 * call's waits for that call, so batches on different streams are correct but do not overlap.  All arguments are validated
 * before anything is launched: on SF_EARG / SF_ESPIN no output is written. */
int sf_vertex_amplitude_batch(int n, const int *two_j, const int *two_dl, const sf_boosters *boosters,
                              double *const *out, sf_stream_t stream);
/* End-to-end variant with HOST buffers (pinned or pageable): copies the four boosters to the device, computes, copies
 * the tensor back and synchronises `stream`.  host_boosters[e] holds n_triples*n_i*n_k_pad doubles. */
int sf_vertex_amplitude_host(const int two_j[10], int two_dl, const double *const host_boosters[4],
                             double *host_out, sf_stream_t stream);

/* Downstream contractions of vertex tensors (Fig. 3; the paper's contract(...)).  All
 * pointers are DEVICE pointers; asynchronous, ordered on `stream`; fixed summation order (bitwise reproducible).
 *   sf_contract_vertices: result[0] = sum_z a[z] b[z] over the n entries of two vertex tensors of the same shape (all five
 *     edges glued).
 *   sf_contract_vectors: result[0] + i result[1] = sum A[i1][i2][i3][i4][i5] psi[0][i1] psi[1][i2] psi[2][i3] psi[3][i4]
 *     psi[4][i5]; A in the layout of sf_vertex_amplitude with n_i[5] entries per index, psi[e] = n_i[e] complex numbers
 *     stored (re, im) interleaved, no conjugation (coherent-state coefficients in the paper; their computation is out of
 *     scope).
 * SF_EARG on a null pointer, n < 0 or an n_i < 1. */
int sf_contract_vertices(const double *a, const double *b, long n, double *result, sf_stream_t stream);
int sf_contract_vectors(const double *A, const int n_i[5], const double *const psi[5], double *result, sf_stream_t stream);

/* sf_contract_vertices for callers that cannot allocate device memory (Fig. 3: result[0] = sum_z a[z] b[z]).
 * Meant for a program that calls the contraction inside a long loop (a sum or a Monte Carlo walk over bulk spins) while all
 * device memory belongs to an allocator of its own (CUDA.jl's pool, PyTorch's caching allocator, a fixed MIG / MPS slice) --
 * there a cudaMalloc made by this library fails or shrinks that pool -- or that cannot take the device-wide synchronisation
 * cudaMalloc / cudaFree bring with them.  sf_contract_vertices gets its partial-sum buffer from the library's growable
 * scratch; this entry point calls no cudaMalloc, no cudaFree and no other allocating routine, needs no sf_init, and keeps
 * its partial sums in a fixed array built into the library's device code: 65 792 bytes that every GPU running this library
 * holds until the process exits.
 *   Limit: n <= sf_contract_noalloc_max_n() = 33 554 432 entries (one slot of the array per 4096 entries; 32^5, the
 *     paper's largest tensors are 21^5).  Beyond it the call returns SF_ELIMIT and launches nothing.
 *   a, b, result: DEVICE pointers, the caller's (n, n and 1 doubles); asynchronous, ordered on `stream`, on the CURRENT device.
 *   First call on each device: looks up the device address of the built-in array (a one-off query that may make the CUDA
 *     runtime load the library's device code).  Make that first call before any stream capture is begun.
 *   The array is shared by all calls on a device and keeps the previous call's contents; each call re-zeroes the one word
 *     that must start at zero, on `stream`, ahead of its kernel.  Calls that can overlap on the GPU (two streams with no
 *     ordering between them, several host threads) race on the array and return wrong sums: keep them on one stream or
 *     order them yourself.  The library's call guard (see Concurrency above) does NOT cover this entry point.
 *   Bitwise reproducible for a given n; equal to sf_contract_vertices up to rounding (a different, also fixed, order).
 * SF_EARG on a null pointer or n < 0, SF_ELIMIT on n above the limit, SF_ECUDA without a device. */
int sf_contract_vertices_noalloc(const double *a, const double *b, long n, double *result, sf_stream_t stream);
long sf_contract_noalloc_max_n(void);

/* Number of kernels the library launched since sf_init / the last reset (bench.py's gpu_launches). */
long sf_launch_count(int reset);
/* Path selection for steps 5-7.  All paths compute the same sum of eq. (3); they differ in the
 * order of the additions only.
 *   0 = automatic: the fastest path that supports the problem's sizes (4, else 3, else 1); when the chosen path runs out of
 *       device memory the next one is tried
 *   1 = staged: per batch of shells, {15j} assembly and the four mode products as separate kernels with intermediates
 *       in global memory, split along i1 when needed; any size
 *   3 = line: persistent per-shell kernel (x-sum of eq. (5) and the k4 product per shell, k3 / k2 products per line /
 *       block of shells by linearity); every intertwiner range <= 16 values.  This is the implementation of the method as
 *       the paper states it (one {15j} assembly and four mode products per shell)
 *   4 = factorised: the sums over the virtual spins are taken one spin at a time with x kept open (Q = sum_l45,
 *       R = sum_{l34 l35}, A' = sum_l23, A = sum_{l24 l25}); same terms, far fewer operations
 * (2 was an earlier on-chip kernel, removed: SF_EARG.)  The vertex calls return SF_EARG when the selected path cannot hold
 * the problem.  sf_last_path() = path the last vertex call took (1, 3 or 4). */
int sf_set_path(int path);
/* Pure host helper (no device needed): the boxes of shell offsets (o23 o24 o25 o34 o35 o45), o = l - j in units of 1, that
 * the factorised path splits the range [shell_lo, shell_hi) of the canonical shell order (eq. (9); l45
 * fastest) into.  boxes[k][0..5] = first offset of each virtual spin, boxes[k][6..11] = number of offsets; at most 11 boxes,
 * disjoint, in ascending shell order, their union is the range.  SF_EARG on a bad range or an odd / negative two_dl. */
int sf_shell_boxes(int two_dl, long shell_lo, long shell_hi, int boxes[16][12], int* n_boxes);
int sf_last_path(void);
/* Recorded launch sequences (default on).  A vertex call is 15-30 small kernel launches.  A call that ran without the library
 * having to grow a scratch block is remembered; when it arrives again with the same arguments (spins, Delta_l, ranges, booster
 * and output POINTERS -- the booster VALUES are read when the kernels run and may change) and unchanged library state, its
 * launches are recorded into a CUDA graph, and every later repetition is one graph launch on the caller's stream (config 0:
 * 0.1 -> 0.03 ms per tensor).  In a fresh context: call 1 allocates (plain), call 2 is remembered (plain), call 3 records and
 * replays, calls 4.. replay.  The result is bit for bit the one of
 * the plain call.  (A call on a stream the caller is capturing is refused: SF_ECAPTURE.)  0 switches the
 * recordings off (every call launches its kernels one by one).  Always SF_OK. */
int sf_set_graphs(int on);

#ifdef __cplusplus
}
#endif
#endif /* SFOAM_H */
