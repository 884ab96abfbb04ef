"""sfoam-b200: thin Python binding of libsfoam.so, the C-ABI CUDA library declared in include/sfoam.h.

Argument marshalling only: every step of the path (the {6j} table, the S arrays, the {15j} assembly, the mode
products and the shell accumulation) runs in the library's CUDA kernels.  PyTorch tensors are used for device memory
and streams; any object with `data_ptr()` (device) works.  There is no CPU fallback: if the library has not been
built, or no CUDA device is present, the calls raise.

Function names are those of the header; spins are 2j integers; `two_j` has the order
(j12 j13 j14 j15 j23 j24 j25 j34 j35 j45) of Listing 8 of the paper.
"""
import ctypes
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libsfoam.so")

SF_OK, SF_ENOTINIT, SF_EARG, SF_ESPIN, SF_ETABLE, SF_ENOMEM, SF_ECUDA, SF_ELIMIT, SF_ECAPTURE = 0, -1, -2, -3, -4, -5, -6, -7, -8


class SfError(RuntimeError):
    def __init__(self, status, what):
        self.status = status
        super().__init__(f"{what}: {_lib().sf_strerror(status).decode()} ({status})")


class _Boosters(ctypes.Structure):
    _fields_ = [("B", ctypes.c_void_p * 4)]


_LIB = None
_I10 = ctypes.c_int * 10
_I5 = ctypes.c_int * 5
_I6 = ctypes.c_int * 6


def _lib():
    global _LIB
    if _LIB is None:
        if not os.path.exists(LIB_PATH):
            raise ImportError(f"{LIB_PATH} is missing: build it with `python -m paper_2107_13952_b200.build` "
                              "(there is no CPU fallback)")
        lib = ctypes.CDLL(LIB_PATH)
        lib.sf_strerror.restype = ctypes.c_char_p
        lib.sf_gamma.restype = ctypes.c_double
        lib.sf_init.argtypes = [ctypes.c_double]
        lib.sf_sixj_table_slots.restype = ctypes.c_long
        lib.sf_launch_count.restype = ctypes.c_long
        lib.sf_graph_replays.restype = ctypes.c_long
        lib.sf_sixj_batch.argtypes = [ctypes.c_void_p, ctypes.c_long, ctypes.c_int, ctypes.c_void_p]
        lib.sf_vertex_work.argtypes = [_I10, ctypes.c_int, ctypes.c_long, ctypes.c_long,
                                       ctypes.POINTER(ctypes.c_double), ctypes.POINTER(ctypes.c_long),
                                       ctypes.POINTER(ctypes.c_double)]
        lib.sf_vertex_terms.argtypes = [_I10, ctypes.c_int, ctypes.c_long, ctypes.c_long,
                                        ctypes.POINTER(ctypes.c_double)]
        lib.sf_factor_work.argtypes = [_I10, ctypes.c_int, ctypes.c_double * 6, ctypes.c_double * 4]
        lib.sf_set_factor_budget.argtypes = [ctypes.c_size_t]
        lib.sf_slice_elems.argtypes = [_I10, ctypes.c_int]
        lib.sf_slice_elems.restype = ctypes.c_long
        lib.sf_fp64_peak.argtypes = [ctypes.c_int, ctypes.POINTER(ctypes.c_double)]
        lib.sf_vertex_amplitude.argtypes = [_I10, ctypes.c_int, ctypes.POINTER(_Boosters), ctypes.c_void_p,
                                            ctypes.c_void_p]
        lib.sf_vertex_amplitude_range.argtypes = [_I10, ctypes.c_int, ctypes.POINTER(_Boosters), ctypes.c_long,
                                                  ctypes.c_long, ctypes.c_void_p, ctypes.c_void_p]
        lib.sf_vertex_amplitude_intertwiners.argtypes = [_I10, ctypes.c_int, ctypes.POINTER(_Boosters), ctypes.c_int * 5,
                                                         ctypes.c_int * 5, ctypes.c_void_p, ctypes.c_void_p]
        lib.sf_vertex_amplitude_batch.argtypes = [ctypes.c_int, ctypes.c_void_p, ctypes.c_void_p, ctypes.c_void_p, ctypes.c_void_p,
                                                  ctypes.c_void_p]
        lib.sf_contract_vertices.argtypes = [ctypes.c_void_p, ctypes.c_void_p, ctypes.c_long, ctypes.c_void_p, ctypes.c_void_p]
        lib.sf_contract_vertices_noalloc.argtypes = [ctypes.c_void_p, ctypes.c_void_p, ctypes.c_long, ctypes.c_void_p,
                                                     ctypes.c_void_p]
        lib.sf_contract_noalloc_max_n.restype = ctypes.c_long
        lib.sf_contract_vectors.argtypes = [ctypes.c_void_p, ctypes.c_int * 5, ctypes.c_void_p * 5, ctypes.c_void_p,
                                            ctypes.c_void_p]
        lib.sf_vertex_amplitude_host.argtypes = [_I10, ctypes.c_int, ctypes.c_void_p * 4, ctypes.c_void_p,
                                                 ctypes.c_void_p]
        lib.sf_set_staged_budget.argtypes = [ctypes.c_size_t]
        _LIB = lib
    return _LIB


def _check(status, what):
    if status != SF_OK:
        raise SfError(status, what)


def _spins(two_j):
    if len(two_j) != 10:
        raise ValueError("two_j must hold the ten boundary spins (12 13 14 15 23 24 25 34 35 45)")
    return _I10(*[int(s) for s in two_j])


def _ptr(t):
    return ctypes.c_void_p(t.data_ptr() if hasattr(t, "data_ptr") else int(t))


def _stream(stream):
    if stream is None:
        return ctypes.c_void_p(0)
    return ctypes.c_void_p(getattr(stream, "cuda_stream", stream))


# ---------------------------------------------------------------------------------------------------------------
# context
# ---------------------------------------------------------------------------------------------------------------
def sf_init(gamma):
    _check(_lib().sf_init(float(gamma)), "sf_init")


def sf_finalize():
    _check(_lib().sf_finalize(), "sf_finalize")


def sf_gamma():
    return _lib().sf_gamma()


def sf_strerror(status):
    return _lib().sf_strerror(int(status)).decode()


def sf_launch_count(reset=False):
    return int(_lib().sf_launch_count(int(bool(reset))))


def sf_set_timing(on):
    _check(_lib().sf_set_timing(int(bool(on))), "sf_set_timing")


def sf_last_stage_ms():
    ms = (ctypes.c_double * 3)()
    _check(_lib().sf_last_stage_ms(ms), "sf_last_stage_ms")
    return list(ms)


def sf_last_kernel_ms():
    """Factorised path: event times (ms) of [k_fz_qp, k_fz_gemm<FzMapR>, k_fz_gemm<FzMapA>, precomputations] of the last
    vertex call made with sf_set_timing(True)."""
    ms = (ctypes.c_double * 4)()
    _check(_lib().sf_last_kernel_ms(ms), "sf_last_kernel_ms")
    return list(ms)


def sf_set_counting(on):
    _check(_lib().sf_set_counting(int(bool(on))), "sf_set_counting")


def sf_set_debug_poison(on):
    _check(_lib().sf_set_debug_poison(int(bool(on))), "sf_set_debug_poison")


def sf_last_dmma():
    """Factorised path: DMMA.8x8x4 warp instructions issued by [k_fz_qp, k_fz_gemm<FzMapR>, k_fz_gemm<FzMapA>] in the last
    vertex call made with sf_set_counting(True)."""
    n = (ctypes.c_double * 3)()
    _check(_lib().sf_last_dmma(n), "sf_last_dmma")
    return list(n)


def sf_shell_boxes(two_dl, shell_lo, shell_hi):
    """Boxes (lo[6], cnt[6]) of shell offsets the factorised path splits [shell_lo, shell_hi) into (host only)."""
    boxes = ((ctypes.c_int * 12) * 16)()
    n = ctypes.c_int(0)
    _check(_lib().sf_shell_boxes(int(two_dl), ctypes.c_long(shell_lo), ctypes.c_long(shell_hi), boxes, ctypes.byref(n)),
           "sf_shell_boxes")
    return [(list(boxes[k][0:6]), list(boxes[k][6:12])) for k in range(n.value)]


def sf_set_path(path):
    """0 = automatic (factorised, else line, else staged), 1 = staged (any size), 3 = line (the per-shell method of the paper
    on chip; intertwiner ranges <= 16 values), 4 = factorised; 3 and 4 raise SF_EARG at call time for shapes they do not
    hold, 2 (a removed kernel) always."""
    _check(_lib().sf_set_path(int(path)), "sf_set_path")


def sf_set_graphs(on):
    """Recorded launch sequences for repeated identical calls (include/sfoam.h): 1 on (default), 0 off."""
    _check(_lib().sf_set_graphs(int(bool(on))), "sf_set_graphs")


def sf_last_path():
    return int(_lib().sf_last_path())


def sf_set_staged_budget(nbytes):
    _lib().sf_set_staged_budget(int(nbytes))


def sf_set_factor_variant(bits):
    """Kernel variants of the factorised path (include/sfoam_debug.h): 0 = default."""
    _lib().sf_set_factor_variant(int(bits))


def sf_graph_replays(reset=False):
    """Vertex calls answered by replaying a recorded launch sequence since sf_init / the last reset (debug hook)."""
    return int(_lib().sf_graph_replays(1 if reset else 0))


def sf_last_qp_kernel():
    """Q/P kernel of the last factorised call: 1 k_fz_qp, 2 k_fz_qp2, 4 k_fz_qp4 (include/sfoam_debug.h)."""
    return int(_lib().sf_last_qp_kernel())


def sf_set_factor_budget(nbytes):
    """Device bytes the factorised path may use for P and R of one pass over i1 (0 = default, a third of the device)."""
    _lib().sf_set_factor_budget(int(nbytes))


# ---------------------------------------------------------------------------------------------------------------
# {6j}
# ---------------------------------------------------------------------------------------------------------------
def sf_sixj_table(two_jmax):
    _check(_lib().sf_sixj_table(int(two_jmax)), "sf_sixj_table")


def sf_sixj_table_slots():
    return int(_lib().sf_sixj_table_slots())


def sf_sixj_table_two_jmax():
    return int(_lib().sf_sixj_table_two_jmax())


def sf_sixj_get(two_j6):
    out = ctypes.c_double()
    _check(_lib().sf_sixj_get(_I6(*[int(s) for s in two_j6]), ctypes.byref(out)), "sf_sixj_get")
    return out.value


def sf_sixj_batch(two_j6, mode=0):
    """two_j6: int array [n, 6] of (a b c d e f) for {a b c; d e f}.  mode 0 = direct evaluation, 1 = table gather."""
    args = np.ascontiguousarray(two_j6, dtype=np.int32).reshape(-1, 6)
    out = np.empty(len(args), dtype=np.float64)
    _check(_lib().sf_sixj_batch(args.ctypes.data, len(args), int(mode), out.ctypes.data), "sf_sixj_batch")
    return out


# ---------------------------------------------------------------------------------------------------------------
# host integer helpers
# ---------------------------------------------------------------------------------------------------------------
def sf_vertex_dims(two_j):
    lo, n = _I5(), _I5()
    _check(_lib().sf_vertex_dims(_spins(two_j), lo, n), "sf_vertex_dims")
    return list(lo), list(n)


def sf_booster_dims(two_j, two_dl, edge):
    """(n_triples, n_i, two_k_base, n_k_pad) of the dense booster tensor B_edge[t][ii][kk]."""
    v = [ctypes.c_int() for _ in range(4)]
    _check(_lib().sf_booster_dims(_spins(two_j), int(two_dl), int(edge), *[ctypes.byref(x) for x in v]),
           "sf_booster_dims")
    return tuple(x.value for x in v)


def sf_booster_krange(two_j, two_dl, edge, t):
    lo, n = ctypes.c_int(), ctypes.c_int()
    _check(_lib().sf_booster_krange(_spins(two_j), int(two_dl), int(edge), int(t), ctypes.byref(lo), ctypes.byref(n)),
           "sf_booster_krange")
    return lo.value, n.value


def sf_booster_kranges(two_j, two_dl, edge):
    """[(two_k_min, n_k)] for every triple t of the edge."""
    nt = (int(two_dl) // 2 + 1) ** 3
    lo, n = (ctypes.c_int * nt)(), (ctypes.c_int * nt)()
    _check(_lib().sf_booster_kranges(_spins(two_j), int(two_dl), int(edge), lo, n), "sf_booster_kranges")
    return list(zip(lo, n))


def sf_vertex_work(two_j, two_dl, shell_lo=0, shell_hi=None):
    """dict(f_con, n_nonempty, n_w): algorithmic contraction flops, non-empty shells, W entries of the shell range."""
    if shell_hi is None:
        shell_hi = (int(two_dl) // 2 + 1) ** 6
    f, ne, nw = ctypes.c_double(), ctypes.c_long(), ctypes.c_double()
    _check(_lib().sf_vertex_work(_spins(two_j), int(two_dl), int(shell_lo), int(shell_hi), ctypes.byref(f),
                                 ctypes.byref(ne), ctypes.byref(nw)), "sf_vertex_work")
    return {"f_con": f.value, "n_nonempty": ne.value, "n_w": nw.value}


def sf_vertex_terms(two_j, two_dl, shell_lo=0, shell_hi=None):
    """Number of (entry, x) summands of eq. (5) over the shell range (device integer kernel); F_asm = 6 * n_terms."""
    if shell_hi is None:
        shell_hi = (int(two_dl) // 2 + 1) ** 6
    n = ctypes.c_double()
    _check(_lib().sf_vertex_terms(_spins(two_j), int(two_dl), int(shell_lo), int(shell_hi), ctypes.byref(n)),
           "sf_vertex_terms")
    return n.value


def sf_factor_work(two_j, two_dl):
    """Useful multiply-adds of the six contractions of the factorised path (Z, Q, P, R, G, A') and the structurally non-zero
    entries of its intermediates (Z, Q, P, R), from the triangle inequalities only (host integer function)."""
    mac, elems = (ctypes.c_double * 6)(), (ctypes.c_double * 4)()
    _check(_lib().sf_factor_work(_spins(two_j), int(two_dl), mac, elems), "sf_factor_work")
    return dict(zip(("Z", "Q", "P", "R", "G", "A"), mac)), dict(zip(("Z", "Q", "P", "R"), elems))


def sf_slice_elems(two_j, two_dl):
    """Entries of the five S arrays of step 4 = {6j} symbols gathered per vertex call (host integer function)."""
    return int(_lib().sf_slice_elems(_spins(two_j), int(two_dl)))


def sf_fp64_peak(kind):
    """Measured FP64 peak in TFLOP/s: kind 0 = DFMA chains, kind 1 = DMMA (mma.sync m8n8k4 f64) chains."""
    v = ctypes.c_double()
    _check(_lib().sf_fp64_peak(int(kind), ctypes.byref(v)), "sf_fp64_peak")
    return v.value


# ---------------------------------------------------------------------------------------------------------------
# the vertex tensor
# ---------------------------------------------------------------------------------------------------------------
def _boosters(boosters):
    if isinstance(boosters, dict):
        boosters = [boosters[e] for e in (2, 3, 4, 5)]
    if len(boosters) != 4:
        raise ValueError("need the four booster tensors of edges 2..5")
    b = _Boosters()
    for e, t in enumerate(boosters):
        b.B[e] = t.data_ptr() if hasattr(t, "data_ptr") else int(t)
    return b


def sf_vertex_amplitude(two_j, two_dl, boosters, out, stream=None):
    """boosters: four DEVICE float64 tensors B_a[t][ii][kk] (edges 2..5; list or {2:..,5:..}); out: DEVICE float64
    tensor of prod(n_i) elements, overwritten with A[i1][i2][i3][i4][i5].  Asynchronous on `stream`."""
    b = _boosters(boosters)
    _check(_lib().sf_vertex_amplitude(_spins(two_j), int(two_dl), ctypes.byref(b), _ptr(out), _stream(stream)),
           "sf_vertex_amplitude")
    return out


def sf_vertex_amplitude_range(two_j, two_dl, boosters, shell_lo, shell_hi, out, stream=None):
    b = _boosters(boosters)
    _check(_lib().sf_vertex_amplitude_range(_spins(two_j), int(two_dl), ctypes.byref(b), int(shell_lo), int(shell_hi),
                                            _ptr(out), _stream(stream)), "sf_vertex_amplitude_range")
    return out


def sf_vertex_amplitude_intertwiners(two_j, two_dl, boosters, i_first, i_count, out, stream=None):
    """The sub-block out[i1][i2][i3][i4][i5] of the vertex tensor over i_count[n] intertwiner values of node n + 1 starting
    at index i_first[n]."""
    b = _boosters(boosters)
    first = (ctypes.c_int * 5)(*[int(v) for v in i_first])
    count = (ctypes.c_int * 5)(*[int(v) for v in i_count])
    _check(_lib().sf_vertex_amplitude_intertwiners(_spins(two_j), int(two_dl), ctypes.byref(b), first, count, _ptr(out),
                                                   _stream(stream)), "sf_vertex_amplitude_intertwiners")
    return out


def sf_vertex_amplitude_batch(two_j, two_dl, boosters, outs, stream=None):
    """Many vertex tensors in one call.  two_j: n lists of ten spins; two_dl: n ints (or one int for all);
    boosters: n quadruples of DEVICE tensors (edges 2..5); outs: n DEVICE float64 tensors, overwritten.  Small tensors are
    computed by one kernel launch (one CTA each), larger ones by the single-tensor path afterwards."""
    n = len(two_j)
    if isinstance(two_dl, int):
        two_dl = [two_dl] * n
    if not (len(two_dl) == len(boosters) == len(outs) == n):
        raise ValueError("two_j, two_dl, boosters and outs must have the same length")
    spins = (ctypes.c_int * (10 * n))(*[int(s) for tj in two_j for s in tj])
    dls = (ctypes.c_int * n)(*[int(d) for d in two_dl])
    barr = (_Boosters * n)()
    for q, b4 in enumerate(boosters):
        if isinstance(b4, dict):
            b4 = [b4[e] for e in (2, 3, 4, 5)]
        for e, t in enumerate(b4):
            barr[q].B[e] = t.data_ptr() if hasattr(t, "data_ptr") else int(t)
    optr = (ctypes.c_void_p * n)(*[o.data_ptr() if hasattr(o, "data_ptr") else int(o) for o in outs])
    _check(_lib().sf_vertex_amplitude_batch(n, spins, dls, barr, optr, _stream(stream)), "sf_vertex_amplitude_batch")
    return outs


def sf_contract_vertices(a, b, result, stream=None):
    """result[0] = sum a b over two vertex tensors of the same shape (device tensors)."""
    _check(_lib().sf_contract_vertices(_ptr(a), _ptr(b), ctypes.c_long(a.numel()), _ptr(result), _stream(stream)),
           "sf_contract_vertices")
    return result


def sf_contract_vertices_noalloc(a, b, result, stream=None):
    """sf_contract_vertices for a caller that cannot allocate device memory (all of it sits in the caller's own pool, or a
    cudaMalloc's device-wide synchronisation is not acceptable where the call is made): the partial sums live in a fixed
    65 792-byte array inside the library instead of cudaMalloc'd scratch.  a.numel() <= sf_contract_noalloc_max_n()
    (33 554 432), else SfError with status SF_ELIMIT.  Needs no sf_init.  All calls on a device share that array: calls
    that may overlap on the GPU race, keep them on one stream.  Make the first call on a device before any stream capture."""
    _check(_lib().sf_contract_vertices_noalloc(_ptr(a), _ptr(b), ctypes.c_long(a.numel()), _ptr(result), _stream(stream)),
           "sf_contract_vertices_noalloc")
    return result


def sf_contract_noalloc_max_n():
    """Largest number of entries sf_contract_vertices_noalloc accepts."""
    return int(_lib().sf_contract_noalloc_max_n())


def sf_contract_vectors(A, psi, result, stream=None):
    """result[0] + i result[1] = sum A[i1..i5] psi[0][i1] ... psi[4][i5]; A a 5-index float64 device tensor, psi five
    complex128 device tensors."""
    n = (ctypes.c_int * 5)(*[int(v) for v in A.shape])
    arr = (ctypes.c_void_p * 5)(*[p.data_ptr() for p in psi])
    _check(_lib().sf_contract_vectors(_ptr(A), n, arr, _ptr(result), _stream(stream)), "sf_contract_vectors")
    return result


def sf_vertex_amplitude_host(two_j, two_dl, host_boosters, host_out, stream=None):
    """End-to-end variant: host_boosters are four HOST float64 arrays (numpy, or pinned torch CPU tensors), host_out
    a HOST float64 array; copies in, computes, copies back and synchronises."""
    if isinstance(host_boosters, dict):
        host_boosters = [host_boosters[e] for e in (2, 3, 4, 5)]
    arr = (ctypes.c_void_p * 4)()
    for e, t in enumerate(host_boosters):
        arr[e] = t.data_ptr() if hasattr(t, "data_ptr") else t.ctypes.data
    optr = host_out.data_ptr() if hasattr(host_out, "data_ptr") else host_out.ctypes.data
    _check(_lib().sf_vertex_amplitude_host(_spins(two_j), int(two_dl), arr, ctypes.c_void_p(optr), _stream(stream)),
           "sf_vertex_amplitude_host")
    return host_out
