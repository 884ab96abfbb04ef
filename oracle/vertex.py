"""EPRL vertex amplitude, eq. (3) of the paper (oracle; test infrastructure).

PAPER.md:52-57:   A_v(j_f, i_e) = (prod_{e=1..5} sqrt(2 i_e + 1))
                                  sum_{l_f, k_e} (prod_{e=2..5} (2 k_e + 1) B4(j_f, i_e; l_f, k_e)) {15j}(l_f, k_e)
with l_1a = j_1a gauge-fixed and the homogeneous cutoff j_f <= l_f <= j_f + Delta_s.

Two levels:
  L0  `vertex_l0_entry`: the literal nested sum for ONE output entry, pure Python, exact fixed-point {15j}.
  L1  `vertex_l1`: steps 4-7 of the algorithm: S arrays of exact {6j}, then the naive C
      loops of vertex_l1.c.  L1 is validated against L0 in tests/test_oracle_vertex.py.

Booster tensors are INPUTS (dense, zero outside the valid k-range):
  B_a[t][ii][kk], a = 2..5, t = triple index in the paper's superscript order,
  ii = (two_i - two_i_min_a)/2, kk = (two_k - two_k_base_a)/2     (layout: DESIGN.md, reading G9).
Output: A[i1][i2][i3][i4][i5] row-major = the paper's column-major A^{i5 i4 i3 i2 i1}.
"""
import ctypes
import math
import os
import subprocess
from multiprocessing import Pool

import numpy as np

from . import fifteenj, ranges, wigner
from .ranges import J12, J13, J14, J15, J23, J24, J25, J34, J35, J45

_HERE = os.path.dirname(os.path.abspath(__file__))


# ------------------------------------------------------------------------------------------------
# layout
# ------------------------------------------------------------------------------------------------

class Layout:
    """Sizes of every array of the problem (two_j[10], two_dl)."""

    def __init__(self, two_j, two_dl):
        if two_dl < 0 or two_dl % 2:
            raise ValueError("two_dl must be a non-negative even integer (reading G5)")
        self.two_j = [int(s) for s in two_j]
        self.two_dl = int(two_dl)
        self.nl = two_dl // 2 + 1
        br = ranges.boundary_ranges(self.two_j)
        if any(n == 0 for _, n in br):
            raise ValueError("a boundary node has an empty intertwiner range")
        self.two_i_min = [lo for lo, _ in br]
        self.n_i = [n for _, n in br]
        self.two_k_base, self.n_k_pad = [], []
        for edge in (2, 3, 4, 5):
            _, _, _, base, pad = ranges.booster_dims(self.two_j, two_dl, edge)
            self.two_k_base.append(base)
            self.n_k_pad.append(pad)
        # bounding range of x from the triad (i1, l25, x) of eq. (5)
        i1s = [self.two_i_min[0] + 2 * a for a in range(self.n_i[0])]
        l25s = [self.two_j[J25] + 2 * o for o in range(self.nl)]
        self.two_x_base = min(abs(i - l) for i in i1s for l in l25s)
        top = max(i + l for i in i1s for l in l25s)
        self.n_x_pad = (top - self.two_x_base) // 2 + 1
        self.n_shells = self.nl ** 6

    def out_shape(self):
        return tuple(self.n_i)

    def booster_shape(self, edge):
        return (self.nl ** 3, self.n_i[edge - 1], self.n_k_pad[edge - 2])

    def s_shapes(self):
        nl, n1, (P2, P3, P4, P5), NX = self.nl, self.n_i[0], self.n_k_pad, self.n_x_pad
        return {
            "S1": (nl, n1, P5, NX),
            "S2": (nl, nl, P4, P5, NX),
            "S3": (nl, nl, nl, P3, P4, NX),
            "S4": (nl, nl, P2, P3, NX),
            "S5": (nl, n1, P2, NX),
        }

    def offsets(self, shell):
        o = []
        for _ in range(6):
            o.append(shell % self.nl)
            shell //= self.nl
        return tuple(reversed(o))


# ------------------------------------------------------------------------------------------------
# step 4: the five S arrays of exact 6j symbols (the five 6j of eq. (5))
# ------------------------------------------------------------------------------------------------

def _fill_slice(args):
    """Fill one l-slice of one S array.  `args` = (name, layout-pickle, l-offset tuple)."""
    name, two_j, two_dl, off = args
    L = Layout(two_j, two_dl)
    j = L.two_j
    i1s = [L.two_i_min[0] + 2 * a for a in range(L.n_i[0])]
    ks = [[L.two_k_base[e] + 2 * q for q in range(L.n_k_pad[e])] for e in range(4)]   # k2,k3,k4,k5 grids
    xs = [L.two_x_base + 2 * q for q in range(L.n_x_pad)]
    six = wigner.sixj
    if name == "S1":     # {i1 l25 x; k5 j14 j15}
        l25 = j[J25] + 2 * off[0]
        return np.array([[[six(i1, l25, x, k5, j[J14], j[J15]) for x in xs] for k5 in ks[3]] for i1 in i1s])
    if name == "S2":     # {j14 k5 x; l35 k4 l45}
        l35, l45 = j[J35] + 2 * off[0], j[J45] + 2 * off[1]
        return np.array([[[six(j[J14], k5, x, l35, k4, l45) for x in xs] for k5 in ks[3]] for k4 in ks[2]])
    if name == "S3":     # {k4 l35 x; k3 l24 l34}
        l24, l34, l35 = j[J24] + 2 * off[0], j[J34] + 2 * off[1], j[J35] + 2 * off[2]
        return np.array([[[six(k4, l35, x, k3, l24, l34) for x in xs] for k4 in ks[2]] for k3 in ks[1]])
    if name == "S4":     # {l24 k3 x; j13 k2 l23}
        l23, l24 = j[J23] + 2 * off[0], j[J24] + 2 * off[1]
        return np.array([[[six(l24, k3, x, j[J13], k2, l23) for x in xs] for k3 in ks[1]] for k2 in ks[0]])
    if name == "S5":     # {k2 j13 x; i1 l25 j12}
        l25 = j[J25] + 2 * off[0]
        return np.array([[[six(k2, j[J13], x, i1, l25, j[J12]) for x in xs] for k2 in ks[0]] for i1 in i1s])
    raise KeyError(name)


def build_s_arrays(L, shell_lo=0, shell_hi=None, processes=1):
    """Dense S1..S5 (double, exact values rounded once); only the l-slices that shells [lo,hi) touch are filled."""
    shell_hi = L.n_shells if shell_hi is None else shell_hi
    need = {k: set() for k in ("S1", "S2", "S3", "S4", "S5")}
    if shell_hi - shell_lo >= L.nl ** 6:
        offs = None
    else:
        offs = [L.offsets(s) for s in range(shell_lo, shell_hi)]
    rng = range(L.nl)
    if offs is None:
        need["S1"] = {(a,) for a in rng}
        need["S5"] = need["S1"]
        need["S2"] = {(a, b) for a in rng for b in rng}
        need["S4"] = need["S2"]
        need["S3"] = {(a, b, c) for a in rng for b in rng for c in rng}
    else:
        for o23, o24, o25, o34, o35, o45 in offs:
            need["S1"].add((o25,))
            need["S5"].add((o25,))
            need["S2"].add((o35, o45))
            need["S3"].add((o24, o34, o35))
            need["S4"].add((o23, o24))
    arrays = {name: np.zeros(shape) for name, shape in L.s_shapes().items()}
    jobs = [(name, L.two_j, L.two_dl, off) for name in arrays for off in sorted(need[name])]
    if processes > 1 and len(jobs) > 8:
        with Pool(processes) as pool:
            results = pool.map(_fill_slice, jobs, chunksize=max(1, len(jobs) // (8 * processes)))
    else:
        results = [_fill_slice(job) for job in jobs]
    for (name, _, _, off), block in zip(jobs, results):
        arrays[name][off] = block
    return arrays


# ------------------------------------------------------------------------------------------------
# L0: literal nested sum of eq. (3) for one output entry
# ------------------------------------------------------------------------------------------------

def vertex_l0_entry(two_j, two_dl, boosters, two_i):
    """A_v(j_f, i_e) for one tuple two_i = (i1..i5), summing eq. (3) term by term over (l_f, k_e).
    boosters = {2: B2, 3: B3, 4: B4, 5: B5} in the dense layout.  Returns (A, sum of |terms|)."""
    L = Layout(two_j, two_dl)
    a_idx = [(ti - lo) // 2 for ti, lo in zip(two_i, L.two_i_min)]
    total, total_abs = 0.0, 0.0
    for offs in ranges.shells(two_dl):
        two_l = ranges.shell_spins(L.two_j, offs)
        kr = [ranges.node_range(two_l, node) for node in (2, 3, 4, 5)]
        if any(n == 0 for _, n in kr):
            continue
        mats = []
        for e, edge in enumerate((2, 3, 4, 5)):
            t = ranges.triple_index(edge, offs, two_dl)
            mats.append(boosters[edge][t][a_idx[edge - 1]])     # row i_a of B_a[t]: a vector over kk
        for k2 in range(kr[0][0], kr[0][0] + 2 * kr[0][1], 2):
            for k3 in range(kr[1][0], kr[1][0] + 2 * kr[1][1], 2):
                for k4 in range(kr[2][0], kr[2][0] + 2 * kr[2][1], 2):
                    for k5 in range(kr[3][0], kr[3][0] + 2 * kr[3][1], 2):
                        ks = (k2, k3, k4, k5)
                        w = 1.0
                        for e, k in enumerate(ks):
                            w *= (k + 1) * mats[e][(k - L.two_k_base[e]) // 2]
                        if w == 0.0:
                            continue
                        total += w * fifteenj.fifteenj(two_l, two_i[0], ks)
                        total_abs += abs(w) * fifteenj.fifteenj_abs_terms(two_l, two_i[0], ks)
    norm = math.sqrt(math.prod(ti + 1 for ti in two_i))
    return norm * total, norm * total_abs


# ------------------------------------------------------------------------------------------------
# L1: S arrays + naive C loops
# ------------------------------------------------------------------------------------------------

_LIBS = {}


def build_c(force=False):
    """Compile vertex_l1.c twice: long double accumulation (parity reference) and double (timed baseline)."""
    src = os.path.join(_HERE, "vertex_l1.c")
    out = {}
    for tag, acc in (("ld", "long double"), ("d", "double")):
        so = os.path.join(_HERE, f"liboracle_l1_{tag}.so")
        if force or not os.path.exists(so) or os.path.getmtime(so) < os.path.getmtime(src):
            subprocess.check_call(["gcc", "-O2", "-fopenmp", "-fPIC", "-shared", "-std=c11",
                                   f"-DACC_T={acc}", "-o", so, src, "-lm"])
        out[tag] = so
    return out


def _lib(tag):
    if tag not in _LIBS:
        lib = ctypes.CDLL(build_c()[tag])
        lib.orc_vertex_range.restype = ctypes.c_long
        _LIBS[tag] = lib
    return _LIBS[tag]


def _iptr(seq):
    return (ctypes.c_int * len(seq))(*[int(v) for v in seq])


def _dptr(a):
    return a.ctypes.data_as(ctypes.POINTER(ctypes.c_double))


def vertex_l1(two_j, two_dl, boosters, shell_lo=0, shell_hi=None, long_double=True, want_abs=True,
              threads=None, s_arrays=None, processes=1):
    """Vertex tensor over shells [shell_lo, shell_hi) of the canonical order.
    Returns dict(A=..., Aabs=... or None, nonempty=int, layout=Layout)."""
    L = Layout(two_j, two_dl)
    shell_hi = L.n_shells if shell_hi is None else shell_hi
    S = s_arrays if s_arrays is not None else build_s_arrays(L, shell_lo, shell_hi, processes=processes)
    Bs = []
    for edge in (2, 3, 4, 5):
        b = np.ascontiguousarray(boosters[edge], dtype=np.float64)
        if b.shape != L.booster_shape(edge):
            raise ValueError(f"booster {edge}: shape {b.shape}, expected {L.booster_shape(edge)}")
        kr = ranges.booster_k_ranges(L.two_j, two_dl, edge)
        for t, (lo, nk) in enumerate(kr):   # entries outside the valid k-range must be zero (reading G9)
            q0 = (lo - L.two_k_base[edge - 2]) // 2 if nk else 0
            mask = np.ones(b.shape[2], dtype=bool)
            mask[q0:q0 + nk] = False
            assert not b[t][:, mask].any(), "booster entry outside the valid k-range is not zero"
        Bs.append(b)
    A = np.zeros(L.out_shape())
    Aabs = np.zeros(L.out_shape()) if want_abs else None
    threads = threads or os.cpu_count() or 1
    n = _lib("ld" if long_double else "d").orc_vertex_range(
        _iptr(L.two_j), ctypes.c_int(two_dl), _iptr(L.two_i_min), _iptr(L.n_i),
        _iptr(L.two_k_base), _iptr(L.n_k_pad), ctypes.c_int(L.two_x_base), ctypes.c_int(L.n_x_pad),
        _dptr(S["S1"]), _dptr(S["S2"]), _dptr(S["S3"]), _dptr(S["S4"]), _dptr(S["S5"]),
        _dptr(Bs[0]), _dptr(Bs[1]), _dptr(Bs[2]), _dptr(Bs[3]),
        ctypes.c_long(shell_lo), ctypes.c_long(shell_hi), ctypes.c_int(threads),
        _dptr(A), _dptr(Aabs) if want_abs else None)
    if n < 0:
        raise MemoryError("oracle C loops failed to allocate")
    return {"A": A, "Aabs": Aabs, "nonempty": int(n), "layout": L}


def bf_normalisation(L):
    """N(i) = prod_{e=1..5} sqrt(2 i_e+1) prod_{a=2..5} (2 i_a+1): with identity boosters and Delta_l = 0,
    eq. (3) gives A[i] = N(i) {15j}(j_f, i_e)   (reading G8)."""
    grids = [np.array([lo + 2 * a + 1 for a in range(n)], dtype=np.float64) for lo, n in zip(L.two_i_min, L.n_i)]
    N = np.ones(L.out_shape())
    for axis, g in enumerate(grids):
        shape = [1] * 5
        shape[axis] = len(g)
        N = N * np.sqrt(g).reshape(shape)
        if axis >= 1:
            N = N * g.reshape(shape)
    return N
