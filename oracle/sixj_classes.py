"""Every distinct {6j} symbol once: representatives of the classes of the 24 tetrahedral symmetries (oracle; test
infrastructure).  The loops are in sixj_classes.c (plain C, integers only); this is the ctypes wrapper.

Used by the exhaustive parity test of the GPU {6j} table (the paper precomputes 6j tables per maximal spin, PAPER.md:103,
207): one symbol per class, each evaluated exactly by wigner.sixj.  Nothing here is shared with the CUDA path.
"""
import ctypes
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_LIB = None


def build_c(force=False):
    src = os.path.join(_HERE, "sixj_classes.c")
    so = os.path.join(_HERE, "liboracle_sixj_classes.so")
    if force or not os.path.exists(so) or os.path.getmtime(so) < os.path.getmtime(src):
        subprocess.check_call(["gcc", "-O2", "-fPIC", "-shared", "-std=c11", "-o", so, src])
    return so


def _lib():
    global _LIB
    if _LIB is None:
        lib = ctypes.CDLL(build_c())
        lib.orc_sixj_classes_ab.restype = ctypes.c_long
        lib.orc_sixj_classes_ab.argtypes = [ctypes.c_int, ctypes.c_int, ctypes.c_int, ctypes.c_void_p, ctypes.c_long]
        _LIB = lib
    return _LIB


def classes_ab(two_jmax, two_a, two_b):
    """int8 array [n, 6]: the representatives (a b c d e f) with the given first two labels and every label <= two_jmax.
    A representative is the lexicographically largest of its 24 images, so a >= every label and b >= c, e, f."""
    n = _lib().orc_sixj_classes_ab(int(two_jmax), int(two_a), int(two_b), None, 0)
    out = np.empty((n, 6), dtype=np.int8)
    if n:
        got = _lib().orc_sixj_classes_ab(int(two_jmax), int(two_a), int(two_b), out.ctypes.data, n)
        assert got == n
    return out


def all_classes(two_jmax):
    """All representatives with labels <= two_jmax, ordered by (a, b) (small two_jmax only: the list grows like two_jmax^6)."""
    parts = [classes_ab(two_jmax, a, b) for a in range(two_jmax + 1) for b in range(a + 1)]
    return np.concatenate(parts) if parts else np.empty((0, 6), dtype=np.int8)
