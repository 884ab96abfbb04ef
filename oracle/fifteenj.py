"""{15j} symbol of the first type, eq. (5) of the paper (oracle; test infrastructure).

PAPER.md:67-95.  The printed equation is partly garbled and its sign exponent is elided
("(-1)^{i_1+k_2+...+j_12+...+l_23+...}").  Reading taken (reading G1): the exponent R is
the sum of ALL fifteen labels.  `brute_force_15j` below pins that reading, sign included, against the
definition of the symbol as the contraction of five 4jm symbols (the notation of eq. (4)).

Argument convention everywhere: `two_l` is the list of ten spins in the order
(12 13 14 15 23 24 25 34 35 45) with the four gauge-fixed entries equal to the boundary spins
(l_1a = j_1a), `two_i1` the boundary intertwiner of node 1 and `two_k = (k2,k3,k4,k5)`.
"""
import itertools

import numpy as np

from . import wigner
from .ranges import J12, J13, J14, J15, J23, J24, J25, J34, J35, J45, NODE_SPINS


def x_range(two_l, two_i1, two_k):
    """Range of the summed spin x: intersection of the five triads of eq. (5) that contain x
    (reading G4: step 1, parity fixed by i1 + l25)."""
    k2, k3, k4, k5 = two_k
    pairs = ((two_i1, two_l[J25]), (k5, two_l[J14]), (k4, two_l[J35]), (k3, two_l[J24]), (k2, two_l[J13]))
    lo = max(abs(a - b) for a, b in pairs)
    hi = min(a + b for a, b in pairs)
    par = (two_i1 + two_l[J25]) % 2
    if any((a + b) % 2 != par for a, b in pairs):
        return range(0)
    return range(lo, hi + 1, 2)


def sixj_factors(two_l, two_i1, two_k, two_x, sixj=wigner.sixj_fixed):
    """The five {6j} of eq. (5), in the order printed."""
    k2, k3, k4, k5 = two_k
    l = two_l
    return (
        sixj(two_i1, l[J25], two_x, k5, l[J14], l[J15]),
        sixj(l[J14], k5, two_x, l[J35], k4, l[J45]),
        sixj(k4, l[J35], two_x, k3, l[J24], l[J34]),
        sixj(l[J24], k3, two_x, l[J13], k2, l[J23]),
        sixj(k2, l[J13], two_x, two_i1, l[J25], l[J12]),
    )


def sign_exponent(two_l, two_i1, two_k):
    """R = i1+k2+k3+k4+k5 + (all ten spins); always an integer (asserted)."""
    two_R = two_i1 + sum(two_k) + sum(two_l)
    assert two_R % 2 == 0, "sum of the fifteen labels must be an integer"
    return two_R // 2


def fifteenj_fixed(two_l, two_i1, two_k):
    """{15j} as a fixed-point integer (value = result / 2^FIXED_BITS): eq. (5) summed term by term."""
    B = wigner.FIXED_BITS
    xs = x_range(two_l, two_i1, two_k)
    if len(xs) == 0:
        return 0
    total = 0
    for two_x in xs:
        prod = (two_x + 1) << B
        for s in sixj_factors(two_l, two_i1, two_k, two_x):
            prod = (prod * s) >> B
        total += prod
    return -total if sign_exponent(two_l, two_i1, two_k) % 2 else total


def fifteenj(two_l, two_i1, two_k):
    """{15j} rounded once to double."""
    return wigner.fixed_to_float(fifteenj_fixed(two_l, two_i1, two_k))


def fifteenj_abs_terms(two_l, two_i1, two_k):
    """sum_x (2x+1) prod |6j|  -- the finest-granularity absolute sum used by the tolerance (reading G15)."""
    total = 0.0
    for two_x in x_range(two_l, two_i1, two_k):
        p = float(two_x + 1)
        for s in sixj_factors(two_l, two_i1, two_k, two_x, sixj=wigner.sixj):
            p *= abs(s)
        total += p
    return total


# ----------------------------------------------------------------------------------------------
# Brute force over magnetic indices: the definition of the symbol as an invariant contraction.
# ----------------------------------------------------------------------------------------------

_LINKS = ((J12, 1, 2), (J13, 1, 3), (J14, 1, 4), (J15, 1, 5), (J23, 2, 3),
          (J24, 2, 4), (J25, 2, 5), (J34, 3, 4), (J35, 3, 5), (J45, 4, 5))


def _node_tensor(two_spins4, two_i):
    """4jm symbol of eq. (4) as a dense array over (m1,m2,m3,m4), m = -j..j ascending."""
    dims = [s + 1 for s in two_spins4]
    T = np.zeros(dims)
    for idx in itertools.product(*[range(d) for d in dims]):
        two_m = [2 * q - s for q, s in zip(idx, two_spins4)]
        if sum(two_m) == 0:
            T[idx] = wigner.fourjm(two_spins4, two_m, two_i)
    return T


def brute_force_15j(two_l, two_intw):
    """Contract five 4jm symbols (one per node, spin orders of ranges.NODE_SPINS, intertwiners
    two_intw = (i1,k2,k3,k4,k5)) over all ten links.  Link (a<b) is contracted with
    sum_m (-1)^{j_ab - m}, node a carrying +m and node b carrying -m.  This is the graph-invariant
    definition of the 15j; eq. (5) is its reduction to 6j symbols."""
    letters = "abcdefghij"
    operands, subs = [], []
    for node in range(1, 6):
        spins = NODE_SPINS[node - 1]
        T = _node_tensor([two_l[s] for s in spins], two_intw[node - 1])
        sub = ""
        for axis, s in enumerate(spins):
            link = next(L for L in _LINKS if L[0] == s)
            sub += letters[s]
            if link[2] == node:
                # second endpoint: carries -m and the phase (-1)^{j-m}; m ascending => flip the axis
                T = np.flip(T, axis=axis)
                two_jl = two_l[s]
                phase = np.array([(-1.0) ** ((two_jl - (2 * q - two_jl)) // 2) for q in range(two_jl + 1)])
                shape = [1] * 4
                shape[axis] = two_jl + 1
                T = T * phase.reshape(shape)
        operands.append(T)
        subs.append(sub)
    return float(np.einsum(",".join(subs) + "->", *operands, optimize=True))
