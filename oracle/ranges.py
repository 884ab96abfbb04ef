"""Intertwiner ranges and shell enumeration (oracle; test infrastructure).

Step 2 of the vertex-tensor algorithm, PAPER.md:168 ("Compute the ranges of the intertwiner
indices"), and the shell cutoff j_f <= l_f <= j_f + Delta_s of PAPER.md:57.  All spins are 2j ints.

Spin order (lexicographic, Listing 8):   two_j = (j12 j13 j14 j15 j23 j24 j25 j34 j35 j45)
Node spin orders (first pair | second pair), read off the booster index sets of step 3
 and the 6j triads of eq. (5):

    node 1: (j12 j13 | j14 j15) -> i1          node 4: (j45 j14 | j24 j34) -> i4 / k4
    node 2: (j23 j24 | j25 j12) -> i2 / k2     node 5: (j15 j25 | j35 j45) -> i5 / k5
    node 3: (j34 j35 | j13 j23) -> i3 / k3

The intertwiner of a node recouples its first pair with its second pair, so its range is the
intersection of the two triangle ranges, in steps of 1 (2 in 2j units).
"""
import itertools

J12, J13, J14, J15, J23, J24, J25, J34, J35, J45 = range(10)

# node -> indices into two_j of (first pair | second pair); node 1 is element 0
NODE_SPINS = (
    (J12, J13, J14, J15),
    (J23, J24, J25, J12),
    (J34, J35, J13, J23),
    (J45, J14, J24, J34),
    (J15, J25, J35, J45),
)

# the six virtual spins in canonical shell order (l23 l24 l25 l34 l35 l45), l45 fastest (eq. (9))
VIRTUAL = (J23, J24, J25, J34, J35, J45)

# booster triples in the paper's superscript order:
#   edge 2: (l23 l24 l25), edge 3: (l34 l35 l23), edge 4: (l45 l24 l34), edge 5: (l25 l35 l45)
EDGE_TRIPLE = {2: (J23, J24, J25), 3: (J34, J35, J23), 4: (J45, J24, J34), 5: (J25, J35, J45)}


def pair_range(two_a, two_b, two_c, two_d):
    """Range (two_min, n) of the spin that recouples (a b) with (c d); n = 0 if empty or parity mismatch."""
    if (two_a + two_b) % 2 != (two_c + two_d) % 2:
        return 0, 0
    lo = max(abs(two_a - two_b), abs(two_c - two_d))
    hi = min(two_a + two_b, two_c + two_d)
    if hi < lo:
        return lo, 0
    return lo, (hi - lo) // 2 + 1


def node_range(two_spins, node):
    """Range of the intertwiner at `node` (1..5) for the 10 spins `two_spins` (boundary j or virtual l)."""
    a, b, c, d = (two_spins[s] for s in NODE_SPINS[node - 1])
    return pair_range(a, b, c, d)


def boundary_ranges(two_j):
    """[(two_i_min, n_i)] for nodes 1..5  (step 2)."""
    return [node_range(two_j, n) for n in range(1, 6)]


def shell_spins(two_j, offsets):
    """Ten spins with the six virtual ones replaced by l = j + offset (offsets in units of 1, canonical order)."""
    two_l = list(two_j)
    for idx, off in zip(VIRTUAL, offsets):
        two_l[idx] = two_j[idx] + 2 * off
    return two_l


def shells(two_dl):
    """All shells in canonical order: offsets (o23,o24,o25,o34,o35,o45), each 0..Delta_l, o45 fastest."""
    n = two_dl // 2 + 1
    return itertools.product(range(n), repeat=6)


def shell_index(offsets, two_dl):
    n = two_dl // 2 + 1
    idx = 0
    for o in offsets:
        idx = idx * n + o
    return idx


def triple_index(edge, offsets, two_dl):
    """t = (u*(dl+1)+v)*(dl+1)+w with (u,v,w) the offsets of the edge's three virtual spins in the
    paper's superscript order."""
    n = two_dl // 2 + 1
    pos = {s: p for p, s in enumerate(VIRTUAL)}
    u, v, w = (offsets[pos[s]] for s in EDGE_TRIPLE[edge])
    return (u * n + v) * n + w


def booster_k_ranges(two_j, two_dl, edge):
    """For booster edge a in 2..5: list over triples t (row-major in the paper's superscript order) of
    (two_k_min, n_k).  The edge's node has three virtual spins and one gauge-fixed boundary spin
    (PAPER.md:122), so its k-range depends on the triple only."""
    n = two_dl // 2 + 1
    out = []
    for u, v, w in itertools.product(range(n), repeat=3):
        two_l = list(two_j)
        for s, o in zip(EDGE_TRIPLE[edge], (u, v, w)):
            two_l[s] = two_j[s] + 2 * o
        out.append(node_range(two_l, edge))
    return out


def booster_dims(two_j, two_dl, edge):
    """(n_triples, n_i, two_i_min, two_k_base, n_k_pad): dense padded layout B_a[t][ii][kk] of SURVEY 8(b)."""
    kr = booster_k_ranges(two_j, two_dl, edge)
    two_i_min, n_i = node_range(two_j, edge)
    nonempty = [(lo, nk) for lo, nk in kr if nk > 0]
    if not nonempty:
        return len(kr), n_i, two_i_min, 0, 0
    base = min(lo for lo, _ in nonempty)
    top = max(lo + 2 * (nk - 1) for lo, nk in nonempty)
    return len(kr), n_i, two_i_min, base, (top - base) // 2 + 1
