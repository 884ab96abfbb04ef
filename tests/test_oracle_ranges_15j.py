"""Pins for oracle/ranges.py and oracle/fifteenj.py.

ranges: brute enumeration of the triangle conditions on small spins, and the workload counts that
SURVEY.md 8(a)/8(c) P2 computed independently.
{15j}: printed exact values (tests/golden/), the brute-force contraction over magnetic indices (which pins the
sign exponent of eq. (5), elided in the text), and the collapse to a single {6j}."""
import itertools
import math
import os
import random

import numpy as np
import pytest

from oracle import fifteenj, ranges, wigner
from oracle.ranges import J12, J13, J14, J15, J23, J24, J25, J34, J35, J45


# ------------------------------------------------------------------------------------------------ ranges

def test_pair_range_brute_force():
    for a, b, c, d in itertools.product(range(0, 7), repeat=4):
        lo, n = ranges.pair_range(a, b, c, d)
        brute = [k for k in range(0, 15) if wigner.is_triad(a, b, k) and wigner.is_triad(c, d, k)]
        assert n == len(brute)
        if n:
            assert lo == brute[0] and brute == list(range(lo, lo + 2 * n, 2))


def test_node_orders_match_eq5_triads():
    # the 6j symbols of eq. (5) couple (i1; j14 j15), (k5; j15 l25), (k4; j14 l45), (k4; l24 l34), (k3; l35 l34),
    # (k2; l24 l23), (k3; j13 l23), (k2; l25 j12), (i1; j13 j12): each pair must be a recoupling pair of its node
    pairs = {1: [{J14, J15}, {J12, J13}], 2: [{J23, J24}, {J25, J12}], 3: [{J34, J35}, {J13, J23}],
             4: [{J45, J14}, {J24, J34}], 5: [{J15, J25}, {J35, J45}]}
    for node, want in pairs.items():
        s = ranges.NODE_SPINS[node - 1]
        assert [set(s[:2]), set(s[2:])] == want or [set(s[2:]), set(s[:2])] == want


def test_listing8_spin_order():
    # Listing 8: js = [5 5 5 5 2 2 2 2 2 2] with j_1a = 5, j_ab = 2 => lexicographic order
    two_j = [10, 10, 10, 10, 4, 4, 4, 4, 4, 4]
    assert [two_j[s] for s in (J12, J13, J14, J15)] == [10] * 4
    assert ranges.boundary_ranges(two_j)[0] == (0, 11)          # node 1: (5 5 | 5 5) -> i1 in 0..10
    assert ranges.boundary_ranges(two_j)[1] == (6, 2)           # node 2: (2 2 | 2 5) -> i2 in {3, 4}


def test_survey_counts_config0():
    two_j = [2] * 10
    assert ranges.boundary_ranges(two_j) == [(0, 3)] * 5
    total_w, nonempty = 0, 0
    for offs in ranges.shells(4):
        two_l = ranges.shell_spins(two_j, offs)
        nk = [ranges.node_range(two_l, n)[1] for n in (2, 3, 4, 5)]
        if all(nk):
            nonempty += 1
            total_w += 3 * math.prod(nk)
    assert nonempty == 729
    assert total_w == 83124
    two_l = ranges.shell_spins(two_j, (1, 0, 0, 0, 0, 2))         # shell (2,1,1,1,1,3)
    assert [ranges.node_range(two_l, n) for n in (2, 3, 4, 5)] == [(2, 2), (2, 2), (4, 1), (4, 1)]


def _vector_counts(two_j, dl):
    """numpy enumeration of all shells: number of non-empty shells and sum of E_W."""
    nl = dl + 1
    o = np.indices((nl,) * 6).reshape(6, -1)
    l = {s: two_j[s] + 2 * o[p] for p, s in enumerate(ranges.VIRTUAL)}
    for s in (J12, J13, J14, J15):
        l[s] = np.full(o.shape[1], two_j[s])
    prod = np.ones(o.shape[1], dtype=np.int64)
    for node in (2, 3, 4, 5):
        a, b, c, d = (l[s] for s in ranges.NODE_SPINS[node - 1])
        lo = np.maximum(np.abs(a - b), np.abs(c - d))
        hi = np.minimum(a + b, c + d)
        n = np.where(hi >= lo, (hi - lo) // 2 + 1, 0)
        prod *= n
    n1 = ranges.boundary_ranges(two_j)[0][1]
    return int((prod > 0).sum()), int(prod.sum()) * n1


def test_survey_counts_config2_config3():
    assert _vector_counts([6] * 10, 8)[0] == 498955               # non-empty shells at dl = 8
    assert _vector_counts([6] * 10, 7)[0] == 256227
    nonempty, total_w = _vector_counts([10] * 10, 10)
    assert nonempty == 1771561 and total_w == 159216924306


def test_vector_counts_agree_with_scalar_code():
    two_j = [8, 7, 12, 3, 8, 5, 9, 12, 3, 7]                      # SURVEY.md 8(d), config 4 base spins
    nonempty, total_w = 0, 0
    for offs in ranges.shells(2):
        two_l = ranges.shell_spins(two_j, offs)
        nk = [ranges.node_range(two_l, n)[1] for n in (2, 3, 4, 5)]
        nonempty += all(nk)
        total_w += math.prod(nk)
    n1 = ranges.boundary_ranges(two_j)[0][1]
    assert _vector_counts(two_j, 1) == (nonempty, total_w * n1)
    assert [n for _, n in ranges.boundary_ranges(two_j)] == [4, 6, 4, 6, 3]


def test_booster_dims_and_triple_index():
    two_j, two_dl = [2] * 10, 4
    for edge in (2, 3, 4, 5):
        kr = ranges.booster_k_ranges(two_j, two_dl, edge)
        assert len(kr) == 27
        nt, n_i, i_min, base, pad = ranges.booster_dims(two_j, two_dl, edge)
        assert (nt, n_i, i_min) == (27, 3, 0)
        for offs in ranges.shells(two_dl):
            t = ranges.triple_index(edge, offs, two_dl)
            assert kr[t] == ranges.node_range(ranges.shell_spins(two_j, offs), edge)
        assert base == min(lo for lo, n in kr if n) and pad >= max(n for _, n in kr)
    # max n_k = 2 j_1a + 1 regardless of Delta_l
    for dl in (0, 2, 5):
        for edge in (2, 3, 4, 5):
            assert max(n for _, n in ranges.booster_k_ranges([6] * 10, 2 * dl, edge)) == 7


# ------------------------------------------------------------------------------------------------ {15j}

def _golden_15j(golden_dir):
    for line in open(os.path.join(golden_dir, "fifteenj_exact_values.txt")):
        if line.startswith("#") or not line.strip():
            continue
        spins, intw, val = (part.split() for part in line.split("|"))
        p, q, r = (int(v) for v in val)
        yield [int(v) for v in spins], [int(v) for v in intw], p / q * math.sqrt(r)


def test_golden_exact_values(golden_dir):
    rows = 0
    for two_l, intw, value in _golden_15j(golden_dir):
        got = fifteenj.fifteenj(two_l, intw[0], intw[1:])
        assert got == pytest.approx(value, rel=4e-16, abs=0), (two_l, intw)
        rows += 1
    assert rows == 16


def test_brute_force_all_spins_half():
    # "brute force on j = 1/2" (BASELINE.json north_star): all 32 entries, sign included
    two_l = [1] * 10
    for intw in itertools.product((0, 2), repeat=5):
        assert fifteenj.fifteenj(two_l, intw[0], intw[1:]) == pytest.approx(
            fifteenj.brute_force_15j(two_l, intw), abs=1e-15)


def test_brute_force_spin_one_and_mixed():
    rng = random.Random(7)
    two_l = [2] * 10
    all_intw = list(itertools.product((0, 2, 4), repeat=5))
    for intw in rng.sample(all_intw, 12):
        assert fifteenj.fifteenj(two_l, intw[0], intw[1:]) == pytest.approx(
            fifteenj.brute_force_15j(two_l, intw), abs=1e-15)
    # non-homogeneous spin sets with half-integers: every node must have an integer spin sum
    done = 0
    while done < 6:
        two_l = [rng.randint(1, 3) for _ in range(10)]
        rs = [ranges.node_range(two_l, n) for n in range(1, 6)]
        if any(n == 0 for _, n in rs):
            continue
        intw = [lo + 2 * rng.randrange(n) for lo, n in rs]
        ref = fifteenj.brute_force_15j(two_l, intw)
        assert fifteenj.fifteenj(two_l, intw[0], intw[1:]) == pytest.approx(ref, abs=1e-15), (two_l, intw)
        done += 1


def test_sign_exponent_is_integer_on_valid_labels():
    rng = random.Random(1)
    for _ in range(200):
        two_l = [rng.randint(1, 9) for _ in range(10)]
        rs = [ranges.node_range(two_l, n) for n in range(1, 6)]
        if any(n == 0 for _, n in rs):
            continue
        intw = [lo + 2 * rng.randrange(n) for lo, n in rs]
        fifteenj.sign_exponent(two_l, intw[0], intw[1:])     # asserts integrality (reading G13)


def test_collapse_to_single_sixj():
    # i1 = 0 and k4 = 0 force j12=j13=a, j14=j15=l45=b, l24=l34=c, l25=l35=d, l23=e, x=d and
    # |{15j}| = |{c k3 d; a k2 e}| / ((2b+1)(2d+1) sqrt((2a+1)(2c+1)))
    rng = random.Random(9)
    done = 0
    while done < 10:
        a, b, c, d, e = (rng.randint(1, 6) for _ in range(5))
        two_l = [0] * 10
        two_l[J12] = two_l[J13] = a
        two_l[J14] = two_l[J15] = two_l[J45] = b
        two_l[J24] = two_l[J34] = c
        two_l[J25] = two_l[J35] = d
        two_l[J23] = e
        rs = [ranges.node_range(two_l, n) for n in range(1, 6)]
        if any(n == 0 for _, n in rs) or rs[0][0] != 0 or rs[3][0] != 0:
            continue
        k2 = rs[1][0] + 2 * rng.randrange(rs[1][1])
        k3 = rs[2][0] + 2 * rng.randrange(rs[2][1])
        k5 = rs[4][0] + 2 * rng.randrange(rs[4][1])
        val = fifteenj.fifteenj(two_l, 0, (k2, k3, 0, k5))
        ref = abs(wigner.sixj(c, k3, d, a, k2, e)) / ((b + 1) * (d + 1) * math.sqrt((a + 1) * (c + 1)))
        assert abs(val) == pytest.approx(ref, rel=1e-14, abs=1e-300), (a, b, c, d, e, k2, k3, k5)
        done += 1
