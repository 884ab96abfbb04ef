"""Pins for oracle/vertex.py (+ vertex_l1.c): eq. (3) of the paper.

  * BF reduction (reading G8): identity boosters, Delta_l = 0  =>  A = N(i) {15j}, with the {15j} values
    of tests/golden/ and of the brute-force contraction
  * one-hot boosters pick a single W entry (pins the irregular k-range indexing)
  * L0 (literal nested sum) == L1 (S arrays + C loops) on tiny inputs
  * multilinearity in each booster, additivity over disjoint shell ranges
  * double vs long double accumulation << tolerance
"""
import itertools
import math
import random

import numpy as np
import pytest

import workloads as wl
from oracle import fifteenj, ranges, vertex
from oracle_dims import dims, spins_valid


def _bf(two_j):
    L = vertex.Layout(two_j, 0)
    edge_dims, _ = dims(two_j, 0)
    B = wl.identity_boosters(edge_dims, L.two_i_min)
    return L, vertex.vertex_l1(two_j, 0, B)


def test_bf_reduction_spin_half_exact_values():
    L, r = _bf([1] * 10)
    A = r["A"]
    assert A.shape == (2,) * 5 and r["nonempty"] == 1
    assert A[0, 0, 0, 0, 0] == pytest.approx(1 / 16, rel=1e-15)
    assert A[1, 1, 1, 1, 1] == pytest.approx(3 ** 2.5 * 3 ** 4 * (-7 / 432), rel=1e-15)
    N = vertex.bf_normalisation(L)
    for idx in itertools.product(range(2), repeat=5):
        intw = [2 * a for a in idx]
        assert A[idx] / N[idx] == pytest.approx(fifteenj.brute_force_15j([1] * 10, intw), abs=1e-15)


@pytest.mark.parametrize("two_j", [2, 3, 4])
def test_bf_reduction_equals_15j(two_j):
    L, r = _bf([two_j] * 10)
    N = vertex.bf_normalisation(L)
    rng = random.Random(two_j)
    n = L.n_i[0]
    for idx in [tuple(rng.randrange(n) for _ in range(5)) for _ in range(40)]:
        intw = [lo + 2 * a for lo, a in zip(L.two_i_min, idx)]
        ref = fifteenj.fifteenj([two_j] * 10, intw[0], intw[1:])
        assert r["A"][idx] / N[idx] == pytest.approx(ref, rel=1e-13, abs=1e-18)


def test_bf_reduction_nonhomogeneous():
    two_j = [8, 7, 12, 3, 8, 5, 9, 12, 3, 7]
    assert spins_valid(two_j)
    L, r = _bf(two_j)
    assert L.n_i == [4, 6, 4, 6, 3]
    N = vertex.bf_normalisation(L)
    for idx in itertools.product(*[range(n) for n in L.n_i]):
        intw = [lo + 2 * a for lo, a in zip(L.two_i_min, idx)]
        ref = fifteenj.fifteenj(two_j, intw[0], intw[1:])
        assert r["A"][idx] / N[idx] == pytest.approx(ref, rel=1e-13, abs=1e-18)


def test_one_hot_boosters_pick_one_w_entry():
    two_j, two_dl = [2] * 10, 4
    L = vertex.Layout(two_j, two_dl)
    edge_dims, k_ranges = dims(two_j, two_dl)
    rng = random.Random(3)
    for _ in range(6):
        offs = tuple(rng.randrange(3) for _ in range(6))
        two_l = ranges.shell_spins(two_j, offs)
        hot, ks, iis = {}, [], []
        for edge in (2, 3, 4, 5):
            t = ranges.triple_index(edge, offs, two_dl)
            lo, nk = k_ranges[edge][t]
            k = lo + 2 * rng.randrange(nk)
            ii = rng.randrange(L.n_i[edge - 1])
            hot[edge] = (t, ii, (k - L.two_k_base[edge - 2]) // 2)
            ks.append(k)
            iis.append(ii)
        B = wl.one_hot_boosters(3, edge_dims, hot)
        A = vertex.vertex_l1(two_j, two_dl, B)["A"]
        # only shells sharing all four triples with `offs` contribute; the triples determine the shell
        expect = np.zeros_like(A)
        for a1 in range(L.n_i[0]):
            i1 = L.two_i_min[0] + 2 * a1
            norm = math.sqrt((i1 + 1) * math.prod(L.two_i_min[e] + 2 * ii + 1 for e, ii in zip((1, 2, 3, 4), iis)))
            expect[(a1, *iis)] = norm * math.prod(k + 1 for k in ks) * fifteenj.fifteenj(two_l, i1, ks)
        assert np.allclose(A, expect, rtol=1e-13, atol=1e-18)
        assert np.count_nonzero(A) <= L.n_i[0]


def _config0():
    c = wl.CONFIGS[0]
    edge_dims, k_ranges = dims(c["two_j"], c["two_dl"])
    return c, wl.random_boosters(c["seed"], 3, edge_dims, k_ranges), edge_dims, k_ranges


def test_l0_equals_l1_config0_entries():
    c, B, _, _ = _config0()
    r = vertex.vertex_l1(c["two_j"], c["two_dl"], B)
    assert r["nonempty"] == 729
    for idx in ((0, 0, 0, 0, 0), (1, 0, 2, 1, 1), (2, 2, 2, 2, 2), (0, 1, 2, 0, 1)):
        a, s = vertex.vertex_l0_entry(c["two_j"], c["two_dl"], B, [2 * v for v in idx])
        assert r["A"][idx] == pytest.approx(a, abs=1e-13 * s)
        assert r["Aabs"][idx] == pytest.approx(s, rel=1e-12)


def test_l0_equals_l1_half_integer_shelled():
    two_j, two_dl = [1] * 10, 2
    edge_dims, k_ranges = dims(two_j, two_dl)
    B = wl.random_boosters(5, 2, edge_dims, k_ranges)
    r = vertex.vertex_l1(two_j, two_dl, B)
    for idx in itertools.product(range(2), repeat=5):
        a, s = vertex.vertex_l0_entry(two_j, two_dl, B, [2 * v for v in idx])
        assert r["A"][idx] == pytest.approx(a, abs=1e-13 * s)


def test_multilinear_and_additive_over_shell_ranges():
    c, B, edge_dims, k_ranges = _config0()
    full = vertex.vertex_l1(c["two_j"], c["two_dl"], B)
    # additivity over disjoint ranges of the canonical shell order
    parts = [vertex.vertex_l1(c["two_j"], c["two_dl"], B, lo, hi) for lo, hi in ((0, 100), (100, 101), (101, 729))]
    assert sum(p["nonempty"] for p in parts) == 729
    assert np.allclose(sum(p["A"] for p in parts), full["A"], rtol=0, atol=1e-13 * full["Aabs"].max())
    # linearity in B3
    B2nd = wl.random_boosters(c["seed"] + 1, 3, edge_dims, k_ranges)
    mix = dict(B)
    mix[3] = 2.0 * B[3] - 0.5 * B2nd[3]
    other = dict(B)
    other[3] = B2nd[3]
    lhs = vertex.vertex_l1(c["two_j"], c["two_dl"], mix)["A"]
    rhs = 2.0 * full["A"] - 0.5 * vertex.vertex_l1(c["two_j"], c["two_dl"], other)["A"]
    assert np.allclose(lhs, rhs, rtol=0, atol=1e-12 * full["Aabs"].max())


def test_double_vs_long_double_far_below_tolerance():
    c, B, _, _ = _config0()
    ld = vertex.vertex_l1(c["two_j"], c["two_dl"], B, long_double=True)
    d = vertex.vertex_l1(c["two_j"], c["two_dl"], B, long_double=False, threads=3)
    assert (np.abs(ld["A"] - d["A"]) <= 1e-14 * ld["Aabs"]).all()


def test_config4_spin_draw_matches_survey():
    two_j, draws = wl.config4_base_spins(spins_valid)
    assert two_j == [8, 7, 12, 3, 8, 5, 9, 12, 3, 7] and draws == 43


def test_layout_rejects_bad_input():
    with pytest.raises(ValueError):
        vertex.Layout([2] * 10, 3)
    with pytest.raises(ValueError):
        vertex.Layout([2, 2, 2, 2, 2, 2, 2, 2, 2, 9], 0)
