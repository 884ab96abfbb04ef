"""Pins for oracle/wigner.py: the exact {6j} and 3jm symbols are checked against what the mathematics fixes
(closed forms, symmetries, orthogonality, Racah and Biedenharn-Elliott identities), against printed exact
values (tests/golden/) and against an independent library (sympy).  A dropped term, a wrong sign or a
transposed argument anywhere in the Racah sum fails at least one of them."""
import itertools
import os
import random
from fractions import Fraction

import pytest

from oracle import wigner
from oracle.wigner import FIXED_BITS, is_triad, sixj, sixj_fixed, sixj_squared

ONE = 1 << FIXED_BITS
TOL = 1 << (FIXED_BITS - 200)      # identities must hold to ~2^-200 in fixed point


def fx_mul(*vals):
    p = ONE
    for v in vals:
        p = (p * v) >> FIXED_BITS
    return p


def random_valid_sixj(rng, jmax):
    """Six spins (2j) satisfying all four triads, built triad by triad."""
    while True:
        a, b, e = (rng.randint(0, jmax) for _ in range(3))
        cs = [c for c in range(abs(a - b), min(a + b, jmax) + 1, 2)]
        fs = [f for f in range(abs(a - e), min(a + e, jmax) + 1, 2)]
        if not cs or not fs:
            continue
        c, f = rng.choice(cs), rng.choice(fs)
        ds = [d for d in range(0, jmax + 1) if is_triad(d, b, f) and is_triad(d, e, c)]
        if ds:
            return a, b, c, rng.choice(ds), e, f


def test_golden_exact_values(golden_dir):
    rows = 0
    for line in open(os.path.join(golden_dir, "sixj_exact_values.txt")):
        if line.startswith("#") or not line.strip():
            continue
        vals = [int(v) for v in line.split()]
        spins, value = vals[:6], Fraction(vals[6], vals[7])
        sign, sq = sixj_squared(*spins)
        assert sq == value * value, spins
        assert sign == (value > 0) - (value < 0), spins
        assert sixj(*spins) == pytest.approx(float(value), rel=1e-15, abs=0)
        rows += 1
    assert rows == 9


def test_closed_form_zero_spin():
    # {a b c; 0 c b} = (-1)^{a+b+c} / sqrt((2b+1)(2c+1))
    for a, b, c in itertools.product(range(0, 13), repeat=3):
        if not is_triad(a, b, c):
            continue
        sign, sq = sixj_squared(a, b, c, 0, c, b)
        assert sq == Fraction(1, (b + 1) * (c + 1))
        assert sign == (-1) ** ((a + b + c) // 2)


def test_vanishes_when_a_triad_fails():
    assert sixj(2, 2, 6, 2, 2, 2) == 0.0       # (1,1,3) not a triangle
    assert sixj(1, 2, 2, 2, 2, 2) == 0.0       # half-integer sum
    assert sixj(2, 2, 2, 2, 2, 6) == 0.0


def test_tetrahedral_symmetries():
    rng = random.Random(11)
    for _ in range(60):
        s = random_valid_sixj(rng, 24)
        ref = sixj_fixed(*s)
        cols = [(s[0], s[3]), (s[1], s[4]), (s[2], s[5])]
        seen = 0
        for perm in itertools.permutations(range(3)):
            pc = [cols[p] for p in perm]
            for flips in ((0, 0, 0), (1, 1, 0), (1, 0, 1), (0, 1, 1)):   # swap upper/lower in two columns
                up = [pc[i][flips[i]] for i in range(3)]
                lo = [pc[i][1 - flips[i]] for i in range(3)]
                assert sixj_fixed(*up, *lo) == ref
                seen += 1
        assert seen == 24


def test_regge_symmetry():
    # {a b c; d e f} = {a, (b+c+e-f)/2, (b+c+f-e)/2; d, (b+e+f-c)/2, (c+e+f-b)/2}   (j units)
    rng = random.Random(5)
    for _ in range(40):
        a, b, c, d, e, f = random_valid_sixj(rng, 20)
        if (b + c + e + f) % 4 != 0:      # need the new 2j values to be integers: (b+c+e-f)/2 in 2j units
            continue
        reg = (a, (b + c + e - f) // 2, (b + c + f - e) // 2, d, (b + e + f - c) // 2, (c + e + f - b) // 2)
        assert sixj_fixed(*reg) == sixj_fixed(a, b, c, d, e, f)


def test_orthogonality():
    # sum_x (2x+1)(2p+1) {a b x; c d p}{a b x; c d q} = delta_pq
    rng = random.Random(3)
    for _ in range(25):
        a, b, c, d = (rng.randint(0, 14) for _ in range(4))
        ps = [p for p in range(0, 40) if is_triad(a, d, p) and is_triad(c, b, p)]
        xs = [x for x in range(0, 40) if is_triad(a, b, x) and is_triad(c, d, x)]
        for p, q in itertools.product(ps[:3], ps[:3]):
            tot = sum((x + 1) * (p + 1) * fx_mul(sixj_fixed(a, b, x, c, d, p), sixj_fixed(a, b, x, c, d, q)) for x in xs)
            assert abs(tot - (ONE if p == q else 0)) < TOL, (a, b, c, d, p, q)


def test_racah_sum_rule():
    # sum_x (-1)^{p+q+x} (2x+1) {a b x; c d p}{a b x; d c q} = {a c q; b d p}
    rng = random.Random(8)
    n = 0
    while n < 25:
        a, b, c, d = (rng.randint(0, 12) for _ in range(4))
        ps = [p for p in range(0, 30) if is_triad(a, d, p) and is_triad(c, b, p)]
        qs = [q for q in range(0, 30) if is_triad(a, c, q) and is_triad(d, b, q)]
        if not ps or not qs:
            continue
        p, q = rng.choice(ps), rng.choice(qs)
        xs = [x for x in range(0, 30) if is_triad(a, b, x) and is_triad(c, d, x)]
        tot = 0
        for x in xs:
            assert (p + q + x) % 2 == 0
            s = -1 if ((p + q + x) // 2) % 2 else 1
            tot += s * (x + 1) * fx_mul(sixj_fixed(a, b, x, c, d, p), sixj_fixed(a, b, x, d, c, q))
        assert abs(tot - sixj_fixed(a, c, q, b, d, p)) < TOL, (a, b, c, d, p, q)
        n += 1


def test_biedenharn_elliott():
    # sum_x (-1)^{S+x}(2x+1){a b x; c d g}{c d x; e f h}{e f x; b a j} = {g h j; e a d}{g h j; f b c}
    rng = random.Random(21)
    n = 0
    while n < 25:
        a, b, c, d, e, f = (rng.randint(0, 10) for _ in range(6))
        gs = [g for g in range(0, 24) if is_triad(a, d, g) and is_triad(c, b, g)]
        hs = [h for h in range(0, 24) if is_triad(c, f, h) and is_triad(e, d, h)]
        js = [j for j in range(0, 24) if is_triad(e, a, j) and is_triad(b, f, j)]
        if not gs or not hs or not js:
            continue
        g, h, j = rng.choice(gs), rng.choice(hs), rng.choice(js)
        if not is_triad(g, h, j):
            continue
        S2 = a + b + c + d + e + f + g + h + j
        tot = 0
        for x in range(0, 24):
            if not (is_triad(a, b, x) and is_triad(c, d, x) and is_triad(e, f, x)):
                continue
            assert (S2 + x) % 2 == 0
            s = -1 if ((S2 + x) // 2) % 2 else 1
            tot += s * (x + 1) * fx_mul(sixj_fixed(a, b, x, c, d, g), sixj_fixed(c, d, x, e, f, h),
                                        sixj_fixed(e, f, x, b, a, j))
        rhs = fx_mul(sixj_fixed(g, h, j, e, a, d), sixj_fixed(g, h, j, f, b, c))
        assert abs(tot - rhs) < TOL, (a, b, c, d, e, f, g, h, j)
        n += 1


def test_against_sympy():
    from sympy import Rational
    from sympy.physics.wigner import wigner_6j

    rng = random.Random(2)
    for _ in range(40):
        s = random_valid_sixj(rng, 30)
        ref = float(wigner_6j(*[Rational(v, 2) for v in s]).evalf(30))
        assert sixj(*s) == pytest.approx(ref, rel=2e-15, abs=1e-300)


def test_large_spin_symmetry_and_orthogonality():
    # the regime of config 4 (two_x up to ~140): exactness must not depend on size
    a, b, c, d = 70, 64, 58, 76
    ps = [p for p in range(0, 160) if is_triad(a, d, p) and is_triad(c, b, p)]
    xs = [x for x in range(0, 160) if is_triad(a, b, x) and is_triad(c, d, x)]
    p = ps[len(ps) // 2]
    tot = sum((x + 1) * (p + 1) * fx_mul(sixj_fixed(a, b, x, c, d, p), sixj_fixed(a, b, x, c, d, p)) for x in xs)
    assert abs(tot - ONE) < TOL


def test_threejm_against_sympy_and_orthogonality():
    from sympy import Rational
    from sympy.physics.wigner import wigner_3j

    rng = random.Random(4)
    n = 0
    while n < 60:
        j1, j2 = rng.randint(0, 8), rng.randint(0, 8)
        j3 = rng.choice(range(abs(j1 - j2), j1 + j2 + 1, 2))
        m1, m2 = rng.choice(range(-j1, j1 + 1, 2)), rng.choice(range(-j2, j2 + 1, 2))
        m3 = -m1 - m2
        if abs(m3) > j3:
            continue
        ref = float(wigner_3j(*[Rational(v, 2) for v in (j1, j2, j3, m1, m2, m3)]))
        assert wigner.threejm(j1, j2, j3, m1, m2, m3) == pytest.approx(ref, rel=1e-14, abs=1e-16)
        n += 1
    # sum_{m1 m2} (2j3+1) (j1 j2 j3; m1 m2 m3)^2 = 1
    for j1, j2, j3 in ((2, 3, 3), (4, 4, 6), (1, 1, 2)):
        for m3 in range(-j3, j3 + 1, 2):
            tot = sum(wigner.threejm(j1, j2, j3, m1, -m3 - m1, m3) ** 2
                      for m1 in range(-j1, j1 + 1, 2) if abs(-m3 - m1) <= j2)
            assert (j3 + 1) * tot == pytest.approx(1.0, rel=1e-14)


def test_sixj_class_representatives_by_brute_force():
    """oracle/sixj_classes.c lists one symbol per class of the 24 tetrahedral symmetries.  Pin: for 2j <= 6 group ALL 7^6
    label tuples with valid triads into orbits of the 24 images written out by hand here (column permutations, upper/lower
    exchange in two columns) and take the largest image of each orbit: the same set, nothing twice; and every image of a
    representative has the same exact value (the symmetries are symmetries of the symbol)."""
    import itertools

    from oracle import sixj_classes

    def images(t):
        a, b, c, d, e, f = t
        cols = [(a, d), (b, e), (c, f)]
        out = set()
        for p in itertools.permutations(cols):
            for fl in ((0, 0, 0), (1, 1, 0), (1, 0, 1), (0, 1, 1)):
                out.add(tuple(p[q][fl[q]] for q in range(3)) + tuple(p[q][1 - fl[q]] for q in range(3)))
        return out

    J = 6
    valid = [t for t in itertools.product(range(J + 1), repeat=6)
             if is_triad(t[0], t[1], t[2]) and is_triad(t[0], t[4], t[5]) and is_triad(t[3], t[1], t[5])
             and is_triad(t[3], t[4], t[2])]
    want = {max(images(t)) for t in valid}
    got = [tuple(int(v) for v in row) for row in sixj_classes.all_classes(J)]
    assert len(got) == len(set(got)) == len(want) and set(got) == want
    assert sum(len(images(t)) for t in want) == len(valid)            # the orbits partition the valid tuples
    for t in got[::7]:
        assert len({sixj_fixed(*im) for im in images(t)}) == 1
    # a larger bound, counts only: every representative is valid, maximal among its images, and below the bound
    J = 12
    reps = sixj_classes.all_classes(J)
    assert reps.max() <= J and reps.min() >= 0
    for row in reps[::97]:
        t = tuple(int(v) for v in row)
        assert t == max(images(t)) and wigner.sixj_parts(*t)[1] != 0
