"""Exact SU(2) recoupling symbols in Python big-integer arithmetic (oracle; test infrastructure).

All spins are passed as integers two_j = 2j.

The paper evaluates Wigner symbols with WIGXJPF/FASTWIGXJ, "prime factorisation and
multi-word integer arithmetic" (ref. [31] PAPER.md:621).  The quantity those
libraries evaluate is the textbook Racah single-sum formula; this file is that formula
written out with Python's unbounded integers, so every intermediate is exact and the only
rounding is the final square root (taken at FIXED_BITS bits, then rounded once to double).

Nothing here is shared with the CUDA path.
"""
from fractions import Fraction
from functools import lru_cache
from math import isqrt

FIXED_BITS = 256  # fixed-point precision used when an irrational value must be represented

_FACT = [1]


def fact(n):
    """n! as an exact integer (n >= 0)."""
    if n < 0:
        raise ValueError("factorial of negative number")
    while len(_FACT) <= n:
        _FACT.append(_FACT[-1] * len(_FACT))
    return _FACT[n]


def is_triad(two_a, two_b, two_c):
    """True iff (a,b,c) can couple: a+b+c integer and |a-b| <= c <= a+b."""
    if (two_a + two_b + two_c) % 2:
        return False
    return abs(two_a - two_b) <= two_c <= two_a + two_b


def delta2(two_a, two_b, two_c):
    """Triangle coefficient squared, Delta^2(a,b,c) = (a+b-c)!(a-b+c)!(-a+b+c)!/(a+b+c+1)!  (exact)."""
    return Fraction(
        fact((two_a + two_b - two_c) // 2) * fact((two_a - two_b + two_c) // 2) * fact((-two_a + two_b + two_c) // 2),
        fact((two_a + two_b + two_c) // 2 + 1),
    )


def sixj_parts(two_a, two_b, two_c, two_d, two_e, two_f):
    """{a b c; d e f} = N * sqrt(D) with N an exact integer (Racah sum) and D an exact rational.

    Racah's formula:  D = D2(abc) D2(aef) D2(dbf) D2(dec),
      N = sum_t (-1)^t (t+1)! / [ prod_i (t-alpha_i)!  prod_j (beta_j-t)! ],
      alpha = (a+b+c, a+e+f, d+b+f, d+e+c),  beta = (a+b+d+e, a+c+d+f, b+c+e+f),
      t from max(alpha) to min(beta).
    Returns (0, 0) when a triad is violated (the symbol vanishes by definition).
    """
    a, b, c, d, e, f = two_a, two_b, two_c, two_d, two_e, two_f
    if min(a, b, c, d, e, f) < 0:
        raise ValueError("negative spin")
    if not (is_triad(a, b, c) and is_triad(a, e, f) and is_triad(d, b, f) and is_triad(d, e, c)):
        return 0, Fraction(0)
    alpha = ((a + b + c) // 2, (a + e + f) // 2, (d + b + f) // 2, (d + e + c) // 2)
    beta = ((a + b + d + e) // 2, (a + c + d + f) // 2, (b + c + e + f) // 2)
    total = 0
    for t in range(max(alpha), min(beta) + 1):
        den = 1
        for al in alpha:
            den *= fact(t - al)
        for be in beta:
            den *= fact(be - t)
        # the seven factorial arguments add up to t, so (t+1)!/den = (t+1) * multinomial is an integer
        term, rem = divmod(fact(t + 1), den)
        assert rem == 0
        total += -term if t % 2 else term
    D = delta2(a, b, c) * delta2(a, e, f) * delta2(d, b, f) * delta2(d, e, c)
    return total, D


@lru_cache(maxsize=None)
def sixj_fixed(two_a, two_b, two_c, two_d, two_e, two_f):
    """{6j} as a fixed-point integer: value = result / 2^FIXED_BITS (error < 2^-(FIXED_BITS-2))."""
    N, D = sixj_parts(two_a, two_b, two_c, two_d, two_e, two_f)
    if N == 0:
        return 0
    # 6j = sign(N) * sqrt(N^2 D), N^2 D exact rational
    q = N * N * D
    r = isqrt((q.numerator << (2 * FIXED_BITS)) // q.denominator)
    return r if N > 0 else -r


def fixed_to_float(v, bits=FIXED_BITS):
    """Round a fixed-point integer to the nearest double (Python int/int division is correctly rounded)."""
    return v / (1 << bits)


def sixj(two_a, two_b, two_c, two_d, two_e, two_f):
    """{6j} rounded once to double."""
    return fixed_to_float(sixj_fixed(two_a, two_b, two_c, two_d, two_e, two_f))


def sixj_squared(two_a, two_b, two_c, two_d, two_e, two_f):
    """(sign, exact rational value of {6j}^2) -- used by pins that compare with printed rationals."""
    N, D = sixj_parts(two_a, two_b, two_c, two_d, two_e, two_f)
    sign = (N > 0) - (N < 0)
    return sign, N * N * D


# ----------------------------------------------------------------------------------------------
# 3jm and 4jm symbols: only needed by the brute-force pin of eq. (5) (fifteenj.brute_force_15j).
# ----------------------------------------------------------------------------------------------

def threejm_parts(two_j1, two_j2, two_j3, two_m1, two_m2, two_m3):
    """Wigner 3jm symbol (j1 j2 j3; m1 m2 m3) = N * sqrt(D), N exact rational, D exact rational.

    Racah's formula:
      (-1)^{j1-j2-m3} sqrt(Delta^2(j1 j2 j3)) sqrt((j1+m1)!(j1-m1)!(j2+m2)!(j2-m2)!(j3+m3)!(j3-m3)!)
        * sum_t (-1)^t / [ t! (j3-j2+t+m1)! (j3-j1+t-m2)! (j1+j2-j3-t)! (j1-t-m1)! (j2-t+m2)! ]
    """
    j1, j2, j3, m1, m2, m3 = two_j1, two_j2, two_j3, two_m1, two_m2, two_m3
    if m1 + m2 + m3 != 0 or not is_triad(j1, j2, j3):
        return Fraction(0), Fraction(0)
    for j, m in ((j1, m1), (j2, m2), (j3, m3)):
        if abs(m) > j or (j + m) % 2:
            return Fraction(0), Fraction(0)
    D = delta2(j1, j2, j3)
    for j, m in ((j1, m1), (j2, m2), (j3, m3)):
        D *= fact((j + m) // 2) * fact((j - m) // 2)
    tmin = max(0, (j2 - j3 - m1) // 2, (j1 - j3 + m2) // 2)
    tmax = min((j1 + j2 - j3) // 2, (j1 - m1) // 2, (j2 + m2) // 2)
    total = Fraction(0)
    for t in range(tmin, tmax + 1):
        den = (fact(t) * fact((j3 - j2 + m1) // 2 + t) * fact((j3 - j1 - m2) // 2 + t)
               * fact((j1 + j2 - j3) // 2 - t) * fact((j1 - m1) // 2 - t) * fact((j2 + m2) // 2 - t))
        total += Fraction(-1 if t % 2 else 1, den)
    if ((j1 - j2 - m3) // 2) % 2:
        total = -total
    return total, D


@lru_cache(maxsize=None)
def threejm(two_j1, two_j2, two_j3, two_m1, two_m2, two_m3):
    """3jm symbol as a double (sqrt of the exact rational taken at FIXED_BITS bits)."""
    N, D = threejm_parts(two_j1, two_j2, two_j3, two_m1, two_m2, two_m3)
    if N == 0:
        return 0.0
    q = N * N * D
    r = isqrt((q.numerator << (2 * FIXED_BITS)) // q.denominator)
    return fixed_to_float(r if N > 0 else -r)


def fourjm(two_j, two_m, two_i):
    """The paper's 4jm symbol with intertwiner i, eq. (4) first line, in the convention

        (j1 j2 j3 j4; m1 m2 m3 m4)^{(i)} = sum_m (-1)^{i-m} (j1 j2 i; m1 m2 m) (i j3 j4; -m m3 m4)

    i.e. i recouples (j1 j2) with (j3 j4)  (the normalisation sqrt(2i+1) is the
    explicit prefactor of eq. (3), not part of the symbol).
    """
    j1, j2, j3, j4 = two_j
    m1, m2, m3, m4 = two_m
    two_m_int = -(m1 + m2)  # the only m for which the first 3jm can be non-zero
    if abs(two_m_int) > two_i or (two_i + two_m_int) % 2:
        return 0.0
    phase = -1.0 if ((two_i - two_m_int) // 2) % 2 else 1.0
    return phase * threejm(j1, j2, two_i, m1, m2, two_m_int) * threejm(two_i, j3, j4, -two_m_int, m3, m4)
