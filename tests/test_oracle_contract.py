"""Pins of the contraction oracle (oracle/contract.py): closed forms and brute force, so that a
transposed index, a conjugation or a dropped factor fails."""
import itertools

import numpy as np
import pytest

from oracle import contract as oc


def _rng(seed):
    return np.random.Generator(np.random.PCG64(seed))


def test_product_tensor_factorises():
    """A = u1 x u2 x u3 x u4 x u5  =>  sum A psi1..psi5 = prod_e (u_e . psi_e), no conjugation."""
    rng = _rng(1)
    dims = (2, 3, 4, 3, 5)
    u = [rng.normal(size=n) for n in dims]
    psi = [rng.normal(size=n) + 1j * rng.normal(size=n) for n in dims]
    A = np.einsum("a,b,c,d,e->abcde", *u)
    val, scale = oc.contract_vectors(A, psi)
    ref = np.prod([np.dot(u[e], psi[e]) for e in range(5)])
    assert abs(val - ref) <= 1e-13 * scale
    # a different vector on every node: swapping two of them must change the result (index order is pinned)
    if dims[1] == dims[3]:
        swapped, _ = oc.contract_vectors(A, [psi[0], psi[3], psi[2], psi[1], psi[4]])
        assert abs(swapped - val) > 1e-6 * abs(val)


def test_one_hot_vectors_pick_one_entry():
    rng = _rng(2)
    dims = (3, 2, 4, 2, 3)
    A = rng.normal(size=dims)
    for idx in [(0, 0, 0, 0, 0), (2, 1, 3, 0, 2), (1, 0, 2, 1, 1)]:
        psi = [np.zeros(n, dtype=complex) for n in dims]
        for e, i in enumerate(idx):
            psi[e][i] = 1.0
        psi[2][idx[2]] = 1j                      # one imaginary unit: the result is i A[idx]
        val, _ = oc.contract_vectors(A, psi)
        assert val == 1j * A[idx]


def test_brute_force_loops():
    rng = _rng(3)
    dims = (2, 2, 3, 2, 2)
    A = rng.normal(size=dims)
    B = rng.normal(size=dims)
    psi = [rng.normal(size=n) + 1j * rng.normal(size=n) for n in dims]
    s, d = 0j, 0.0
    for idx in itertools.product(*[range(n) for n in dims]):
        term = A[idx]
        for e in range(5):
            term = term * psi[e][idx[e]]
        s += term
        d += A[idx] * B[idx]
    val, scale = oc.contract_vectors(A, psi)
    assert abs(val - s) <= 1e-14 * scale
    dot, dscale = oc.contract_vertices(A, B)
    assert abs(dot - d) <= 1e-14 * dscale


def test_vertex_vertex_closed_forms():
    rng = _rng(4)
    A = rng.normal(size=(3, 3, 3, 3, 3))
    nrm, scale = oc.contract_vertices(A, A)
    assert nrm == pytest.approx(np.linalg.norm(A.ravel()) ** 2, rel=1e-14) and scale == pytest.approx(nrm, rel=1e-15)
    ones = np.ones((2, 3, 2, 3, 2))
    assert oc.contract_vertices(ones, ones)[0] == 72.0
    # orthogonal by construction: even and odd entries
    E = np.zeros(32); E[0::2] = 1.0
    O = np.zeros(32); O[1::2] = 1.0
    assert oc.contract_vertices(E.reshape(2, 2, 2, 2, 2), O.reshape(2, 2, 2, 2, 2))[0] == 0.0
    # exact summation: catastrophic cancellation that a naive left-to-right fp64 sum gets wrong
    a = np.array([1e16, 1.0, -1e16] + [0.0] * 29).reshape(2, 2, 2, 2, 2)
    assert oc.contract_vertices(a, np.ones_like(a))[0] == 1.0


def test_linearity_in_each_vector():
    rng = _rng(5)
    dims = (2, 3, 2, 3, 2)
    A = rng.normal(size=dims)
    psi = [rng.normal(size=n) + 1j * rng.normal(size=n) for n in dims]
    phi = rng.normal(size=dims[3]) + 1j * rng.normal(size=dims[3])
    c = 0.7 - 1.3j
    base, scale = oc.contract_vectors(A, psi)
    other, _ = oc.contract_vectors(A, psi[:3] + [phi] + psi[4:])
    both, _ = oc.contract_vectors(A, psi[:3] + [psi[3] + c * phi] + psi[4:])
    assert abs(both - (base + c * other)) <= 1e-13 * scale * (1 + abs(c))
