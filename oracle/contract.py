"""ORACLE (test infrastructure, not the product path): downstream contractions of vertex tensors, plain definitions.

    contract_vertices(A, B) = sum_{i1..i5} A[i1..i5] B[i1..i5]                    PAPER.md:365 (Fig. 3, left)
    contract_vectors(A, psi) = sum_{i1..i5} A[i1..i5] psi1[i1] ... psi5[i5]        PAPER.md:253, 365 (Fig. 3, right):
                                                                                 contract(v, cs5, cs4, cs3, cs2, cs1)

A is the vertex tensor in the library's layout out[i1][i2][i3][i4][i5] (= the paper's column-major A^{i5 i4 i3 i2 i1},
PAPER.md:182-186), psi_e a complex vector over the intertwiners of node e (coherent-state coefficients in the paper; any
complex vector here).  Sums are exact sums of fp64 products (math.fsum), so the result does not depend on an order.
Each function also returns the sum of |terms| (the scale of the fp64 forward error bound).
Pinned by tests/test_oracle_contract.py (closed forms for product tensors, one-hot vectors, brute-force loops).
Shares no code with the CUDA path.
"""
import math

import numpy as np


def contract_vertices(A, B):
    a = np.asarray(A, dtype=np.float64).ravel()
    b = np.asarray(B, dtype=np.float64).ravel()
    assert a.shape == b.shape
    t = a * b
    return math.fsum(t), math.fsum(np.abs(t))


def contract_vectors(A, psi):
    A = np.asarray(A, dtype=np.float64)
    assert A.ndim == 5 and len(psi) == 5
    psi = [np.asarray(p, dtype=np.complex128) for p in psi]
    for e in range(5):
        assert psi[e].shape == (A.shape[e],)
    # the full list of terms A[i1..i5] psi1[i1] ... psi5[i5], summed exactly (real and imaginary parts apart)
    w = psi[0][:, None, None, None, None] * psi[1][None, :, None, None, None] * psi[2][None, None, :, None, None] \
        * psi[3][None, None, None, :, None] * psi[4][None, None, None, None, :]
    t = (A * w).ravel()
    return complex(math.fsum(t.real), math.fsum(t.imag)), math.fsum(np.abs(t))
