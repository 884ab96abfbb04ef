"""GPU parity of the downstream contractions (sf_contract_vertices, sf_contract_vectors) against
oracle/contract.py through the C ABI: |gpu - oracle| <= 1e-12 * sum|terms| (fp64 sums of up to 4e6 products in a fixed
order against an exact sum), shapes from 1 entry to 21^5, ragged shapes, a real vertex tensor, determinism, errors."""
import numpy as np
import pytest
import torch

import paper_2107_13952_b200 as sf
import workloads as wl
from oracle import contract as oc

pytestmark = pytest.mark.gpu
TOL = 1e-12


@pytest.fixture(scope="module", autouse=True)
def ctx():
    sf.sf_init(wl.GAMMA)
    yield


def _gpu_vectors(A, psi):
    Ad = torch.from_numpy(A).cuda()
    pd = [torch.from_numpy(p).cuda() for p in psi]
    res = torch.full((2,), float("nan"), dtype=torch.float64, device="cuda")
    sf.sf_contract_vectors(Ad, pd, res, torch.cuda.current_stream())
    torch.cuda.synchronize()
    r = res.cpu().numpy()
    return complex(r[0], r[1])


def _gpu_dot(A, B):
    res = torch.full((1,), float("nan"), dtype=torch.float64, device="cuda")
    sf.sf_contract_vertices(torch.from_numpy(A).cuda(), torch.from_numpy(B).cuda(), res, torch.cuda.current_stream())
    torch.cuda.synchronize()
    return float(res.cpu()[0])


@pytest.mark.parametrize("dims", [(1, 1, 1, 1, 1), (3, 3, 3, 3, 3), (2, 5, 3, 7, 4), (11, 11, 11, 11, 11), (13, 1, 9, 2, 17),
                                  (2, 3, 2, 3, 70), (1, 2, 3, 1, 1500), (21, 21, 21, 21, 21)])
def test_vectors_and_vertices_match_the_oracle(dims):
    rng = np.random.Generator(np.random.PCG64(sum(dims)))
    A = rng.normal(size=dims)
    B = rng.normal(size=dims)
    psi = [rng.normal(size=n) + 1j * rng.normal(size=n) for n in dims]
    ref, scale = oc.contract_vectors(A, psi)
    got = _gpu_vectors(A, psi)
    assert abs(got - ref) <= TOL * scale, (got, ref)
    dref, dscale = oc.contract_vertices(A, B)
    dgot = _gpu_dot(A, B)
    assert abs(dgot - dref) <= TOL * dscale
    assert _gpu_vectors(A, psi) == got and _gpu_dot(A, B) == dgot          # fixed summation order


def test_one_hot_vectors_and_product_tensor():
    rng = np.random.Generator(np.random.PCG64(9))
    dims = (4, 3, 5, 2, 6)
    A = rng.normal(size=dims)
    idx = (3, 1, 4, 0, 5)
    psi = [np.zeros(n, dtype=complex) for n in dims]
    for e, i in enumerate(idx):
        psi[e][i] = 1.0
    psi[4][idx[4]] = 1j
    assert _gpu_vectors(A, psi) == 1j * A[idx]
    u = [rng.normal(size=n) for n in dims]
    phi = [rng.normal(size=n) + 1j * rng.normal(size=n) for n in dims]
    T = np.einsum("a,b,c,d,e->abcde", *u)
    ref = np.prod([np.dot(u[e], phi[e]) for e in range(5)])
    _, scale = oc.contract_vectors(T, phi)
    assert abs(_gpu_vectors(T, phi) - ref) <= TOL * scale


def test_on_a_computed_vertex_tensor():
    """The path the paper's Listing 3 takes: compute a vertex tensor, then contract it with five complex vectors."""
    cfg = wl.config2(1)
    two_j, two_dl = cfg["two_j"], cfg["two_dl"]
    edge_dims, k_ranges = {}, {}
    for edge in (2, 3, 4, 5):
        _, n_i_e, base, pad = sf.sf_booster_dims(two_j, two_dl, edge)
        edge_dims[edge] = (n_i_e, base, pad)
        k_ranges[edge] = sf.sf_booster_kranges(two_j, two_dl, edge)
    B = wl.random_boosters(cfg["seed"], two_dl // 2 + 1, edge_dims, k_ranges)
    Bdev = {e: torch.from_numpy(b).cuda() for e, b in B.items()}
    _, n_i = sf.sf_vertex_dims(two_j)
    out = torch.zeros(tuple(n_i), dtype=torch.float64, device="cuda")
    st = torch.cuda.current_stream()
    sf.sf_vertex_amplitude(two_j, two_dl, Bdev, out, st)
    rng = np.random.Generator(np.random.PCG64(12))
    psi = [rng.normal(size=n) + 1j * rng.normal(size=n) for n in n_i]
    res = torch.zeros(2, dtype=torch.float64, device="cuda")
    sf.sf_contract_vectors(out, [torch.from_numpy(p).cuda() for p in psi], res, st)      # same stream: ordered after the tensor
    nrm = torch.zeros(1, dtype=torch.float64, device="cuda")
    sf.sf_contract_vertices(out, out, nrm, st)
    torch.cuda.synchronize()
    A = out.cpu().numpy()
    ref, scale = oc.contract_vectors(A, psi)
    r = res.cpu().numpy()
    assert abs(complex(r[0], r[1]) - ref) <= TOL * scale
    dref, dscale = oc.contract_vertices(A, A)
    assert abs(float(nrm.cpu()[0]) - dref) <= TOL * dscale


def test_errors():
    A = torch.zeros(32, dtype=torch.float64, device="cuda").reshape(2, 2, 2, 2, 2)
    res = torch.zeros(2, dtype=torch.float64, device="cuda")
    lib = sf._lib()
    import ctypes
    n = (ctypes.c_int * 5)(2, 2, 0, 2, 2)
    arr = (ctypes.c_void_p * 5)(*[A.data_ptr()] * 5)
    assert lib.sf_contract_vectors(ctypes.c_void_p(A.data_ptr()), n, arr, ctypes.c_void_p(res.data_ptr()), None) == sf.SF_EARG
    assert lib.sf_contract_vertices(None, ctypes.c_void_p(A.data_ptr()), ctypes.c_long(4), ctypes.c_void_p(res.data_ptr()),
                                    None) == sf.SF_EARG
