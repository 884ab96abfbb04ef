"""sf_contract_vertices_noalloc against sf_contract_vertices (the existing path), on a GPU.

sf_contract_vertices_noalloc is the two-vertex contraction sum_z a[z] b[z] for a caller that cannot
allocate device memory where it makes the call: typically a long sum or Monte Carlo walk over bulk spins inside a program
whose allocator (CUDA.jl's pool, PyTorch's caching allocator, a fixed MIG / MPS slice) already owns the whole GPU, so that a
cudaMalloc coming from this library fails or eats into that pool, or a caller that cannot take the device-wide
synchronisation a cudaMalloc / cudaFree implies.  Its partial sums live in a fixed 65 792-byte array inside the library
instead of the context's cudaMalloc'd scratch, which caps the input at sf_contract_noalloc_max_n() entries.

Checked here: the same value as the existing path within the tolerance of tests/test_gpu_contract.py (1e-12 * sum|terms|;
the two add in different fixed orders) on two calls in a row -- the second call finds the first call's ticket and partial
sums in the shared array, so a large input is followed by a small one and the other way round --, bitwise repeatability,
that the device's free memory does not move across the calls, and the refusal beyond the limit.

This file is named so that pytest collects it last (a failure here under -x hides no other test), and it passes alone in
a fresh process as well as after the rest of the suite (it assumes nothing about the library's state except what its own
fixture sets up)."""
import ctypes

import numpy as np
import pytest
import torch

import paper_2107_13952_b200 as sf
import workloads as wl

pytestmark = pytest.mark.gpu
TOL = 1e-12          # of sum|a b|: the tolerance tests/test_gpu_contract.py uses for the same contraction


@pytest.fixture(scope="module", autouse=True)
def ctx():
    sf.sf_init(wl.GAMMA)          # the existing path needs the context (its scratch); the new entry point does not
    yield


def _pair(n, seed):
    rng = np.random.Generator(np.random.PCG64(seed))
    a, b = rng.normal(size=n), rng.normal(size=n)
    return a, b, float(np.abs(a * b).sum())


def _existing(ad, bd, st):
    res = torch.full((1,), float("nan"), dtype=torch.float64, device="cuda")
    sf.sf_contract_vertices(ad, bd, res, st)
    return res


# (first call, second call): the paper's tensor sizes 3^5, 11^5, 21^5, one entry, exactly one and two chunks of 4096, one past a
# chunk; each order so that the second call meets a larger / smaller grid's leftovers in the shared array
PAIRS = [(21 ** 5, 3 ** 5), (3 ** 5, 21 ** 5), (11 ** 5, 1), (1, 11 ** 5), (4096, 4097), (8192, 4095), (4097, 7 ** 5)]


@pytest.mark.parametrize("n1,n2", PAIRS)
def test_two_calls_in_a_row_match_the_existing_path(n1, n2):
    st = torch.cuda.current_stream()
    cases = []
    for n, seed in ((n1, 1000 + n1), (n2, 2000 + n2)):
        a, b, scale = _pair(n, seed)
        ad, bd = torch.from_numpy(a).cuda(), torch.from_numpy(b).cuda()
        cases.append((ad, bd, scale, _existing(ad, bd, st)))
    outs = [torch.full((1,), float("nan"), dtype=torch.float64, device="cuda") for _ in cases]
    sf.sf_contract_vertices_noalloc(cases[0][0], cases[0][1], outs[0], st)        # set-up call of this device, if it is the first
    torch.cuda.synchronize()
    for o in outs:
        o.fill_(float("nan"))
    torch.cuda.synchronize()
    free_before = torch.cuda.mem_get_info()[0]
    for (ad, bd, _, _), o in zip(cases, outs):                                    # two calls back to back on one stream
        sf.sf_contract_vertices_noalloc(ad, bd, o, st)
    torch.cuda.synchronize()
    assert torch.cuda.mem_get_info()[0] == free_before, "device memory moved across allocation-free calls"
    for (ad, bd, scale, ref), o in zip(cases, outs):
        got, want = float(o.cpu()[0]), float(ref.cpu()[0])
        assert np.isfinite(got)
        assert abs(got - want) <= TOL * scale, (ad.numel(), got, want, scale)
    # the same two calls again, other way round: bit for bit the same sums (fixed order, nothing left over from earlier calls)
    again = [torch.full((1,), float("nan"), dtype=torch.float64, device="cuda") for _ in cases]
    for (ad, bd, _, _), o in reversed(list(zip(cases, again))):
        sf.sf_contract_vertices_noalloc(ad, bd, o, st)
    torch.cuda.synchronize()
    for o, o2 in zip(outs, again):
        assert float(o.cpu()[0]) == float(o2.cpu()[0])


def test_exact_small_sums():
    """Integers: both paths are exact, so equality is exact -- and a one-hot b picks one entry of a."""
    st = torch.cuda.current_stream()
    n = 3 * 4096 + 5
    a = torch.arange(n, dtype=torch.float64, device="cuda") % 17 - 8
    b = torch.arange(n, dtype=torch.float64, device="cuda") % 5 - 2
    res = torch.zeros(1, dtype=torch.float64, device="cuda")
    sf.sf_contract_vertices_noalloc(a, b, res, st)
    torch.cuda.synchronize()
    av, bv = np.arange(n) % 17 - 8, np.arange(n) % 5 - 2
    assert float(res.cpu()[0]) == float((av * bv).sum()) == float(_existing(a, b, st).cpu()[0])
    hot = torch.zeros(n, dtype=torch.float64, device="cuda")
    hot[n - 2] = 1.0
    sf.sf_contract_vertices_noalloc(a, hot, res, st)
    torch.cuda.synchronize()
    assert float(res.cpu()[0]) == float(av[n - 2])


def test_limit_and_bad_arguments():
    lib = sf._lib()
    nmax = sf.sf_contract_noalloc_max_n()
    assert nmax == 8192 * 4096
    a = torch.ones(8, dtype=torch.float64, device="cuda")
    res = torch.full((1,), 123.0, dtype=torch.float64, device="cuda")
    pa, pr = ctypes.c_void_p(a.data_ptr()), ctypes.c_void_p(res.data_ptr())
    # beyond the limit: refused before anything is launched (the pointers are never dereferenced, the result is untouched)
    assert lib.sf_contract_vertices_noalloc(pa, pa, ctypes.c_long(nmax + 1), pr, None) == sf.SF_ELIMIT
    assert b"fixed built-in scratch" in lib.sf_strerror(sf.SF_ELIMIT)
    with pytest.raises(sf.SfError) as e:
        sf.sf_contract_vertices_noalloc(_FakeTensor(a.data_ptr(), nmax + 1), a, res)
    assert e.value.status == sf.SF_ELIMIT
    assert lib.sf_contract_vertices_noalloc(None, pa, ctypes.c_long(8), pr, None) == sf.SF_EARG
    assert lib.sf_contract_vertices_noalloc(pa, pa, ctypes.c_long(-1), pr, None) == sf.SF_EARG
    torch.cuda.synchronize()
    assert float(res.cpu()[0]) == 123.0
    # an empty sum is a valid call: 0.0, written by the kernel
    assert lib.sf_contract_vertices_noalloc(pa, pa, ctypes.c_long(0), pr, None) == sf.SF_OK
    torch.cuda.synchronize()
    assert float(res.cpu()[0]) == 0.0


class _FakeTensor:
    """A device pointer with a claimed size: enough for the binding, never dereferenced by a refused call."""

    def __init__(self, ptr, n):
        self._ptr, self._n = ptr, n

    def data_ptr(self):
        return self._ptr

    def numel(self):
        return self._n


def test_at_the_limit():
    """n = the maximum (2 x 268 MB of input): every slot of the built-in array is used."""
    st = torch.cuda.current_stream()
    n = sf.sf_contract_noalloc_max_n()
    g = torch.Generator(device="cuda")
    g.manual_seed(5)
    a = torch.randn(n, dtype=torch.float64, device="cuda", generator=g)
    b = torch.randn(n, dtype=torch.float64, device="cuda", generator=g)
    res = torch.zeros(1, dtype=torch.float64, device="cuda")
    sf.sf_contract_vertices_noalloc(a, b, res, st)
    ref = _existing(a, b, st)
    torch.cuda.synchronize()
    scale = float((a * b).abs().sum().cpu())
    assert abs(float(res.cpu()[0]) - float(ref.cpu()[0])) <= TOL * scale
