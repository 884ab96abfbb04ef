"""GPU parity of the batched many-vertex entry point ("many vertex tensors with few shells") against
the oracle: sf_vertex_amplitude_batch computes n small vertex tensors in one kernel launch, one CTA per tensor; the oracle is
a loop over vertex_l1.  Tolerance of north_star: |A_gpu - A_oracle| <= 1e-11 * sum|terms| entry by entry."""
import random

import numpy as np
import pytest
import torch

import paper_2107_13952_b200 as sf
import workloads as wl
from oracle import ranges
from gpu_common import assert_parity, boosters_for, run_oracle, to_device

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module", autouse=True)
def ctx():
    sf.sf_init(wl.GAMMA)
    yield


def _mixed_small_problems(n, seed):
    """Seeded random boundary spins (integer and half-integer mixed, 2j <= 6) with Delta_l in 0..2."""
    rng = random.Random(seed)
    cfgs = []
    while len(cfgs) < n:
        two_j = [rng.randrange(0, 7) for _ in range(10)]
        two_dl = 2 * rng.randrange(0, 3)
        if not all(m > 0 for _, m in ranges.boundary_ranges(two_j)):
            continue
        cfg = dict(two_j=two_j, two_dl=two_dl, boosters="random", seed=5000 + len(cfgs), name=f"mixed{len(cfgs)}")
        try:
            boosters_for(cfg)
        except sf.SfError:
            continue                                  # a booster edge without any valid k
        cfgs.append(cfg)
    return cfgs


def _run_batch(cfgs):
    Bs = [boosters_for(c) for c in cfgs]
    Bdev = [to_device(B) for B in Bs]
    outs = [torch.full(tuple(sf.sf_vertex_dims(c["two_j"])[1]), float("nan"), dtype=torch.float64, device="cuda") for c in cfgs]
    before = sf.sf_launch_count(reset=True)
    sf.sf_vertex_amplitude_batch([c["two_j"] for c in cfgs], [c["two_dl"] for c in cfgs], Bdev, outs, torch.cuda.current_stream())
    torch.cuda.synchronize()
    return Bs, [o.cpu().numpy() for o in outs], sf.sf_launch_count()


def test_batch_of_64_mixed_small_spin_sets_matches_the_oracle():
    cfgs = _mixed_small_problems(64, seed=581) + [wl.CONFIGS[0], wl.config1(1), wl.config1(4), wl.config2(1)]
    Bs, A, launches = _run_batch(cfgs)
    for cfg, B, Ag in zip(cfgs, Bs, A):
        Ao, Aabs = run_oracle(cfg["two_j"], cfg["two_dl"], B, processes=1)
        assert_parity(Ag, Ao, Aabs, what=f"batch {cfg['name']} {cfg['two_j']} dl {cfg['two_dl']}")


def test_small_tensors_share_one_launch():
    """Tensors that fit one SM (here config 0 and the smallest BF tensors) are computed by exactly ONE kernel launch."""
    cfgs = [wl.CONFIGS[0]] * 6 + [wl.config1(1), wl.config1(2), dict(two_j=[2] * 10, two_dl=2, boosters="random", seed=3, name="j1dl1")]
    Bs, A, launches = _run_batch(cfgs)
    assert launches == 1, f"{launches} launches"
    for cfg, B, Ag in zip(cfgs, Bs, A):
        Ao, Aabs = run_oracle(cfg["two_j"], cfg["two_dl"], B, processes=1)
        assert_parity(Ag, Ao, Aabs, what=f"batch {cfg['name']}")


def test_batch_equals_single_calls_and_is_deterministic():
    cfgs = _mixed_small_problems(24, seed=7) + [wl.CONFIGS[0]] * 3
    Bs, A1, _ = _run_batch(cfgs)
    _, A2, _ = _run_batch(cfgs)
    sf.sf_sixj_table(12)            # with a resident table the S arrays are gathered from it where the arguments fit
    try:
        _, A3, _ = _run_batch(cfgs)
    finally:
        sf.sf_sixj_table(-1)
    for a, b in zip(A1, A3):
        assert np.abs(a - b).max() <= 1e-13 * max(np.abs(a).max(), 1e-300)
    for a, b in zip(A1, A2):
        assert np.array_equal(a, b), "not bitwise reproducible run to run"
    for cfg, B, Ab in zip(cfgs, Bs, A1):
        out = torch.zeros(Ab.shape, dtype=torch.float64, device="cuda")
        sf.sf_vertex_amplitude(cfg["two_j"], cfg["two_dl"], to_device(B), out, torch.cuda.current_stream())
        torch.cuda.synchronize()
        single = out.cpu().numpy()
        scale = max(np.abs(single).max(), 1e-300)
        assert np.abs(single - Ab).max() <= 1e-12 * scale


def test_batch_with_a_tensor_too_large_for_one_sm_and_error_behaviour():
    """config 2 at Delta_l = 3 (4096 shells, S arrays beyond one SM's shared memory) rides along: it is computed by the
    single-tensor path after the batch kernel; invalid arguments are refused before anything is written."""
    cfgs = [wl.CONFIGS[0], wl.config2(3), wl.config1(2)]
    Bs, A, launches = _run_batch(cfgs)
    assert launches > 1
    for cfg, B, Ag in zip(cfgs, Bs, A):
        Ao, Aabs = run_oracle(cfg["two_j"], cfg["two_dl"], B)
        assert_parity(Ag, Ao, Aabs, what=f"batch {cfg['name']}")
    # errors: an odd node (SF_ESPIN), an odd two_dl (SF_EARG); nothing is written
    good = wl.CONFIGS[0]
    Bdev = to_device(boosters_for(good))
    outs = [torch.zeros(3 ** 5, dtype=torch.float64, device="cuda") for _ in range(2)]
    for bad_j, bad_dl, status in [([2] * 9 + [3], 4, sf.SF_ESPIN), ([2] * 10, 3, sf.SF_EARG)]:
        with pytest.raises(sf.SfError) as e:
            sf.sf_vertex_amplitude_batch([good["two_j"], bad_j], [good["two_dl"], bad_dl], [Bdev, Bdev], outs)
        assert e.value.status == status
    torch.cuda.synchronize()
    assert all((o == 0).all() for o in outs)
    sf.sf_vertex_amplitude_batch([], [], [], [])       # an empty batch is a no-op
