"""GPU parity of the vertex tensor (steps 4-7 of the algorithm) against the oracle, through the
C ABI, on the five workloads of BASELINE.json (small ones in full, large ones on shell sub-ranges the oracle finishes
in seconds), for the staged, the per-shell line and the factorised path (the automatic choice), plus edge cases,
additivity, determinism and error behaviour.
"""
import itertools
import random

import numpy as np
import pytest
import torch

import paper_2107_13952_b200 as sf
import workloads as wl
from oracle import ranges
from oracle import vertex as ov
from gpu_common import TOL, abi_dims, assert_parity, boosters_for, run_gpu, run_oracle, to_device

pytestmark = pytest.mark.gpu

PATHS = [pytest.param(1, id="staged"), pytest.param(3, id="line"), pytest.param(0, id="auto")]
TAKEN = {1: 1, 3: 3, 0: 4}      # automatic selection takes the factorised path wherever it fits


@pytest.fixture(scope="module", autouse=True)
def ctx():
    sf.sf_init(wl.GAMMA)
    yield
    sf.sf_set_path(0)
    sf.sf_sixj_table(-1)


@pytest.fixture(params=PATHS)
def path(request):
    sf.sf_set_path(request.param)
    yield request.param
    sf.sf_set_path(0)


def _full(cfg, what):
    B = boosters_for(cfg)
    Ag = run_gpu(cfg["two_j"], cfg["two_dl"], B)
    Ao, Aabs = run_oracle(cfg["two_j"], cfg["two_dl"], B)
    return assert_parity(Ag, Ao, Aabs, what=what), Ag, Ao


def test_config0_full(path):
    worst, Ag, Ao = _full(wl.CONFIGS[0], "config 0")
    assert Ag.shape == (3,) * 5 and np.abs(Ao).max() > 0
    assert sf.sf_last_path() == TAKEN[path]


@pytest.mark.parametrize("two_j", list(range(1, 15)))
def test_config1_bf_sweep(path, two_j):
    """Identity boosters, Delta_l = 0  =>  A = N(i) {15j}  (reading G8)."""
    cfg = wl.config1(two_j)
    worst, Ag, Ao = _full(cfg, cfg["name"])
    if two_j == 1:      # printed exact values, SURVEY.md 8(c) P5
        assert Ag[0, 0, 0, 0, 0] == pytest.approx(1 / 16, rel=1e-13)
        assert Ag[1, 1, 1, 1, 1] == pytest.approx(3 ** 2.5 * 3 ** 4 * (-7 / 432), rel=1e-13)


@pytest.mark.parametrize("two_j", list(range(15, 21)))
def test_config1_bf_large_spins_full_tensor(two_j):
    """The upper end of BASELINE.json's config 1 (j = 15/2 .. 10; up to 21^5 entries), automatic path, full tensors: with
    test_config1_bf_sweep every 2j = 1 .. 20 of the sweep is compared entrywise with the oracle."""
    cfg = wl.config1(two_j)
    worst, Ag, Ao = _full(cfg, cfg["name"])
    assert Ag.shape == (two_j + 1,) * 5
    assert sf.sf_last_path() == 4


def test_config1_bf_j10_staged_path():
    """The largest BF tensor on the staged path (the fallback for shapes the other paths do not hold)."""
    cfg = wl.config1(20)
    sf.sf_set_path(1)
    try:
        _full(cfg, cfg["name"])
    finally:
        sf.sf_set_path(0)


@pytest.mark.parametrize("dl", [0, 1, 2])
def test_config2_small_shell_counts_full(path, dl):
    cfg = wl.config2(dl)
    _full(cfg, cfg["name"])


@pytest.mark.parametrize("dl,lo,n", [(4, 7000, 40), (8, 531441 - 25, 25), (8, 0, 12), (7, 100000, 30)])
def test_config2_sub_ranges(path, dl, lo, n):
    """Larger Delta_l on contiguous shell sub-ranges (Delta_l = 7, 8 contain empty shells: reading G10)."""
    cfg = wl.config2(dl)
    B = boosters_for(cfg)
    Ag = run_gpu(cfg["two_j"], cfg["two_dl"], B, lo, lo + n)
    Ao, Aabs = run_oracle(cfg["two_j"], cfg["two_dl"], B, lo, lo + n)
    assert_parity(Ag, Ao, Aabs, what=f"{cfg['name']} shells [{lo},{lo + n})")


def test_config3_scattered_shells(path):
    """The headline workload (j = 5, Delta_l = 10) on single shells spread over the grid, and one short range."""
    cfg = wl.CONFIGS[3]
    B = boosters_for(cfg)
    Bdev = to_device(B)
    rng = random.Random(3)
    picks = [0, 11 ** 6 - 1] + [rng.randrange(11 ** 6) for _ in range(3)]
    for s in picks:
        Ag = run_gpu(cfg["two_j"], cfg["two_dl"], B, s, s + 1, Bdev=Bdev)
        Ao, Aabs = run_oracle(cfg["two_j"], cfg["two_dl"], B, s, s + 1)
        assert_parity(Ag, Ao, Aabs, what=f"config 3 shell {s}")
    lo = 11 ** 5 * 3 + 11 ** 2 * 5 + 7
    Ag = run_gpu(cfg["two_j"], cfg["two_dl"], B, lo, lo + 9, Bdev=Bdev)
    Ao, Aabs = run_oracle(cfg["two_j"], cfg["two_dl"], B, lo, lo + 9)
    assert_parity(Ag, Ao, Aabs, what="config 3 short range")
    assert sf.sf_last_path() == TAKEN[path]


def test_config3_blocks_and_ragged_ranges():
    """The headline workload at its bench launch configuration (automatic path = factorised), on ranges that are whole
    boxes of virtual spins (all (l34 l35 l45) of one (l23 l24 l25): 1331 shells) and on ragged ranges that the
    library splits into up to 11 boxes."""
    cfg = wl.CONFIGS[3]
    B = boosters_for(cfg)
    Bdev = to_device(B)
    nl3 = 11 ** 3
    for lo, hi in [(nl3 * 700, nl3 * 701), (nl3 * 1330, nl3 * 1331), (nl3 * 5 + 777, nl3 * 6 + 1500),
                   (11 ** 5 * 4 - 40, 11 ** 5 * 4 + 2000)]:
        Ag = run_gpu(cfg["two_j"], cfg["two_dl"], B, lo, hi, Bdev=Bdev)
        assert sf.sf_last_path() == 4
        Ao, Aabs = run_oracle(cfg["two_j"], cfg["two_dl"], B, lo, hi)
        assert_parity(Ag, Ao, Aabs, what=f"config 3 shells [{lo},{hi})")


@pytest.mark.parametrize("bits", [pytest.param(1, id="R-booster-stationary"), pytest.param(8, id="R-gather-gemm"), pytest.param(2, id="qp-gen1"),
                                  pytest.param(4, id="qp-gen2"), pytest.param(0, id="default")])
def test_factorised_kernel_variants_against_the_oracle(bits):
    """Every kernel variant of the factorised path (sf_set_factor_variant, include/sfoam_debug.h: the fallbacks the
    default falls back to for shapes its kernels do not hold) against the oracle: config 0 and a half-integer set in
    full, config 2 (Delta_l = 3) in full, a whole (l23 l24 l25) block and a ragged range of config 3, a config 4 block."""
    sf.sf_set_path(4)
    sf.sf_set_factor_variant(bits)
    try:
        for cfg, what in [(wl.CONFIGS[0], "config 0"), (wl.config2(3), "config 2 dl 3"),
                          (dict(two_j=[4, 3, 1, 4, 2, 5, 5, 5, 4, 3], two_dl=4, boosters="random", seed=77), "half-integer")]:
            B = boosters_for(cfg)
            Ag = run_gpu(cfg["two_j"], cfg["two_dl"], B)
            assert sf.sf_last_path() == 4
            Ao, Aabs = run_oracle(cfg["two_j"], cfg["two_dl"], B)
            assert_parity(Ag, Ao, Aabs, what=f"variant {bits}: {what}")
        cfg = wl.CONFIGS[3]
        B = boosters_for(cfg)
        Bdev = to_device(B)
        nl3 = 11 ** 3
        for lo, hi in [(nl3 * 613, nl3 * 614), (nl3 * 9 + 1200, nl3 * 10 + 300)]:
            Ag = run_gpu(cfg["two_j"], cfg["two_dl"], B, lo, hi, Bdev=Bdev)
            Ao, Aabs = run_oracle(cfg["two_j"], cfg["two_dl"], B, lo, hi)
            assert_parity(Ag, Ao, Aabs, what=f"variant {bits}: config 3 shells [{lo},{hi})")
        cfg = _config4(2)
        B = boosters_for(cfg)
        Ag = run_gpu(cfg["two_j"], cfg["two_dl"], B, 7 ** 3 * 100, 7 ** 3 * 101)
        Ao, Aabs = run_oracle(cfg["two_j"], cfg["two_dl"], B, 7 ** 3 * 100, 7 ** 3 * 101)
        assert_parity(Ag, Ao, Aabs, what=f"variant {bits}: config 4 lambda 2 block")
    finally:
        sf.sf_set_factor_variant(0)
        sf.sf_set_path(0)


def test_recorded_launch_sequences_replay_the_plain_call():
    """sf_set_graphs (include/sfoam.h): from the third identical call on, a vertex call replays a recorded CUDA graph.  The
    replay must equal the plain call bit for bit, follow booster VALUES changed in place, and be dropped when a setting
    changes (here: the path)."""
    cfg = wl.config2(2)
    two_j, two_dl = cfg["two_j"], cfg["two_dl"]
    B = boosters_for(cfg)
    Bdev = to_device(B)
    _, n_i = sf.sf_vertex_dims(two_j)
    out = torch.full(tuple(n_i), float("nan"), dtype=torch.float64, device="cuda")
    st = torch.cuda.current_stream()

    def call():
        out.fill_(float("nan"))
        sf.sf_vertex_amplitude(two_j, two_dl, Bdev, out, st)
        torch.cuda.synchronize()
        return out.cpu().numpy().copy()

    try:
        sf.sf_set_graphs(0)
        plain = call()
        sf.sf_set_graphs(1)
        runs = [call() for _ in range(5)]                 # 1: plain, 2: plain + remembered, 3: recorded + replayed, 4, 5: replayed
        for r in runs:
            assert np.array_equal(r, plain)
        n0 = sf.sf_launch_count()
        call()
        assert sf.sf_launch_count() > n0                  # a replay still reports the launches it stands for
        # new booster values behind the same pointers
        Bdev[3].mul_(-2.0)
        scaled = call()
        sf.sf_set_graphs(0)
        assert np.array_equal(call(), scaled)
        assert np.abs(scaled + 2.0 * plain).max() <= 1e-12 * np.abs(plain).max()      # multilinear in every booster
        sf.sf_set_graphs(1)
        # another path: the recordings of the old setting must not be replayed
        for _ in range(3):
            call()
        sf.sf_set_path(3)
        line = call()
        assert sf.sf_last_path() == 3
        assert np.abs(line - scaled).max() <= 1e-12 * np.abs(scaled).max()
        Ao, Aabs = run_oracle(two_j, two_dl, {e: Bdev[e].cpu().numpy() for e in Bdev})
        assert_parity(scaled, Ao, Aabs, what="replayed call")
    finally:
        sf.sf_set_graphs(1)
        sf.sf_set_path(0)


def test_calls_on_two_streams_share_the_scratch_buffers_safely():
    """The library has one set of scratch buffers; calls on different streams are serialised by an event (include/sfoam.h,
    Concurrency).  Two different problems issued back to back on two streams, no synchronisation in between, must both
    come out bit for bit as when they run alone."""
    cfgs = [wl.config2(4), wl.config2(3), wl.CONFIGS[0]]
    prob = []
    for cfg in cfgs:
        B = boosters_for(cfg)
        prob.append((cfg["two_j"], cfg["two_dl"], to_device(B), sf.sf_vertex_dims(cfg["two_j"])[1]))
    alone = []
    for two_j, two_dl, Bdev, n_i in prob:
        out = torch.full(tuple(n_i), float("nan"), dtype=torch.float64, device="cuda")
        sf.sf_vertex_amplitude(two_j, two_dl, Bdev, out, torch.cuda.current_stream())
        torch.cuda.synchronize()
        alone.append(out.cpu().numpy())
    streams = [torch.cuda.Stream() for _ in prob]
    for rep in range(3):
        outs = []
        for (two_j, two_dl, Bdev, n_i), st in zip(prob, streams):
            out = torch.full(tuple(n_i), float("nan"), dtype=torch.float64, device="cuda")
            torch.cuda.synchronize()                      # the fill is done; from here on only the library orders the streams
            outs.append(out)
        for (two_j, two_dl, Bdev, n_i), st, out in zip(prob, streams, outs):
            sf.sf_vertex_amplitude(two_j, two_dl, Bdev, out, st)
        torch.cuda.synchronize()
        for out, ref in zip(outs, alone):
            assert np.array_equal(out.cpu().numpy(), ref)


QP4_CLASSES = [      # (two_j, two_dl, shells or None = all): one spin set per instantiation k_fz_qp4<LDZ, N5T, N4T> (sf_factor_qp4.cu)
    pytest.param([11, 0, 0, 11, 9, 2, 0, 13, 10, 11], 2, None, id="ldz52-n5t1-n4t1"),
    pytest.param([0, 10, 12, 12, 11, 13, 8, 9, 0, 10], 2, None, id="ldz52-n5t1-n4t2"),
    pytest.param([13, 5, 2, 8, 0, 6, 11, 10, 11, 8], 2, None, id="ldz52-n5t2-n4t1"),
    pytest.param([1, 1, 9, 11, 4, 8, 11, 13, 8, 12], 2, None, id="ldz52-n5t2-n4t2"),
    pytest.param([3, 12, 3, 12, 3, 7, 13, 3, 12, 13], 2, None, id="ldz68-n5t2-n4t1"),
    pytest.param([13, 10, 13, 12, 12, 9, 14, 8, 14, 12], 2, (21, 27), id="ldz68-n5t2-n4t2"),
]


@pytest.mark.parametrize("two_j,two_dl,shells", QP4_CLASSES)
def test_qp4_template_classes_against_the_oracle(two_j, two_dl, shells):
    """k_fz_qp4 is compiled for one or two tiles of i5 and of i4 and two strides of its Z slab; the five workloads reach two
    of the six instantiations.  One irregular spin set per instantiation (found by a seeded search over 2j <= 14), each on
    the factorised path with the Q/P kernel checked, against the oracle."""
    cfg = dict(two_j=two_j, two_dl=two_dl, boosters="random", seed=4100 + sum(two_j))
    B = boosters_for(cfg)
    sf.sf_set_path(4)
    try:
        if shells is None:
            Ag = run_gpu(two_j, two_dl, B)
            Ao, Aabs = run_oracle(two_j, two_dl, B)
        else:
            Ag = run_gpu(two_j, two_dl, B, shells[0], shells[1])
            Ao, Aabs = run_oracle(two_j, two_dl, B, shells[0], shells[1])
        assert sf.sf_last_path() == 4 and sf.sf_last_qp_kernel() == 4
        assert np.abs(Ao).max() > 0
        assert_parity(Ag, Ao, Aabs, what=f"qp4 class {two_j}")
    finally:
        sf.sf_set_path(0)


def test_paths_agree_on_a_full_tensor():
    """Config 2, Delta_l = 4 (15 625 shells) in full: the factorised and the per-shell line path give the same tensor to
    rounding, and both match the oracle."""
    cfg = wl.config2(4)
    B = boosters_for(cfg)
    Bdev = to_device(B)
    sf.sf_set_path(4)
    A4 = run_gpu(cfg["two_j"], cfg["two_dl"], B, Bdev=Bdev)
    sf.sf_set_path(3)
    A3 = run_gpu(cfg["two_j"], cfg["two_dl"], B, Bdev=Bdev)
    sf.sf_set_path(0)
    Ao, Aabs = run_oracle(cfg["two_j"], cfg["two_dl"], B)
    assert_parity(A4, Ao, Aabs, what="config 2 dl=4, factorised")
    assert_parity(A3, Ao, Aabs, what="config 2 dl=4, line")


def test_config3_full_size_factorised_equals_line():
    """All 1 771 561 shells of the headline workload, in the launch configuration bench.py times: the factorised path and
    the per-shell line path (each compared with the oracle on sub-ranges above) give the same tensor to rounding.  A
    property that holds at any size: both are the sum of eq. (3), in different orders."""
    cfg = wl.CONFIGS[3]
    B = boosters_for(cfg)
    Bdev = to_device(B)
    sf.sf_sixj_table(60)
    sf.sf_set_path(4)
    A4 = run_gpu(cfg["two_j"], cfg["two_dl"], B, Bdev=Bdev)
    assert sf.sf_last_path() == 4
    sf.sf_set_path(3)
    A3 = run_gpu(cfg["two_j"], cfg["two_dl"], B, Bdev=Bdev)
    sf.sf_set_path(0)
    sf.sf_sixj_table(-1)
    assert np.isfinite(A4).all() and np.abs(A4).max() > 0
    # FP64 sums of ~1e9 terms per entry in two different orders; measured 8e-15 of the largest entry
    assert np.abs(A4 - A3).max() <= 1e-12 * np.abs(A3).max()


def _config4(lam):
    base, _ = wl.config4_base_spins(lambda tj: all(n > 0 for _, n in ranges.boundary_ranges(tj)))
    assert base == [8, 7, 12, 3, 8, 5, 9, 12, 3, 7]
    return wl.config4(base, lam)


@pytest.mark.parametrize("lam,n", [(1, 60), (2, 6), (3, 1), (4, 1), (6, 1)])
def test_config4_sub_ranges(path, lam, n):
    if path == 3 and lam > 1:
        pytest.skip("the line path holds intertwiner ranges of at most 16 values")
    cfg = _config4(lam)
    B = boosters_for(cfg)
    lo = 7 ** 6 // 2 + 11
    Ag = run_gpu(cfg["two_j"], cfg["two_dl"], B, lo, lo + n)
    Ao, Aabs = run_oracle(cfg["two_j"], cfg["two_dl"], B, lo, lo + n)
    assert_parity(Ag, Ao, Aabs, what=f"{cfg['name']} shells [{lo},{lo + n})")


# (lambda, first shell, number of shells): whole (l34 l35 l45) blocks of 7^3 shells, whole (l35 l45) planes and whole l45
# lines followed by a ragged tail, so that the boxes the factorised path runs have 7 offsets per virtual spin (c34 = c35 =
# c45 = 7, two k-steps over l45) as in the full tensors bench.py times; the oracle cost grows like lambda^5, so the larger
# spins get planes instead of blocks
CONFIG4_RANGES = [(2, 343 * 170, 343 + 60), (3, 343 * 171, 343 + 60), (4, 343 * 5, 343 + 23), (5, 343 * 200 + 49, 49 * 2 + 17),
                  (6, 343 * 342 + 49 * 3, 49 + 7 + 3)]


@pytest.mark.parametrize("lam,lo,n", CONFIG4_RANGES)
def test_config4_blocks_planes_and_ragged_tails(lam, lo, n):
    """BASELINE.json config 4 (js * lambda) for every lambda = 2 .. 6 on the automatic (factorised) path."""
    cfg = _config4(lam)
    B = boosters_for(cfg)
    Ag = run_gpu(cfg["two_j"], cfg["two_dl"], B, lo, lo + n)
    assert sf.sf_last_path() == 4
    boxes = sf.sf_shell_boxes(cfg["two_dl"], lo, lo + n)
    assert any(cnt[5] == 7 and cnt[4] == 7 for _, cnt in boxes)
    Ao, Aabs = run_oracle(cfg["two_j"], cfg["two_dl"], B, lo, lo + n, processes=16)
    assert np.abs(Ao).max() > 0
    assert_parity(Ag, Ao, Aabs, what=f"{cfg['name']} shells [{lo},{lo + n})")


@pytest.mark.parametrize("lam", [2, 3])
def test_config4_full_tensor_factorised_equals_staged(lam):
    """All 117 649 shells of config 4 at lambda = 2, 3: the factorised path (the one bench.py times) and the staged per-shell
    path (compared with the oracle on sub-ranges above) give the same tensor to rounding."""
    cfg = _config4(lam)
    B = boosters_for(cfg)
    Bdev = to_device(B)
    sf.sf_set_path(4)
    A4 = run_gpu(cfg["two_j"], cfg["two_dl"], B, Bdev=Bdev)
    sf.sf_set_path(1)
    A1 = run_gpu(cfg["two_j"], cfg["two_dl"], B, Bdev=Bdev)
    sf.sf_set_path(0)
    assert np.isfinite(A4).all() and np.abs(A4).max() > 0
    assert np.abs(A4 - A1).max() <= 1e-12 * np.abs(A1).max()


def test_factorised_path_small_memory_budget_takes_the_multi_pass_branches():
    """With a P/R budget of a few hundred KB (sf_set_factor_budget) small problems run one i1 per pass, several passes: the
    branch the full-size workloads take (config 3: 5 + 5 + 1 values of i1), here on tensors the oracle computes in full."""
    cases = [wl.config2(2), wl.config2(3), dict(two_j=[4, 3, 1, 4, 2, 5, 5, 5, 4, 3], two_dl=4, boosters="random", seed=77),
             _config4(1)]
    sf.sf_set_path(4)
    try:
        for cfg in cases:
            B = boosters_for(cfg)
            Bdev = to_device(B)
            n = (cfg["two_dl"] // 2 + 1) ** 6
            lo, hi = (0, n) if n <= 4096 else (n // 2, n // 2 + 343 + 20)
            Ao, Aabs = run_oracle(cfg["two_j"], cfg["two_dl"], B, lo, hi)
            ref = run_gpu(cfg["two_j"], cfg["two_dl"], B, lo, hi, Bdev=Bdev)
            for budget in (1, 300 * 1024, 3 * 1024 * 1024):
                sf.sf_set_factor_budget(budget)
                Ag = run_gpu(cfg["two_j"], cfg["two_dl"], B, lo, hi, Bdev=Bdev)
                sf.sf_set_factor_budget(0)
                assert_parity(Ag, Ao, Aabs, what=f"{cfg.get('name')} budget {budget}")
                assert np.abs(Ag - ref).max() <= 1e-13 * max(Aabs.max(), 1e-300)
    finally:
        sf.sf_set_factor_budget(0)
        sf.sf_set_path(0)


def test_config3_full_tensor_against_the_cached_oracle_tensor(golden_dir):
    """ALL 1 771 561 shells of the headline workload (BASELINE.json config 3), the tensor bench.py times, entry by entry
    against the oracle's full tensor: tests/golden/config3_full.npz, written by tests/golden/make_config3_full.py from
    `oracle/` alone (long double, ~2 h of CPU) and keyed by the hash of the inputs.  Both the automatic (factorised) path and
    the per-shell line path, at the tolerance of north_star."""
    import hashlib
    import os
    f = os.path.join(golden_dir, "config3_full.npz")
    assert os.path.exists(f), "tests/golden/config3_full.npz is missing: run tests/golden/make_config3_full.py"
    z = np.load(f)
    cfg = wl.CONFIGS[3]
    B = boosters_for(cfg)
    h = hashlib.sha256()
    h.update(np.asarray(list(cfg["two_j"]) + [cfg["two_dl"]], dtype=np.int64).tobytes())
    for edge in (2, 3, 4, 5):
        h.update(np.ascontiguousarray(B[edge], dtype=np.float64).tobytes())
    assert h.hexdigest() == str(z["input_sha256"]), "the cached oracle tensor was computed from different inputs"
    assert int(z["nonempty"]) == 11 ** 6
    Ao, Aabs = z["A"], z["Aabs"]
    Bdev = to_device(B)
    sf.sf_sixj_table(60)
    try:
        for path in (0, 3):
            sf.sf_set_path(path)
            Ag = run_gpu(cfg["two_j"], cfg["two_dl"], B, Bdev=Bdev)
            assert sf.sf_last_path() == TAKEN[path]
            assert_parity(Ag, Ao, Aabs, what=f"config 3, all shells, path {TAKEN[path]}")
    finally:
        sf.sf_set_path(0)
        sf.sf_sixj_table(-1)


@pytest.mark.parametrize("name", ["config2_dl8", "config4_lam1", "config4_lam2"])
def test_secondary_workloads_full_tensor_against_the_cached_oracle_tensor(golden_dir, name):
    """The other tensors bench.py times (its `other_workloads` rows), in full and entry by entry against the oracle: config 2
    at Delta_l = 8 (all 9^6 = 531 441 shells) and config 4 at lambda = 1, 2 (all 7^6 = 117 649 shells each).  The files
    tests/golden/<name>_full.npz are written by tests/golden/make_full_tensor.py from `oracle/` alone (exact-{6j} S arrays, long
    double loops) and keyed by the hash of the inputs.  Automatic path (what bench.py runs), S arrays gathered from the table
    and evaluated directly, at the tolerance of north_star."""
    import hashlib
    import os
    f = os.path.join(golden_dir, name + "_full.npz")
    assert os.path.exists(f), f"{f} is missing: run tests/golden/make_full_tensor.py"
    z = np.load(f)
    cfg = wl.config2(8) if name == "config2_dl8" else _config4(int(name[-1]))
    B = boosters_for(cfg)
    h = hashlib.sha256()
    h.update(np.asarray(list(cfg["two_j"]) + [cfg["two_dl"]], dtype=np.int64).tobytes())
    for edge in (2, 3, 4, 5):
        h.update(np.ascontiguousarray(B[edge], dtype=np.float64).tobytes())
    assert h.hexdigest() == str(z["input_sha256"]), "the cached oracle tensor was computed from different inputs"
    Ao, Aabs = z["A"], z["Aabs"]
    assert int(z["nonempty"]) > 0 and np.abs(Ao).max() > 0
    Bdev = to_device(B)
    sf.sf_set_path(0)
    try:
        for table in (60, -1):
            sf.sf_sixj_table(table)
            Ag = run_gpu(cfg["two_j"], cfg["two_dl"], B, Bdev=Bdev)
            assert sf.sf_last_path() == 4                      # the factorised path, as in bench.py
            assert_parity(Ag, Ao, Aabs, what=f"{name}, all shells, table {table}")
    finally:
        sf.sf_sixj_table(-1)


def test_table_and_direct_slices_agree(path):
    """With a resident table the S arrays are gathered from it; the tensor must not change beyond rounding."""
    cfg = wl.config2(2)
    B = boosters_for(cfg)
    sf.sf_sixj_table(-1)
    A0 = run_gpu(cfg["two_j"], cfg["two_dl"], B)
    sf.sf_sixj_table(30)
    A1 = run_gpu(cfg["two_j"], cfg["two_dl"], B)
    sf.sf_sixj_table(-1)
    Ao, Aabs = run_oracle(cfg["two_j"], cfg["two_dl"], B)
    assert_parity(A1, Ao, Aabs, what="table-gathered slices")
    assert np.abs(A1 - A0).max() <= 1e-13 * Aabs.max()


def test_additivity_and_determinism(path):
    cfg = wl.config2(3)
    B = boosters_for(cfg)
    Bdev = to_device(B)
    two_j, two_dl = cfg["two_j"], cfg["two_dl"]
    full = run_gpu(two_j, two_dl, B, Bdev=Bdev)
    again = run_gpu(two_j, two_dl, B, Bdev=Bdev)
    assert np.array_equal(full, again), "not bitwise reproducible run to run"
    cuts = [0, 1, 777, 2048, 4095, 4096]
    parts = sum(run_gpu(two_j, two_dl, B, a, b, Bdev=Bdev) for a, b in zip(cuts[:-1], cuts[1:]))
    scale = np.abs(full).max()
    assert np.abs(parts - full).max() <= 1e-12 * scale
    empty = run_gpu(two_j, two_dl, B, 100, 100, Bdev=Bdev)
    assert (empty == 0).all()


def test_one_hot_boosters_pick_one_w_entry(path):
    """B_a = e_i e_k^T at one triple each  =>  A[i1, i2..i5] = prod sqrt(2i+1) prod (2k_a+1) {15j}  (pin P6(ii))."""
    from oracle import fifteenj
    two_j, two_dl = [2] * 10, 4
    edge_dims, k_ranges = abi_dims(two_j, two_dl)
    lo_i, n_i = sf.sf_vertex_dims(two_j)
    rng = random.Random(11)
    for _ in range(4):
        offs = tuple(rng.randrange(3) for _ in range(6))
        two_l = ranges.shell_spins(two_j, offs)
        hot, ks, iis = {}, [], []
        for edge in (2, 3, 4, 5):
            t = ranges.triple_index(edge, offs, two_dl)
            klo, nk = k_ranges[edge][t]
            k = klo + 2 * rng.randrange(nk)
            ii = rng.randrange(n_i[edge - 1])
            hot[edge] = (t, ii, (k - edge_dims[edge][1]) // 2)
            ks.append(k)
            iis.append(ii)
        A = run_gpu(two_j, two_dl, wl.one_hot_boosters(3, edge_dims, hot))
        for a1 in range(n_i[0]):
            i1 = lo_i[0] + 2 * a1
            norm = np.sqrt(np.prod([i1 + 1] + [lo_i[e + 1] + 2 * iis[e] + 1 for e in range(4)]))
            ref = norm * np.prod([k + 1 for k in ks]) * fifteenj.fifteenj(two_l, i1, ks)
            assert A[(a1, *iis)] == pytest.approx(ref, rel=1e-12, abs=1e-16)
        mask = np.ones_like(A, dtype=bool)
        mask[(slice(None), *iis)] = False
        assert (A[mask] == 0).all()


def test_half_integer_nonhomogeneous_full(path):
    two_j, two_dl = [4, 3, 1, 4, 2, 5, 5, 5, 4, 3], 4
    cfg = dict(two_j=two_j, two_dl=two_dl, boosters="random", seed=77)
    B = boosters_for(cfg)
    Ag = run_gpu(two_j, two_dl, B)
    Ao, Aabs = run_oracle(two_j, two_dl, B)
    assert_parity(Ag, Ao, Aabs, what="half-integer non-homogeneous")


def test_random_small_spin_sets_full(path):
    """Seeded random boundary spins (integer and half-integer mixed, 2j <= 5) with random Delta_l <= 2, full tensors:
    irregular ranges, empty k-ranges for some triples, one-value intertwiner ranges."""
    rng = random.Random(2107)
    done = 0
    while done < 8:
        two_j = [rng.randrange(0, 6) for _ in range(10)]
        two_dl = 2 * rng.randrange(0, 3)
        if not all(n > 0 for _, n in ranges.boundary_ranges(two_j)):
            continue
        cfg = dict(two_j=two_j, two_dl=two_dl, boosters="random", seed=1000 + done)
        try:
            B = boosters_for(cfg)
        except sf.SfError:
            continue                                  # a booster edge without any valid k: nothing to contract
        try:
            Ag = run_gpu(two_j, two_dl, B)
        except sf.SfError as e:
            if path == 3 and e.status == sf.SF_EARG:
                done += 1
                continue                              # the line path does not hold this shape
            raise
        Ao, Aabs = run_oracle(two_j, two_dl, B)
        assert_parity(Ag, Ao, Aabs, what=f"random spins {two_j} dl {two_dl}")
        done += 1


def _run_sub(two_j, two_dl, Bdev, first, count):
    out = torch.full(tuple(count), float("nan"), dtype=torch.float64, device="cuda")
    sf.sf_vertex_amplitude_intertwiners(two_j, two_dl, Bdev, first, count, out, torch.cuda.current_stream())
    torch.cuda.synchronize()
    return out.cpu().numpy()


@pytest.mark.parametrize("which", ["config0", "config2_dl2", "half_integer"])
def test_reduced_intertwiner_ranges(path, which):
    """the tensor for a reduced set of boundary intertwiners = the sub-block of the full tensor; batches
    over i1 joined at the end give the full tensor."""
    if which == "config0":
        cfg = wl.CONFIGS[0]
    elif which == "config2_dl2":
        cfg = wl.config2(2)
    else:
        cfg = dict(two_j=[4, 3, 1, 4, 2, 5, 5, 5, 4, 3], two_dl=4, boosters="random", seed=77)
    two_j, two_dl = cfg["two_j"], cfg["two_dl"]
    B = boosters_for(cfg)
    Bdev = to_device(B)
    Ao, Aabs = run_oracle(two_j, two_dl, B)
    _, n_i = sf.sf_vertex_dims(two_j)
    rng = random.Random(41)
    for _ in range(4):
        first = [rng.randrange(n) for n in n_i]
        count = [rng.randrange(1, n - f + 1) for n, f in zip(n_i, first)]
        sl = tuple(slice(f, f + c) for f, c in zip(first, count))
        assert_parity(_run_sub(two_j, two_dl, Bdev, first, count), Ao[sl], Aabs[sl], what=f"{which} block {first} {count}")
    # batches over i1, joined (the paper's way of splitting a tensor that does not fit)
    full = run_gpu(two_j, two_dl, B, Bdev=Bdev)
    joined = np.concatenate([_run_sub(two_j, two_dl, Bdev, [a, 0, 0, 0, 0], [1] + list(n_i[1:])) for a in range(n_i[0])], axis=0)
    assert_parity(joined, Ao, Aabs, what=f"{which} joined i1 batches")
    assert np.abs(joined - full).max() <= 1e-13 * max(Aabs.max(), 1e-300)
    for bad_first, bad_count in [([0] * 5, [n_i[0] + 1] + list(n_i[1:])), ([0, 0, -1, 0, 0], list(n_i)), ([0] * 5, [1, 1, 0, 1, 1])]:
        with pytest.raises(sf.SfError) as e:
            sf.sf_vertex_amplitude_intertwiners(two_j, two_dl, Bdev, bad_first, bad_count,
                                                torch.zeros(8, dtype=torch.float64, device="cuda"))
        assert e.value.status == sf.SF_EARG


def test_many_shells_small_spins(path):
    """Delta_l = 13 on j = 1 (14 values per virtual spin, 7.5 M shells; most of them empty): more than 12 offsets per
    spin takes the general-size branch of the factorised Q phase."""
    cfg = dict(two_j=[2] * 10, two_dl=26, boosters="random", seed=4242)
    B = boosters_for(cfg)
    Bdev = to_device(B)
    nl3 = 14 ** 3
    for lo, hi in [(3, 203), (0, nl3), (nl3 * 15 + 7, nl3 * 16 + 500)]:
        Ag = run_gpu(cfg["two_j"], cfg["two_dl"], B, lo, hi, Bdev=Bdev)
        Ao, Aabs = run_oracle(cfg["two_j"], cfg["two_dl"], B, lo, hi)
        assert np.abs(Ao).max() > 0
        assert_parity(Ag, Ao, Aabs, what=f"j=1 dl=13 shells [{lo},{hi})")


def test_factorised_path_reads_only_what_it_wrote():
    """The intermediates of the factorised path are written and read through the same range predicates; with the arrays
    pre-filled with NaN patterns (sf_set_debug_poison) the tensor must come out bit for bit the same."""
    cases = [wl.CONFIGS[0], wl.config2(3), wl.config1(5), dict(two_j=[4, 3, 1, 4, 2, 5, 5, 5, 4, 3], two_dl=4, boosters="random", seed=77),
             _config4(2)]
    sf.sf_set_path(4)
    try:
        for cfg in cases:
            B = boosters_for(cfg)
            Bdev = to_device(B)
            n = (cfg["two_dl"] // 2 + 1) ** 6
            for lo, hi in [(None, None), (n // 3, n // 3 + 57 if n > 100 else n)]:
                clean = run_gpu(cfg["two_j"], cfg["two_dl"], B, lo, hi, Bdev=Bdev)
                sf.sf_set_debug_poison(True)
                poisoned = run_gpu(cfg["two_j"], cfg["two_dl"], B, lo, hi, Bdev=Bdev)
                sf.sf_set_debug_poison(False)
                assert np.isfinite(poisoned).all() and np.array_equal(clean, poisoned), cfg.get("name")
        # the headline workload on one block of shells and on a ragged range
        cfg = wl.CONFIGS[3]
        B = boosters_for(cfg)
        Bdev = to_device(B)
        for lo, hi in [(11 ** 3 * 40, 11 ** 3 * 41), (11 ** 5 * 7 - 300, 11 ** 5 * 7 + 900)]:
            clean = run_gpu(cfg["two_j"], cfg["two_dl"], B, lo, hi, Bdev=Bdev)
            sf.sf_set_debug_poison(True)
            poisoned = run_gpu(cfg["two_j"], cfg["two_dl"], B, lo, hi, Bdev=Bdev)
            sf.sf_set_debug_poison(False)
            assert np.array_equal(clean, poisoned)
    finally:
        sf.sf_set_debug_poison(False)
        sf.sf_set_path(0)


def test_errors(path):
    two_j = [2] * 10
    B = to_device(boosters_for(wl.CONFIGS[0]))
    out = torch.zeros(3 ** 5, dtype=torch.float64, device="cuda")
    # the last: the largest {6j} label 2 (j + Delta_l) = 260 is beyond the validated envelope of the {6j} evaluation
    for bad_j, bad_dl, status in [([2] * 9 + [3], 4, sf.SF_ESPIN), (two_j, 3, sf.SF_EARG), (two_j, -2, sf.SF_EARG),
                                  ([130] * 10, 0, sf.SF_EARG)]:
        with pytest.raises(sf.SfError) as e:
            sf.sf_vertex_amplitude(bad_j, bad_dl, B, out)
        assert e.value.status == status
    with pytest.raises(sf.SfError) as e:
        sf.sf_vertex_amplitude_range(two_j, 4, B, 10, 5, out)
    assert e.value.status == sf.SF_EARG
    with pytest.raises(sf.SfError) as e:
        sf.sf_vertex_amplitude_range(two_j, 4, B, 0, 730, out)
    assert e.value.status == sf.SF_EARG
    assert (out == 0).all()          # untouched on error


def test_host_entry_point_matches_device_entry_point():
    cfg = wl.CONFIGS[0]
    B = boosters_for(cfg)
    Ad = run_gpu(cfg["two_j"], cfg["two_dl"], B)
    hb = [torch.from_numpy(B[e]).pin_memory() for e in (2, 3, 4, 5)]
    ho = torch.empty(3 ** 5, dtype=torch.float64).pin_memory()
    sf.sf_vertex_amplitude_host(cfg["two_j"], cfg["two_dl"], hb, ho, torch.cuda.current_stream())
    assert np.array_equal(ho.numpy().reshape(Ad.shape), Ad)
