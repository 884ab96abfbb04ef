"""CPU-side checks of the C-ABI library (no compute calls: there is no GPU here).

  * libsfoam.so loads and exports every function include/sfoam.h declares
  * the pure host integer helpers (step 2 of the algorithm) agree with the oracle's range code
    and with the counts of SURVEY.md 8(a)/8(c) P2
  * without a CUDA device the compute entry points fail loudly (no CPU fallback)
"""
import ctypes
import os
import re

import pytest

import paper_2107_13952_b200 as sf
from paper_2107_13952_b200 import build as sf_build
from oracle import ranges

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module", autouse=True)
def built():
    sf_build.build()


def test_every_declared_symbol_is_exported():
    header = open(os.path.join(ROOT, "include", "sfoam.h")).read()
    header = re.sub(r"/\*.*?\*/", "", header, flags=re.S)
    names = set(re.findall(r"\b(sf_[a-z0-9_]+)\s*\(", header))
    assert {"sf_init", "sf_sixj_table", "sf_vertex_amplitude", "sf_vertex_amplitude_range",
            "sf_vertex_amplitude_host", "sf_sixj_get", "sf_vertex_dims", "sf_booster_dims"} <= names
    lib = ctypes.CDLL(sf.LIB_PATH)
    for n in sorted(names):
        assert hasattr(lib, n), f"{n} declared in sfoam.h but not exported"


SPIN_SETS = [([2] * 10, 4), ([1] * 10, 2), ([6] * 10, 6), ([10] * 10, 4),
             ([8, 7, 12, 3, 8, 5, 9, 12, 3, 7], 4), ([4, 3, 1, 4, 2, 5, 5, 5, 4, 3], 2)]


@pytest.mark.parametrize("two_j,two_dl", SPIN_SETS)
def test_dims_match_oracle_ranges(two_j, two_dl):
    br = ranges.boundary_ranges(two_j)
    lo, n = sf.sf_vertex_dims(two_j)
    assert lo == [r[0] for r in br] and n == [r[1] for r in br]
    for edge in (2, 3, 4, 5):
        nt, n_i, _, base, pad = ranges.booster_dims(two_j, two_dl, edge)
        assert sf.sf_booster_dims(two_j, two_dl, edge) == (nt, n_i, base, pad)
        kr = ranges.booster_k_ranges(two_j, two_dl, edge)
        got = sf.sf_booster_kranges(two_j, two_dl, edge)
        for t, (klo, nk) in enumerate(kr):
            assert got[t][1] == nk
            if nk:
                assert got[t][0] == klo
            if t % 7 == 0:
                one = sf.sf_booster_krange(two_j, two_dl, edge, t)
                assert one[1] == nk and (nk == 0 or one[0] == klo)


def test_error_codes_of_host_helpers():
    with pytest.raises(sf.SfError) as e:
        sf.sf_vertex_dims([1, 1, 1, 2, 1, 1, 1, 1, 1, 1])       # node 1 has an odd spin sum
    assert e.value.status == sf.SF_ESPIN
    with pytest.raises(sf.SfError) as e:
        sf.sf_vertex_dims([10, 0, 1, 1, 2, 2, 2, 2, 2, 2])      # node 1: (j12 j13) -> 10, (j14 j15) -> 0..2: empty
    assert e.value.status == sf.SF_ESPIN
    with pytest.raises(sf.SfError) as e:
        sf.sf_booster_dims([2] * 10, 3, 2)                      # odd two_dl
    assert e.value.status == sf.SF_EARG
    with pytest.raises(sf.SfError) as e:
        sf.sf_booster_dims([2] * 10, 2, 6)                      # bad edge
    assert e.value.status == sf.SF_EARG
    with pytest.raises(sf.SfError) as e:
        sf.sf_vertex_dims([-2] + [2] * 9)
    assert e.value.status == sf.SF_EARG


def test_work_counts_match_survey_and_oracle():
    # config 0 sum of E_W = 83 124, 729 shells all non-empty
    w = sf.sf_vertex_work([2] * 10, 4)
    assert w["n_nonempty"] == 729 and w["n_w"] == 83124
    # independent count with the oracle's range code
    two_j, two_dl = [2] * 10, 4
    tot_w, tot_f = 0, 0
    n = [r[1] for r in ranges.boundary_ranges(two_j)]
    for offs in ranges.shells(two_dl):
        two_l = ranges.shell_spins(two_j, offs)
        K = [ranges.node_range(two_l, node)[1] for node in (2, 3, 4, 5)]
        if 0 in K:
            continue
        tot_w += n[0] * K[0] * K[1] * K[2] * K[3]
        tot_f += 2 * (n[0] * K[0] * K[1] * K[2] * K[3] * n[4] + n[0] * K[0] * K[1] * K[2] * n[3] * n[4]
                      + n[0] * K[0] * K[1] * n[2] * n[3] * n[4] + n[0] * K[0] * n[1] * n[2] * n[3] * n[4])
    assert tot_w == w["n_w"] and tot_f == w["f_con"]
    # config 2, Delta_l = 7: 262 144 shells, 256 227 non-empty
    assert sf.sf_vertex_work([6] * 10, 14)["n_nonempty"] == 256227
    # additivity over a split of the range
    a = sf.sf_vertex_work([6] * 10, 4, 0, 300)
    b = sf.sf_vertex_work([6] * 10, 4, 300, 729)
    c = sf.sf_vertex_work([6] * 10, 4)
    assert a["f_con"] + b["f_con"] == c["f_con"] and a["n_nonempty"] + b["n_nonempty"] == c["n_nonempty"]


def test_no_cpu_fallback():
    import torch
    if torch.cuda.is_available():
        pytest.skip("a CUDA device is present; the loud-failure path is for boxes without one")
    with pytest.raises(sf.SfError) as e:
        sf.sf_init(1.2)
    assert e.value.status == sf.SF_ECUDA
    with pytest.raises(sf.SfError) as e:
        sf.sf_sixj_table(10)
    assert e.value.status == sf.SF_ENOTINIT
    with pytest.raises(sf.SfError) as e:
        sf.sf_sixj_get([2, 2, 2, 2, 2, 2])
    assert e.value.status == sf.SF_ENOTINIT


def test_shell_boxes_tile_the_range_exactly():
    """Host logic of the factorised path: a range of the canonical shell order (l45 fastest, eq. (9)) is a
    disjoint, ordered union of at most 11 boxes of offsets."""
    import itertools
    import random
    rng = random.Random(5)
    for nl in (1, 2, 3, 4):
        n = nl ** 6
        cases = [(0, n), (0, 0), (n, n), (0, 1), (n - 1, n)] + [tuple(sorted((rng.randrange(n + 1), rng.randrange(n + 1))))
                                                                 for _ in range(40)]
        for lo, hi in cases:
            boxes = sf.sf_shell_boxes(2 * (nl - 1), lo, hi)
            assert len(boxes) <= 11
            shells = []
            for blo, cnt in boxes:
                assert all(c >= 1 for c in cnt) and all(0 <= a and a + c <= nl for a, c in zip(blo, cnt))
                for o in itertools.product(*[range(a, a + c) for a, c in zip(blo, cnt)]):
                    s = 0
                    for d in o:
                        s = s * nl + d
                    shells.append(s)
            # box order = shell order between boxes; inside a box the offsets enumerate a sorted set
            assert sorted(shells) == list(range(lo, hi)), (nl, lo, hi, boxes)
            firsts = [min(sh) for sh in _box_shell_sets(boxes, nl)]
            assert firsts == sorted(firsts)
    with pytest.raises(sf.SfError):
        sf.sf_shell_boxes(3, 0, 1)
    with pytest.raises(sf.SfError):
        sf.sf_shell_boxes(2, 5, 4)


def _box_shell_sets(boxes, nl):
    import itertools
    out = []
    for blo, cnt in boxes:
        ss = []
        for o in itertools.product(*[range(a, a + c) for a, c in zip(blo, cnt)]):
            s = 0
            for d in o:
                s = s * nl + d
            ss.append(s)
        out.append(ss)
    return out
