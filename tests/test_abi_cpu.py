"""CPU-side checks of the C-ABI library (no compute calls: there is no GPU here).

  * libsfoam.so loads and exports every function include/sfoam.h and include/sfoam_debug.h declare
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
    header = open(os.path.join(ROOT, "include", "sfoam.h")).read() + open(os.path.join(ROOT, "include", "sfoam_debug.h")).read()
    header = re.sub(r"/\*.*?\*/", "", header, flags=re.S)
    names = set(re.findall(r"\b(sf_[a-z0-9_]+)\s*\(", header))
    assert {"sf_init", "sf_sixj_table", "sf_vertex_amplitude", "sf_vertex_amplitude_range",
            "sf_vertex_amplitude_host", "sf_sixj_get", "sf_vertex_dims", "sf_booster_dims"} <= names
    lib = ctypes.CDLL(sf.LIB_PATH)
    for n in sorted(names):
        assert hasattr(lib, n), f"{n} declared in include/*.h but not exported"


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


def _tri(a, b, c):
    return ((a + b + c) % 2 == 0) & (c >= abs(a - b)) & (c <= a + b)


def _factor_work_bruteforce(two_j, two_dl):
    """The counts sf_factor_work returns, by dense boolean masks over every index of every contraction of the factorised
    chain (K-f): a term counts when the triads among the labels of both operands hold."""
    import numpy as np
    from oracle.ranges import J12, J13, J14, J15, J23, J24, J25, J34, J35, J45
    nl, j = two_dl // 2 + 1, two_j
    br = ranges.boundary_ranges(two_j)
    n1, n2, n3, n4, n5 = [b[1] for b in br]
    lv = {s: j[s] + 2 * np.arange(nl) for s in (J23, J24, J25, J34, J35, J45)}
    i1 = br[0][0] + 2 * np.arange(n1)
    ks = []
    for e in (2, 3, 4, 5):
        _, _, _, base, pad = ranges.booster_dims(two_j, two_dl, e)
        ks.append(base + 2 * np.arange(pad))
    k2, k3, k4, k5 = ks
    x = np.arange(min(abs(a - b) for a in i1 for b in lv[J25]), max(a + b for a in i1 for b in lv[J25]) + 1, 2)

    def m(spec, *vals):
        """boolean triad mask with one axis per array argument (scalars broadcast)"""
        arrs = [v for v in vals if not np.isscalar(v)]
        nd, out, pos = len(arrs), [], 0
        for v in vals:
            if np.isscalar(v):
                out.append(v)
            else:
                sh = [1] * nd
                sh[pos] = len(v)
                out.append(v.reshape(sh))
                pos += 1
        return _tri(*out).astype(np.int64)

    I = np.einsum
    t_i1_l25_x = m("", i1, lv[J25], x)
    t_k5_l25 = m("", k5, lv[J25], j[J15])
    t_k5_x = m("", k5, j[J14], x)
    t_k4_l45 = m("", j[J14], k4, lv[J45])
    t_l35_k5_l45 = m("", lv[J35], k5, lv[J45])
    t_l35_k4_x = m("", lv[J35], k4, x)
    t_l24_l34_k4 = m("", lv[J24], lv[J34], k4)
    t_k3_l35_l34 = m("", k3, lv[J35], lv[J34])
    t_k3_l24_x = m("", k3, lv[J24], x)
    t_k3_l23 = m("", j[J13], k3, lv[J23])
    t_k2_l23_l24 = _tri(lv[J23].reshape(1, -1, 1), lv[J24].reshape(1, 1, -1), k2.reshape(-1, 1, 1)).astype(np.int64)
    t_k2_l25 = m("", k2, lv[J25], j[J12])
    t_k2_x = m("", k2, j[J13], x)
    zc = I("abx,ub,ux,kd,cud,ckx->bacdkx", t_i1_l25_x, t_k5_l25, t_k5_x, t_k4_l45, t_l35_k5_l45, t_l35_k4_x)
    zmask = (zc > 0).astype(np.int64)
    qc = I("bacdkx,kd,efk->bacefkx", zmask, t_k4_l45, t_l24_l34_k4)
    qmask = (qc > 0).astype(np.int64)
    pc = I("bacefkx,ckx,efk,gcf,gex->ebagxfc", qmask, t_l35_k4_x, t_l24_l34_k4, t_k3_l35_l34, t_k3_l24_x)
    pmask = (pc > 0).astype(np.int64)
    rc = I("ebagxfc,gcf,gh->ebagxh", pmask, t_k3_l35_l34, t_k3_l23)
    rmask = (rc > 0).astype(np.int64)
    gc = I("whe,wb,wx,abx,gex,gh->ebagxh", t_k2_l23_l24, t_k2_l25, t_k2_x, t_i1_l25_x, t_k3_l24_x, t_k3_l23)
    mac = {"Z": zc.sum() * n5, "Q": qc.sum() * n5 * n4, "P": pc.sum() * n5 * n4, "R": rc.sum() * n3 * n4 * n5,
           "G": gc.sum() * n2, "A": ((gc > 0) * rmask).sum() * n2 * n3 * n4 * n5}
    elems = {"Z": zmask.sum() * n5, "Q": qmask.sum() * n4 * n5, "P": pmask.sum() * n4 * n5, "R": rmask.sum() * n3 * n4 * n5}
    return mac, elems


@pytest.mark.parametrize("two_j,two_dl", [([2] * 10, 4), ([1] * 10, 2), ([6] * 10, 4), ([4, 3, 1, 4, 2, 5, 5, 5, 4, 3], 4),
                                          ([8, 7, 12, 3, 8, 5, 9, 12, 3, 7], 2)])
def test_factor_work_matches_dense_mask_count(two_j, two_dl):
    """The roofline numerator of the factorised path (bench.py) = useful multiply-adds on valid index ranges: the host
    counter of the library against a dense brute-force count."""
    mac, elems = sf.sf_factor_work(two_j, two_dl)
    bmac, belems = _factor_work_bruteforce(two_j, two_dl)
    for k in mac:
        assert mac[k] == bmac[k], (k, mac[k], bmac[k])
    for k in elems:
        assert elems[k] == belems[k], (k, elems[k], belems[k])
