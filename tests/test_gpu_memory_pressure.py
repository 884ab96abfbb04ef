"""The factorised path next to another tenant of the device memory (sf_vertex_factor.cu, the P / R pass-size loop).

When the device refuses the P + R blocks of a pass, the pass is halved until they fit.  The refused size is remembered, so
that the following identical calls neither repeat the failing allocation (a device synchronisation, a free and a failed
cudaMalloc per call) nor keep changing the library state -- which would keep them from ever being recorded and replayed
(sf_set_graphs).  Checked: same tensor as without the other tenant, and the repeated calls do reach the replay."""
import numpy as np
import pytest
import torch

import paper_2107_13952_b200 as sf
import workloads as wl
from gpu_common import boosters_for, to_device

pytestmark = pytest.mark.gpu
GB = 1 << 30


def test_refused_pass_size_is_remembered_and_calls_get_recorded():
    cfg = wl.CONFIGS[3]                                   # j = 5, Delta_l = 10: P + R take 11.7 GB per i1, 47 GB for the default pass of 4
    two_j, two_dl = cfg["two_j"], cfg["two_dl"]
    sf.sf_init(wl.GAMMA)
    sf.sf_set_path(4)
    sf.sf_set_graphs(1)
    Bdev = to_device(boosters_for(cfg))
    _, n_i = sf.sf_vertex_dims(two_j)
    st = torch.cuda.current_stream()
    ref = torch.zeros(tuple(n_i), dtype=torch.float64, device="cuda")
    sf.sf_vertex_amplitude(two_j, two_dl, Bdev, ref, st)
    torch.cuda.synchronize()
    assert sf.sf_last_path() == 4
    hog = None
    try:
        sf.sf_finalize()                                  # give the scratch of earlier calls back: the pass size is decided afresh
        sf.sf_init(wl.GAMMA)
        sf.sf_set_path(4)
        torch.cuda.empty_cache()
        free, _ = torch.cuda.mem_get_info()
        leave = 30 * GB                                   # room for two i1 per pass (23.5 GB) and the other arrays (1.5 GB), not for four
        assert free > leave + GB
        hog = torch.empty(free - leave, dtype=torch.uint8, device="cuda")
        out = torch.zeros_like(ref)
        sf.sf_graph_replays(reset=True)
        for call in range(6):
            out.fill_(float("nan"))
            sf.sf_vertex_amplitude(two_j, two_dl, Bdev, out, st)
            torch.cuda.synchronize()
            assert sf.sf_last_path() == 4
            err = float((out - ref).abs().max())
            assert err <= 1e-13 * float(ref.abs().max()), (call, err)
        # call 1 shrinks the pass and allocates, call 2 is remembered, call 3 records: at least calls 4..6 are replays
        assert sf.sf_graph_replays() >= 3, sf.sf_graph_replays()
    finally:
        del hog
        sf.sf_finalize()                                  # forgets the refused size as well
        torch.cuda.empty_cache()
        sf.sf_init(wl.GAMMA)
        sf.sf_set_path(0)


def test_a_new_context_after_finalize_starts_clean():
    """sf_finalize + sf_init: what the library cached about the device and its scratch in the first context (SM count, memory
    size, shared-memory attributes already raised, the zeroed ticket block of the contractions) is not carried over: all
    paths, the batch call and both contractions give the same bits in the second context."""
    cfg = wl.CONFIGS[0]
    two_j, two_dl = cfg["two_j"], cfg["two_dl"]
    Bdev = to_device(boosters_for(cfg))
    _, n_i = sf.sf_vertex_dims(two_j)
    st = torch.cuda.current_stream()
    psi = [torch.full((n,), 0.5 + 0.25j, dtype=torch.complex128, device="cuda") for n in n_i]

    def everything():
        res = []
        for path in (1, 3, 4):
            sf.sf_set_path(path)
            out = torch.full(tuple(n_i), float("nan"), dtype=torch.float64, device="cuda")
            sf.sf_vertex_amplitude(two_j, two_dl, Bdev, out, st)
            res.append(out)
        sf.sf_set_path(0)
        outb = torch.full(tuple(n_i), float("nan"), dtype=torch.float64, device="cuda")
        sf.sf_vertex_amplitude_batch([two_j], [two_dl], [Bdev], [outb], st)
        r1 = torch.zeros(1, dtype=torch.float64, device="cuda")
        r2 = torch.zeros(2, dtype=torch.float64, device="cuda")
        sf.sf_contract_vertices(res[0], outb, r1, st)
        sf.sf_contract_vectors(res[0], psi, r2, st)
        torch.cuda.synchronize()
        return res + [outb, r1, r2]

    sf.sf_init(wl.GAMMA)
    first = everything()
    sf.sf_finalize()
    sf.sf_init(wl.GAMMA)
    second = everything()
    for a, b in zip(first, second):
        assert torch.equal(a, b)
