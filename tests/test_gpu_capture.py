"""Stream capture and the C ABI (include/sfoam.h, "Stream capture"): every entry point that works in the library's scratch
refuses a stream the caller is capturing with SF_ECAPTURE, issues no CUDA work (the capture stays valid, ends normally and
replays), and works again, with unchanged results, once the capture has ended."""
import numpy as np
import pytest
import torch

import paper_2107_13952_b200 as sf
import workloads as wl
from gpu_common import boosters_for, to_device

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module", autouse=True)
def ctx():
    sf.sf_init(wl.GAMMA)
    sf.sf_set_path(0)
    yield


def test_captured_stream_is_refused_and_the_capture_survives():
    cfg = wl.CONFIGS[0]
    two_j, two_dl = cfg["two_j"], cfg["two_dl"]
    Bdev = to_device(boosters_for(cfg))
    _, n_i = sf.sf_vertex_dims(two_j)
    n_shells = (two_dl // 2 + 1) ** 6
    out = torch.zeros(tuple(n_i), dtype=torch.float64, device="cuda")
    res = torch.zeros(2, dtype=torch.float64, device="cuda")
    psi = [torch.ones(n, dtype=torch.complex128, device="cuda") for n in n_i]
    host_B = [b.cpu().numpy() for b in (Bdev[e] for e in (2, 3, 4, 5))]
    host_out = np.zeros(tuple(n_i))
    sf.sf_vertex_amplitude(two_j, two_dl, Bdev, out, torch.cuda.current_stream())
    sf.sf_contract_vertices(out, out, res, torch.cuda.current_stream())
    torch.cuda.synchronize()
    before, nrm_before = out.clone(), float(res.cpu()[0])

    calls = {
        "sf_vertex_amplitude": lambda st: sf.sf_vertex_amplitude(two_j, two_dl, Bdev, out, st),
        "sf_vertex_amplitude_range": lambda st: sf.sf_vertex_amplitude_range(two_j, two_dl, Bdev, 0, n_shells, out, st),
        "sf_vertex_amplitude_intertwiners": lambda st: sf.sf_vertex_amplitude_intertwiners(two_j, two_dl, Bdev, [0] * 5, list(n_i),
                                                                                          out, st),
        "sf_vertex_amplitude_batch": lambda st: sf.sf_vertex_amplitude_batch([two_j], [two_dl], [Bdev], [out], st),
        "sf_vertex_amplitude_host": lambda st: sf.sf_vertex_amplitude_host(two_j, two_dl, host_B, host_out, st),
        "sf_contract_vertices": lambda st: sf.sf_contract_vertices(out, out, res, st),
        "sf_contract_vectors": lambda st: sf.sf_contract_vectors(out, psi, res, st),
    }
    x = torch.arange(8, dtype=torch.float64, device="cuda")
    y = torch.zeros_like(x)
    s = torch.cuda.Stream()
    g = torch.cuda.CUDAGraph()
    refused = {}
    with torch.cuda.graph(g, stream=s):
        y.copy_(x * 3.0)                                     # the caller's own work, so that the graph is not empty
        st = torch.cuda.current_stream()
        for name, call in calls.items():
            with pytest.raises(sf.SfError) as e:
                call(st)
            refused[name] = e.value.status
    assert refused == {name: sf.SF_ECAPTURE for name in calls}, refused
    assert b"captured" in sf._lib().sf_strerror(sf.SF_ECAPTURE)
    y.zero_()
    g.replay()                                               # the capture ended normally and holds the caller's work only
    torch.cuda.synchronize()
    assert torch.equal(y, x * 3.0)
    assert torch.equal(out, before)                          # nothing of the refused calls ran
    # outside the capture the same calls work and give the same bits as before
    out.fill_(float("nan"))
    sf.sf_vertex_amplitude(two_j, two_dl, Bdev, out, torch.cuda.current_stream())
    sf.sf_contract_vertices(out, out, res, torch.cuda.current_stream())
    torch.cuda.synchronize()
    assert torch.equal(out, before) and float(res.cpu()[0]) == nrm_before
