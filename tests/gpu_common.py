"""Shared helpers of the GPU parity tests: run the CUDA path through the C-ABI binding and the oracle on the same
seeded inputs, compare entry by entry with the tolerance of north_star:

    |A_gpu - A_oracle| <= 1e-11 * sum|terms|      (FP64; reading G15 of DESIGN.md: terms at the finest (l_f, k_e, x)
                                                   granularity, which the oracle returns as Aabs)
"""
import numpy as np
import torch

import paper_2107_13952_b200 as sf
import workloads as wl
from oracle import vertex as ov

TOL = 1e-11


def abi_dims(two_j, two_dl):
    """edge_dims / k_ranges in the form workloads/ expects, from the C-ABI host helpers."""
    edge_dims, k_ranges = {}, {}
    for edge in (2, 3, 4, 5):
        _, n_i, base, pad = sf.sf_booster_dims(two_j, two_dl, edge)
        edge_dims[edge] = (n_i, base, pad)
        k_ranges[edge] = sf.sf_booster_kranges(two_j, two_dl, edge)
    return edge_dims, k_ranges


def boosters_for(cfg):
    two_j, two_dl = cfg["two_j"], cfg["two_dl"]
    edge_dims, k_ranges = abi_dims(two_j, two_dl)
    if cfg["boosters"] == "identity":
        lo, _ = sf.sf_vertex_dims(two_j)
        return wl.identity_boosters(edge_dims, lo)
    return wl.random_boosters(cfg["seed"], two_dl // 2 + 1, edge_dims, k_ranges)


def to_device(B):
    return {e: torch.from_numpy(np.ascontiguousarray(b)).cuda() for e, b in B.items()}


def run_gpu(two_j, two_dl, B, lo=None, hi=None, Bdev=None):
    _, n_i = sf.sf_vertex_dims(two_j)
    Bdev = Bdev if Bdev is not None else to_device(B)
    out = torch.full(tuple(n_i), float("nan"), dtype=torch.float64, device="cuda")
    stream = torch.cuda.current_stream()
    if lo is None:
        sf.sf_vertex_amplitude(two_j, two_dl, Bdev, out, stream)
    else:
        sf.sf_vertex_amplitude_range(two_j, two_dl, Bdev, lo, hi, out, stream)
    torch.cuda.synchronize()
    return out.cpu().numpy()


def run_oracle(two_j, two_dl, B, lo=0, hi=None, processes=8):
    r = ov.vertex_l1(two_j, two_dl, B, shell_lo=lo, shell_hi=hi, long_double=True, want_abs=True,
                     processes=processes)
    return r["A"], r["Aabs"]


def assert_parity(Ag, Ao, Aabs, tol=TOL, what=""):
    assert Ag.shape == Ao.shape
    assert np.isfinite(Ag).all(), f"{what}: non-finite output"
    err = np.abs(Ag - Ao)
    bound = tol * Aabs
    bad = err > bound
    # an entry whose every term vanishes must be exactly zero on both sides
    worst = float((err / np.maximum(Aabs, 1e-300)).max()) if err.size else 0.0
    assert not bad.any(), f"{what}: {int(bad.sum())} entries exceed {tol}*sum|terms|; worst ratio {worst:.3e}"
    return worst
