"""Writes tests/golden/<name>_full.npz: the FULL vertex tensor of one of the secondary workloads bench.py times
(BASELINE.json config 2: homogeneous j = 3, Delta_l = 0..8; config 4: the seeded non-homogeneous spins scaled by
lambda, Delta_l = 6), as the ORACLE computes it -- the same recipe as make_config3_full.py for the headline workload.

Calls only `oracle/` and the seeded input generator `workloads/` (which holds none of the method's arithmetic): exact
big-integer {6j} for the five S arrays (oracle/vertex.py::build_s_arrays), then the naive per-shell C loops of
oracle/vertex_l1.c (steps 5-7) with long double accumulation over contiguous chunks of the canonical shell
order, the chunk tensors summed in long double in chunk order (eq. (3) is additive over shells).  No value in
the file comes from the CUDA path.

    A, Aabs        float64 [n1,n2,n3,n4,n5]  the tensor out[i1][i2][i3][i4][i5] and sum|terms| (reading G15)
    input_sha256   hash of (two_j, two_dl, the four booster arrays): the key the test checks
    nonempty       number of non-empty shells

    python tests/golden/make_full_tensor.py --config 2 --sub 8       # config2_dl8_full.npz   (~9 min on 8 cores)
    python tests/golden/make_full_tensor.py --config 4 --sub 1       # config4_lam1_full.npz  (~1 min)
    python tests/golden/make_full_tensor.py --config 4 --sub 2       # config4_lam2_full.npz  (~11 min)
"""
import argparse
import hashlib
import os
import sys
import time

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(os.path.dirname(HERE))
sys.path.insert(0, ROOT)

import workloads as wl                      # noqa: E402
from oracle import ranges                   # noqa: E402
from oracle import vertex as ov             # noqa: E402


def workload(config, sub):
    if config == 2:
        return wl.config2(sub), f"config2_dl{sub}"
    if config == 4:
        base, _ = wl.config4_base_spins(lambda tj: all(n > 0 for _, n in ranges.boundary_ranges(tj)))
        return wl.config4(base, sub), f"config4_lam{sub}"
    raise SystemExit("--config 2 (with --sub Delta_l) or --config 4 (with --sub lambda)")


def inputs(cfg):
    two_j, two_dl = cfg["two_j"], cfg["two_dl"]
    edge_dims, k_ranges = {}, {}
    for edge in (2, 3, 4, 5):
        _, n_i, _, base, pad = ranges.booster_dims(two_j, two_dl, edge)
        edge_dims[edge] = (n_i, base, pad)
        k_ranges[edge] = ranges.booster_k_ranges(two_j, two_dl, edge)
    return two_j, two_dl, wl.random_boosters(cfg["seed"], two_dl // 2 + 1, edge_dims, k_ranges)


def input_hash(two_j, two_dl, B):
    h = hashlib.sha256()
    h.update(np.asarray(list(two_j) + [two_dl], dtype=np.int64).tobytes())
    for edge in (2, 3, 4, 5):
        h.update(np.ascontiguousarray(B[edge], dtype=np.float64).tobytes())
    return h.hexdigest()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--config", type=int, required=True)
    ap.add_argument("--sub", type=int, required=True, help="Delta_l of config 2, lambda of config 4")
    ap.add_argument("--threads", type=int, default=os.cpu_count() or 1)
    ap.add_argument("--nchunks", type=int, default=27)
    args = ap.parse_args()
    cfg, name = workload(args.config, args.sub)
    two_j, two_dl, B = inputs(cfg)
    key = input_hash(two_j, two_dl, B)
    L = ov.Layout(two_j, two_dl)
    t0 = time.time()
    S = ov.build_s_arrays(L, 0, L.n_shells, processes=args.threads)
    print(f"{name}: S arrays (exact 6j) {time.time() - t0:.1f} s", flush=True)
    A = np.zeros(L.out_shape(), dtype=np.longdouble)
    Aabs = np.zeros(L.out_shape(), dtype=np.longdouble)
    nonempty = 0
    n = L.n_shells
    for c in range(args.nchunks):
        lo, hi = n * c // args.nchunks, n * (c + 1) // args.nchunks
        t = time.time()
        r = ov.vertex_l1(two_j, two_dl, B, lo, hi, long_double=True, want_abs=True, threads=args.threads, s_arrays=S)
        A += r["A"]
        Aabs += r["Aabs"]
        nonempty += r["nonempty"]
        print(f"{name}: chunk {c + 1}/{args.nchunks} shells [{lo},{hi}): {time.time() - t:.1f} s", flush=True)
    out = os.path.join(HERE, name + "_full.npz")
    np.savez_compressed(out, A=A.astype(np.float64), Aabs=Aabs.astype(np.float64), input_sha256=key, nonempty=nonempty,
                        two_j=np.asarray(two_j), two_dl=two_dl)
    print(f"wrote {out}: {nonempty} non-empty shells, key {key}, {time.time() - t0:.0f} s")


if __name__ == "__main__":
    main()
