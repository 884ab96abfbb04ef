"""Writes tests/golden/config3_full.npz: the FULL vertex tensor of the headline workload (BASELINE.json config 3,
homogeneous j = 5, Delta_l = 10, all 11^6 = 1 771 561 shells) as the ORACLE computes it.

Calls only `oracle/` (and the seeded input generator `workloads/`, which holds none of the method's arithmetic):
exact big-integer {6j} for the five S arrays (oracle/vertex.py::build_s_arrays), then the naive per-shell C loops of
oracle/vertex_l1.c (steps 5-7) with long double accumulation, over contiguous chunks of the canonical
shell order (the paper's own decomposition over shells; eq. (3) is additive over shells).  The chunk
tensors are summed in long double in chunk order.  No value in the file comes from the CUDA path.

    A     float64 [11,11,11,11,11]   the tensor, out[i1][i2][i3][i4][i5]
    Aabs  float64 [11,11,11,11,11]   sum of |terms| at the finest (l_f, k_e, x) granularity (reading G15)
    input_sha256                     hash of (two_j, two_dl, the four booster arrays): the key the test checks
    nonempty                         number of non-empty shells

Cost: about 2 hours on 8 cores (long double + the |terms| pass run at ~260 shells/s); chunks are checkpointed under
--ckpt so an interrupted run resumes.

    python tests/golden/make_config3_full.py [--threads N] [--ckpt DIR] [--chunks-per-run K]
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

OUT = os.path.join(HERE, "config3_full.npz")


def inputs():
    cfg = wl.CONFIGS[3]
    two_j, two_dl = cfg["two_j"], cfg["two_dl"]
    edge_dims, k_ranges = {}, {}
    for edge in (2, 3, 4, 5):
        _, n_i, _, base, pad = ranges.booster_dims(two_j, two_dl, edge)
        edge_dims[edge] = (n_i, base, pad)
        k_ranges[edge] = ranges.booster_k_ranges(two_j, two_dl, edge)
    B = wl.random_boosters(cfg["seed"], two_dl // 2 + 1, edge_dims, k_ranges)
    return two_j, two_dl, B


def input_hash(two_j, two_dl, B):
    h = hashlib.sha256()
    h.update(np.asarray(list(two_j) + [two_dl], dtype=np.int64).tobytes())
    for edge in (2, 3, 4, 5):
        h.update(np.ascontiguousarray(B[edge], dtype=np.float64).tobytes())
    return h.hexdigest()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--threads", type=int, default=os.cpu_count() or 1)
    ap.add_argument("--ckpt", default=os.path.join(HERE, ".config3_full_ckpt"))
    ap.add_argument("--nchunks", type=int, default=121)
    args = ap.parse_args()

    two_j, two_dl, B = inputs()
    key = input_hash(two_j, two_dl, B)
    L = ov.Layout(two_j, two_dl)
    os.makedirs(args.ckpt, exist_ok=True)
    t0 = time.time()
    S = ov.build_s_arrays(L, 0, L.n_shells, processes=args.threads)
    print(f"S arrays (exact 6j): {time.time() - t0:.1f} s", flush=True)

    A = np.zeros(L.out_shape(), dtype=np.longdouble)
    Aabs = np.zeros(L.out_shape(), dtype=np.longdouble)
    nonempty = 0
    n = L.n_shells
    for c in range(args.nchunks):
        lo, hi = n * c // args.nchunks, n * (c + 1) // args.nchunks
        f = os.path.join(args.ckpt, f"{key[:16]}_{args.nchunks}_{c}.npz")
        if os.path.exists(f):
            z = np.load(f)
            a, ab, ne = z["A"], z["Aabs"], int(z["nonempty"])
        else:
            t = time.time()
            r = ov.vertex_l1(two_j, two_dl, B, lo, hi, long_double=True, want_abs=True, threads=args.threads,
                             s_arrays=S)
            a, ab, ne = r["A"], r["Aabs"], r["nonempty"]
            np.savez(f + ".tmp.npz", A=a, Aabs=ab, nonempty=ne)
            os.replace(f + ".tmp.npz", f)
            print(f"chunk {c + 1}/{args.nchunks} shells [{lo},{hi}): {time.time() - t:.1f} s", flush=True)
        A += a
        Aabs += ab
        nonempty += ne
    np.savez_compressed(OUT, A=A.astype(np.float64), Aabs=Aabs.astype(np.float64), input_sha256=key,
                        nonempty=nonempty, two_j=np.asarray(two_j), two_dl=two_dl)
    print(f"wrote {OUT}: {nonempty} non-empty shells, key {key}, {time.time() - t0:.0f} s")


if __name__ == "__main__":
    main()
