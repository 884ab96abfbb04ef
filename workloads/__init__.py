"""Seeded synthetic inputs for the five workloads of BASELINE.json (shared by the oracle and the CUDA path).

This module holds NONE of the method's arithmetic: no triangle inequalities, no Wigner symbols, no
contraction.  Everything that depends on the method (intertwiner ranges, validity of a spin set) is passed
in by the caller, who gets it either from `oracle.ranges` (tests) or from the C-ABI helpers
`sf_vertex_dims` / `sf_booster_dims` / `sf_booster_krange` (bench, smoke).

Recipe: the paper's workloads are homogeneous spin sweeps
(Fig. 2 / Listing 6) and the scaled spin set js*lambda; real booster
tensors need the out-of-scope SL(2,C) integrals, so boosters are synthetic:
    B_a[t][i][k] = z * (1 + u + v + w)^(-1.5),  z ~ N(0,1) iid on the valid (i,k) entries, 0 elsewhere,
with (u,v,w) the shell offsets (units of 1) of the edge's three virtual spins.  Generation order: edge 2..5,
then t row-major, then i, then valid k ascending, all from numpy.random.Generator(PCG64(seed)).
"""
import numpy as np

BASE_SEED = 210713952
GAMMA = 1.2   # Immirzi parameter named by the configs; a label only: boosters are inputs


def config_seed(config, sub=0):
    return BASE_SEED + 1000 * config + sub


def homogeneous(two_j):
    return [int(two_j)] * 10


CONFIGS = {
    0: dict(name="config0_j1_dl2", two_j=homogeneous(2), two_dl=4, boosters="random", seed=config_seed(0)),
    3: dict(name="config3_j5_dl10", two_j=homogeneous(10), two_dl=20, boosters="random", seed=config_seed(3)),
}


def config1(two_j):
    """BF sweep: homogeneous spin j = two_j/2 (two_j = 1..20), Delta_l = 0, identity boosters."""
    return dict(name=f"config1_bf_2j{two_j}", two_j=homogeneous(two_j), two_dl=0, boosters="identity", seed=None)


def config2(dl):
    """Homogeneous j = 3, Delta_l = dl in 0..8."""
    return dict(name=f"config2_j3_dl{dl}", two_j=homogeneous(6), two_dl=2 * dl, boosters="random",
                seed=config_seed(2, dl))


def config4_base_spins(is_valid, seed=BASE_SEED):
    """Ten spins 2j drawn uniformly from {2..12} (j in {1, 3/2, ..., 6}), resampled until `is_valid(two_j)`
    (every node's four spins admit a non-empty intertwiner range; predicate supplied by the caller)."""
    rng = np.random.Generator(np.random.PCG64(seed))
    draws = 0
    while True:
        two_j = [int(v) for v in rng.integers(2, 13, size=10)]
        draws += 1
        if is_valid(two_j):
            return two_j, draws


def config4(base_two_j, lam):
    """Non-homogeneous sweep: base spins scaled by lambda = 1..6, Delta_l = 6."""
    return dict(name=f"config4_lam{lam}", two_j=[int(s) * lam for s in base_two_j], two_dl=12,
                boosters="random", seed=config_seed(4, lam))


def random_boosters(seed, nl, edge_dims, k_ranges):
    """Synthetic boosters {2: B2, 3: B3, 4: B4, 5: B5}, each float64 [nl^3][n_i][n_k_pad].

    edge_dims[a] = (n_i, two_k_base, n_k_pad);  k_ranges[a][t] = (two_k_min, n_k)  for a in 2..5.
    """
    rng = np.random.Generator(np.random.PCG64(seed))
    out = {}
    for edge in (2, 3, 4, 5):
        n_i, base, pad = edge_dims[edge]
        B = np.zeros((nl ** 3, n_i, pad))
        t = 0
        for u in range(nl):
            for v in range(nl):
                for w in range(nl):
                    lo, nk = k_ranges[edge][t]
                    if nk > 0:
                        q0 = (lo - base) // 2
                        B[t, :, q0:q0 + nk] = rng.standard_normal((n_i, nk)) * (1.0 + u + v + w) ** -1.5
                    t += 1
        out[edge] = B
    return out


def identity_boosters(edge_dims, two_i_min):
    """delta_{ik} boosters for Delta_l = 0 (one triple): B_a[0][ii][kk] = 1 iff two_i == two_k."""
    out = {}
    for edge in (2, 3, 4, 5):
        n_i, base, pad = edge_dims[edge]
        B = np.zeros((1, n_i, pad))
        for ii in range(n_i):
            kk = (two_i_min[edge - 1] + 2 * ii - base) // 2
            if 0 <= kk < pad:
                B[0, ii, kk] = 1.0
        out[edge] = B
    return out


def one_hot_boosters(nl, edge_dims, hot):
    """All-zero boosters except B_a[t_a][ii_a][kk_a] = 1 for hot[a] = (t_a, ii_a, kk_a)."""
    out = {}
    for edge in (2, 3, 4, 5):
        n_i, _, pad = edge_dims[edge]
        B = np.zeros((nl ** 3, n_i, pad))
        t, ii, kk = hot[edge]
        B[t, ii, kk] = 1.0
        out[edge] = B
    return out
