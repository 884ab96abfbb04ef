"""Helper for tests: problem dimensions from the ORACLE's range code, in the form workloads/ expects."""
from oracle import ranges


def dims(two_j, two_dl):
    edge_dims, k_ranges = {}, {}
    for edge in (2, 3, 4, 5):
        _, n_i, _, base, pad = ranges.booster_dims(two_j, two_dl, edge)
        edge_dims[edge] = (n_i, base, pad)
        k_ranges[edge] = ranges.booster_k_ranges(two_j, two_dl, edge)
    return edge_dims, k_ranges


def spins_valid(two_j):
    return all(n > 0 for _, n in ranges.boundary_ranges(two_j))
