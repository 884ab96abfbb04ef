"""CPU oracle for the EPRL vertex-amplitude hot path of arXiv 2107.13952.

TEST INFRASTRUCTURE, NOT PRODUCT CODE.  Only `tests/`, `__graft_entry__.smoke()`
and `bench.py`'s cpu_baseline / `--impl reference` legs may import anything
from this package.  It shares no code, header, table or helper with
`paper_2107_13952_b200/` (the CUDA path) and neither imports the other.

Contents (each function cites the PAPER.md passage it restates):

  wigner.py     exact {6j} (Racah formula, Python big integers / Fractions),
                exact 3jm and the paper's 4jm symbol of eq. (4)          [pinned]
  ranges.py     intertwiner ranges, step 2 of the algorithm, PAPER.md:168 [pinned]
  fifteenj.py   {15j} of eq. (5) by direct summation over x (exact fixed
                point), plus the brute-force magnetic-index contraction
                that pins its sign                                       [pinned]
  vertex.py     eq. (3): level L0 = literal nested sum (tiny inputs),
                level L1 = per-shell W + naive mode products (C loops)   [pinned]
  vertex_l1.c   the naive C loops behind L1 (steps 5-7)
  contract.py   downstream contractions vertex x vertex and vertex x five
                complex vectors, exact sums       [pinned]

Parity status: every function here is pinned by `tests/test_oracle_*.py`
(closed forms, identities, printed exact values under tests/golden/, brute
force).  Nothing is "parity unpinned".
"""
