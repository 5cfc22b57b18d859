"""CPU ORACLE for the k-nearest-neighbour lists that feed the sparse atom attention  --  TEST INFRASTRUCTURE, NOT THE
PRODUCT.  Only `tests/`, `__graft_entry__.smoke()` and `bench.py`'s cpu_baseline / `--impl reference` legs may import
this file.  It shares no code with the CUDA path and imports nothing from it.

What it computes (Design-CP, arxiv/paper_2607_05439; citations are /root/reference/PAPER.md lines):

  PAPER.md:303 (section A)   "The kNN indices are computed once per denoising step from the current noised coordinates
      X^(t) via a single cdist call" ... "the spatially closest atoms ... until the per-query budget k = n_attn-keys
      (default k = 128) is filled"
  PAPER.md:454 (section C.3) "A naive implementation computes an [L, L] distance matrix and takes the top-k per row";
      the distributed version is a chunked cdist + a running top-k merge with the same result.

Definition (the plain one: full distance row, then the k smallest): for query atom l,
  d2(l, m) = (x_m0 - x_l0)^2 + (x_m1 - x_l1)^2 + (x_m2 - x_l2)^2,
  idx[l, :] = the k atoms m with the smallest d2(l, m), ordered by (d2, m) ascending; the query itself (d2 = 0) is
  part of its own list, as in the paper's budget ("the query atom plus ...").
Readings: squared Euclidean distance (same order as cdist's Euclidean); ties broken by the
smaller atom index, which makes the result unique; floating point decides an integer here, so the distance is taken
in the KERNEL's precision and operation order -- IEEE binary32, every operation rounded to nearest, no fused
multiply-add: t = x_m - x_l per coordinate, d2 = (t0*t0 + t1*t1) + t2*t2 -- which numpy float32 arithmetic reproduces
bit for bit.  The structured budget of the paper (n_seq sequence-local atoms, inter-chain quota) is not part of this
function (no formulas in the paper; SURVEY.md 8(f) f4 names the cdist + top-k core only).

Pins (tests/test_oracle_pins.py): integer lattice points (exact distances, neighbours known in closed form), a
pure-Python brute force using `struct`-rounded binary32 arithmetic, scipy's cKDTree (fp64) on well-separated random
points, translation by exactly representable offsets, k = 1 returns the query itself.
"""
from __future__ import annotations

import numpy as np


def squared_distances_row(x: np.ndarray, l: int) -> np.ndarray:
    """d2(l, .) in binary32 with the operation order stated above."""
    x = np.asarray(x, dtype=np.float32)
    t = x - x[l]                                   # float32 subtraction, one rounding per coordinate
    s0 = t[:, 0] * t[:, 0]
    s1 = t[:, 1] * t[:, 1]
    s2 = t[:, 2] * t[:, 2]
    return (s0 + s1) + s2                          # float32 throughout (numpy does not fuse)


def knn_rows(x, k: int, rows) -> np.ndarray:
    x = np.asarray(x, dtype=np.float32)
    L = x.shape[0]
    k = min(k, L)
    out = np.empty((len(rows), k), dtype=np.int32)
    ar = np.arange(L)
    for n, l in enumerate(rows):
        d2 = squared_distances_row(x, l)
        order = np.lexsort((ar, d2))               # primary key d2, ties by the smaller index
        out[n] = order[:k]
    return out


def knn(x, k: int) -> np.ndarray:
    return knn_rows(x, k, list(range(np.asarray(x).shape[0])))
