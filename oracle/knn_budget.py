"""CPU ORACLE for the STRUCTURED neighbour budget of the sparse atom attention  --  TEST INFRASTRUCTURE, NOT THE PRODUCT.
Only `tests/`, `__graft_entry__.smoke()` and `bench.py`'s cpu_baseline / `--impl reference` legs may import this file.
It shares no code with the CUDA path and imports nothing from it.

What it computes (Design-CP, arxiv/paper_2607_05439; citations are /root/reference/PAPER.md lines):

  PAPER.md:303  "the O(L k) atom-level attention ... draws its k neighbours from a structured budget: a fixed number
      n_seq of per-residue sequence-local neighbours (default n_seq = 2, namely the query atom plus its immediate
      flanking residues' atoms), and the spatially closest atoms beyond those, until the per-query budget
      k = n_attn-keys (default k = 128) is filled.  ...  When the input is a multi-chain assembly with more than three
      chains, the budget is split into an intra-chain quota of k - max(32, k/4) neighbours and an inter-chain quota of
      at least 32 neighbours, ensuring that every query atom always retains at least 32 context atoms outside its own
      chain"
  PAPER.md:454  the [L] token identifiers and chain assignments are the inputs of the masking; distances as in
      oracle/knn.py (one cdist, top-k per row)

Readings (#26) -- the text fixes the quantities, these fix the rest:
  * order relation: every "closest" below means smallest (d2, atom index), d2 the binary32 squared distance of
    oracle/knn.py (floating point decides an integer: same precision and operation order as the kernel);
  * sequence-local set S(l): the atoms of the query's own chain whose residue id differs from the query's by at most
    n_seq - 1 (n_seq = 2: the query's residue and its two flanking residues; n_seq = 1: its own residue; n_seq = 0:
    empty).  S is taken first; if it has more than k atoms, its k closest are the list;
  * at most three chains: the list is S plus the closest atoms outside S until it has k entries;
  * more than three chains (counted over the whole chain-id vector): q_out = min(max(32, floor(k / 4)), k - 1) -- the
    query itself always stays in its list.  The other chains come first in the accounting, because the text states
    the guarantee ("always retains at least 32 context atoms outside its own chain"): n_out = min(q_out, number of
    foreign atoms) closest foreign atoms; the own chain gets the remaining k - n_out entries -- S first (its closest
    members if S alone is larger), then the closest same-chain atoms outside S; if the own chain is smaller than that,
    the remainder goes back to the other chains.  The list always has min(k, L) entries;
  * output order: the selected atoms by (d2, index) ascending (the attention is invariant to the order of its slots;
    this makes the list unique), the query itself included (d2 = 0).

Pins (tests/test_oracle_pins.py): n_seq = 0 with at most three chains is oracle/knn.py; a hand-built four-chain
lattice where both quotas bind (counts and members known in closed form), a short own chain (inter fills), few
foreign atoms (intra fills); a far-away flanking residue that only the sequence-local rule can bring in; a second,
pure-Python implementation (struct-rounded binary32, selection by repeated minimum extraction); chain relabelling and
exact translations change nothing.
"""
from __future__ import annotations

import numpy as np

from .knn import squared_distances_row


def knn_budget_rows(x, residue_id, chain_id, k: int, rows, n_seq: int = 2) -> np.ndarray:
    x = np.asarray(x, dtype=np.float32)
    rid = np.asarray(residue_id, dtype=np.int64)
    cid = np.asarray(chain_id, dtype=np.int64)
    L = x.shape[0]
    k = min(k, L)
    split = np.unique(cid).size > 3
    q_out = min(max(32, k // 4), k - 1)
    ar = np.arange(L)
    out = np.empty((len(rows), k), dtype=np.int32)
    for n, l in enumerate(rows):
        d2 = squared_distances_row(x, l)
        order = np.lexsort((ar, d2))                                  # all atoms, closest first
        same = cid == cid[l]
        seq = same & (np.abs(rid - rid[l]) <= n_seq - 1) if n_seq >= 1 else np.zeros(L, dtype=bool)
        S = [m for m in order if seq[m]]
        if not split:
            rest = [m for m in order if not seq[m]]
            sel = (S + rest)[:k]                                      # S first (its closest if it is larger than k)
        else:
            A = S + [m for m in order if same[m] and not seq[m]]      # own chain: S first, then by distance
            B = [m for m in order if not same[m]]                     # other chains
            n_out = min(len(B), q_out)
            n_in = min(len(A), k - n_out)
            n_out = min(len(B), k - n_in)                             # what the own chain cannot fill
            sel = A[:n_in] + B[:n_out]
        sel = np.asarray(sel, dtype=np.int64)
        out[n] = sel[np.lexsort((sel, d2[sel]))]
    return out


def knn_budget(x, residue_id, chain_id, k: int, n_seq: int = 2) -> np.ndarray:
    return knn_budget_rows(x, residue_id, chain_id, k, list(range(np.asarray(x).shape[0])), n_seq)
