"""CPU fp64 ORACLE for the sparse (k-neighbour) atom-level attention with pair bias  --  TEST INFRASTRUCTURE,
NOT THE PRODUCT.  Only `tests/`, `__graft_entry__.smoke()` and `bench.py`'s cpu_baseline / `--impl reference`
legs may import this file.  It shares no code with the CUDA path and imports nothing from it.

What it computes (Design-CP, arxiv/paper_2607_05439; citations are /root/reference/PAPER.md lines):

  PAPER.md:58 (section 3.1)  "Atom-level attention is sparse in computation: each query atom attends to a budget
      of k neighbours ... The relevant slice of P is gathered at those k indices and then projected to the
      per-head bias, so the attention computation itself is O(L k)."
  PAPER.md:303 (section A)   the block "consumes a [L, k, c_atompair] slice rather than a [L, L, c_atompair] tensor";
      k = n_attn-keys (default 128).
  PAPER.md:456 (section C.3) "K/V/B entries are gathered at those ... indices, and the resulting ... logits are
      merged into the running softmax"
  The per-pair arithmetic is the dense layer's (oracle/pair_bias_attention.py, steps 1-7); only the key set of
  query l changes: keys m = idx[l, j], j = 0..k-1, pair features p_slice[l, j, :] = P[l, idx[l, j], :].

Steps, for query atom l (plain definition, one atom at a time, every intermediate materialised):
  1-2. q, k, v, g from the atom single track a [L, c_atom], exactly as single_track() of the dense oracle
  3.   b_j^h = LayerNorm(p_slice[l, j, :]) . W_b[:, h]                       j over the VALID neighbours
  4.   l_j^h = (q_l^h . k_{idx[l,j]}^h) / sqrt(c) + b_j^h
  5.   a_j^h = softmax over the valid j
  6.   o_l^h = sum_j a_j^h v_{idx[l,j]}^h
  7.   out_l = (g_l (.) [o_l^0 .. o_l^{H-1}]) W_o
Readings: a negative index marks an unused slot of the budget (masked out; the paper always
fills the budget); an atom with no valid neighbour gets out_l = 0; a neighbour listed twice counts
twice (the softmax runs over slots, not over distinct atoms).

Pins (tests/test_oracle_pins.py, `-m "not gpu"`): with idx[l] = a permutation of ALL atoms and p_slice the matching
gather of a dense P, the result equals the (pinned) dense oracle; pure-Python brute force on tiny inputs;
invariance under a permutation of the slots; a masked slot equals a shorter list; k = 1 returns the gated value of
the single neighbour.  No function in this file is "parity unpinned".
"""
from __future__ import annotations

import numpy as np

from oracle.pair_bias_attention import _f64, layer_norm, single_track


def sparse_atom_attention_rows(a, p_rows, idx_rows, row_idx, w, H: int, c: int, eps: float = 1e-5) -> np.ndarray:
    """Steps 1-7 for the query atoms `row_idx`; p_rows [n, k, c_atompair] and idx_rows [n, k] are their slices."""
    q, kk, v, g = single_track(a, w, H, c, eps)                 # [L, H, c] x 3, [L, H*c]
    w_b, w_o = _f64(w["w_b"]), _f64(w["w_o"])
    gamma, beta = _f64(w["ln_z_gamma"]), _f64(w["ln_z_beta"])
    out = np.zeros((len(row_idx), w_o.shape[1]))
    for n, l in enumerate(row_idx):
        slots = [j for j in range(idx_rows.shape[1]) if idx_rows[n, j] >= 0]
        if not slots:
            continue
        m = np.asarray([int(idx_rows[n, j]) for j in slots])
        bias = layer_norm(_f64(p_rows[n, slots, :]), gamma, beta, eps) @ w_b          # [k_valid, H]
        logits = np.einsum("hd,jhd->jh", q[l], kk[m]) / np.sqrt(float(c)) + bias      # [k_valid, H]
        e = np.exp(logits - logits.max(axis=0, keepdims=True))
        attn = e / e.sum(axis=0, keepdims=True)
        o = np.einsum("jh,jhd->hd", attn, v[m])                                       # [H, c]
        out[n] = (g[l] * o.reshape(-1)) @ w_o
    return out


def sparse_atom_attention(a, p_slice, idx, w, H: int, c: int, eps: float = 1e-5) -> np.ndarray:
    """All query atoms: a [L, c_atom], p_slice [L, k, c_atompair], idx [L, k] (int, < 0 = unused slot)."""
    L = np.asarray(a).shape[0]
    return sparse_atom_attention_rows(a, np.asarray(p_slice), np.asarray(idx), list(range(L)), w, H, c, eps)
