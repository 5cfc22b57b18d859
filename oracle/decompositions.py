"""CPU fp64 ORACLE for Design-CP's decompositions  --  TEST INFRASTRUCTURE, NOT THE PRODUCT.

Separate fp64 code path that states what the row-shard and 2D-grid emulations mean
(only tests/, smoke() and bench.py's CPU legs may import it; it shares nothing with the CUDA path).

  * shard_range       PAPER.md:72 Eq. 1 and :337 Eq. 5:
                        I_p = floor(I/P) + [p < I mod P],  start_p = p*floor(I/P) + min(p, I mod P)
  * row(P)            PAPER.md:77-86 section 3.2: stripe p does cross-attention of its query rows
                      against ALL keys, with the bias from its row stripe Z^(p); outputs concatenated.
  * grid(P), G=sqrt(P) PAPER.md:90 section 3.3, :446-450 section C.2: rows and keys cut into G blocks
                      (Eq. 5 on both axes, reading #11 in DESIGN.md); block (r, cb) yields a partial
                      online-softmax state from quadrant Z^(r,cb) only; the G states of a row block are
                      merged left to right ("merges the partial output into a running total via an
                      online softmax"); P must be a perfect square.
  * merge             running softmax statistics (Milakov & Gimelshein):
                        m' = max(m_a, m_b), l' = l_a e^{m_a-m'} + l_b e^{m_b-m'}, acc' likewise.

Pins: tests/test_oracle_pins.py (Eq. 5 closed-form properties exhaustively for I<=200, P<=17;
merge algebra; row/grid agreement with the dense definition to 1e-12).
"""
from __future__ import annotations

import math

import numpy as np

from . import pair_bias_attention as dense

F64 = np.float64


def shard_range(n: int, parts: int, p: int):
    """Eq. 5: (start_p, I_p) of shard p of n items over `parts` shards."""
    if not (1 <= parts and 0 <= p < parts):
        raise ValueError("need 1 <= parts and 0 <= p < parts")
    base, rem = n // parts, n % parts
    length = base + (1 if p < rem else 0)
    start = p * base + min(p, rem)
    return start, length


def grid_side(parts: int) -> int:
    """the 2D scheme needs a perfect-square device count."""
    g = math.isqrt(parts)
    if g * g != parts:
        raise ValueError("grid decomposition needs a perfect-square number of parts")
    return g


def partial_state(q_rows, k_blk, v_blk, b_blk, c: int):
    """Partial online-softmax state of query rows against ONE key block.

    q_rows [R, H, c], k_blk/v_blk [J, H, c], b_blk [R, J, H]  ->
    m [R, H] = max_j l,  l [R, H] = sum_j e^{l-m},  acc [R, H, c] = sum_j e^{l-m} v_j
    """
    R, H, _ = q_rows.shape
    m = np.empty((R, H), dtype=F64)
    lsum = np.empty((R, H), dtype=F64)
    acc = np.empty((R, H, c), dtype=F64)
    for r in range(R):
        lg = dense.logits_row(q_rows[r], k_blk, b_blk[r], c)       # [H, J]
        m[r] = lg.max(axis=1)
        e = np.exp(lg - m[r][:, None])
        lsum[r] = e.sum(axis=1)
        for h in range(H):
            acc[r, h] = e[h] @ v_blk[:, h, :]
    return m, lsum, acc


def merge(a, b):
    """Merge two partial states (m, l, acc) of the same rows over disjoint key sets."""
    m_a, l_a, acc_a = a
    m_b, l_b, acc_b = b
    m = np.maximum(m_a, m_b)
    fa, fb = np.exp(m_a - m), np.exp(m_b - m)
    return m, l_a * fa + l_b * fb, acc_a * fa[..., None] + acc_b * fb[..., None]


def finalize(state, g_rows, w_o):
    """Steps 6-7 from a merged state: o = acc / l, out = (g (.) o) W_o."""
    _, lsum, acc = state
    o = acc / lsum[..., None]
    R = o.shape[0]
    return (g_rows * o.reshape(R, -1)) @ np.asarray(w_o, dtype=F64)


def row_decomposition(s, z, w, H: int, c: int, parts: int, eps: float = 1e-5) -> np.ndarray:
    """row(P): Eq. 2 per stripe, stripes concatenated (the paper's ALLGATHER)."""
    I = np.asarray(s).shape[0]
    outs = []
    for p in range(parts):
        start, length = shard_range(I, parts, p)
        rows = range(start, start + length)
        outs.append(dense.pair_bias_attention_rows(s, z[start:start + length], rows, w, H, c, eps))
    return np.concatenate(outs, axis=0)


def grid_decomposition(s, z, w, H: int, c: int, parts: int, eps: float = 1e-5,
                       first_block_offset: bool = False) -> np.ndarray:
    """grid(P): G x G quadrants, partial states merged over key blocks.

    Merge order: ascending key block cb = 0..G-1 (canonical, reading #13 in DESIGN.md); with
    `first_block_offset` the order is rotated to start at cb = r, the block a transpose-then-ring
    schedule visits first -- same result up to rounding.
    """
    G = grid_side(parts)
    q, k, v, g = dense.single_track(s, w, H, c, eps)
    I = q.shape[0]
    out = np.empty((I, np.asarray(w["w_o"]).shape[1]), dtype=F64)
    for r in range(G):
        r0, rl = shard_range(I, G, r)
        order = [(r + t) % G for t in range(G)] if first_block_offset else list(range(G))
        state = None
        for cb in order:
            c0, cl = shard_range(I, G, cb)
            quad = z[r0:r0 + rl, c0:c0 + cl]                         # Z^(r,cb)  [I_r, I_c, c_z]
            b_blk = np.stack([dense.pair_bias_row(quad[t], w, eps) for t in range(rl)]) \
                if rl and cl else np.zeros((rl, cl, H))
            part = partial_state(q[r0:r0 + rl], k[c0:c0 + cl], v[c0:c0 + cl], b_blk, c)
            state = part if state is None else merge(state, part)    # first block initialises
        out[r0:r0 + rl] = finalize(state, g[r0:r0 + rl], w["w_o"])
    return out


def key_split_states(s, z_rows, row_idx, w, H: int, c: int, key_chunks: int, eps: float = 1e-5):
    """Partial states of the given query rows for each of `key_chunks` Eq.-5 key chunks.

    Returns a list of (m [R,H], l [R,H], acc [R,H,c]); used to check the CUDA path's exported
    partial states and its merge kernel.
    """
    q, k, v, _ = dense.single_track(s, w, H, c, eps)
    I = k.shape[0]
    rows = list(row_idx)
    states = []
    for cb in range(key_chunks):
        c0, cl = shard_range(I, key_chunks, cb)
        b_blk = np.stack([dense.pair_bias_row(np.asarray(z_rows[t])[c0:c0 + cl], w, eps)
                          for t in range(len(rows))])
        states.append(partial_state(q[rows], k[c0:c0 + cl], v[c0:c0 + cl], b_blk, c))
    return states
