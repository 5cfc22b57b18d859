"""CPU fp64 ORACLE for a stack of non-triangular Pairformer blocks  --  TEST INFRASTRUCTURE, NOT THE PRODUCT.
Only `tests/`, `__graft_entry__.smoke()` and `bench.py`'s cpu_baseline / `--impl reference` legs may import this file.
It shares no code with the CUDA path and imports nothing from it.

What it computes (Design-CP, arxiv/paper_2607_05439; citations are /root/reference/PAPER.md lines):

  PAPER.md:289 (section A.1)  "The Pairformer block ... is, in this codebase, an AttentionPairBias (16 heads, optional
                              QK-norm) followed by a Transition module; both stock configurations explicitly disable
                              the ... triangle multiplication and triangle attention paths"
  PAPER.md:293                "Two non-triangular Pairformer blocks (each 16-head AttentionPairBias + Transition) then
                              refine (S, Z)"  (token initialiser; :295 two more in the diffusion token encoder)
  PAPER.md:381-409            the Transition on the pair track: Eq. 6 / Algorithm 1, already residual (Z <- Z + A)

Reading (#23): block b, in the order the paper names its parts,
      S <- S + AttentionPairBias_b(S, Z)          (oracle/pair_bias_attention.py; residual on the single track)
      Z <- Z + Transition_b(Z)                    (oracle/pair_transition.py, Eq. 6)
  and block b + 1 sees the updated (S, Z).  The paper gives no formula for a single-track transition, the conditional
  layer norm or QK-norm: they are not part of this stack.
Storage reading: a device pipeline that keeps S and Z in bf16 rounds them once per block when they are written back;
`round_store` (a callable applied to the new S and the new Z of every block, default identity) lets a test state that
precision explicitly.  It is an argument, not arithmetic of this module.

Pins (tests/test_oracle_pins.py): W_o = 0 and W_3 = 0 leave (S, Z) unchanged for any depth; the single-track update of
block 1 equals the independent pure-Python brute force (oracle/brute.py) on the ORIGINAL Z and that of block 2 the
brute force on (S_1, Z_1) -- so a swapped order (transition before attention) or a stale Z fails; Z_2 equals the
transition applied twice.
"""
from __future__ import annotations

from typing import Callable, Optional, Sequence, Tuple

import numpy as np

from .pair_bias_attention import pair_bias_attention
from .pair_transition import pair_transition


def pairformer_block(s, z, w_attn: dict, w_tr: dict, H: int, c: int, eps: float = 1e-5,
                     round_store: Optional[Callable[[np.ndarray], np.ndarray]] = None) -> Tuple[np.ndarray, np.ndarray]:
    """One block: s [I, c_s], z [I, I, c_z] -> (s', z').  w_attn: the layer's weights (w_q ... ln_z_beta), w_tr: w1, w2,
    w3, gamma, beta of the transition."""
    rs = round_store if round_store is not None else (lambda x: x)
    s = np.asarray(s, dtype=np.float64)
    z = np.asarray(z, dtype=np.float64)
    s_new = rs(s + pair_bias_attention(s, z, w_attn, H, c, eps))                      # AttentionPairBias, residual
    z_new = rs(pair_transition(z, w_tr["w1"], w_tr["w2"], w_tr["w3"], w_tr["gamma"], w_tr["beta"], eps))   # Eq. 6
    return s_new, z_new


def pairformer_stack(s, z, blocks: Sequence[Tuple[dict, dict]], H: int, c: int, eps: float = 1e-5,
                     round_store: Optional[Callable[[np.ndarray], np.ndarray]] = None) -> Tuple[np.ndarray, np.ndarray]:
    """`blocks` = [(w_attn, w_tr), ...] applied in order; returns the final (s, z)."""
    for w_attn, w_tr in blocks:
        s, z = pairformer_block(s, z, w_attn, w_tr, H, c, eps, round_store)
    return np.asarray(s, dtype=np.float64), np.asarray(z, dtype=np.float64)
