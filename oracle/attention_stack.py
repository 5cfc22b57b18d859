"""CPU fp64 ORACLE for the diffusion transformer's attention stack on a resident pair tensor  --  TEST INFRASTRUCTURE,
NOT THE PRODUCT.  Only `tests/`, `__graft_entry__.smoke()` and `bench.py`'s cpu_baseline / `--impl reference` legs may
import this file.  It shares no code with the CUDA path and imports nothing from it.

What it computes (Design-CP, arxiv/paper_2607_05439; citations are /root/reference/PAPER.md lines):

  PAPER.md:294 (section A.1)  "Diffusion transformer (one call per recycling iteration).  Eighteen sequential
                              AttentionPairBiasDiffusion + ConditionedTransitionBlock blocks (16 heads each, 0.10
                              dropout) update the token-level latent A_I in R^{B x I x c_token} using the local pair
                              bias derived from Z.  This is the stage that dominates per-step compute"
  PAPER.md:285                c_token = 768
  PAPER.md:58, :83 (Eq. 2)    the attention with pair bias itself (oracle/pair_bias_attention.py)

Reading (#25): block b = 1 .. n, each with its own weights (projections, pair LayerNorm affine,
W_b, optional LayerNorm on the latent and query bias),
      A <- A + AttentionPairBias_b(A, Z)
  with Z READ-ONLY: every block derives its own bias LN_b(Z) W_b^b from the same pair tensor, and block b + 1 sees the
  latent block b wrote.  Dropout is the identity at inference.  The paper gives no formulas for the conditional (AdaLN)
  normalisation nor for the ConditionedTransitionBlock: they are not part of this stack.
Storage reading: a device pipeline that keeps A in bf16 rounds it once per block when it is written back; `round_store`
(a callable applied to the new A of every block, default identity) states that precision.  It is an argument, not
arithmetic of this module.

Pins (tests/test_oracle_pins.py): W_o = 0 leaves A unchanged for any depth; one block equals A + the dense oracle;
block 2's update equals the independent pure-Python brute force (oracle/brute.py) on the latent block 1 wrote and the
ORIGINAL Z -- a stack that fed block 2 the original latent, or another block's weights, fails; Z is not written;
`round_store` is applied once per block.
"""
from __future__ import annotations

from typing import Callable, Optional, Sequence

import numpy as np

from .pair_bias_attention import pair_bias_attention


def attention_stack(a, z, blocks: Sequence[dict], H: int, c: int, eps: float = 1e-5,
                    round_store: Optional[Callable[[np.ndarray], np.ndarray]] = None) -> np.ndarray:
    """a [I, c_token], z [I, I, c_z] (read-only), blocks = [weights of block 1, ...] -> the final latent [I, c_token]."""
    rs = round_store if round_store is not None else (lambda x: x)
    a = np.asarray(a, dtype=np.float64)
    z = np.asarray(z, dtype=np.float64)
    for w in blocks:
        a = np.asarray(rs(a + pair_bias_attention(a, z, w, H, c, eps)), dtype=np.float64)   # PAPER.md:294; residual
    return a
