"""CPU fp64 ORACLE for the pairwise SwiGLU transition  --  TEST INFRASTRUCTURE, NOT THE PRODUCT.
Only `tests/`, `__graft_entry__.smoke()` and `bench.py`'s cpu_baseline / `--impl reference` legs may import this file.
It shares no code with the CUDA path and imports nothing from it.

What it computes (Design-CP, arxiv/paper_2607_05439; citations are /root/reference/PAPER.md lines):

  PAPER.md:381-385 (section B.3, Eq. 6)   Transition(Z) = W_3 ( SiLU(W_1 LN(Z)) (.) W_2 LN(Z) ),
      W_1, W_2 in R^{c_z x 4 c_z}, W_3 in R^{4 c_z x c_z};  residual  Z <- Z + Transition(Z)
  PAPER.md:387-409 (Algorithm 1)          N <- LayerNorm(Z); A <- W_1 N; B <- W_2 N; A <- SiLU(A); A <- A (.) B;
                                          A <- W_3 A; Z <- Z + A          (the order followed below, per pair)

Readings: LayerNorm over the channel axis with affine gamma, beta, population variance,
eps = 1e-5 (the same LayerNorm reading as the attention layer); the weights act on the channel axis of every pair
independently (row vector convention: n W_1 with W_1 stored [c_z, 4 c_z]); no biases; SiLU(x) = x / (1 + e^{-x}).

Pins (tests/test_oracle_pins.py): torch fp64 layer_norm + silu + matmul composition (library routines), pure-Python
brute force, W_3 = 0 and W_1 = 0 give Z back, linearity in W_3, per-pair independence / permutation of pairs.
"""
from __future__ import annotations

import numpy as np


def pair_transition(z, w1, w2, w3, gamma, beta, eps: float = 1e-5) -> np.ndarray:
    """z [..., c_z] -> z + Transition(z), Algorithm 1 step by step (every intermediate materialised)."""
    z = np.asarray(z, dtype=np.float64)
    w1, w2, w3 = (np.asarray(w, dtype=np.float64) for w in (w1, w2, w3))
    gamma, beta = np.asarray(gamma, dtype=np.float64), np.asarray(beta, dtype=np.float64)
    mu = z.mean(axis=-1, keepdims=True)
    d = z - mu
    var = (d * d).mean(axis=-1, keepdims=True)
    n = d / np.sqrt(var + eps) * gamma + beta          # N <- LayerNorm(Z)
    a = n @ w1                                         # A <- W_1 N
    b = n @ w2                                         # B <- W_2 N
    a = a / (1.0 + np.exp(-a))                         # A <- SiLU(A)
    a = a * b                                          # A <- A (.) B
    a = a @ w3                                         # A <- W_3 A
    return z + a                                       # Z <- Z + A
