"""CPU fp64 ORACLE for attention with pair bias  --  TEST INFRASTRUCTURE, NOT THE PRODUCT.

Only `tests/`, `__graft_entry__.smoke()` and `bench.py`'s cpu_baseline / `--impl reference`
legs may import this file.  It shares no code with the CUDA path (`paper_2607_05439_b200/`),
and imports nothing from it.  Plain numpy, float64, one query row at a time, every
intermediate materialised, no blocking / fusion / reordering beyond what is written below.

What it computes (Design-CP, arxiv/paper_2607_05439; citations are /root/reference/PAPER.md lines):

  PAPER.md:58 (section 3.1)  "a learned projection of Z produces a per-head pair bias
      B in R^{I x I x H} that is added to the attention logits before the softmax,
      softmax(Q K^T / sqrt(d) + B)"
  PAPER.md:81-83 (section 3.2, Eq. 2)  Attn^(p) = softmax(Q^(p) K^T / sqrt(d) + B^(p)) V,
      B^(p) = f_B(Z^(p)) in R^{I_p x I x H}: the FIRST index of Z is the query.
  BASELINE.json config 0  out = W_o . ( sigmoid(s W_g) (.) softmax(Q K^T / sqrt(c) + LN(z) W_b) V )

The seven steps (readings of silent points are listed in DESIGN.md):
  1. s~_i = s_i                     (or LayerNorm(s_i; gamma_s, beta_s) when LN_s weights are given)
  2. q_i = s~_i W_q (+ b_q),  k_i = s~_i W_k,  v_i = s~_i W_v,  g_i = 1/(1+exp(-s~_i W_g))
     head h owns channels h*c .. h*c+c-1
  3. per pair: mu = mean_k z_ijk, var = mean_k (z_ijk-mu)^2 (population),
     zhat_ijk = (z_ijk-mu)/sqrt(var+eps)*gamma_k + beta_k,   b_ij^h = sum_k zhat_ijk W_b[k,h]
  4. l_ij^h = (q_i^h . k_j^h)/sqrt(c) + b_ij^h            i = query = first index of z
  5. a_ij^h = exp(l_ij^h - max_j l_ij^h) / sum_j exp(l_ij^h - max_j l_ij^h)
  6. o_i^h = sum_j a_ij^h v_j^h
  7. out_i = (g_i (.) [o_i^0 .. o_i^{H-1}]) W_o

Decompositions (PAPER.md:72 Eq. 1, :337 Eq. 5, :90 section 3.3, :446 section C.2) live in
`oracle/decompositions.py`.

Pins (tests/test_oracle_pins.py, all `-m "not gpu"`): worked example with closed-form LN
(tests/golden/worked_example.txt), pure-Python brute force on I<=16 (oracle/brute.py),
uniform-attention closed form, single-key limit, one-hot orientation limit, LayerNorm
invariances, torch fp64 layer_norm + scaled_dot_product_attention composition, permutation
equivariance, cyclic copy-shift invariance, decomposition agreement.  No function in this
file is "parity unpinned".
"""
from __future__ import annotations

import numpy as np

F64 = np.float64


def _f64(x):
    return np.ascontiguousarray(np.asarray(x, dtype=F64))


def layer_norm(x: np.ndarray, gamma: np.ndarray, beta: np.ndarray, eps: float) -> np.ndarray:
    """Step 3 (and step 1 when LN_s is given): LayerNorm over the LAST axis, population variance."""
    mu = x.mean(axis=-1, keepdims=True)
    d = x - mu
    var = (d * d).mean(axis=-1, keepdims=True)
    return d / np.sqrt(var + eps) * gamma + beta


def single_track(s, w, H: int, c: int, eps: float = 1e-5):
    """Steps 1-2: q, k, v, g from the single track.  Returns arrays [I, H, c] (g: [I, H*c])."""
    s = _f64(s)
    if w.get("ln_s_gamma") is not None:
        s = layer_norm(s, _f64(w["ln_s_gamma"]), _f64(w["ln_s_beta"]), eps)
    I = s.shape[0]
    q = s @ _f64(w["w_q"])
    if w.get("b_q") is not None:
        q = q + _f64(w["b_q"])
    k = s @ _f64(w["w_k"])
    v = s @ _f64(w["w_v"])
    g = 1.0 / (1.0 + np.exp(-(s @ _f64(w["w_g"]))))
    return q.reshape(I, H, c), k.reshape(I, H, c), v.reshape(I, H, c), g


def pair_bias_row(z_i, w, eps: float = 1e-5) -> np.ndarray:
    """Step 3 for one query row: z_i [J, c_z] -> b_i [J, H]."""
    zhat = layer_norm(_f64(z_i), _f64(w["ln_z_gamma"]), _f64(w["ln_z_beta"]), eps)
    return zhat @ _f64(w["w_b"])


def logits_row(q_i, k, b_i, c: int) -> np.ndarray:
    """Step 4 for one query row: q_i [H, c], k [J, H, c], b_i [J, H] -> l [H, J]."""
    H = q_i.shape[0]
    l = np.empty((H, k.shape[0]), dtype=F64)
    for h in range(H):
        l[h] = (k[:, h, :] @ q_i[h]) / np.sqrt(F64(c)) + b_i[:, h]
    return l


def pair_bias_attention_rows(s, z_rows, row_idx, w, H: int, c: int, eps: float = 1e-5) -> np.ndarray:
    """The layer for the query rows `row_idx` only.

    s       [I, c_s]            full single track (keys/values come from ALL tokens)
    z_rows  [len(row_idx), I, c_z]   z[row_idx[r], :, :]  -- rows of z index queries
    returns [len(row_idx), c_s]
    A row's output needs only s and z[i, :, :], so evaluating a subset of rows is exact.
    """
    q, k, v, g = single_track(s, w, H, c, eps)
    w_o = _f64(w["w_o"])
    I = k.shape[0]
    out = np.empty((len(row_idx), w_o.shape[1]), dtype=F64)
    for r, i in enumerate(row_idx):
        b_i = pair_bias_row(z_rows[r], w, eps)                 # step 3  [I, H]
        l = logits_row(q[i], k, b_i, c)                        # step 4  [H, I]
        m = l.max(axis=1, keepdims=True)                       # step 5
        e = np.exp(l - m)
        a = e / e.sum(axis=1, keepdims=True)
        o = np.empty((H, c), dtype=F64)                        # step 6
        for h in range(H):
            o[h] = a[h] @ v[:, h, :]
        out[r] = (g[i] * o.reshape(H * c)) @ w_o               # step 7
    return out


def pair_bias_attention(s, z, w, H: int, c: int, eps: float = 1e-5) -> np.ndarray:
    """The whole layer: s [I, c_s], z [I, I, c_z] -> out [I, c_s] (fp64)."""
    I = np.asarray(s).shape[0]
    return pair_bias_attention_rows(s, z, range(I), w, H, c, eps)
