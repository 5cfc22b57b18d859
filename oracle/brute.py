"""Deliberately naive pure-Python brute force of the layer (I <= 16) -- TEST INFRASTRUCTURE.

Written independently of `oracle/pair_bias_attention.py`: nested loops over Python lists,
`math.exp`, materialises the full [H][I][I] logits.  It exists only to pin the numpy oracle
(tests/test_oracle_pins.py::test_brute_force_*).  Equations: PAPER.md:58, :83 (Eq. 2) and
BASELINE.json config 0's formula; readings in DESIGN.md.
"""
import math


def brute_force(s, z, w_q, w_k, w_v, w_g, w_b, w_o, gamma, beta, H, c, eps=1e-5,
                ln_s=None, b_q=None):
    """All arguments are nested Python lists of floats; returns out as a list of lists."""
    I, c_s = len(s), len(s[0])
    c_z = len(z[0][0])
    D = H * c
    if ln_s is not None:
        gs, bs = ln_s
        s2 = []
        for i in range(I):
            mu = sum(s[i]) / c_s
            var = sum((x - mu) ** 2 for x in s[i]) / c_s
            s2.append([(s[i][t] - mu) / math.sqrt(var + eps) * gs[t] + bs[t] for t in range(c_s)])
        s = s2

    def proj(W, i, col):
        return sum(s[i][t] * W[t][col] for t in range(c_s))

    q = [[proj(w_q, i, e) + (b_q[e] if b_q is not None else 0.0) for e in range(D)] for i in range(I)]
    k = [[proj(w_k, i, e) for e in range(D)] for i in range(I)]
    v = [[proj(w_v, i, e) for e in range(D)] for i in range(I)]
    g = [[1.0 / (1.0 + math.exp(-proj(w_g, i, e))) for e in range(D)] for i in range(I)]

    # logits[h][i][j]
    logits = [[[0.0] * I for _ in range(I)] for _ in range(H)]
    for i in range(I):
        for j in range(I):
            zz = z[i][j]
            mu = sum(zz) / c_z
            var = sum((x - mu) ** 2 for x in zz) / c_z
            zh = [(zz[t] - mu) / math.sqrt(var + eps) * gamma[t] + beta[t] for t in range(c_z)]
            for h in range(H):
                bias = sum(zh[t] * w_b[t][h] for t in range(c_z))
                dot = sum(q[i][h * c + d] * k[j][h * c + d] for d in range(c))
                logits[h][i][j] = dot / math.sqrt(c) + bias

    out = []
    for i in range(I):
        gated = [0.0] * D
        for h in range(H):
            row = logits[h][i]
            mx = max(row)
            ex = [math.exp(x - mx) for x in row]
            tot = sum(ex)
            for d in range(c):
                o = sum(ex[j] / tot * v[j][h * c + d] for j in range(I))
                gated[h * c + d] = g[i][h * c + d] * o
        out.append([sum(gated[e] * w_o[e][t] for e in range(D)) for t in range(len(w_o[0]))])
    return out


def brute_force_sparse(a, p_slice, idx, w_q, w_k, w_v, w_g, w_b, w_o, gamma, beta, H, c, eps=1e-5):
    """Sparse k-neighbour atom attention, same naive style: nested loops over Python
    lists, `math.exp`.  a [L][c_atom], p_slice [L][k][c_atompair], idx [L][k] (negative = unused slot).
    Pins `oracle/sparse_atom_attention.py` (tests/test_oracle_pins.py::test_sparse_brute_force)."""
    L, c_s = len(a), len(a[0])
    c_p = len(p_slice[0][0])
    D = H * c

    def proj(W, i, col):
        return sum(a[i][t] * W[t][col] for t in range(c_s))

    out = []
    for l in range(L):
        gated = [0.0] * D
        slots = [j for j in range(len(idx[l])) if idx[l][j] >= 0]
        for h in range(H):
            if not slots:
                continue
            logit = []
            for j in slots:
                m = idx[l][j]
                pp = p_slice[l][j]
                mu = sum(pp) / c_p
                var = sum((x - mu) ** 2 for x in pp) / c_p
                bias = sum(((pp[t] - mu) / math.sqrt(var + eps) * gamma[t] + beta[t]) * w_b[t][h] for t in range(c_p))
                dot = sum(proj(w_q, l, h * c + d) * proj(w_k, m, h * c + d) for d in range(c))
                logit.append(dot / math.sqrt(c) + bias)
            mx = max(logit)
            ex = [math.exp(x - mx) for x in logit]
            tot = sum(ex)
            for d in range(c):
                o = sum(ex[n] / tot * proj(w_v, idx[l][j], h * c + d) for n, j in enumerate(slots))
                gated[h * c + d] = o / (1.0 + math.exp(-proj(w_g, l, h * c + d)))
        out.append([sum(gated[e] * w_o[e][t] for e in range(D)) for t in range(len(w_o[0]))])
    return out
