"""Pins for the CPU fp64 oracle (`-m "not gpu"`): each test fixes the oracle against something
other than itself -- a hand-derived worked example, brute force, closed forms, invariants,
library routines -- so that a dropped term, a wrong sign/index or a transposed operand fails.
Citations: PAPER.md:58, :72 (Eq. 1), :83 (Eq. 2), :90, :337 (Eq. 5); SURVEY.md section 8(c).
"""
import math
import os

import numpy as np
import pytest
import torch

from oracle import brute
from oracle import decompositions as dec
from oracle import pair_bias_attention as orc

HERE = os.path.dirname(os.path.abspath(__file__))


def rand_problem(rng, I, c_s, c_z, H, c, ln_s=False, b_q=False):
    D = H * c
    w = {
        "w_q": rng.normal(size=(c_s, D)) / math.sqrt(c_s),
        "w_k": rng.normal(size=(c_s, D)) / math.sqrt(c_s),
        "w_v": rng.normal(size=(c_s, D)) / math.sqrt(c_s),
        "w_g": rng.normal(size=(c_s, D)) / math.sqrt(c_s),
        "w_b": rng.normal(size=(c_z, H)) / math.sqrt(c_z),
        "w_o": rng.normal(size=(D, c_s)) / math.sqrt(D),
        "ln_z_gamma": 1 + 0.1 * rng.normal(size=c_z),
        "ln_z_beta": 0.1 * rng.normal(size=c_z),
    }
    if ln_s:
        w["ln_s_gamma"] = 1 + 0.1 * rng.normal(size=c_s)
        w["ln_s_beta"] = 0.1 * rng.normal(size=c_s)
    if b_q:
        w["b_q"] = 0.1 * rng.normal(size=D)
    s = rng.normal(size=(I, c_s))
    z = rng.normal(size=(I, I, c_z))
    return s, z, w


# ---------------------------------------------------------------- worked example (golden file)
def _golden():
    vals = {}
    with open(os.path.join(HERE, "golden", "worked_example.txt")) as f:
        for line in f:
            if line.startswith("#") or not line.strip():
                continue
            k, v = line.split()
            vals[k] = float(v)
    return vals


def _worked_problem():
    s = np.array([[1.0], [-0.5]])
    z = np.array([[[1.0, 3.0], [2.0, 0.0]], [[0.0, 4.0], [5.0, 1.0]]])
    w = {"w_q": [[2.0]], "w_k": [[1.0]], "w_v": [[3.0]], "w_g": [[0.0]], "w_o": [[2.0]],
         "w_b": [[0.75], [-0.25]], "ln_z_gamma": [1.0, 1.0], "ln_z_beta": [0.0, 0.0]}
    return s, z, w


def test_worked_example_matches_golden():
    g = _golden()
    s, z, w = _worked_problem()
    out = orc.pair_bias_attention(s, z, w, H=1, c=1, eps=1e-5)
    assert out.shape == (2, 1)
    assert abs(out[0, 0] - g["out0"]) < 1e-13
    assert abs(out[1, 0] - g["out1"]) < 1e-13
    # the golden values themselves follow the hand derivation written in the file header
    r, rp = 1 / math.sqrt(1 + 1e-5 / 1.0), 1 / math.sqrt(1 + 1e-5 / 4.0)
    assert abs(r - g["r"]) < 1e-15 and abs(rp - g["r_prime"]) < 1e-15
    a00 = 1 / (1 + math.exp((-1 + r) - (2 - r)))
    a10 = 1 / (1 + math.exp((0.5 + rp) - (-1 - rp)))
    assert abs(a00 - g["a00"]) < 1e-15 and abs(a10 - g["a10"]) < 1e-15
    assert abs(4.5 * a00 - 1.5 - g["out0"]) < 1e-13 and abs(4.5 * a10 - 1.5 - g["out1"]) < 1e-13
    # bias rows of the worked example: b00=-r, b01=+r, b10=-r', b11=+r'
    b0 = orc.pair_bias_row(z[0], w, 1e-5)[:, 0]
    b1 = orc.pair_bias_row(z[1], w, 1e-5)[:, 0]
    assert np.allclose(b0, [-r, r], atol=1e-15) and np.allclose(b1, [-rp, rp], atol=1e-15)


# ---------------------------------------------------------------- brute force on tiny inputs
@pytest.mark.parametrize("I,c_s,c_z,H,c,ln_s,b_q", [
    (5, 6, 3, 2, 4, False, False),     # H*c != c_s, c_z not a power of two
    (16, 8, 5, 3, 2, True, True),      # optional LN_s and b_q
    (7, 4, 1, 1, 3, False, False),     # c_z = 1
    (1, 3, 4, 2, 2, False, False),     # single token
])
def test_brute_force_agreement(I, c_s, c_z, H, c, ln_s, b_q):
    rng = np.random.default_rng(100 + I)
    s, z, w = rand_problem(rng, I, c_s, c_z, H, c, ln_s, b_q)
    out = orc.pair_bias_attention(s, z, w, H, c)
    ref = brute.brute_force(
        s.tolist(), z.tolist(), w["w_q"].tolist(), w["w_k"].tolist(), w["w_v"].tolist(),
        w["w_g"].tolist(), w["w_b"].tolist(), w["w_o"].tolist(), w["ln_z_gamma"].tolist(),
        w["ln_z_beta"].tolist(), H, c,
        ln_s=(w["ln_s_gamma"].tolist(), w["ln_s_beta"].tolist()) if ln_s else None,
        b_q=w["b_q"].tolist() if b_q else None)
    ref = np.array(ref)
    assert np.max(np.abs(out - ref)) <= 1e-12 * max(1.0, np.max(np.abs(ref)))


# ---------------------------------------------------------------- closed forms
def test_uniform_attention_closed_form():
    """W_b = 0 and identical keys (W_k = 0) => uniform attention => out_i = (g_i * mean_j v_j) W_o."""
    rng = np.random.default_rng(1)
    I, c_s, c_z, H, c = 23, 12, 6, 3, 4
    s, z, w = rand_problem(rng, I, c_s, c_z, H, c)
    w["w_b"] = np.zeros_like(w["w_b"])
    w["ln_z_beta"] = np.zeros_like(w["ln_z_beta"])
    w["w_k"] = np.zeros_like(w["w_k"])
    out = orc.pair_bias_attention(s, z, w, H, c)
    g = 1 / (1 + np.exp(-(s @ w["w_g"])))
    ref = (g * (s @ w["w_v"]).mean(axis=0)) @ w["w_o"]
    assert np.max(np.abs(out - ref)) < 1e-13


def test_constant_values_closed_form():
    """All v_j equal u (rows of s equal except through W_v... use W_v rows so that v_j=u) => o_i = u."""
    rng = np.random.default_rng(2)
    I, c_s, c_z, H, c = 11, 5, 4, 2, 3
    s, z, w = rand_problem(rng, I, c_s, c_z, H, c)
    s[:, 0] = 1.0                       # constant feature
    w["w_v"][1:, :] = 0.0               # v_j = W_v[0,:] for every j
    out = orc.pair_bias_attention(s, z, w, H, c)
    g = 1 / (1 + np.exp(-(s @ w["w_g"])))
    ref = (g * w["w_v"][0]) @ w["w_o"]
    assert np.max(np.abs(out - ref)) < 1e-13


def test_single_key_limit():
    rng = np.random.default_rng(3)
    s, z, w = rand_problem(rng, 1, 7, 5, 2, 3)
    out = orc.pair_bias_attention(s, z, w, 2, 3)
    g = 1 / (1 + np.exp(-(s @ w["w_g"])))
    assert np.max(np.abs(out - (g * (s @ w["w_v"])) @ w["w_o"])) < 1e-14


def test_one_hot_limit_pins_orientation_of_z():
    """Bias +50 at j = pi(i), -50 elsewhere => out_i -> (g_i * v_pi(i)) W_o; a transposed z fails."""
    rng = np.random.default_rng(4)
    I, c_s, c_z, H, c = 9, 6, 2, 2, 3
    s, _, w = rand_problem(rng, I, c_s, c_z, H, c)
    pi = np.roll(np.arange(I), 2)                    # non-involutive permutation (a 9-cycle shift)
    assert not np.array_equal(pi[pi], np.arange(I))
    # c_z = 2: LN(z) = (+r, -r) or (-r, +r); with W_b = (A, -A) the bias is +-2 A r for every head
    z = np.zeros((I, I, 2))
    z[..., 0], z[..., 1] = -1.0, 1.0                  # bias = -2Ar
    for i in range(I):
        z[i, pi[i]] = (1.0, -1.0)                     # bias = +2Ar at j = pi(i)
    w["ln_z_gamma"] = np.ones(2)
    w["ln_z_beta"] = np.zeros(2)
    w["w_b"] = np.tile(np.array([[25.0], [-25.0]]), (1, H))
    out = orc.pair_bias_attention(s, z, w, H, c)
    g = 1 / (1 + np.exp(-(s @ w["w_g"])))
    v = s @ w["w_v"]
    ref = (g * v[pi]) @ w["w_o"]
    assert np.max(np.abs(out - ref)) < 1e-12
    wrong = (g * v[np.argsort(pi)]) @ w["w_o"]       # what a transposed read of z would give
    assert np.max(np.abs(out - wrong)) > 1e-3
    out_t = orc.pair_bias_attention(s, np.swapaxes(z, 0, 1).copy(), w, H, c)
    assert np.max(np.abs(out_t - ref)) > 1e-3


def test_layernorm_invariances():
    """z_ij -> a_ij z_ij + t_ij 1 (a > 0) leaves the bias unchanged for eps = 0; c_z = 1 => zhat = beta."""
    rng = np.random.default_rng(5)
    I, c_s, c_z, H, c = 8, 5, 7, 2, 2
    s, z, w = rand_problem(rng, I, c_s, c_z, H, c)
    a = rng.uniform(0.5, 3.0, size=(I, I, 1))
    t = rng.normal(size=(I, I, 1))
    o1 = orc.pair_bias_attention(s, z, w, H, c, eps=0.0)
    o2 = orc.pair_bias_attention(s, a * z + t, w, H, c, eps=0.0)
    assert np.max(np.abs(o1 - o2)) < 1e-12
    # c_z = 1: constant bias per head => equals bias-free attention (softmax shift invariance)
    s, z, w = rand_problem(rng, I, c_s, 1, H, c)
    w0 = dict(w)
    w0["w_b"] = np.zeros_like(w["w_b"])
    assert np.max(np.abs(orc.pair_bias_attention(s, z, w, H, c)
                         - orc.pair_bias_attention(s, z, w0, H, c))) < 1e-13


def test_library_composition_torch_fp64():
    """Third independent check: torch fp64 layer_norm + linear + scaled_dot_product_attention."""
    rng = np.random.default_rng(6)
    I, c_s, c_z, H, c = 96, 24, 16, 4, 6
    s, z, w = rand_problem(rng, I, c_s, c_z, H, c, ln_s=True, b_q=True)
    out = orc.pair_bias_attention(s, z, w, H, c, eps=1e-5)
    T = lambda x: torch.tensor(np.asarray(x), dtype=torch.float64)
    F = torch.nn.functional
    st = F.layer_norm(T(s), (c_s,), T(w["ln_s_gamma"]), T(w["ln_s_beta"]), 1e-5)
    q = (st @ T(w["w_q"]) + T(w["b_q"])).view(I, H, c).transpose(0, 1)
    k = (st @ T(w["w_k"])).view(I, H, c).transpose(0, 1)
    v = (st @ T(w["w_v"])).view(I, H, c).transpose(0, 1)
    b = F.layer_norm(T(z), (c_z,), T(w["ln_z_gamma"]), T(w["ln_z_beta"]), 1e-5) @ T(w["w_b"])
    o = F.scaled_dot_product_attention(q[None], k[None], v[None], attn_mask=b.permute(2, 0, 1)[None])[0]
    o = o.transpose(0, 1).reshape(I, H * c)
    ref = (torch.sigmoid(st @ T(w["w_g"])) * o) @ T(w["w_o"])
    assert np.max(np.abs(out - ref.numpy())) < 1e-12


# ---------------------------------------------------------------- symmetry
def test_permutation_equivariance():
    rng = np.random.default_rng(7)
    I, c_s, c_z, H, c = 17, 6, 5, 2, 3
    s, z, w = rand_problem(rng, I, c_s, c_z, H, c)
    pi = rng.permutation(I)
    o = orc.pair_bias_attention(s, z, w, H, c)
    op = orc.pair_bias_attention(s[pi], z[pi][:, pi], w, H, c)
    assert np.max(np.abs(op - o[pi])) < 1e-12


def test_cyclic_copy_shift_invariance():
    """Noise-free generator with a cyclic copy table E[a,b] = F[(b-a) mod C] is invariant under
    copy shifts => the output is periodic over copies (echoes the paper's symmetric assemblies,
    PAPER.md:325-327)."""
    import dcp_synth as syn
    cfg = syn.small_config("cyc", I=5 * 4, c_s=6, c_z=4, H=2, c=3, structured=True, copies=5, seed=11)
    w = {k: v.double().numpy() for k, v in syn.make_weights(cfg).items()}
    # noise-free s: repeat the ASU block exactly
    rng = np.random.default_rng(8)
    a = rng.normal(size=(cfg.n_res, cfg.c_s))
    s = np.tile(a, (cfg.copies, 1))
    z = syn.make_z(cfg, noise=0.0, cyclic_copy_table=True).double().numpy()
    o = orc.pair_bias_attention(s, z, w, cfg.H, cfg.c)
    o = o.reshape(cfg.copies, cfg.n_res, -1)
    assert np.max(np.abs(o - o[0:1])) < 1e-12


# ---------------------------------------------------------------- Eq. 5 planner
def test_shard_range_closed_form_exhaustive():
    for n in range(0, 201):
        for P in range(1, 18):
            tot, prev_end, sizes = 0, 0, []
            for p in range(P):
                st, ln = dec.shard_range(n, P, p)
                assert st == prev_end                      # start_{p+1} = start_p + I_p
                assert ln == n // P + (1 if p < n % P else 0)   # Eq. 1
                prev_end = st + ln
                tot += ln
                sizes.append(ln)
            assert tot == n and max(sizes) - min(sizes) <= 1
    # the paper's examples of uneven splits
    assert [dec.shard_range(67, 4, p)[1] for p in range(4)] == [17, 17, 17, 16]
    assert [dec.shard_range(600, 7, p)[1] for p in range(7)] == [86, 86, 86, 86, 86, 85, 85]


def test_grid_needs_perfect_square():
    assert dec.grid_side(16) == 4 and dec.grid_side(1) == 1
    for bad in (2, 3, 8, 15):
        with pytest.raises(ValueError):
            dec.grid_side(bad)


# ---------------------------------------------------------------- merge operator
def test_merge_algebra_and_extremes():
    rng = np.random.default_rng(9)
    R, H, c = 4, 3, 5

    def state(shift):
        m = rng.normal(size=(R, H)) + shift
        return m, rng.uniform(0.5, 2, size=(R, H)), rng.normal(size=(R, H, c))

    a, b, cst = state(0), state(80.0), state(-80.0)
    ab_c = dec.merge(dec.merge(a, b), cst)
    a_bc = dec.merge(a, dec.merge(b, cst))
    ba = dec.merge(b, a)
    for x, y in zip(ab_c, a_bc):
        assert np.all(np.isfinite(x)) and np.allclose(x, y, rtol=1e-12, atol=0)
    for x, y in zip(dec.merge(a, b), ba):
        assert np.allclose(x, y, rtol=1e-14, atol=0)
    m2, l2, acc2 = dec.merge(a, a)                       # self-merge doubles l and acc, keeps m
    assert np.array_equal(m2, a[0]) and np.allclose(l2, 2 * a[1]) and np.allclose(acc2, 2 * a[2])


# ---------------------------------------------------------------- decompositions agree with the dense definition
@pytest.mark.parametrize("I", [12, 13, 30])
def test_row_and_grid_agree_with_dense(I):
    rng = np.random.default_rng(10 + I)
    c_s, c_z, H, c = 6, 5, 2, 3
    s, z, w = rand_problem(rng, I, c_s, c_z, H, c)
    o = orc.pair_bias_attention(s, z, w, H, c)
    scale = np.max(np.abs(o))
    for P in list(range(1, I + 1, max(1, I // 6))) + [I]:
        assert np.max(np.abs(dec.row_decomposition(s, z, w, H, c, P) - o)) <= 1e-12 * scale
    for P in (1, 4, 9, 16):
        if math.isqrt(P) <= I:
            assert np.max(np.abs(dec.grid_decomposition(s, z, w, H, c, P) - o)) <= 1e-12 * scale
            assert np.max(np.abs(dec.grid_decomposition(s, z, w, H, c, P, first_block_offset=True) - o)) \
                <= 1e-12 * scale
    with pytest.raises(ValueError):
        dec.grid_decomposition(s, z, w, H, c, 8)


def test_key_split_states_merge_to_dense():
    rng = np.random.default_rng(11)
    I, c_s, c_z, H, c = 21, 6, 4, 2, 3
    s, z, w = rand_problem(rng, I, c_s, c_z, H, c)
    rows = [0, 5, 20]
    states = dec.key_split_states(s, z[rows], rows, w, H, c, key_chunks=4)
    st = states[0]
    for nxt in states[1:]:
        st = dec.merge(st, nxt)
    _, _, _, g = orc.single_track(s, w, H, c)
    out = dec.finalize(st, g[rows], w["w_o"])
    ref = orc.pair_bias_attention_rows(s, z[rows], rows, w, H, c)
    assert np.max(np.abs(out - ref)) < 1e-12


# ---------------------------------------------------------------- generator determinism
def test_input_generator_is_seed_deterministic():
    import dcp_synth as syn
    cfg = syn.small_config("g", I=60 * 2, c_s=8, c_z=4, H=2, c=4, dtype="bf16", structured=True, seed=5)
    z1, z2 = syn.make_z(cfg, chunk_rows=16), syn.make_z(cfg, chunk_rows=16)
    assert torch.equal(z1, z2)
    assert torch.equal(syn.make_s(cfg), syn.make_s(cfg))
    w1, w2 = syn.make_weights(cfg), syn.make_weights(cfg)
    assert all(torch.equal(w1[k], w2[k]) for k in w1)
    cfg2 = syn.small_config("g", I=60 * 2, c_s=8, c_z=4, H=2, c=4, dtype="bf16", structured=True, seed=6)
    assert not torch.equal(z1, syn.make_z(cfg2, chunk_rows=16))


# ---------------------------------------------------------------- sparse k-neighbour atom attention
def _sparse_problem(rng, L, k, c_s=12, c_p=6, H=2, c=4):
    from oracle import sparse_atom_attention as spo  # noqa: F401
    a, P, w = rand_problem(rng, L, c_s, c_p, H, c)
    idx = np.stack([rng.choice(L, size=k, replace=False) for _ in range(L)])
    p_slice = np.stack([P[l, idx[l]] for l in range(L)])
    return a, P, p_slice, idx, w


def test_sparse_full_budget_equals_dense_oracle():
    """idx[l] = a permutation of ALL atoms, p_slice the matching gather of a dense P  =>  the dense layer."""
    from oracle import sparse_atom_attention as spo
    rng = np.random.default_rng(41)
    L, H, c = 17, 3, 4
    a, P, p_slice, idx, w = _sparse_problem(rng, L, L, H=H, c=c)
    dense = orc.pair_bias_attention(a, P, w, H, c)
    sparse = spo.sparse_atom_attention(a, p_slice, idx, w, H, c)
    assert np.max(np.abs(dense - sparse)) <= 1e-12 * max(1.0, np.max(np.abs(dense)))


def test_sparse_brute_force():
    from oracle import sparse_atom_attention as spo
    rng = np.random.default_rng(42)
    L, k, H, c = 7, 3, 2, 3
    a, P, p_slice, idx, w = _sparse_problem(rng, L, k, c_s=5, c_p=4, H=H, c=c)
    idx[2, 1] = -1                      # an unused slot
    idx[4, :] = -1                      # an atom without neighbours: out = 0
    idx[5, 2] = idx[5, 0]               # a neighbour listed twice counts twice
    p_slice[5, 2] = p_slice[5, 0]
    tl = lambda x: np.asarray(x).tolist()
    ref = brute.brute_force_sparse(tl(a), tl(p_slice), tl(idx), tl(w["w_q"]), tl(w["w_k"]), tl(w["w_v"]), tl(w["w_g"]),
                                   tl(w["w_b"]), tl(w["w_o"]), tl(w["ln_z_gamma"]), tl(w["ln_z_beta"]), H, c)
    got = spo.sparse_atom_attention(a, p_slice, idx, w, H, c)
    assert np.max(np.abs(got - np.asarray(ref))) <= 1e-12
    assert np.all(got[4] == 0.0)


def test_sparse_slot_permutation_and_masking():
    from oracle import sparse_atom_attention as spo
    rng = np.random.default_rng(43)
    L, k, H, c = 11, 5, 2, 4
    a, P, p_slice, idx, w = _sparse_problem(rng, L, k, H=H, c=c)
    base = spo.sparse_atom_attention(a, p_slice, idx, w, H, c)
    perm = rng.permutation(k)
    assert np.max(np.abs(spo.sparse_atom_attention(a, p_slice[:, perm], idx[:, perm], w, H, c) - base)) <= 1e-13
    # a masked slot == a shorter list (whatever the pair features stored in the masked slot)
    idx2, p2 = idx.copy(), p_slice.copy()
    idx2[:, 3] = -1
    p2[:, 3] = 1e6
    keep = [0, 1, 2, 4]
    short = spo.sparse_atom_attention(a, p_slice[:, keep], idx[:, keep], w, H, c)
    assert np.max(np.abs(spo.sparse_atom_attention(a, p2, idx2, w, H, c) - short)) <= 1e-13


def test_sparse_single_neighbour_closed_form():
    """k = 1: softmax over one slot is 1, so out_l = (sigmoid(a_l W_g) (.) a_m W_v) W_o with m = idx[l, 0]."""
    from oracle import sparse_atom_attention as spo
    rng = np.random.default_rng(44)
    L, H, c = 9, 2, 3
    a, P, p_slice, idx, w = _sparse_problem(rng, L, 1, H=H, c=c)
    got = spo.sparse_atom_attention(a, p_slice, idx, w, H, c)
    gate = 1.0 / (1.0 + np.exp(-(a @ w["w_g"])))
    ref = (gate * (a[idx[:, 0]] @ w["w_v"])) @ w["w_o"]
    assert np.max(np.abs(got - ref)) <= 1e-12


# ---------------------------------------------------------------- k nearest neighbours
def test_knn_integer_lattice_closed_form():
    """Points on the integer line 0..n-1 (exact binary32 distances): the neighbours of l are l, then l-1 / l+1
    (the smaller index first on the tie), l-2 / l+2, ..."""
    from oracle import knn as ko
    n, k = 23, 7
    x = np.zeros((n, 3), dtype=np.float32)
    x[:, 1] = np.arange(n)
    got = ko.knn(x, k)
    for l in range(n):
        cand = sorted(range(n), key=lambda m: (abs(m - l), m))[:k]
        assert got[l].tolist() == cand


def test_knn_brute_force_binary32():
    """Pure-Python brute force with every operation rounded to binary32 through struct (independent of numpy)."""
    import struct
    from oracle import knn as ko
    f32 = lambda v: struct.unpack("f", struct.pack("f", v))[0]
    rng = np.random.default_rng(51)
    L, k = 40, 9
    x = (rng.normal(size=(L, 3)) * 7).astype(np.float32)
    x[7] = x[3]                                    # an exact duplicate point: tie broken by index
    got = ko.knn(x, k)
    xs = [[float(v) for v in row] for row in x]
    for l in range(L):
        d = []
        for m in range(L):
            t = [f32(xs[m][a] - xs[l][a]) for a in range(3)]
            s = [f32(t[a] * t[a]) for a in range(3)]
            d.append((f32(f32(s[0] + s[1]) + s[2]), m))
        assert got[l].tolist() == [m for _, m in sorted(d)[:k]]


def test_knn_matches_kdtree_and_is_translation_invariant():
    from scipy.spatial import cKDTree
    from oracle import knn as ko
    rng = np.random.default_rng(52)
    L, k = 300, 16
    x = rng.uniform(-20, 20, size=(L, 3)).astype(np.float32)
    got = ko.knn(x, k)
    _, ref = cKDTree(x.astype(np.float64)).query(x.astype(np.float64), k=k)
    for l in range(L):                             # fp64 vs binary32 can only differ on near-ties: compare as sets
        assert len(set(got[l].tolist()) ^ set(ref[l].tolist())) <= 2
    assert np.array_equal(got[:, 0], np.arange(L))                 # the query itself comes first (d2 = 0)
    xi = np.round(x * 8) / 8                        # multiples of 1/8: a shift by 64 is exact in binary32
    assert np.array_equal(ko.knn(xi, k), ko.knn((xi + np.float32(64.0)).astype(np.float32), k))
    assert np.array_equal(ko.knn(x, 1)[:, 0], np.arange(L))


# ---------------------------------------------------------------- pairwise SwiGLU transition (Eq. 6, Alg. 1)
def _transition_problem(rng, n_pairs=37, c_z=12):
    z = rng.normal(size=(n_pairs, c_z)) * 1.5 + 0.3
    w1 = rng.normal(size=(c_z, 4 * c_z)) / math.sqrt(c_z)
    w2 = rng.normal(size=(c_z, 4 * c_z)) / math.sqrt(c_z)
    w3 = rng.normal(size=(4 * c_z, c_z)) / math.sqrt(4 * c_z)
    gamma, beta = 1 + 0.1 * rng.normal(size=c_z), 0.1 * rng.normal(size=c_z)
    return z, w1, w2, w3, gamma, beta


def test_transition_matches_torch_composition():
    from oracle import pair_transition as pto
    z, w1, w2, w3, gamma, beta = _transition_problem(np.random.default_rng(61))
    tz = torch.from_numpy(z)
    n = torch.nn.functional.layer_norm(tz, (z.shape[-1],), torch.from_numpy(gamma), torch.from_numpy(beta), 1e-5)
    ref = tz + (torch.nn.functional.silu(n @ torch.from_numpy(w1)) * (n @ torch.from_numpy(w2))) @ torch.from_numpy(w3)
    assert np.max(np.abs(pto.pair_transition(z, w1, w2, w3, gamma, beta) - ref.numpy())) <= 1e-12


def test_transition_brute_force():
    from oracle import pair_transition as pto
    z, w1, w2, w3, gamma, beta = _transition_problem(np.random.default_rng(62), n_pairs=5, c_z=3)
    got = pto.pair_transition(z, w1, w2, w3, gamma, beta)
    c = z.shape[1]
    for p in range(z.shape[0]):
        row = [float(v) for v in z[p]]
        mu = sum(row) / c
        var = sum((v - mu) ** 2 for v in row) / c
        n = [(row[t] - mu) / math.sqrt(var + 1e-5) * gamma[t] + beta[t] for t in range(c)]
        h = []
        for j in range(4 * c):
            a = sum(n[t] * w1[t][j] for t in range(c))
            b = sum(n[t] * w2[t][j] for t in range(c))
            h.append(a / (1.0 + math.exp(-a)) * b)
        for t in range(c):
            assert abs(got[p][t] - (row[t] + sum(h[j] * w3[j][t] for j in range(4 * c)))) <= 1e-12


def test_transition_special_cases():
    from oracle import pair_transition as pto
    rng = np.random.default_rng(63)
    z, w1, w2, w3, gamma, beta = _transition_problem(rng)
    assert np.array_equal(pto.pair_transition(z, w1, w2, 0 * w3, gamma, beta), z)          # W_3 = 0: the residual only
    assert np.max(np.abs(pto.pair_transition(z, 0 * w1, w2, w3, gamma, beta) - z)) <= 1e-15  # SiLU(0) = 0
    t1 = pto.pair_transition(z, w1, w2, w3, gamma, beta) - z
    t2 = pto.pair_transition(z, w1, w2, 2.5 * w3, gamma, beta) - z
    assert np.max(np.abs(t2 - 2.5 * t1)) <= 1e-12                                            # linear in W_3
    perm = rng.permutation(z.shape[0])                                                       # pairs are independent
    assert np.max(np.abs(pto.pair_transition(z[perm], w1, w2, w3, gamma, beta)
                         - pto.pair_transition(z, w1, w2, w3, gamma, beta)[perm])) <= 1e-13
    # LayerNorm invariance: a per-pair affine rescale of z changes only the residual term (up to the eps term)
    zs = 3.0 * z + 7.0
    t3 = pto.pair_transition(zs, w1, w2, w3, gamma, beta, eps=0.0) - zs
    assert np.max(np.abs(t3 - (pto.pair_transition(z, w1, w2, w3, gamma, beta, eps=0.0) - z))) <= 1e-11


# ---------------------------------------------------------------- Pairformer stack (oracle/pairformer_stack.py)
def _stack_problem(rng, I=5, c_s=6, c_z=4, H=2, c=3, n_blocks=2):
    s, z, _ = rand_problem(rng, I, c_s, c_z, H, c)
    blocks = []
    for _ in range(n_blocks):
        _, _, w = rand_problem(rng, I, c_s, c_z, H, c)
        _, w1, w2, w3, gamma, beta = _transition_problem(rng, n_pairs=1, c_z=c_z)
        blocks.append((w, {"w1": w1, "w2": w2, "w3": 3.0 * w3, "gamma": gamma, "beta": beta}))   # a transition that moves z a lot
    return s, z, blocks


def _brute_attention(s, z, w, H, c):
    tl = lambda x: np.asarray(x).tolist()
    return np.array(brute.brute_force(tl(s), tl(z), tl(w["w_q"]), tl(w["w_k"]), tl(w["w_v"]), tl(w["w_g"]), tl(w["w_b"]),
                                      tl(w["w_o"]), tl(w["ln_z_gamma"]), tl(w["ln_z_beta"]), H, c))


def test_stack_identity_when_output_weights_vanish():
    from oracle import pairformer_stack as pso
    s, z, blocks = _stack_problem(np.random.default_rng(71), n_blocks=3)
    for w, t in blocks:
        w["w_o"] = np.zeros_like(w["w_o"])
        t["w3"] = np.zeros_like(t["w3"])
    s3, z3 = pso.pairformer_stack(s, z, blocks, 2, 3)
    assert np.array_equal(s3, s) and np.array_equal(z3, z)


def test_stack_order_against_brute_force():
    """Attention of block b reads the Z that block b - 1 left (not the original, not the one its own transition writes)."""
    from oracle import pairformer_stack as pso
    H, c = 2, 3
    s, z, blocks = _stack_problem(np.random.default_rng(72), n_blocks=2)
    s1, z1 = pso.pairformer_stack(s, z, blocks[:1], H, c)
    s2, z2 = pso.pairformer_stack(s, z, blocks, H, c)
    t0, t1 = blocks[0][1], blocks[1][1]
    # the transition really moves z (otherwise the order pins below would be vacuous)
    assert np.max(np.abs(z1 - z)) > 0.5
    assert np.max(np.abs(s1 - (s + _brute_attention(s, z, blocks[0][0], H, c)))) <= 1e-12      # block 1: original z
    assert np.max(np.abs(s1 - (s + _brute_attention(s, z1, blocks[0][0], H, c)))) > 1e-3       # ... not the updated one
    assert np.max(np.abs(s2 - (s1 + _brute_attention(s1, z1, blocks[1][0], H, c)))) <= 1e-12   # block 2: (s1, z1)
    # the pair track: the transition applied block by block (torch composition as the independent routine)
    def tr(zz, t):
        tz = torch.from_numpy(zz)
        n = torch.nn.functional.layer_norm(tz, (zz.shape[-1],), torch.from_numpy(t["gamma"]), torch.from_numpy(t["beta"]), 1e-5)
        return (tz + (torch.nn.functional.silu(n @ torch.from_numpy(t["w1"])) * (n @ torch.from_numpy(t["w2"])))
                @ torch.from_numpy(t["w3"])).numpy()
    assert np.max(np.abs(z1 - tr(z, t0))) <= 1e-12
    assert np.max(np.abs(z2 - tr(tr(z, t0), t1))) <= 1e-11


def test_stack_round_store_is_applied_once_per_block():
    from oracle import pairformer_stack as pso
    H, c = 2, 3
    s, z, blocks = _stack_problem(np.random.default_rng(73), n_blocks=2)
    bf = lambda x: torch.from_numpy(np.asarray(x)).to(torch.bfloat16).double().numpy()
    s2, z2 = pso.pairformer_stack(bf(s), bf(z), blocks, H, c, round_store=bf)
    assert np.array_equal(bf(s2), s2) and np.array_equal(bf(z2), z2)
    s1, z1 = pso.pairformer_block(bf(s), bf(z), *blocks[0], H, c, round_store=bf)
    s2b, z2b = pso.pairformer_block(s1, z1, *blocks[1], H, c, round_store=bf)
    assert np.array_equal(s2, s2b) and np.array_equal(z2, z2b)


# ------------------------------------------------------------------ attention stack on a read-only pair tensor
def _attn_stack_problem(rng, I=5, c_s=6, c_z=4, H=2, c=3, n_blocks=3):
    s, z, _ = rand_problem(rng, I, c_s, c_z, H, c)
    return s, z, [rand_problem(rng, I, c_s, c_z, H, c)[2] for _ in range(n_blocks)]


def test_attention_stack_identity_and_single_block():
    from oracle import attention_stack as aso
    from oracle import pair_bias_attention as orc
    H, c = 2, 3
    a, z, blocks = _attn_stack_problem(np.random.default_rng(81))
    z0 = z.copy()
    one = aso.attention_stack(a, z, blocks[:1], H, c)
    assert np.array_equal(one, a + orc.pair_bias_attention(a, z, blocks[0], H, c))
    assert np.array_equal(z, z0)                                        # Z is read-only
    dead = [dict(w, w_o=np.zeros_like(w["w_o"])) for w in blocks]
    assert np.array_equal(aso.attention_stack(a, z, dead, H, c), a)     # W_o = 0: identity at any depth


def test_attention_stack_order_against_brute_force():
    """Block b reads the latent block b - 1 wrote, its OWN weights, and the original Z."""
    from oracle import attention_stack as aso
    H, c = 2, 3
    a, z, blocks = _attn_stack_problem(np.random.default_rng(82))
    a1 = aso.attention_stack(a, z, blocks[:1], H, c)
    a2 = aso.attention_stack(a, z, blocks[:2], H, c)
    a3 = aso.attention_stack(a, z, blocks, H, c)
    assert np.max(np.abs(a1 - (a + _brute_attention(a, z, blocks[0], H, c)))) <= 1e-12
    assert np.max(np.abs(a2 - (a1 + _brute_attention(a1, z, blocks[1], H, c)))) <= 1e-12
    assert np.max(np.abs(a3 - (a2 + _brute_attention(a2, z, blocks[2], H, c)))) <= 1e-12
    # the plausible mistakes move the result by far more than rounding
    assert np.max(np.abs(a2 - (a1 + _brute_attention(a, z, blocks[1], H, c)))) > 1e-3      # stale latent
    assert np.max(np.abs(a2 - (a1 + _brute_attention(a1, z, blocks[0], H, c)))) > 1e-3     # another block's weights
    assert np.max(np.abs(a2 - (a + _brute_attention(a1, z, blocks[1], H, c)))) > 1e-3      # residual onto the wrong latent


def test_attention_stack_round_store_once_per_block():
    from oracle import attention_stack as aso
    H, c = 2, 3
    a, z, blocks = _attn_stack_problem(np.random.default_rng(83))
    bf = lambda x: torch.from_numpy(np.asarray(x)).to(torch.bfloat16).double().numpy()
    a3 = aso.attention_stack(bf(a), bf(z), blocks, H, c, round_store=bf)
    assert np.array_equal(bf(a3), a3)
    step = bf(a)
    for w in blocks:
        step = aso.attention_stack(step, bf(z), [w], H, c, round_store=bf)
    assert np.array_equal(a3, step)
    assert np.max(np.abs(a3 - aso.attention_stack(bf(a), bf(z), blocks, H, c))) > 0          # the rounding is really there


# ------------------------------------------------------------------ structured neighbour budget
def _four_chain_lattice(n_per_chain=(60, 60, 60, 60), gap=100.0):
    """Chains = parallel lines of unit-spaced atoms along x, chain c at y = gap * c; residue = 4 consecutive atoms."""
    xs, rid, cid = [], [], []
    for ch, n in enumerate(n_per_chain):
        for a in range(n):
            xs.append((float(a), gap * ch, 0.0)); rid.append(a // 4); cid.append(ch)
    return np.array(xs, dtype=np.float32), np.array(rid), np.array(cid)


def test_knn_budget_reduces_to_plain_knn():
    from oracle import knn as ko
    from oracle import knn_budget as kb
    rng = np.random.default_rng(91)
    x = rng.normal(size=(70, 3)).astype(np.float32) * 3
    rid, cid = np.arange(70) // 5, np.arange(70) // 30          # three chains: no quota
    assert np.array_equal(kb.knn_budget(x, rid, cid, 16, n_seq=0), ko.knn(x, 16))
    assert np.array_equal(kb.knn_budget(x, rid, np.zeros(70, int), 70, n_seq=2), ko.knn(x, 70))   # k = L: everything


def test_knn_budget_quotas_bind_on_a_four_chain_lattice():
    from oracle import knn_budget as kb
    k = 48                                                       # q_out = max(32, 12) = 32, the own chain gets 16
    x, rid, cid = _four_chain_lattice()
    l = 30                                                       # middle of chain 0, residue 7 (atoms 28..31)
    row = kb.knn_budget_rows(x, rid, cid, k, [l], n_seq=2)[0]
    intra = [m for m in row if cid[m] == 0]
    inter = [m for m in row if cid[m] != 0]
    assert len(intra) == 16 and len(inter) == 32                 # both quotas bind (pure kNN would stay in chain 0)
    # intra: S = residues 6..8 = atoms 24..35 (12 atoms), then the closest others: 23, 36 (d = 7, 6) -> 36 first, 23, 37, 22
    assert sorted(intra) == [22, 23] + list(range(24, 36)) + [36, 37]
    # inter: chain 1 is the closest foreign chain (y = 100): its 32 atoms nearest x = 30, ties by the smaller index
    assert sorted(inter) == [60 + a for a in range(14, 46)]     # |a - 30| <= 15, and a = 14 (idx 74) wins the tie with 46
    assert row[0] == l and len(set(row.tolist())) == k
    d2 = ((x[row] - x[l]) ** 2).sum(1)
    assert np.all(np.diff(d2) >= 0)                              # output ordered by distance
    # three chains only: no split, the list is S + the closest atoms, all in chain 0
    keep = cid < 3
    row3 = kb.knn_budget_rows(x[keep], rid[keep], cid[keep], k, [l], n_seq=2)[0]
    assert all(cid[m] == 0 for m in row3) and sorted(row3.tolist()) == list(range(6, 54)) or sorted(row3.tolist()) == list(range(7, 55))


def test_knn_budget_short_chain_and_few_foreign_atoms():
    from oracle import knn_budget as kb
    k = 48
    x, rid, cid = _four_chain_lattice((10, 60, 60, 60))          # own chain has 10 < q_in atoms: the others fill
    row = kb.knn_budget_rows(x, rid, cid, k, [3], n_seq=2)[0]
    assert sum(cid[m] == 0 for m in row) == 10 and sum(cid[m] != 0 for m in row) == 38
    x, rid, cid = _four_chain_lattice((60, 5, 5, 5))             # 15 foreign atoms < q_out: the own chain fills
    row = kb.knn_budget_rows(x, rid, cid, k, [30], n_seq=2)[0]
    assert sum(cid[m] != 0 for m in row) == 15 and sum(cid[m] == 0 for m in row) == 33
    x, rid, cid = _four_chain_lattice((20, 4, 4, 4))             # k = L
    assert sorted(kb.knn_budget_rows(x, rid, cid, 32, [0], n_seq=2)[0].tolist()) == list(range(32))


def test_knn_budget_sequence_local_atoms_come_first():
    from oracle import knn_budget as kb
    rng = np.random.default_rng(92)
    L, k = 80, 8
    x = rng.normal(size=(L, 3)).astype(np.float32)
    rid, cid = np.arange(L) // 4, np.zeros(L, int)
    x[36:40] += 1000.0                                           # residue 9, flanking residue 8 of atom 33, moved far away
    row2 = kb.knn_budget_rows(x, rid, cid, k, [33], n_seq=2)[0]
    assert set(range(28, 40)) >= set(row2.tolist()) and len(row2) == k     # S = residues 7..9 = 12 atoms >= k: its 8 closest
    row1 = kb.knn_budget_rows(x, rid, cid, 16, [33], n_seq=2)[0]
    assert set(range(28, 40)) <= set(row1.tolist())              # all of S, the far residue included, + 4 spatial ones
    row0 = kb.knn_budget_rows(x, rid, cid, 16, [33], n_seq=1)[0]
    assert set(range(32, 36)) <= set(row0.tolist()) and not (set(range(36, 40)) & set(row0.tolist()))
    cid2 = cid.copy(); cid2[36:40] = 1                           # the flanking residue belongs to another chain: not local
    assert not (set(range(36, 40)) & set(kb.knn_budget_rows(x, rid, cid2, 16, [33], n_seq=2)[0].tolist()))


def test_knn_budget_brute_force_binary32():
    """A second implementation: struct-rounded binary32 distances, selection by repeated extraction of the minimum."""
    import struct
    from oracle import knn_budget as kb
    f32 = lambda v: struct.unpack("f", struct.pack("f", v))[0]
    rng = np.random.default_rng(93)
    for L, k, n_chains, n_seq in ((90, 40, 5, 2), (64, 36, 4, 1), (50, 12, 2, 2), (77, 33, 6, 0)):
        x = (rng.integers(-6, 7, size=(L, 3)) * 0.37).astype(np.float32)      # many exact ties
        cid = np.sort(rng.integers(0, n_chains, size=L)); rid = np.arange(L) // 3
        got = kb.knn_budget(x, rid, cid, k, n_seq=n_seq)
        split = len(set(cid.tolist())) > 3
        q_out = min(max(32, k // 4), k - 1)
        for l in range(L):
            d2 = []
            for m in range(L):
                t = [f32(float(x[m, a]) - float(x[l, a])) for a in range(3)]
                d2.append(f32(f32(f32(t[0] * t[0]) + f32(t[1] * t[1])) + f32(t[2] * t[2])))
            pool = set(range(L))
            def take(pred, n):
                got_ = []
                while len(got_) < n:
                    cand = [m for m in pool if pred(m)]
                    if not cand:
                        break
                    b = min(cand, key=lambda m: (d2[m], m)); pool.discard(b); got_.append(b)
                return got_
            local = lambda m: n_seq >= 1 and cid[m] == cid[l] and abs(rid[m] - rid[l]) <= n_seq - 1
            if not split:
                sel = take(local, k)
                sel += take(lambda m: True, k - len(sel))
            else:
                out_ = take(lambda m: cid[m] != cid[l], q_out)         # the foreign quota is served first ...
                sel = take(local, k - len(out_))                       # ... then the own chain, sequence-local atoms first
                sel += take(lambda m: cid[m] == cid[l], k - len(out_) - len(sel))
                sel += out_
                sel += take(lambda m: True, k - len(sel))              # a small own chain: the others fill
            want = sorted(sel, key=lambda m: (d2[m], m))
            assert got[l].tolist() == want, (L, k, l)


def test_knn_budget_invariances():
    from oracle import knn_budget as kb
    rng = np.random.default_rng(94)
    L, k = 120, 40
    x = rng.normal(size=(L, 3)).astype(np.float32) * 4
    rid, cid = np.arange(L) // 6, np.arange(L) // 24             # five chains
    base = kb.knn_budget(x, rid, cid, k)
    assert np.array_equal(kb.knn_budget(x, rid, (cid * 7 + 3) % 11, k), base)          # chain labels are only labels
    assert np.array_equal(kb.knn_budget(x, rid + 1000, cid, k), base)                  # so are residue offsets
    xi = np.round(x * 8) / 8                                                           # exactly representable grid
    assert np.array_equal(kb.knn_budget(xi + np.float32(16.0), rid, cid, k), kb.knn_budget(xi, rid, cid, k))
    for l in range(L):
        assert base[l, 0] == l and len(set(base[l].tolist())) == k
        assert sum(cid[m] != cid[l] for m in base[l]) >= 32                            # PAPER.md:303 "at least 32"
