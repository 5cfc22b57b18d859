"""GPU parity of the sparse k-neighbour atom attention against the fp64
oracle, through the C ABI.  bf16 tolerances of BASELINE.json (rel-L2 <= 1e-2, max-abs <= 2e-2)."""
import numpy as np
import pytest
import torch

import dcp_synth as syn
from oracle import sparse_atom_attention as spo
from tests import util

pytestmark = pytest.mark.gpu
DEV = "cuda:0"


def _dcp():
    import paper_2607_05439_b200 as dcp
    return dcp


def _problem(L, k, H=4, c_atom=128, seed=11, structured=False, copies=60, ln_s=False, b_q=False):
    cfg = syn.small_config("sp", I=L, c_s=c_atom, c_z=16, H=H, c=32, dtype="bf16", seed=seed, structured=structured,
                           copies=copies)
    w = syn.make_weights(cfg, DEV, with_ln_s=ln_s, with_b_q=b_q)
    a = syn.make_s(cfg, DEV)
    idx = util.neighbour_lists(cfg, k, DEV)
    p = syn.make_p_slice(cfg, idx, DEV)
    return cfg, a, p, idx, w


def _oracle(cfg, a, p, idx, w, rows=None):
    rows = list(range(cfg.I)) if rows is None else list(rows)
    r = torch.as_tensor(rows, device=a.device)
    return spo.sparse_atom_attention_rows(util.np64(a), util.np32(p.index_select(0, r)),
                                          idx.index_select(0, r).cpu().numpy(), rows, util.weights_np(w), cfg.H, cfg.c)


@pytest.mark.parametrize("L,k,H,c_atom,ln_s,b_q", [
    (300, 128, 4, 128, False, False),   # the paper's default budget k = 128
    (77, 33, 4, 64, True, True),        # ragged k (two passes, partial second), optional LN_s + b_q, mma.sync GEMM fallback
    (40, 40, 2, 128, False, False),     # k = L: every atom attends to all atoms
    (129, 1, 3, 72, False, False),      # single neighbour, odd head count, c_atom not a multiple of 64
    (600, 512, 4, 128, False, False),   # the largest supported budget
    (200, 64, 8, 128, False, False),    # H = 8: one 512-byte row per warp-level load
    (90, 48, 16, 64, False, False),     # H = 16: slot-per-lane kernel
])
def test_sparse_small_shapes(L, k, H, c_atom, ln_s, b_q):
    dcp = _dcp()
    cfg, a, p, idx, w = _problem(L, k, H=H, c_atom=c_atom, seed=100 + L, ln_s=ln_s, b_q=b_q)
    out = dcp.dcp_sparse_atom_attention(a, p, idx, w, cfg.H, cfg.c)
    util.check_close(out, _oracle(cfg, a, p, idx, w), "bf16", f"sparse L={L} k={k}")
    again = dcp.dcp_sparse_atom_attention(a, p, idx, w, cfg.H, cfg.c)
    assert torch.equal(out, again)      # run-to-run bitwise repeatable (no atomics)


def test_sparse_masked_slots_and_empty_rows():
    dcp = _dcp()
    cfg, a, p, idx, w = _problem(96, 64, seed=7)
    g = torch.Generator(device="cpu").manual_seed(5)
    mask = (torch.rand(idx.shape, generator=g) < 0.3).to(DEV)
    idx = torch.where(mask, torch.full_like(idx, -1), idx)
    idx[5] = -1                                            # an atom without valid neighbours: out = 0
    p = torch.where(mask[..., None], torch.full_like(p, 300.0), p)   # whatever sits in a masked slot is ignored
    out = dcp.dcp_sparse_atom_attention(a, p, idx.contiguous(), w, cfg.H, cfg.c)
    util.check_close(out, _oracle(cfg, a, p, idx, w), "bf16", "sparse masked")
    assert torch.all(out[5] == 0)


def test_sparse_out_of_range_indices_are_unused_slots():
    """An index >= L is treated like a negative one (include/designcp.h): same output as with -1 there, for both
    kernels (rows kernel H = 4, slot-per-lane kernel H = 16) and for the gather."""
    dcp = _dcp()
    for H in (4, 16):
        cfg, a, p, idx, w = _problem(80, 48, H=H, seed=23)
        g = torch.Generator(device="cpu").manual_seed(6)
        mask = (torch.rand(idx.shape, generator=g) < 0.25).to(DEV)
        big = torch.where(mask, torch.full_like(idx, cfg.I + 1000), idx).contiguous()
        big[3, 0] = 2 ** 31 - 1
        neg = torch.where(big >= cfg.I, torch.full_like(idx, -1), big).contiguous()
        assert torch.equal(dcp.dcp_sparse_atom_attention(a, p, big, w, cfg.H, cfg.c),
                           dcp.dcp_sparse_atom_attention(a, p, neg, w, cfg.H, cfg.c))
    P = syn.make_z(cfg, DEV)
    assert torch.equal(dcp.dcp_gather_pair_slice(P, big), dcp.dcp_gather_pair_slice(P, neg))
    from paper_2607_05439_b200 import binding
    st = binding.raw().dcp_gather_pair_slice(P.data_ptr(), 0, big.data_ptr(), p.data_ptr(), cfg.I, big.shape[1], 16, 7, None)
    assert st == 1                                         # unknown dtype code


def test_sparse_full_budget_matches_dense_layer():
    """k = L with every atom listed once: the sparse kernel and the dense atom-level kernel compute the same layer."""
    dcp = _dcp()
    L = 160
    cfg = syn.small_config("spd", I=L, c_s=128, c_z=16, H=4, c=32, dtype="bf16", seed=9)
    w = syn.make_weights(cfg, DEV)
    a = syn.make_s(cfg, DEV)
    P = syn.make_z(cfg, DEV)
    g = torch.Generator(device="cpu").manual_seed(3)
    idx = torch.stack([torch.randperm(L, generator=g) for _ in range(L)]).to(torch.int32).to(DEV)
    p_slice = torch.gather(P, 1, idx.long()[..., None].expand(-1, -1, cfg.c_z)).contiguous()
    sparse = dcp.dcp_sparse_atom_attention(a, p_slice, idx, w, cfg.H, cfg.c)
    dense = dcp.dcp_atom_pair_bias_attention(a, P, w, cfg.H, cfg.c)
    ref = util.oracle_rows(cfg, a, P, w, range(L))
    util.check_close(sparse, ref, "bf16", "sparse, full budget")
    util.check_close(dense, ref, "bf16", "dense")


def test_gather_pair_slice_and_full_chain():
    """coordinates -> dcp_knn -> dcp_gather_pair_slice (dense P) -> dcp_sparse_atom_attention, against the oracles:
    the gather is byte work (bit-exact against torch.gather), the chain is checked against the sparse oracle."""
    dcp = _dcp()
    cfg = syn.small_config("chain", I=480, c_s=128, c_z=16, H=4, c=32, dtype="bf16", seed=13, structured=True, copies=60)
    w = syn.make_weights(cfg, DEV)
    a = syn.make_s(cfg, DEV)
    P = syn.make_z(cfg, DEV)
    x = syn.make_atom_coords(cfg, DEV)
    idx = dcp.dcp_knn(x, 64)
    idx[3, 10:] = -1                                        # a partly filled budget
    p_slice = dcp.dcp_gather_pair_slice(P, idx)
    ref_slice = torch.gather(P, 1, idx.long().clamp(min=0)[..., None].expand(-1, -1, cfg.c_z))
    ref_slice = torch.where((idx < 0)[..., None], torch.zeros_like(ref_slice), ref_slice)
    assert torch.equal(p_slice, ref_slice)
    out = dcp.dcp_sparse_atom_attention(a, p_slice, idx, w, cfg.H, cfg.c)
    util.check_close(out, _oracle(cfg, a, p_slice, idx, w), "bf16", "knn -> gather -> sparse attention")
    pf = dcp.dcp_gather_pair_slice(P.float(), idx)          # fp32 rows (64 bytes) gather too
    assert torch.equal(pf, ref_slice.float())


def test_sparse_c4_sampled_rows():
    """C4's atoms (L = 24000, c_atom 128, H 4, c 32) with the paper's budget k = 128: sampled rows vs the oracle."""
    dcp = _dcp()
    cfg = syn.CONFIGS["C4"]
    w = syn.make_weights(cfg, DEV)
    a = syn.make_s(cfg, DEV)
    idx = util.neighbour_lists(cfg, 128, DEV)
    p = syn.make_p_slice(cfg, idx, DEV)
    out = dcp.dcp_sparse_atom_attention(a, p, idx, w, cfg.H, cfg.c)
    rows = syn.sample_rows(cfg.I, 200, boundaries=[400, 12000], seed=1)
    util.check_close(out.index_select(0, torch.as_tensor(rows, device=DEV)), _oracle(cfg, a, p, idx, w, rows), "bf16",
                     "sparse C4 sampled")
    assert torch.isfinite(out.float()).all()


def test_sparse_error_paths():
    dcp = _dcp()
    cfg, a, p, idx, w = _problem(64, 32, seed=2)
    with pytest.raises(dcp.DcpError) as e:      # fp32 storage is not instantiated
        dcp.dcp_sparse_atom_attention(a.float(), p.float(), idx, {k: v.float() for k, v in w.items()}, cfg.H, cfg.c)
    assert e.value.status == 2
    with pytest.raises(dcp.DcpError) as e:      # head dim other than 32
        dcp.dcp_sparse_atom_attention(a, p, idx, w, 8, 16)
    assert e.value.status == 2
    ws = torch.empty(256, dtype=torch.uint8, device=DEV)
    with pytest.raises(dcp.DcpError) as e:      # workspace too small
        dcp.dcp_sparse_atom_attention(a, p, idx, w, cfg.H, cfg.c, workspace=ws)
    assert e.value.status == 3
