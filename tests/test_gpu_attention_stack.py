"""GPU parity of the attention stack on a read-only pair tensor (the diffusion
transformer's eighteen sequential AttentionPairBias blocks over the c_token = 768 latent) through the C ABI against
oracle/attention_stack.py.  The device keeps the latent in bf16 and rounds it once per block; the oracle is given that
rounding (`round_store`).  Per block, started from the oracle's own (bf16-exact) latent: BASELINE.json's bf16 bounds on the
block's update (max-abs <= 2e-2, times the update's RMS where that exceeds 1: the bound is stated for O(1) outputs and
deep blocks of a growing latent produce larger ones) plus one bf16 ulp of the stored latent (2^-7 |ref|: both sides round
their sum to bf16 and may land on neighbouring values); the update itself, seen through that storage, within 2e-2 rel-L2.  The whole chain: the per-block errors add, n_blocks x the bounds
on the norms."""
import numpy as np
import pytest
import torch

import dcp_synth as syn
from oracle import attention_stack as aso
from oracle import pair_bias_attention as orc
from tests import util

pytestmark = pytest.mark.gpu
DEV = "cuda:0"


def _dcp():
    import paper_2607_05439_b200 as dcp
    return dcp


def _bf(x):
    return torch.from_numpy(np.asarray(x)).to(torch.bfloat16).double().numpy()


def _blocks(cfg, n, with_ln_s=False):
    return [syn.make_weights(syn.small_config("blk", I=cfg.I, c_s=cfg.c_s, c_z=cfg.c_z, H=cfg.H, c=cfg.c, dtype="bf16",
                                              seed=cfg.seed + 101 * (b + 1)), DEV,
                             with_ln_s=with_ln_s == "all" or (with_ln_s == "odd" and b % 2 == 1))
            for b in range(n)]


@pytest.mark.parametrize("I,copies,c_s,c,n_blocks,ln_s", [
    (96, 12, 768, 48, 1, False),     # c_token = 768 = H * c: the diffusion transformer's widths
    (75, 15, 768, 48, 3, "odd"),     # ragged I, every other block with a LayerNorm on the latent
    (60, 60, 768, 48, 18, "all"),    # the paper's depth; every block normalises the latent it reads (the paper's blocks
                                     # all have a layer-norm path) -- without it a residual stream of 18
                                     # random-weight blocks grows until the softmax is one-hot and ill-conditioned
    (131, 1, 384, 24, 4, False),     # another instantiated head size, c_s != 768
])
def test_attention_stack_matches_oracle(I, copies, c_s, c, n_blocks, ln_s):
    dcp = _dcp()
    cfg = syn.small_config("astack", I=I, c_s=c_s, c_z=128, H=16, c=c, dtype="bf16", seed=7 + I, structured=copies > 1,
                           copies=copies)
    a0, z = syn.make_s(cfg, DEV), syn.make_z(cfg, DEV)
    z_before = z.clone()
    blocks = _blocks(cfg, n_blocks, ln_s)
    ob = [util.weights_np(w) for w in blocks]
    zn = util.np64(z)
    # ---- every block on its own, from the oracle's latent entering it
    a_ref = util.np64(a0)
    for b in range(n_blocks):
        a_in = a_ref
        a_ref = aso.attention_stack(a_in, zn, ob[b:b + 1], cfg.H, cfg.c, round_store=_bf)
        a1 = torch.from_numpy(a_in).to(torch.bfloat16).to(DEV)
        dcp.dcp_attention_stack(a1, z, blocks[b:b + 1], cfg.H, cfg.c)
        got = util.np64(a1)
        upd_ref = a_ref - a_in
        rel = np.linalg.norm((got - a_in) - upd_ref) / np.linalg.norm(upd_ref)
        assert rel <= 2e-2, f"block {b}: update rel-L2 {rel:.3e}"          # the update as seen through bf16 storage of a + update
        rms = max(1.0, float(np.sqrt(np.mean(upd_ref ** 2))))             # BASELINE's max-abs is stated for O(1) outputs
        bad = np.abs(got - a_ref) > util.TOL_BF16_MAXABS * rms + 2.0 ** -7 * np.abs(a_ref)
        assert not bad.any(), (f"block {b}: {bad.sum()} elements out of tolerance, max-abs {np.abs(got - a_ref).max():.3e}, "
                               f"update rms {rms:.2f}")
    # ---- the chain in one call
    a = a0.clone()
    dcp.dcp_attention_stack(a, z, blocks, cfg.H, cfg.c)
    torch.cuda.synchronize()
    assert torch.equal(z, z_before), "the pair tensor is read-only"
    got = util.np64(a)
    assert np.all(np.isfinite(got))
    rel = np.linalg.norm(got - a_ref) / np.linalg.norm(a_ref)
    assert rel <= n_blocks * util.TOL_BF16_RELL2, f"chain: rel-L2 {rel:.3e}"
    upd, upd_ref = got - util.np64(a0), a_ref - util.np64(a0)
    assert np.linalg.norm(upd - upd_ref) / np.linalg.norm(upd_ref) <= max(5e-2, n_blocks * util.TOL_BF16_RELL2)
    # ---- repeatable bit for bit; block by block == one call
    a2 = a0.clone()
    for w in blocks:
        dcp.dcp_attention_stack(a2, z, [w], cfg.H, cfg.c)
    assert torch.equal(a2, a)


def test_attention_stack_one_block_is_the_layer_plus_residual():
    """One block against the layer call: the stack adds the residual in fp32 before the single rounding, the layer call
    returns the rounded output -- they agree to one rounding of the layer output."""
    dcp = _dcp()
    cfg = syn.small_config("astack1", I=120, c_s=768, c_z=128, H=16, c=48, dtype="bf16", seed=3, structured=True, copies=60)
    a0, z = syn.make_s(cfg, DEV), syn.make_z(cfg, DEV)
    (w,) = _blocks(cfg, 1)
    o = dcp.dcp_pair_bias_attention(a0, z, w, cfg.H, cfg.c)
    a = a0.clone()
    dcp.dcp_attention_stack(a, z, [w], cfg.H, cfg.c)
    two_step = (a0.float() + o.float())
    assert float((a.float() - two_step).abs().max()) <= 2.0 ** -7 * float(two_step.abs().max()) + 2.0 ** -8 * float(o.abs().max())


def test_attention_stack_full_size_block_sampled():
    """At C2's size with the diffusion transformer's width (I = 3000, c_token = 768: the shape bench.py --workload D2
    times): three blocks on the device; block 3 is checked on sampled rows against the oracle started from the device's
    own latent after two blocks (a row of block 3 needs that whole latent for K / V, and z[i, :, :])."""
    dcp = _dcp()
    cfg = syn.small_config("D2", I=3000, c_s=768, c_z=128, H=16, c=48, dtype="bf16", seed=2, structured=True, copies=60)
    a0, z = syn.make_s(cfg, DEV), syn.make_z(cfg, DEV)
    blocks = _blocks(cfg, 3)
    a2 = a0.clone()
    dcp.dcp_attention_stack(a2, z, blocks[:2], cfg.H, cfg.c)
    a3 = a2.clone()
    dcp.dcp_attention_stack(a3, z, blocks[2:], cfg.H, cfg.c)
    full = a0.clone()
    dcp.dcp_attention_stack(full, z, blocks, cfg.H, cfg.c)
    assert torch.equal(full, a3)
    rows = syn.sample_rows(cfg.I, 32, boundaries=(32, 1000, 2976), seed=5)
    idx = torch.as_tensor(rows, device=DEV)
    upd_ref = orc.pair_bias_attention_rows(util.np64(a2), util.np32(z.index_select(0, idx)), rows, util.weights_np(blocks[2]),
                                           cfg.H, cfg.c)
    a2r = util.np64(a2.index_select(0, idx))
    ref = _bf(a2r + upd_ref)
    got = util.np64(a3.index_select(0, idx))
    rel = np.linalg.norm((got - a2r) - upd_ref) / np.linalg.norm(upd_ref)
    assert rel <= 2e-2, f"update rel-L2 {rel:.3e}"
    assert np.all(np.abs(got - ref) <= util.TOL_BF16_MAXABS + 2.0 ** -7 * np.abs(ref)), np.abs(got - ref).max()
    del z
    torch.cuda.empty_cache()


def test_attention_stack_error_paths():
    dcp = _dcp()
    cfg = syn.small_config("aserr", I=64, c_s=768, c_z=128, H=16, c=48, dtype="bf16", seed=5)
    a, z = syn.make_s(cfg, DEV), syn.make_z(cfg, DEV)
    blocks = _blocks(cfg, 1)
    with pytest.raises(dcp.DcpError) as e:
        dcp.dcp_attention_stack(a, z, blocks, cfg.H, cfg.c, workspace=torch.empty(256, dtype=torch.uint8, device=DEV))
    assert e.value.status == 3
    with pytest.raises(dcp.DcpError):
        dcp.dcp_attention_stack(a, z, [], cfg.H, cfg.c)
    cfg32 = syn.CONFIGS["C0"]
    s32, z32, w32 = util.make_problem(cfg32, DEV)
    with pytest.raises(dcp.DcpError) as e:                 # fp32 has no tensor-core kernel: the stack is bf16 only
        dcp.dcp_attention_stack(s32, z32, [w32], cfg32.H, cfg32.c)
    assert e.value.status == 2
    out = dcp.dcp_attention_stack(a, z, blocks, cfg.H, cfg.c)
    assert torch.isfinite(out.float()).all()


# ------------------------------------------------------------------ the same stack with a bias cache
@pytest.mark.parametrize("I,copies,c,n_blocks", [
    (96, 12, 48, 1),
    (75, 15, 48, 3),       # ragged I: the last query / key tiles of the cache are partly out of range
    (131, 1, 24, 4),
    (60, 60, 48, 18),      # the paper's depth in ONE pass: 304 projection columns, split into a single-buffered Y part
                           # (ones + 6 blocks) and a double-buffered X part (12 blocks) of tensor memory
    (40, 1, 48, 16),       # the smallest split: Y = ones + 4 blocks, X = 12 blocks
    (48, 12, 48, 23),      # the widest pass: Y = 256 columns (ones + 15 blocks), X = 128 (8 blocks)
    (36, 12, 48, 25),      # two passes over z (23 + 2 blocks)
    (300, 60, 32, 16),
])
def test_attention_stack_cached_matches_oracle_and_streaming(I, copies, c, n_blocks):
    """One pass over z writes every block's bias tiles (fp16), the blocks then read those: per block from the oracle's
    latent at the same bounds as the streaming stack, and the chain close to the streaming call (they differ by the
    fp16 rounding of the bias only)."""
    dcp = _dcp()
    c_s = 768 if c == 48 else 384
    cfg = syn.small_config("cstack", I=I, c_s=c_s, c_z=128, H=16, c=c, dtype="bf16", seed=31 + I, structured=copies > 1,
                           copies=copies)
    a0, z = syn.make_s(cfg, DEV), syn.make_z(cfg, DEV)
    z_before = z.clone()
    blocks = _blocks(cfg, n_blocks, "all")
    ob = [util.weights_np(w) for w in blocks]
    zn = util.np64(z)
    a_ref = util.np64(a0)
    for b in range(n_blocks):
        a_in = a_ref
        a_ref = aso.attention_stack(a_in, zn, ob[b:b + 1], cfg.H, cfg.c, round_store=_bf)
        a1 = torch.from_numpy(a_in).to(torch.bfloat16).to(DEV)
        dcp.dcp_attention_stack_cached(a1, z, blocks[b:b + 1], cfg.H, cfg.c)
        got = util.np64(a1)
        upd_ref = a_ref - a_in
        rel = np.linalg.norm((got - a_in) - upd_ref) / np.linalg.norm(upd_ref)
        assert rel <= 2e-2, f"block {b}: update rel-L2 {rel:.3e}"
        rms = max(1.0, float(np.sqrt(np.mean(upd_ref ** 2))))
        bad = np.abs(got - a_ref) > util.TOL_BF16_MAXABS * rms + 2.0 ** -7 * np.abs(a_ref)
        assert not bad.any(), f"block {b}: {bad.sum()} elements out of tolerance, max-abs {np.abs(got - a_ref).max():.3e}"
    a_c, a_s = a0.clone(), a0.clone()
    dcp.dcp_attention_stack_cached(a_c, z, blocks, cfg.H, cfg.c)
    dcp.dcp_attention_stack(a_s, z, blocks, cfg.H, cfg.c)
    torch.cuda.synchronize()
    assert torch.equal(z, z_before)
    gc, gs = util.np64(a_c), util.np64(a_s)
    assert np.all(np.isfinite(gc))
    assert np.linalg.norm(gc - a_ref) / np.linalg.norm(a_ref) <= n_blocks * util.TOL_BF16_RELL2
    assert np.linalg.norm(gc - gs) / np.linalg.norm(gs) <= n_blocks * 2e-3, "cached and streaming stacks drift apart"
    again = a0.clone()
    dcp.dcp_attention_stack_cached(again, z, blocks, cfg.H, cfg.c)
    assert torch.equal(again, a_c)


def test_attention_stack_cached_full_size_block_sampled():
    """The configuration bench.py --workload D2 --cached times (I = 3000, c_token = 768: 94 x 188 cache tiles per block,
    282 work units with three key segments each): 17 blocks on the device, in one pass with split projection columns and,
    as 16 + 1 blocks, in two calls; block 17 checked on sampled rows against the oracle started from the device's own
    latent after 16 blocks, and the call as a whole equal to 16 + 1 blocks in two calls."""
    dcp = _dcp()
    cfg = syn.small_config("D2", I=3000, c_s=768, c_z=128, H=16, c=48, dtype="bf16", seed=2, structured=True, copies=60)
    a0, z = syn.make_s(cfg, DEV), syn.make_z(cfg, DEV)
    blocks = _blocks(cfg, 17)
    cache = torch.empty(dcp.dcp_attention_stack_cache_bytes(cfg.I, 17), dtype=torch.uint8, device=DEV)
    a16 = a0.clone()
    dcp.dcp_attention_stack_cached(a16, z, blocks[:16], cfg.H, cfg.c, bias_cache=cache)
    a17 = a16.clone()
    dcp.dcp_attention_stack_cached(a17, z, blocks[16:], cfg.H, cfg.c, bias_cache=cache)
    full = a0.clone()
    dcp.dcp_attention_stack_cached(full, z, blocks, cfg.H, cfg.c, bias_cache=cache)
    assert torch.equal(full, a17)
    assert bool(torch.isfinite(full.float()).all())
    rows = syn.sample_rows(cfg.I, 32, boundaries=(32, 1000, 2976), seed=6)
    idx = torch.as_tensor(rows, device=DEV)
    upd_ref = orc.pair_bias_attention_rows(util.np64(a16), util.np32(z.index_select(0, idx)), rows, util.weights_np(blocks[16]),
                                           cfg.H, cfg.c)
    a16r = util.np64(a16.index_select(0, idx))
    ref = _bf(a16r + upd_ref)
    got = util.np64(a17.index_select(0, idx))
    rel = np.linalg.norm((got - a16r) - upd_ref) / np.linalg.norm(upd_ref)
    assert rel <= 2e-2, f"update rel-L2 {rel:.3e}"
    assert np.all(np.abs(got - ref) <= util.TOL_BF16_MAXABS + 2.0 ** -7 * np.abs(ref)), np.abs(got - ref).max()
    del z, cache
    torch.cuda.empty_cache()


def test_attention_stack_cached_error_paths():
    dcp = _dcp()
    cfg = syn.small_config("cserr", I=64, c_s=768, c_z=128, H=16, c=48, dtype="bf16", seed=5)
    a, z = syn.make_s(cfg, DEV), syn.make_z(cfg, DEV)
    blocks = _blocks(cfg, 2)
    with pytest.raises(dcp.DcpError) as e:                 # cache too small
        dcp.dcp_attention_stack_cached(a, z, blocks, cfg.H, cfg.c, bias_cache=torch.empty(1024, dtype=torch.uint8, device=DEV))
    assert e.value.status == 3
    cfg4 = syn.small_config("cserr4", I=64, c_s=128, c_z=16, H=4, c=32, dtype="bf16", seed=5)
    with pytest.raises(dcp.DcpError) as e:                 # the atom shape has no bias cache
        dcp.dcp_attention_stack_cached(syn.make_s(cfg4, DEV), syn.make_z(cfg4, DEV), [syn.make_weights(cfg4, DEV)], cfg4.H, cfg4.c)
    assert e.value.status == 2
    assert dcp.dcp_attention_stack_cache_bytes(3000, 18) == 18 * 94 * 188 * 8 * 512 * 4
