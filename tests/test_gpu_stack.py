"""GPU parity of the Pairformer stack (first step) through the C ABI against
oracle/pairformer_stack.py.  The device keeps S and Z in bf16 and rounds them once per block; the oracle is given
that storage rounding explicitly (`round_store`).  Tolerances: BASELINE.json's bf16 bound rel-L2 <= 1e-2 on both
tracks after the whole stack, and elementwise n_blocks x the per-layer bounds (errors of consecutive blocks add up;
DESIGN.md 6.7): |ds| <= n (2e-2 + 2^-8 |s|), |dz| <= n (2e-2 + 2^-8 |z|)."""
import math

import numpy as np
import pytest
import torch

import dcp_synth as syn
from oracle import pairformer_stack as pso
from tests import util

pytestmark = pytest.mark.gpu
DEV = "cuda:0"


def _dcp():
    import paper_2607_05439_b200 as dcp
    return dcp


def _bf16_round(x):
    return torch.from_numpy(np.asarray(x)).to(torch.bfloat16).double().numpy()


def _blocks(cfg, n_blocks, scale_w3=1.0):
    blocks = []
    for b in range(n_blocks):
        wa = syn.make_weights(syn.small_config("blk", I=cfg.I, c_s=cfg.c_s, c_z=cfg.c_z, H=cfg.H, c=cfg.c, dtype="bf16",
                                               seed=cfg.seed + 31 * (b + 1)), DEV)
        g = torch.Generator(device="cpu").manual_seed(1000 + cfg.seed + b)
        n = lambda *s, std=1.0: (torch.randn(*s, generator=g) * std).to(torch.bfloat16).to(DEV)
        c_z = cfg.c_z
        wt = {"w1": n(c_z, 4 * c_z, std=1 / math.sqrt(c_z)), "w2": n(c_z, 4 * c_z, std=1 / math.sqrt(c_z)),
              "w3": n(4 * c_z, c_z, std=scale_w3 / math.sqrt(4 * c_z)),
              "gamma": (1 + 0.1 * torch.randn(c_z, generator=g)).to(torch.bfloat16).to(DEV),
              "beta": (0.1 * torch.randn(c_z, generator=g)).to(torch.bfloat16).to(DEV)}
        blocks.append((wa, wt))
    return blocks


def _oracle(s, z, blocks, H, c):
    ob = [({k: util.np64(v) for k, v in wa.items()}, {k: util.np64(v) for k, v in wt.items()}) for wa, wt in blocks]
    return pso.pairformer_stack(util.np64(s), util.np64(z), ob, H, c, round_store=_bf16_round)


@pytest.mark.parametrize("I,copies,n_blocks", [(96, 12, 1), (180, 60, 2), (75, 15, 4)])
def test_stack_matches_oracle(I, copies, n_blocks):
    dcp = _dcp()
    cfg = syn.small_config("stack", I=I, c_s=384, c_z=128, H=16, c=48, dtype="bf16", seed=11 + I, structured=True,
                           copies=copies)
    s0, z0 = syn.make_s(cfg, DEV), syn.make_z(cfg, DEV)
    blocks = _blocks(cfg, n_blocks)
    s_ref, z_ref = _oracle(s0, z0, blocks, cfg.H, cfg.c)
    s, z = s0.clone(), z0.clone()
    dcp.dcp_pairformer_stack(s, z, blocks, cfg.H, cfg.c)
    torch.cuda.synchronize()
    gs, gz = util.np64(s), util.np64(z)
    assert np.all(np.isfinite(gs)) and np.all(np.isfinite(gz))
    for name, got, ref, x0 in (("s", gs, s_ref, util.np64(s0)), ("z", gz, z_ref, util.np64(z0))):
        rel = np.linalg.norm(got - ref) / np.linalg.norm(ref)
        assert rel <= 1e-2, f"{name}: rel-L2 {rel:.3e}"
        bad = np.abs(got - ref) > n_blocks * (2e-2 + 2.0 ** -8 * np.abs(ref))
        assert not bad.any(), f"{name}: {bad.sum()} elements out of tolerance, max-abs {np.abs(got - ref).max():.3e}"
        # the stack's own contribution (final - initial) carries signal and agrees
        upd, upd_ref = got - x0, ref - x0
        assert np.linalg.norm(upd_ref) > 0.1 * np.linalg.norm(x0) or name == "s"
        assert np.linalg.norm(upd - upd_ref) / np.linalg.norm(upd_ref) <= 5e-2, name
    # repeatable bit for bit
    s2, z2 = s0.clone(), z0.clone()
    dcp.dcp_pairformer_stack(s2, z2, blocks, cfg.H, cfg.c)
    assert torch.equal(s, s2) and torch.equal(z, z2)


def test_stack_equals_the_calls_it_is_made_of():
    """One block == dcp_pair_bias_attention + residual + dcp_pair_transition issued by hand (bitwise)."""
    dcp = _dcp()
    cfg = syn.small_config("stack1", I=120, c_s=384, c_z=128, H=16, c=48, dtype="bf16", seed=5, structured=True, copies=60)
    s0, z0 = syn.make_s(cfg, DEV), syn.make_z(cfg, DEV)
    (wa, wt), = _blocks(cfg, 1)
    s, z = s0.clone(), z0.clone()
    dcp.dcp_pairformer_stack(s, z, [(wa, wt)], cfg.H, cfg.c)
    o = dcp.dcp_pair_bias_attention(s0, z0, wa, cfg.H, cfg.c)
    s_hand = (s0.float() + o.float()).to(torch.bfloat16)
    z_hand = dcp.dcp_pair_transition(z0, wt["w1"], wt["w2"], wt["w3"], wt["gamma"], wt["beta"])
    assert torch.equal(s, s_hand) and torch.equal(z, z_hand)


def test_stack_error_paths():
    dcp = _dcp()
    cfg = syn.small_config("stackerr", I=64, c_s=384, c_z=128, H=16, c=48, dtype="bf16", seed=5)
    s, z = syn.make_s(cfg, DEV), syn.make_z(cfg, DEV)
    blocks = _blocks(cfg, 1)
    with pytest.raises(dcp.DcpError):                       # workspace too small
        dcp.dcp_pairformer_stack(s, z, blocks, cfg.H, cfg.c, workspace=torch.empty(256, dtype=torch.uint8, device=DEV))
    with pytest.raises(dcp.DcpError):                       # no blocks
        dcp.dcp_pairformer_stack(s, z, [], cfg.H, cfg.c)
    cfg32 = syn.small_config("stackf32", I=64, c_s=128, c_z=64, H=4, c=32, dtype="f32", seed=5)
    with pytest.raises(dcp.DcpError):                       # fp32 / c_z = 64: the transition is not instantiated
        dcp.dcp_pairformer_stack(syn.make_s(cfg32, DEV), syn.make_z(cfg32, DEV),
                                 [(syn.make_weights(cfg32, DEV), blocks[0][1])], cfg32.H, cfg32.c)


def test_stack_full_size_block_sampled():
    """One block at C2's full size (I = 3000: the shape bench.py --workload P2 times): sampled query rows of S and the
    same rows of Z against the oracle's block (the attention rows oracle + the transition of those rows' pairs)."""
    dcp = _dcp()
    from oracle import pair_bias_attention as orc
    from oracle import pair_transition as pto
    cfg = syn.CONFIGS["C2"]
    s0, z0 = syn.make_s(cfg, DEV), syn.make_z(cfg, DEV)
    (wa, wt), = _blocks(cfg, 1)
    rows = syn.sample_rows(cfg.I, 24, boundaries=(32, 1000, 2000), seed=3)
    idx = torch.as_tensor(rows, device=DEV)
    z_rows0 = util.np64(z0.index_select(0, idx))
    s_ref = util.np64(s0)[np.asarray(rows)] + orc.pair_bias_attention_rows(
        util.np64(s0), z_rows0, rows, {k: util.np64(v) for k, v in wa.items()}, cfg.H, cfg.c)
    z_ref = pto.pair_transition(z_rows0, *[util.np64(wt[k]) for k in ("w1", "w2", "w3", "gamma", "beta")])
    s, z = s0.clone(), z0
    dcp.dcp_pairformer_stack(s, z, [(wa, wt)], cfg.H, cfg.c)
    torch.cuda.synchronize()
    for name, got, ref in (("s", util.np64(s.index_select(0, idx)), s_ref), ("z", util.np64(z.index_select(0, idx)), z_ref)):
        rel = np.linalg.norm(got - ref) / np.linalg.norm(ref)
        assert rel <= 1e-2, f"{name}: rel-L2 {rel:.3e}"
        assert np.all(np.abs(got - ref) <= 2e-2 + 2.0 ** -8 * np.abs(ref)), f"{name}: max-abs {np.abs(got - ref).max():.3e}"
