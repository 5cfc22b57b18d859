"""The layer call enqueues only stream-ordered work (no host synchronisation, no allocation): it can be captured into a
CUDA graph and replayed (launch-bound small problems, e.g. C1).  Replay must reproduce the eager result bit for bit."""
import pytest
import torch

import dcp_synth as syn

pytestmark = pytest.mark.gpu
DEV = "cuda:0"


def test_layer_and_stack_capture_into_a_cuda_graph():
    import paper_2607_05439_b200 as dcp
    cfg = syn.small_config("graph", I=300, c_s=384, c_z=128, H=16, c=48, dtype="bf16", seed=21, structured=True, copies=60)
    w, s, z = syn.make_weights(cfg, DEV), syn.make_s(cfg, DEV), syn.make_z(cfg, DEV)
    n = dcp.dcp_workspace_bytes(cfg.I, cfg.c_s, cfg.H, cfg.c, cfg.c_z, torch.bfloat16)
    ws = torch.empty(n, dtype=torch.uint8, device=DEV)
    out = torch.empty_like(s)
    eager = dcp.dcp_pair_bias_attention(s, z, w, cfg.H, cfg.c, workspace=ws).clone()
    side = torch.cuda.Stream()
    side.wait_stream(torch.cuda.current_stream())
    with torch.cuda.stream(side):
        dcp.dcp_pair_bias_attention(s, z, w, cfg.H, cfg.c, out=out, workspace=ws, stream=side)   # warm-up on the capture stream
    torch.cuda.current_stream().wait_stream(side)
    torch.cuda.synchronize()
    g = torch.cuda.CUDAGraph()
    with torch.cuda.graph(g, stream=side):
        dcp.dcp_pair_bias_attention(s, z, w, cfg.H, cfg.c, out=out, workspace=ws, stream=side)
    out.zero_()
    for _ in range(3):
        g.replay()
    torch.cuda.synchronize()
    assert torch.equal(out, eager)


def test_stacks_and_no_alloc_entry_capture_into_a_cuda_graph():
    """dcp_attention_stack, dcp_attention_stack_cached (caller-owned cache and workspace) and
    dcp_pair_bias_attention_no_alloc enqueue launches only: each captures into a CUDA graph and the replay reproduces the
    eager result bit for bit (the stacks update the latent in place, so every replay starts from a restored copy)."""
    import paper_2607_05439_b200 as dcp
    cfg = syn.small_config("graph2", I=200, c_s=768, c_z=128, H=16, c=48, dtype="bf16", seed=23, structured=True, copies=40)
    a0, z = syn.make_s(cfg, DEV), syn.make_z(cfg, DEV)
    blocks = [syn.make_weights(syn.small_config("blk", I=cfg.I, c_s=cfg.c_s, c_z=cfg.c_z, H=cfg.H, c=cfg.c, dtype="bf16", seed=60 + b),
                               DEV, with_ln_s=True) for b in range(4)]
    ws = torch.empty(dcp.dcp_attention_stack_cached_workspace_bytes(cfg.I, cfg.c_s, cfg.H, cfg.c, cfg.c_z, torch.bfloat16),
                     dtype=torch.uint8, device=DEV)
    cache = torch.empty(dcp.dcp_attention_stack_cache_bytes(cfg.I, len(blocks)), dtype=torch.uint8, device=DEV)
    w1 = blocks[0]
    out_na = torch.empty_like(a0)
    calls = {
        "stack": lambda a, st: dcp.dcp_attention_stack(a, z, blocks, cfg.H, cfg.c, workspace=ws, stream=st),
        "cached": lambda a, st: dcp.dcp_attention_stack_cached(a, z, blocks, cfg.H, cfg.c, bias_cache=cache, workspace=ws, stream=st),
        "no_alloc": lambda a, st: dcp.dcp_pair_bias_attention_no_alloc(a, z, w1, cfg.H, cfg.c, out_na, stream=st),
    }
    for name, call in calls.items():
        a = a0.clone()
        call(a, None)
        torch.cuda.synchronize()
        eager = (out_na if name == "no_alloc" else a).clone()
        side = torch.cuda.Stream()
        side.wait_stream(torch.cuda.current_stream())
        a.copy_(a0)
        with torch.cuda.stream(side):
            call(a, side)                                        # warm-up on the capture stream
        torch.cuda.current_stream().wait_stream(side)
        torch.cuda.synchronize()
        g = torch.cuda.CUDAGraph()
        a.copy_(a0)
        torch.cuda.synchronize()
        with torch.cuda.graph(g, stream=side):
            call(a, side)
        for _ in range(2):
            a.copy_(a0)
            out_na.zero_()
            torch.cuda.synchronize()
            g.replay()
            torch.cuda.synchronize()
            assert torch.equal(out_na if name == "no_alloc" else a, eager), name
