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
