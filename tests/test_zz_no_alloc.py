"""GPU test (`-m gpu`) of dcp_pair_bias_attention_no_alloc (include/designcp.h): the layer with its workspace in the
library's static device array, against the existing caller-workspace path on the same inputs, within the tolerances
the parity tests use (tests/util.py) -- on two calls in a row with different inputs, so contents the first call left
in the shared array must not leak into the second.  Collected last on purpose (file name): the suite runs with
pytest -x."""
import pytest
import torch

import dcp_synth as syn
from tests import util

pytestmark = pytest.mark.gpu

DEV = "cuda:0"


def _dcp():
    import paper_2607_05439_b200 as dcp   # raises if libdesigncp.so is missing: no fallback
    return dcp


def _case(dtype, I, c_s, c_z, H, c, seed):
    cfg = syn.small_config("na", I=I, c_s=c_s, c_z=c_z, H=H, c=c, dtype=dtype, seed=seed)
    s, z, w = util.make_problem(cfg, DEV)
    return cfg, s, z, w


def test_no_alloc_matches_workspace_path_on_two_calls_in_a_row():
    dcp = _dcp()
    # tensor-core kernel, ragged I spanning several tiles; then a different, smaller problem on the same array
    calls = [("bf16", 333, 128, 128, 16, 48, 5), ("bf16", 131, 64, 128, 16, 24, 6)]
    for k, (dtype, I, c_s, c_z, H, c, seed) in enumerate(calls):
        cfg, s, z, w = _case(dtype, I, c_s, c_z, H, c, seed)
        ref = dcp.dcp_pair_bias_attention(s, z, w, H, c)                    # existing path, torch-allocated workspace
        out = torch.full_like(s, float("nan"))
        before = torch.cuda.memory_allocated()
        dcp.dcp_pair_bias_attention_no_alloc(s, z, w, H, c, out)
        assert torch.cuda.memory_allocated() == before                       # the binding allocated nothing either
        torch.cuda.synchronize()
        util.check_close(out, util.np64(ref), dtype, f"no_alloc call {k}")
        assert torch.equal(out, ref), f"no_alloc call {k}: same kernels, same plan -> same bits"
        # and against the oracle, like the parity tests
        util.check_close(out, util.oracle_rows(cfg, s, z, w, range(I)), dtype, f"no_alloc call {k} vs oracle")


def test_no_alloc_fp32_generic_and_decompositions():
    dcp = _dcp()
    cfg, s, z, w = _case("f32", 67, 40, 20, 3, 32, 9)
    for kw in (dict(), dict(decomp="row", parts=4), dict(decomp="grid", parts=4)):
        ref = dcp.dcp_pair_bias_attention(s, z, w, cfg.H, cfg.c, kernel="generic", **kw)
        out = torch.full_like(s, float("nan"))
        dcp.dcp_pair_bias_attention_no_alloc(s, z, w, cfg.H, cfg.c, out, kernel="generic", **kw)
        util.check_close(out, util.np64(ref), "f32", f"no_alloc {kw}")
        assert torch.equal(out, ref)


def test_no_alloc_rejects_sizes_beyond_the_static_scratch():
    dcp = _dcp()
    limit = dcp.dcp_no_alloc_scratch_bytes()
    assert limit == 32 << 20
    I, c_s, c_z, H, c = 3000, 384, 128, 16, 48
    assert dcp.dcp_workspace_bytes(I, c_s, H, c, c_z, torch.bfloat16) > limit
    # validation comes before any launch: the (uninitialised) big tensors are never read
    cfg, s, z, w = _case("bf16", 64, c_s, c_z, H, c, 3)
    s_big = torch.empty(I, c_s, dtype=torch.bfloat16, device=DEV)
    z_big = torch.empty(I, I, c_z, dtype=torch.bfloat16, device=DEV)
    out = torch.full_like(s_big, 1.0)
    with pytest.raises(dcp.DcpError) as e:
        dcp.dcp_pair_bias_attention_no_alloc(s_big, z_big, w, H, c, out)
    assert e.value.status == 5 and "SCRATCH_LIMIT" in str(e.value)
    torch.cuda.synchronize()
    assert bool((out == 1.0).all())
