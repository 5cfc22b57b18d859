"""`-m "not gpu"`: the C-ABI library loads, exports every symbol include/designcp.h declares, and its
host-only entry points (planner, workspace sizing, argument validation) behave -- no compute calls."""
import ctypes
import os
import re

import pytest
import torch

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _ensure_built():
    import __graft_entry__ as ge
    ge.build()


def test_library_exports_every_declared_symbol():
    _ensure_built()
    hdr = open(os.path.join(ROOT, "include", "designcp.h")).read()
    declared = set(re.findall(r"\b(dcp_[a-z_0-9]+)\s*\(", hdr))
    assert {"dcp_pair_bias_attention", "dcp_atom_pair_bias_attention", "dcp_partial_states",
            "dcp_merge_states", "dcp_shard_range", "dcp_workspace_bytes"} <= declared
    lib = ctypes.CDLL(os.path.join(ROOT, "paper_2607_05439_b200", "libdesigncp.so"))
    for name in sorted(declared):
        assert hasattr(lib, name), f"libdesigncp.so does not export {name}"
    from paper_2607_05439_b200 import binding
    assert set(binding.EXPORTS) == declared


def test_shard_range_matches_eq5_and_oracle():
    _ensure_built()
    import paper_2607_05439_b200 as dcp
    from oracle import decompositions as dec
    for n in (1, 7, 64, 67, 600, 3000):
        for P in (1, 2, 3, 4, 7, 8, 16, 17):
            if P > n:
                continue
            for p in range(P):
                assert dcp.dcp_shard_range(n, P, p) == dec.shard_range(n, P, p)
    with pytest.raises(dcp.DcpError):
        dcp.dcp_shard_range(10, 0, 0)
    with pytest.raises(dcp.DcpError):
        dcp.dcp_shard_range(10, 4, 4)


def test_workspace_bytes_and_validation_without_gpu():
    _ensure_built()
    import paper_2607_05439_b200 as dcp
    b1 = dcp.dcp_workspace_bytes(3000, 384, 16, 48, 128, torch.bfloat16)
    b4 = dcp.dcp_workspace_bytes(3000, 384, 16, 48, 128, torch.bfloat16, "grid", 16)
    assert b4 > b1 > 5 * 3000 * 768 * 2
    # states: [slots][I][H] x2 + [slots][I][D] fp32
    assert b4 - b1 >= 3 * 3000 * (2 * 16 + 768) * 4
    for bad in (dict(decomp="grid", parts=8), dict(decomp="row", parts=3001), dict(decomp="grid", parts=0)):
        with pytest.raises(dcp.DcpError) as e:
            dcp.dcp_workspace_bytes(3000, 384, 16, 48, 128, torch.bfloat16, **bad)
        assert e.value.status == 1
    with pytest.raises(dcp.DcpError) as e:      # c_z * sizeof(elt) % 16 != 0
        dcp.dcp_workspace_bytes(64, 128, 4, 32, 3, torch.float32)
    assert e.value.status == 1
    with pytest.raises(dcp.DcpError) as e:      # D not a multiple of 32: no kernel instantiated
        dcp.dcp_workspace_bytes(64, 128, 3, 7, 64, torch.float32)
    assert e.value.status == 2
    assert dcp.status_string(0) == "DCP_OK" and dcp.version() >= 100
    assert dcp.dcp_kernel_supported("generic", torch.float32, 4, 32, 64)


def test_product_does_not_import_oracle():
    """The product path must not route through the oracle (or any CPU fallback)."""
    pkg = os.path.join(ROOT, "paper_2607_05439_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                src = open(os.path.join(dirpath, f)).read()
                assert not re.search(r"^\s*(from|import)\s+oracle\b", src, re.M), f
                assert "oracle/" not in src or f.endswith((".cu", ".cuh", ".h")), f
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith(".py"):
            src = open(os.path.join(ROOT, "oracle", f)).read()
            assert not re.search(r"^\s*(from|import)\s+paper_2607_05439_b200\b", src, re.M), f
