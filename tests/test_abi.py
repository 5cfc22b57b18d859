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
    s1 = dcp.dcp_plan_units(3000, 16, 48, 128, torch.bfloat16)[2]
    s4 = dcp.dcp_plan_units(3000, 16, 48, 128, torch.bfloat16, "grid", 16)[2]
    assert s4 > s1 and b4 - b1 >= (s4 - s1) * 3000 * (2 * 16 + 768) * 4
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


def test_plan_units_are_a_pure_function_of_the_key_cut():
    """Host logic behind the bitwise decomposition contract: the segments a key chunk is cut into
    depend on (I, number of chunks) only -- never on the row partition -- so row(P) and the G x G grid cut a row's keys
    exactly like monolithic(key_split = 1 resp. G); the tile height may differ (it changes no row's arithmetic)."""
    _ensure_built()
    import paper_2607_05439_b200 as dcp
    bf = torch.bfloat16
    for I in (131, 600, 3000, 12000, 27180):
        seg1, tq1, slots1 = dcp.dcp_plan_units(I, 16, 48, 128, bf)
        assert slots1 == seg1 and 25 <= tq1 <= 32 and 1 <= seg1 <= 16
        for P in (2, 7, 8, 16):
            if P > I:
                continue
            seg, tq, slots = dcp.dcp_plan_units(I, 16, 48, 128, bf, "row", P)
            assert (seg, slots) == (seg1, slots1) and 25 <= tq <= 32
        for G in (2, 4):
            segk, _, slotsk = dcp.dcp_plan_units(I, 16, 48, 128, bf, key_split=G)
            segg, _, slotsg = dcp.dcp_plan_units(I, 16, 48, 128, bf, "grid", G * G)
            assert (segg, slotsg) == (segk, slotsk) and slotsg == G * segg
    # the headline config: 3 segments x 97 tiles of 31 rows = 291 units for 148 SMs (two waves)
    assert dcp.dcp_plan_units(3000, 16, 48, 128, bf) == (3, 31, 3)
    # forced values are honoured, clamped to whole key tiles; the atom and generic kernels have one tiling
    assert dcp.dcp_plan_units(3000, 16, 48, 128, bf, key_segments=5, tile=(28, 16))[:2] == (5, 28)
    assert dcp.dcp_plan_units(300, 16, 48, 128, bf, key_segments=64)[0] == 300 // 16
    assert dcp.dcp_plan_units(24000, 4, 32, 16, bf)[1] == 64
    assert dcp.dcp_plan_units(64, 4, 32, 64, torch.float32, key_split=2) == (1, 0, 2)
    with pytest.raises(dcp.DcpError) as e:
        dcp.dcp_plan_units(3000, 16, 48, 128, bf, tile=(24, 16))
    assert e.value.status == 2


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
