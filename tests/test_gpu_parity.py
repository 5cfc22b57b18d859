"""GPU parity tests (`-m gpu`): the CUDA path, called through the C ABI, against the fp64 oracle on the
same seeded inputs.  Tolerances are BASELINE.json's (tests/util.py).  Small cases compare every element;
the full-size configs compare sampled query rows (a row's output needs only s and z[i,:,:], so a sampled
row is exact).  Edge cases: ragged tails, uneven shards, I smaller than a tile, I = 1.
"""
import numpy as np
import pytest
import torch

import dcp_synth as syn
from tests import util

pytestmark = pytest.mark.gpu

DEV = "cuda:0"


def _dcp():
    import paper_2607_05439_b200 as dcp   # raises if libdesigncp.so is missing: no fallback
    return dcp


# kernels to exercise for a storage dtype (the MMA kernel is bf16-only)
def kernels_for(dtype, H=16, c=48, c_z=128):
    if dtype == "f32":
        return ["generic"]
    ok = _dcp().dcp_kernel_supported("mma", torch.bfloat16, H, c, c_z)
    return ["generic", "mma"] if ok else ["generic"]


# ------------------------------------------------------------------ config 0 (fp32), all decompositions
def test_c0_fp32_all_decompositions():
    dcp = _dcp()
    cfg = syn.CONFIGS["C0"]
    s, z, w = util.make_problem(cfg, DEV)
    ref = util.oracle_rows(cfg, s, z, w, range(cfg.I))
    mono = dcp.dcp_pair_bias_attention(s, z, w, cfg.H, cfg.c, kernel="generic")
    util.check_close(mono, ref, "f32", "C0 monolithic")
    row = dcp.dcp_pair_bias_attention(s, z, w, cfg.H, cfg.c, decomp="row", parts=4, kernel="generic")
    grid = dcp.dcp_pair_bias_attention(s, z, w, cfg.H, cfg.c, decomp="grid", parts=4, kernel="generic")
    util.check_close(row, ref, "f32", "C0 row(4)")
    util.check_close(grid, ref, "f32", "C0 grid(2x2)")
    # decomposition contract: row(P) == monolithic bitwise; grid(GxG) == monolithic(key_split=G) bitwise
    assert torch.equal(row, mono)
    mono_k2 = dcp.dcp_pair_bias_attention(s, z, w, cfg.H, cfg.c, key_split=2, kernel="generic")
    assert torch.equal(grid, mono_k2)
    rel = (grid - mono).abs().max().item() / mono.abs().max().item()
    assert rel <= 1e-6, rel


# ------------------------------------------------------------------ ragged / odd small shapes, fp32 and bf16
@pytest.mark.parametrize("dtype,I,c_s,c_z,H,c,ln_s,b_q", [
    ("f32", 67, 40, 20, 3, 32, True, True),      # tail tiles, uneven shards, D=96 != c_s, optional LN_s + b_q
    ("f32", 1, 16, 4, 1, 32, False, False),      # single token
    ("f32", 5, 24, 8, 2, 16, False, False),      # I smaller than any tile
    ("bf16", 131, 64, 32, 4, 24, False, False),  # ragged, c = 24
    ("bf16", 200, 128, 16, 4, 32, True, False),  # atom-like widths
    ("bf16", 131, 64, 128, 16, 24, False, False),  # tensor-core kernel shapes: ragged I, c = 24 (padded to 32)
    ("bf16", 77, 96, 128, 16, 48, True, True),     # tensor-core kernel, c = 48, LN_s + b_q, I < 3 tiles
    ("bf16", 200, 64, 128, 16, 32, False, False),  # tensor-core kernel, c = 32
    ("bf16", 9, 32, 128, 16, 48, False, False),    # tensor-core kernel, I smaller than a tile
])
def test_small_shapes_all_decompositions(dtype, I, c_s, c_z, H, c, ln_s, b_q):
    dcp = _dcp()
    cfg = syn.small_config("t", I=I, c_s=c_s, c_z=c_z, H=H, c=c, dtype=dtype, seed=21 + I)
    s, z, w = util.make_problem(cfg, DEV, with_ln_s=ln_s, with_b_q=b_q)
    ref = util.oracle_rows(cfg, s, z, w, range(I))
    for kern in kernels_for(dtype, H, c, c_z):
        try:
            mono = dcp.dcp_pair_bias_attention(s, z, w, H, c, kernel=kern)
        except dcp.DcpError as e:
            if kern == "mma" and e.status == 2:   # shape not instantiated for the MMA kernel
                continue
            raise
        util.check_close(mono, ref, dtype, f"{kern} mono I={I}")
        for P in sorted({1, 2, 3, 7, I} & set(range(1, I + 1))):
            row = dcp.dcp_pair_bias_attention(s, z, w, H, c, decomp="row", parts=P, kernel=kern)
            util.check_close(row, ref, dtype, f"{kern} row({P}) I={I}")
            assert torch.equal(row, mono), f"{kern} row({P}) != monolithic bitwise"
        for P in (1, 4, 9):
            G = int(round(P ** 0.5))
            if G > I:
                continue
            grid = dcp.dcp_pair_bias_attention(s, z, w, H, c, decomp="grid", parts=P, kernel=kern)
            util.check_close(grid, ref, dtype, f"{kern} grid({P}) I={I}")
            mk = dcp.dcp_pair_bias_attention(s, z, w, H, c, key_split=G, kernel=kern)
            assert torch.equal(grid, mk), f"{kern} grid({P}) != monolithic(key_split={G}) bitwise"


# ------------------------------------------------------------------ config 1 (bf16, I=600) in full
def test_c1_bf16_full():
    dcp = _dcp()
    cfg = syn.CONFIGS["C1"]
    s, z, w = util.make_problem(cfg, DEV)
    ref = util.oracle_rows(cfg, s, z, w, range(cfg.I))
    for kern in kernels_for("bf16", cfg.H, cfg.c, cfg.c_z):
        mono = dcp.dcp_pair_bias_attention(s, z, w, cfg.H, cfg.c, kernel=kern)
        util.check_close(mono, ref, "bf16", f"C1 {kern} monolithic")
        for decomp, P in (("row", 8), ("row", 7), ("grid", 4), ("grid", 16)):
            o = dcp.dcp_pair_bias_attention(s, z, w, cfg.H, cfg.c, decomp=decomp, parts=P, kernel=kern)
            util.check_close(o, ref, "bf16", f"C1 {kern} {decomp}({P})")
            if decomp == "row":
                assert torch.equal(o, mono)
        # run-to-run bitwise repeatability (no atomics)
        again = dcp.dcp_pair_bias_attention(s, z, w, cfg.H, cfg.c, kernel=kern)
        assert torch.equal(again, mono)


# ------------------------------------------------------------------ full-size configs: SURVEY.md 8(c)'s acceptance protocol
def protocol_rows(dcp, I, tile, shard_counts, count, seed):
    """Query rows SURVEY.md 8(c) asks for at sizes the oracle cannot cover in full: the first and last row of the tensor,
    both sides of every stripe / row-block boundary, and every query-tile class of every shard -- first and last row of
    its first tile, of an interior tile and of its last (possibly ragged) tile -- topped up with seeded random rows."""
    rows = set()
    for parts in shard_counts:
        for p in range(parts):
            b, n = dcp.dcp_shard_range(I, parts, p)
            last_tile = b + (n - 1) // tile * tile
            mid_tile = b + (n // tile // 2) * tile
            rows |= {b - 1, b, b + 1, b + tile - 1, b + tile, mid_tile, mid_tile + tile - 1, last_tile - 1, last_tile,
                     b + n - 2, b + n - 1}
    rows = {r for r in rows if 0 <= r < I}
    extra = 0
    while len(rows) < count:                       # seeded random rows until the protocol's count is reached
        extra += count - len(rows)
        rows |= set(syn.sample_rows(I, extra + 2, seed=seed))
    return sorted(rows)


def _oracle_rows_chunked(cfg, s, z, w, rows, chunk=256):
    return np.concatenate([util.oracle_rows(cfg, s, z, w, rows[i:i + chunk]) for i in range(0, len(rows), chunk)], axis=0)


def test_c2_bf16_full_output():
    """C2 (the headline config, I = 3000) over the FULL output, all three decompositions ("C1, C2 over
    the full output"): monolithic, 8 stripes of 375, 4 x 4 grid of 750^2 quadrants."""
    dcp = _dcp()
    cfg = syn.CONFIGS["C2"]
    s, z, w = util.make_problem(cfg, DEV)
    ref = _oracle_rows_chunked(cfg, s, z, w, list(range(cfg.I)))
    mono = dcp.dcp_pair_bias_attention(s, z, w, cfg.H, cfg.c)
    util.check_close(mono, ref, "bf16", "C2 monolithic (full output)")
    row = dcp.dcp_pair_bias_attention(s, z, w, cfg.H, cfg.c, decomp="row", parts=8)
    assert torch.equal(row, mono), "row(8) != monolithic bitwise"
    grid = dcp.dcp_pair_bias_attention(s, z, w, cfg.H, cfg.c, decomp="grid", parts=16)
    util.check_close(grid, ref, "bf16", "C2 grid(4x4) (full output)")
    assert torch.equal(grid, dcp.dcp_pair_bias_attention(s, z, w, cfg.H, cfg.c, key_split=4))
    del z
    torch.cuda.empty_cache()


@pytest.mark.parametrize("name,decomps,tile", [
    ("C3", [("monolithic", 1), ("row", 16), ("grid", 16)], 32),
    ("C4", [("monolithic", 1), ("row", 16), ("grid", 16)], 64),
])
def test_full_size_sampled_rows(name, decomps, tile):
    """C3 / C4 on >= 256 sampled query rows (a row's output needs only s and z[i, :, :], so a sampled row is exact)."""
    dcp = _dcp()
    cfg = syn.CONFIGS[name]
    free, _ = torch.cuda.mem_get_info()
    if cfg.z_bytes() * 1.15 > free:
        pytest.skip(f"{name}: z needs {cfg.z_bytes() / 1e9:.1f} GB")
    s, z, w = util.make_problem(cfg, DEV)
    shard_counts = {1}
    for _, P in decomps:
        shard_counts |= {P, int(round(P ** 0.5))}
    rows = protocol_rows(dcp, cfg.I, tile, sorted(shard_counts), 256, cfg.seed)
    assert len(rows) >= 256 and rows[0] == 0 and rows[-1] == cfg.I - 1
    ref = _oracle_rows_chunked(cfg, s, z, w, rows)
    idx = torch.as_tensor(rows, device=DEV)
    atom = name == "C4"
    mono = None
    for decomp, P in decomps:
        out = dcp.dcp_pair_bias_attention(s, z, w, cfg.H, cfg.c, decomp=decomp, parts=P, atom=atom)
        util.check_close(out.index_select(0, idx), ref, "bf16", f"{name} {decomp}({P})")
        assert torch.isfinite(out.float()).all()
        if decomp == "monolithic":
            mono = out
        elif decomp == "row":
            assert torch.equal(out, mono), f"{name} row({P}) != monolithic bitwise"
    del z
    torch.cuda.empty_cache()


# ------------------------------------------------------------------ partial states and the merge kernel
@pytest.mark.parametrize("dtype,c_z,H,c", [("f32", 32, 4, 24), ("bf16", 32, 4, 24), ("bf16", 128, 16, 24),
                                           ("bf16", 16, 4, 32)])   # last: the atom-level tensor-core kernel
def test_partial_states_and_merge(dtype, c_z, H, c):
    from oracle import decompositions as dec
    dcp = _dcp()
    cfg = syn.small_config("ps", I=150, c_s=64, c_z=c_z, H=H, c=c, dtype=dtype, seed=33)
    s, z, w = util.make_problem(cfg, DEV)
    q0, q1 = 37, 101
    rows = list(range(q0, q1))
    states = dec.key_split_states(util.np64(s), util.np32(z[q0:q1]), rows, util.weights_np(w), cfg.H, cfg.c, 3)
    got = []
    tol = 2e-5 if dtype == "f32" else 3e-2
    for kern in kernels_for(dtype, cfg.H, cfg.c, cfg.c_z):
        got = []
        for cb in range(3):
            k0, kl = dcp.dcp_shard_range(cfg.I, 3, cb)
            try:
                m, l, acc = dcp.dcp_partial_states(s, z, w, cfg.H, cfg.c, q0, q1, k0, k0 + kl, kernel=kern)
            except dcp.DcpError as e:
                if kern == "mma" and e.status == 2:
                    got = None
                    break
                raise
            got.append((m, l, acc))
            om, ol, oacc = states[cb]
            # the state is defined up to its reference m (reading 19): l/acc are compared after rescaling to
            # the oracle's m.  fp32 kernel: m is the row maximum.  bf16 tensor-core kernel: the reference follows the
            # running maximum lazily -- never above it, at most 8 log2 units (8 ln 2) below it.
            f = np.exp(util.np64(m) - om)
            dm = util.np64(m) - om
            if dtype == "f32":
                assert np.max(np.abs(dm)) <= 1e-4
            else:
                assert dm.max() <= 0.1 and dm.min() >= -(8.0 * np.log(2.0) + 0.1)
            assert np.max(np.abs(util.np64(l) * f - ol) / ol) <= tol
            a = util.np64(acc).reshape(len(rows), cfg.H, cfg.c) * f[..., None]
            assert np.max(np.abs(a - oacc)) <= tol * max(1.0, np.max(np.abs(oacc)))
        if got is None:
            continue
        M = torch.stack([g[0] for g in got]); L = torch.stack([g[1] for g in got]); A = torch.stack([g[2] for g in got])
        mm, ll, aa = dcp.dcp_merge_states(M, L, A, cfg.H, cfg.c)
        st = (util.np64(M[0]), util.np64(L[0]), util.np64(A[0]).reshape(len(rows), cfg.H, cfg.c))
        for t in (1, 2):
            st = dec.merge(st, (util.np64(M[t]), util.np64(L[t]), util.np64(A[t]).reshape(len(rows), cfg.H, cfg.c)))
        assert np.array_equal(util.np64(mm), st[0])
        assert np.max(np.abs(util.np64(ll) - st[1]) / st[1]) <= 1e-6
        assert np.max(np.abs(util.np64(aa).reshape(st[2].shape) - st[2])) <= 1e-6 * max(1.0, np.max(np.abs(st[2])))


def test_merge_extremes_no_nan():
    dcp = _dcp()
    rows, H, c = 5, 2, 4
    g = torch.Generator(device="cpu").manual_seed(3)
    m = torch.randn(3, rows, H, generator=g)
    m[1] += 80.0
    m[2] -= 80.0
    l = torch.rand(3, rows, H, generator=g) + 0.5
    acc = torch.randn(3, rows, H * c, generator=g)
    mm, ll, aa = dcp.dcp_merge_states(m.to(DEV), l.to(DEV), acc.to(DEV), H, c)
    assert torch.isfinite(mm).all() and torch.isfinite(ll).all() and torch.isfinite(aa).all()
    assert torch.equal(mm.cpu(), m.max(dim=0).values)


# ------------------------------------------------------------------ strided view, host entry
def test_ldz_strided_view_and_host_entry():
    dcp = _dcp()
    cfg = syn.small_config("ld", I=96, c_s=64, c_z=32, H=4, c=24, dtype="bf16", seed=44)
    s, z, w = util.make_problem(cfg, DEV)
    ref = util.oracle_rows(cfg, s, z, w, range(cfg.I))
    # z as a view of a wider tensor: row pitch (I + 8) * c_z elements
    big = torch.zeros(cfg.I, cfg.I + 8, cfg.c_z, dtype=z.dtype, device=DEV)
    big[:, :cfg.I] = z
    out = dcp.dcp_pair_bias_attention(s, big, w, cfg.H, cfg.c, ldz=(cfg.I + 8) * cfg.c_z)
    util.check_close(out, ref, "bf16", "strided z")
    base = dcp.dcp_pair_bias_attention(s, z, w, cfg.H, cfg.c)
    assert torch.equal(out, base)
    # host entry: pinned host buffers, copies inside the call
    sh, zh = s.cpu().pin_memory(), z.cpu().pin_memory()
    oh = torch.empty(cfg.I, cfg.c_s, dtype=s.dtype).pin_memory()
    ws = torch.empty(dcp.dcp_workspace_bytes(cfg.I, cfg.c_s, cfg.H, cfg.c, cfg.c_z, s.dtype), dtype=torch.uint8, device=DEV)
    dcp.dcp_pair_bias_attention_host(sh, zh, w, cfg.H, cfg.c, oh, torch.empty_like(s), torch.empty_like(z),
                                     torch.empty_like(s), ws)
    torch.cuda.synchronize()
    assert torch.equal(oh, base.cpu())


# ------------------------------------------------------------------ error paths of the C ABI (need device pointers)
def test_error_paths():
    dcp = _dcp()
    cfg = syn.small_config("e", I=32, c_s=32, c_z=8, H=2, c=16, dtype="f32", seed=5)
    s, z, w = util.make_problem(cfg, DEV)
    with pytest.raises(dcp.DcpError) as e:
        dcp.dcp_pair_bias_attention(s, z, w, cfg.H, cfg.c, decomp="grid", parts=8)      # not a perfect square
    assert e.value.status == 1
    with pytest.raises(dcp.DcpError) as e:
        dcp.dcp_pair_bias_attention(s, z, w, cfg.H, cfg.c, decomp="row", parts=33)      # parts > I
    assert e.value.status == 1
    with pytest.raises(dcp.DcpError) as e:
        dcp.dcp_pair_bias_attention(s, z, w, cfg.H, cfg.c, workspace=torch.empty(256, dtype=torch.uint8, device=DEV))
    assert e.value.status == 3
    with pytest.raises(dcp.DcpError) as e:
        dcp.dcp_pair_bias_attention(s, z, w, 3, 7)                                      # D = 21: unsupported
    assert e.value.status in (1, 2)
    with pytest.raises(dcp.DcpError) as e:
        dcp.dcp_pair_bias_attention(s, z, w, cfg.H, cfg.c, kernel="mma")                # fp32 has no MMA kernel
    assert e.value.status == 2
    w2 = dict(w)
    w2["ln_s_gamma"] = w["ln_z_gamma"]                                                  # gamma without beta
    with pytest.raises(dcp.DcpError):
        dcp.dcp_pair_bias_attention(s, z, w2, cfg.H, cfg.c)
    # still healthy afterwards
    out = dcp.dcp_pair_bias_attention(s, z, w, cfg.H, cfg.c)
    assert torch.isfinite(out).all() and dcp.dcp_last_launch_count() > 0


# ------------------------------------------------------------------ the ring's visiting order (SURVEY.md 8c reading 13)
@pytest.mark.parametrize("dtype,c_z,H,c,kern", [("f32", 32, 4, 24, "generic"), ("bf16", 128, 16, 48, "mma")])
def test_merge_in_rotated_ring_order(dtype, c_z, H, c, kern):
    """Row block r of a G x G grid merged in the order a ring visits its key blocks -- starting at block c = r
    ("bundles the K/V/B shift") -- instead of ascending c: the device merge of the device's own
    quadrant states, fed in rotated order, agrees with the oracle's rotated-order grid and with the canonical order
    within tolerance (not bitwise: the fold is not associative)."""
    from oracle import decompositions as dec
    dcp = _dcp()
    G = 3
    cfg = syn.small_config("ring", I=150, c_s=64, c_z=c_z, H=H, c=c, dtype=dtype, seed=41)
    s, z, w = util.make_problem(cfg, DEV)
    ref_rot = dec.grid_decomposition(util.np64(s), util.np32(z), util.weights_np(w), cfg.H, cfg.c, G * G, first_block_offset=True)
    ref = util.oracle_rows(cfg, s, z, w, range(cfg.I))
    assert np.max(np.abs(ref_rot - ref)) <= 1e-10
    wn = util.weights_np(w)
    g = 1.0 / (1.0 + np.exp(-(util.np64(s) @ wn["w_g"])))
    out_rot, out_can = np.zeros_like(ref), np.zeros_like(ref)
    for r in range(G):
        q0, ql = dcp.dcp_shard_range(cfg.I, G, r)
        st = []
        for cb in range(G):
            k0, kl = dcp.dcp_shard_range(cfg.I, G, cb)
            st.append(dcp.dcp_partial_states(s, z, w, cfg.H, cfg.c, q0, q0 + ql, k0, k0 + kl, kernel=kern))
        for order, dst in (([(r + t) % G for t in range(G)], out_rot), (list(range(G)), out_can)):
            M = torch.stack([st[cb][0] for cb in order]); L = torch.stack([st[cb][1] for cb in order])
            A = torch.stack([st[cb][2] for cb in order])
            _, ll, aa = dcp.dcp_merge_states(M, L, A, cfg.H, cfg.c)
            o = util.np64(aa).reshape(ql, cfg.H, cfg.c) / util.np64(ll)[..., None]
            dst[q0:q0 + ql] = (g[q0:q0 + ql] * o.reshape(ql, -1)) @ wn["w_o"]
    tol = 1e-5 if dtype == "f32" else util.TOL_BF16_MAXABS
    assert np.max(np.abs(out_rot - ref)) <= tol and np.max(np.abs(out_can - ref)) <= tol
    assert np.max(np.abs(out_rot - out_can)) <= (1e-6 if dtype == "f32" else 1e-4) * max(1.0, np.max(np.abs(ref)))


def test_merge_of_empty_states_is_the_identity():
    dcp = _dcp()
    rows, H, c = 4, 2, 4
    g = torch.Generator(device="cpu").manual_seed(8)
    m = torch.randn(3, rows, H, generator=g); l = torch.rand(3, rows, H, generator=g) + 0.5
    acc = torch.randn(3, rows, H * c, generator=g)
    for empty in ((0, 1), (1, 2), (0, 1, 2)):
        mm, ll, aa = m.clone(), l.clone(), acc.clone()
        for e in empty:
            mm[e] = -float("inf"); ll[e] = 0.0; aa[e] = 0.0
        mo, lo, ao = dcp.dcp_merge_states(mm.to(DEV), ll.to(DEV), aa.to(DEV), H, c)
        assert not torch.isnan(mo).any() and not torch.isnan(lo).any() and not torch.isnan(ao).any()
        keep = [i for i in range(3) if i not in empty]
        if len(keep) == 1:
            assert torch.equal(mo.cpu(), m[keep[0]]) and torch.equal(lo.cpu(), l[keep[0]]) and torch.equal(ao.cpu(), acc[keep[0]])
        else:
            assert torch.isinf(mo).all() and (lo == 0).all() and (ao == 0).all()


# ------------------------------------------------------------------ dcp_plan: tile and key_segments
def test_plan_tile_and_key_segments():
    dcp = _dcp()
    cfg = syn.small_config("plan", I=300, c_s=64, c_z=128, H=16, c=48, dtype="bf16", seed=17)
    s, z, w = util.make_problem(cfg, DEV)
    ref = util.oracle_rows(cfg, s, z, w, range(cfg.I))
    base = dcp.dcp_pair_bias_attention(s, z, w, cfg.H, cfg.c)
    for tq in (32, 31, 28, 25):        # any query-tile height 25..32: the tiling changes no row's arithmetic
        assert torch.equal(dcp.dcp_pair_bias_attention(s, z, w, cfg.H, cfg.c, tile=(tq, 16)), base), tq
        assert torch.equal(dcp.dcp_pair_bias_attention(s, z, w, cfg.H, cfg.c, tile=(tq, 0), decomp="grid", parts=9),
                           dcp.dcp_pair_bias_attention(s, z, w, cfg.H, cfg.c, decomp="grid", parts=9)), tq
    for bad in ((64, 16), (32, 32), (128, 0), (24, 16), (33, 0)):
        with pytest.raises(dcp.DcpError) as e:
            dcp.dcp_pair_bias_attention(s, z, w, cfg.H, cfg.c, tile=bad)
        assert e.value.status == 2
    with pytest.raises(dcp.DcpError) as e:
        dcp.dcp_pair_bias_attention(s, z, w, cfg.H, cfg.c, key_segments=65)
    assert e.value.status == 1
    for ks in (1, 2, 5, 64):           # 64 is clamped to the whole key tiles of a chunk
        mono = dcp.dcp_pair_bias_attention(s, z, w, cfg.H, cfg.c, key_segments=ks)
        util.check_close(mono, ref, "bf16", f"key_segments={ks}")
        row = dcp.dcp_pair_bias_attention(s, z, w, cfg.H, cfg.c, decomp="row", parts=7, key_segments=ks)
        assert torch.equal(row, mono), f"row(7) != monolithic bitwise at key_segments={ks}"
        grid = dcp.dcp_pair_bias_attention(s, z, w, cfg.H, cfg.c, decomp="grid", parts=9, key_segments=ks)
        assert torch.equal(grid, dcp.dcp_pair_bias_attention(s, z, w, cfg.H, cfg.c, key_split=3, key_segments=ks))
        util.check_close(grid, ref, "bf16", f"grid(9) key_segments={ks}")
    cfg0 = syn.CONFIGS["C0"]
    s0, z0, w0 = util.make_problem(cfg0, DEV)
    assert torch.equal(dcp.dcp_pair_bias_attention(s0, z0, w0, cfg0.H, cfg0.c, tile=(8, 32)),
                       dcp.dcp_pair_bias_attention(s0, z0, w0, cfg0.H, cfg0.c))


# ------------------------------------------------------------------ seeded fuzz over shapes, decompositions and unit plans
def test_fuzz_decompositions_and_unit_plans():
    """Forty seeded random problems on the tensor-core kernels (token shape, every fourth the atom shape; ragged I from 1
    to 420, every instantiated head size, random stripes / grids / key splits / forced segments / tile heights): each result against the oracle, and the
    bitwise contract row(P) == monolithic, grid(G x G) == monolithic(key_split = G) for equal key segments."""
    dcp = _dcp()
    rng = np.random.default_rng(2025)
    for case in range(40):
        I = int(rng.integers(1, 421))
        atom = case % 4 == 3                       # every fourth case: the atom-level kernel's shape
        c = 32 if atom else int(rng.choice([24, 32, 48]))
        c_s = int(rng.choice([32, 64, 96]))
        cfg = syn.small_config("fuzz", I=I, c_s=c_s, c_z=16 if atom else 128, H=4 if atom else 16, c=c, dtype="bf16",
                               seed=1000 + case)
        s, z, w = util.make_problem(cfg, DEV, with_ln_s=bool(rng.integers(0, 2)), with_b_q=bool(rng.integers(0, 2)))
        ref = util.oracle_rows(cfg, s, z, w, range(I))
        ks = int(rng.choice([0, 0, 1, 2, 3, 7]))
        tq = 0 if atom else int(rng.choice([0, 0, 25, 27, 30, 31, 32]))
        kw = dict(key_segments=ks, tile=(tq, 0))
        mono = dcp.dcp_pair_bias_attention(s, z, w, cfg.H, cfg.c, **kw)
        util.check_close(mono, ref, "bf16", f"fuzz {case}: I={I} c={c} ks={ks} tq={tq}")
        P = int(rng.integers(1, min(I, 9) + 1))
        row = dcp.dcp_pair_bias_attention(s, z, w, cfg.H, cfg.c, decomp="row", parts=P, key_segments=ks,
                                          tile=(0 if atom else int(rng.choice([0, 26, 32])), 0))
        assert torch.equal(row, mono), f"fuzz {case}: row({P}) != monolithic (I={I}, ks={ks})"
        G = int(rng.integers(1, min(I, 4) + 1))
        grid = dcp.dcp_pair_bias_attention(s, z, w, cfg.H, cfg.c, decomp="grid", parts=G * G, **kw)
        mk = dcp.dcp_pair_bias_attention(s, z, w, cfg.H, cfg.c, key_split=G, key_segments=ks)
        assert torch.equal(grid, mk), f"fuzz {case}: grid({G * G}) != monolithic(key_split={G}) (I={I}, ks={ks})"
        util.check_close(grid, ref, "bf16", f"fuzz {case}: grid({G * G})")
