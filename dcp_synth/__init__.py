"""Seeded synthetic inputs for the pair-bias attention layer (Design-CP's one-GPU core).

This module is the ONLY code shared by the CPU oracle (`oracle/`) and the CUDA path
(`paper_2607_05439_b200/`).  It holds no arithmetic of the method itself: it only draws
random tensors with the shapes, value distributions and copy/residue block structure of
the paper's icosahedral workloads (PAPER.md:118-120 "60 x 210 residues", :152, :323;
BASELINE.json `configs`), and rounds them once to the storage dtype.

Recipe:
  * token index  i = copy * n + res,  copy in [0, copies), res in [0, n)   (copies = 60)
  * s[i]   = a[res] + 0.1 * N(0,1)                 a ~ N(0,1)  [n, c_s]
  * z[i,j] = E[copy(i), copy(j)] + R[res(i), res(j)] + 0.1 * N(0,1)
             E ~ N(0,1) [copies, copies, c_z],  R ~ N(0,1) [n, n, c_z]
  * weights: W_q, W_k, W_v, W_g [c_s, H*c], W_o [H*c, c_s], W_b [c_z, H]  ~ N(0, 1/fan_in)
             (variance 1/fan_in), gamma = 1 + 0.1 N(0,1), beta = 0.1 N(0,1)
  * config 0 is iid: s ~ N(0,1), z ~ N(0,1), no block structure.

Everything is generated with `torch` generators so the same code runs on the CPU (tests,
oracle) and on the GPU (z of 2.3-36.9 GB must be born in HBM).  CPU and CUDA generators give
different bit streams; each is deterministic per seed.  Parity tests always hand the oracle
the exact stored bits (read back from the device), never a re-generation.
"""
from __future__ import annotations

import dataclasses
import math
from typing import Dict, Optional

import torch

COPIES = 60  # icosahedral point group order: 60 ASU copies


@dataclasses.dataclass(frozen=True)
class LayerConfig:
    """Shape of one pair-bias attention layer call (BASELINE.json `configs`)."""

    name: str
    I: int          # tokens (or L atoms)
    c_s: int        # single-track width (c_atom for the atom variant)
    c_z: int        # pair width (c_atompair for the atom variant)
    H: int          # heads
    c: int          # head dim
    dtype: str      # "f32" | "bf16"  storage type
    seed: int
    structured: bool = True   # icosahedral copy/residue block structure
    copies: int = COPIES

    @property
    def D(self) -> int:
        return self.H * self.c

    @property
    def n_res(self) -> int:
        return self.I // self.copies if self.structured else self.I

    def z_bytes(self) -> int:
        return self.I * self.I * self.c_z * (4 if self.dtype == "f32" else 2)


# BASELINE.json configs 0..4 (C0..C4)
CONFIGS: Dict[str, LayerConfig] = {
    "C0": LayerConfig("C0", I=64, c_s=128, c_z=64, H=4, c=32, dtype="f32", seed=0, structured=False),
    "C1": LayerConfig("C1", I=600, c_s=384, c_z=128, H=16, c=24, dtype="bf16", seed=1),
    "C2": LayerConfig("C2", I=3000, c_s=384, c_z=128, H=16, c=48, dtype="bf16", seed=2),
    "C3": LayerConfig("C3", I=12000, c_s=384, c_z=128, H=16, c=48, dtype="bf16", seed=3),
    "C4": LayerConfig("C4", I=24000, c_s=128, c_z=16, H=4, c=32, dtype="bf16", seed=4),
}


def torch_dtype(name: str) -> torch.dtype:
    return {"f32": torch.float32, "bf16": torch.bfloat16}[name]


def _gen(seed: int, device) -> torch.Generator:
    g = torch.Generator(device=device)
    g.manual_seed(int(seed))
    return g


def make_weights(cfg: LayerConfig, device="cpu", with_ln_s: bool = False,
                 with_b_q: bool = False) -> Dict[str, torch.Tensor]:
    """Layer weights, drawn on the CPU in fp32 (tiny), rounded once to the storage dtype.

    Draw order is fixed: W_q, W_k, W_v, W_g, W_b, W_o, gamma_z, beta_z, gamma_s, beta_s, b_q.
    """
    g = _gen(cfg.seed * 1000003 + 17, "cpu")
    dt = torch_dtype(cfg.dtype)
    D = cfg.D

    def n(*shape, std=1.0):
        return torch.randn(*shape, generator=g, dtype=torch.float32) * std

    w = {}
    for k in ("w_q", "w_k", "w_v", "w_g"):
        w[k] = n(cfg.c_s, D, std=1.0 / math.sqrt(cfg.c_s))
    w["w_b"] = n(cfg.c_z, cfg.H, std=1.0 / math.sqrt(cfg.c_z))
    w["w_o"] = n(D, cfg.c_s, std=1.0 / math.sqrt(D))
    w["ln_z_gamma"] = 1.0 + 0.1 * n(cfg.c_z)
    w["ln_z_beta"] = 0.1 * n(cfg.c_z)
    gs, bs, bq = 1.0 + 0.1 * n(cfg.c_s), 0.1 * n(cfg.c_s), 0.1 * n(D)
    if with_ln_s:
        w["ln_s_gamma"], w["ln_s_beta"] = gs, bs
    if with_b_q:
        w["b_q"] = bq
    return {k: v.to(dt).to(device).contiguous() for k, v in w.items()}


def make_s(cfg: LayerConfig, device="cpu") -> torch.Tensor:
    """Single track s [I, c_s] in the storage dtype."""
    g = _gen(cfg.seed * 1000003 + 1, "cpu")
    if not cfg.structured:
        s = torch.randn(cfg.I, cfg.c_s, generator=g, dtype=torch.float32)
    else:
        n = cfg.n_res
        assert n * cfg.copies == cfg.I, "structured configs need I = copies * n_res"
        a = torch.randn(n, cfg.c_s, generator=g, dtype=torch.float32)
        s = a.repeat(cfg.copies, 1) + 0.1 * torch.randn(cfg.I, cfg.c_s, generator=g, dtype=torch.float32)
    return s.to(torch_dtype(cfg.dtype)).to(device).contiguous()


def _tables(cfg: LayerConfig, device):
    g = _gen(cfg.seed * 1000003 + 2, "cpu")
    n = cfg.n_res
    E = torch.randn(cfg.copies, cfg.copies, cfg.c_z, generator=g, dtype=torch.float32)
    R = torch.randn(n, n, cfg.c_z, generator=g, dtype=torch.float32)
    return E.to(device), R.to(device)


def fill_z(cfg: LayerConfig, out: torch.Tensor, chunk_rows: int = 0,
           noise: float = 0.1, cyclic_copy_table: bool = False) -> torch.Tensor:
    """Fill `out` ([I, I, c_z], storage dtype, on any device) with the pair tensor, in row chunks.

    Chunk r (rows [r*chunk, (r+1)*chunk)) draws its noise from a generator seeded
    (seed, r) on out's device, so a fill is repeatable for a fixed device type and chunk size.
    `cyclic_copy_table` replaces E[a,b] by F[(b-a) mod copies] (used by the oracle's
    copy-shift invariance pin; SURVEY.md 8c "Symmetry").
    """
    I, cz = cfg.I, cfg.c_z
    assert tuple(out.shape) == (I, I, cz)
    dev = out.device
    if not cfg.structured:
        chunk = chunk_rows or I
        for r, i0 in enumerate(range(0, I, chunk)):
            i1 = min(I, i0 + chunk)
            g = _gen(cfg.seed * 1000003 + 1000 + r, dev)
            out[i0:i1] = torch.randn(i1 - i0, I, cz, generator=g, device=dev, dtype=torch.float32).to(out.dtype)
        return out
    n = cfg.n_res
    E, R = _tables(cfg, dev)
    if cyclic_copy_table:
        F = E[0]  # [copies, c_z]
        a = torch.arange(cfg.copies, device=dev)
        E = F[(a[None, :] - a[:, None]) % cfg.copies]
    idx = torch.arange(I, device=dev)
    copy_j, res_j = idx // n, idx % n
    if chunk_rows <= 0:
        # ~256 MB of fp32 temporaries per chunk
        chunk_rows = max(1, min(I, (64 << 20) // max(1, I * cz)))
    for r, i0 in enumerate(range(0, I, chunk_rows)):
        i1 = min(I, i0 + chunk_rows)
        ci, ri = copy_j[i0:i1], res_j[i0:i1]
        blk = E[ci][:, copy_j] + R[ri][:, res_j]
        if noise != 0.0:
            g = _gen(cfg.seed * 1000003 + 1000 + r, dev)
            blk += noise * torch.randn(i1 - i0, I, cz, generator=g, device=dev, dtype=torch.float32)
        out[i0:i1] = blk.to(out.dtype)
        del blk
    return out


def make_z(cfg: LayerConfig, device="cpu", **kw) -> torch.Tensor:
    out = torch.empty(cfg.I, cfg.I, cfg.c_z, dtype=torch_dtype(cfg.dtype), device=device)
    return fill_z(cfg, out, **kw)


def small_config(name: str, I: int, c_s: int, c_z: int, H: int, c: int, dtype: str = "f32",
                 seed: int = 7, structured: bool = False, copies: int = COPIES) -> LayerConfig:
    """Helper for tests: arbitrary small shapes (ragged tails, odd sizes)."""
    return LayerConfig(name, I=I, c_s=c_s, c_z=c_z, H=H, c=c, dtype=dtype, seed=seed,
                       structured=structured, copies=copies)


def sample_rows(I: int, count: int, boundaries=(), seed: int = 0):
    """Query rows for sampled parity at sizes the oracle cannot cover in full: first/last row,
    both sides of every given boundary, plus seeded random rows."""
    rows = {0, I - 1}
    for b in boundaries:
        for r in (b - 1, b):
            if 0 <= r < I:
                rows.add(int(r))
    g = _gen(seed + 99, "cpu")
    while len(rows) < min(count, I):
        rows.add(int(torch.randint(0, I, (1,), generator=g)))
    return sorted(rows)


# ------------------------------------------------------------------ sparse k-neighbour atom attention
def make_atom_coords(cfg: LayerConfig, device="cpu") -> torch.Tensor:
    """Synthetic atom coordinates [L, 3] (fp32) of an icosahedral-shaped assembly: one ASU chain drawn as a
    self-avoiding-ish random walk (1.5 A steps), copied `copies` times with seeded random rotations and centres on
    a sphere whose radius keeps neighbouring copies in contact.  Input recipe only (stands in for the noised
    coordinates X^(t) of PAPER.md:303); nothing of the method's arithmetic."""
    g = _gen(cfg.seed * 1000003 + 5, "cpu")
    n = cfg.n_res if cfg.structured else cfg.I
    copies = cfg.copies if cfg.structured else 1
    steps = torch.randn(n, 3, generator=g, dtype=torch.float32)
    steps = 1.5 * steps / steps.norm(dim=1, keepdim=True)
    asu = torch.cumsum(steps, dim=0)
    asu = asu - asu.mean(dim=0, keepdim=True)
    rad = float(asu.norm(dim=1).max())
    out = []
    for _ in range(copies):
        qm, _r = torch.linalg.qr(torch.randn(3, 3, generator=g, dtype=torch.float32))
        ctr = torch.randn(3, generator=g, dtype=torch.float32)
        ctr = ctr / ctr.norm() * (rad * math.sqrt(copies) / 2.0 if copies > 1 else 0.0)
        out.append(asu @ qm.T + ctr)
    return torch.cat(out, dim=0).to(device).contiguous()


def make_atom_topology(cfg: LayerConfig, device="cpu", atoms_per_residue: int = 8):
    """(residue_id, chain_id, n_chains): the [L] int32 token and chain assignments of the synthetic assembly (the inputs
    PAPER.md:454 names) -- every ASU copy is one chain, `atoms_per_residue` consecutive atoms form a residue, residue ids
    run on across chains (global token index).  Unstructured configs: one chain."""
    L = cfg.I
    a = torch.arange(L, dtype=torch.int32)
    n = cfg.n_res if cfg.structured else L
    residue_id = (a // atoms_per_residue).to(torch.int32)
    chain_id = (a // n).to(torch.int32) if cfg.structured else torch.zeros(L, dtype=torch.int32)
    return residue_id.to(device).contiguous(), chain_id.to(device).contiguous(), (cfg.copies if cfg.structured else 1)


def make_p_slice(cfg: LayerConfig, idx: torch.Tensor, device="cpu", noise: float = 0.1, chunk: int = 4096) -> torch.Tensor:
    """Pair features of the listed neighbours, p_slice[l, j] = P[l, idx[l, j]] with the same recipe as the dense
    pair tensor (E[copy, copy] + R[atom, atom] + 0.1 N(0, 1)), built directly in slice form [L, k, c_z]."""
    L, k = idx.shape
    out = torch.empty(L, k, cfg.c_z, dtype=torch_dtype(cfg.dtype), device=device)
    if not cfg.structured:
        g = _gen(cfg.seed * 1000003 + 6, device)
        out.copy_(torch.randn(L, k, cfg.c_z, generator=g, device=device, dtype=torch.float32))
        return out
    n = cfg.n_res
    E, R = _tables(cfg, device)
    for r, i0 in enumerate(range(0, L, chunk)):
        i1 = min(L, i0 + chunk)
        rows = torch.arange(i0, i1, device=device)
        m = idx[i0:i1].long().clamp(min=0)
        blk = E[(rows // n)[:, None], m // n] + R[(rows % n)[:, None], m % n]
        g = _gen(cfg.seed * 1000003 + 2000 + r, device)
        blk += noise * torch.randn(i1 - i0, k, cfg.c_z, generator=g, device=device, dtype=torch.float32)
        out[i0:i1] = blk.to(out.dtype)
    return out


# ------------------------------------------------------------------ LayerNorm edge cases (per-pair affine shifts)
def affine_pairs(z: torch.Tensor, a: float, t: float, seed: int = 0, n_const: int = 0) -> torch.Tensor:
    """Edge-case inputs for the pair LayerNorm: every pair (leading dims of z; the last dim is the channel axis) becomes
    a * z + t_pair * 1 with t_pair = +-|t| * U(0.5, 1) (seeded sign and magnitude), computed in fp32 and rounded once to
    z's dtype; `n_const` seeded pairs are then overwritten by a constant across channels (variance exactly 0).
    LayerNorm is invariant under such a map up to the epsilon term and the storage rounding ("LN axis
    and affine"), so the layer's output barely moves while |mean| / sigma of a pair grows to |t| / (1.4 a)."""
    g = _gen(seed * 7919 + 3, "cpu")
    lead = z.shape[:-1]
    n = int(torch.tensor(lead).prod()) if len(lead) else 1
    sign = torch.where(torch.rand(n, generator=g) < 0.5, -1.0, 1.0)
    mag = 0.5 + 0.5 * torch.rand(n, generator=g)
    tp = (float(t) * sign * mag).reshape(*lead, 1).to(z.device)
    out = (float(a) * z.float() + tp).to(z.dtype)
    if n_const > 0:
        flat = out.reshape(n, z.shape[-1])
        pick = torch.randperm(n, generator=g)[:min(n_const, n)].to(z.device)
        flat[pick] = flat[pick][:, :1].expand(-1, z.shape[-1]).clone()
        out = flat.reshape(z.shape)
    return out.contiguous()
