"""Shared helpers for the GPU parity tests: marshal the exact stored bits to the fp64 oracle."""
import numpy as np
import torch

import dcp_synth as syn
from oracle import pair_bias_attention as orc

# BASELINE.json tolerances (north_star): fp32 max-abs <= 1e-5; bf16 rel-L2 <= 1e-2 and max-abs <= 2e-2
TOL_F32_MAXABS = 1e-5
TOL_BF16_RELL2 = 1e-2
TOL_BF16_MAXABS = 2e-2


def np64(t: torch.Tensor) -> np.ndarray:
    return t.detach().float().cpu().double().numpy()


def np32(t: torch.Tensor) -> np.ndarray:
    return t.detach().float().cpu().numpy()


def weights_np(w):
    return {k: np64(v) for k, v in w.items()}


def make_problem(cfg, device, with_ln_s=False, with_b_q=False):
    w = syn.make_weights(cfg, device, with_ln_s=with_ln_s, with_b_q=with_b_q)
    s = syn.make_s(cfg, device)
    z = syn.make_z(cfg, device)
    return s, z, w


def oracle_rows(cfg, s, z, w, rows):
    """fp64 oracle on the exact stored bits, for the given query rows (reads back only z[rows])."""
    rows = list(rows)
    idx = torch.as_tensor(rows, device=z.device)
    z_rows = np32(z.index_select(0, idx))
    return orc.pair_bias_attention_rows(np64(s), z_rows, rows, weights_np(w), cfg.H, cfg.c)


def check_close(out: torch.Tensor, ref: np.ndarray, dtype: str, what: str = ""):
    got = np64(out)
    err = np.abs(got - ref)
    maxabs = float(err.max())
    rel = float(np.linalg.norm(got - ref) / max(np.linalg.norm(ref), 1e-300))
    assert np.all(np.isfinite(got)), f"{what}: non-finite output"
    if dtype == "f32":
        assert maxabs <= TOL_F32_MAXABS, f"{what}: max-abs {maxabs:.3e} > {TOL_F32_MAXABS}"
    else:
        assert rel <= TOL_BF16_RELL2, f"{what}: rel-L2 {rel:.3e} > {TOL_BF16_RELL2}"
        assert maxabs <= TOL_BF16_MAXABS, f"{what}: max-abs {maxabs:.3e} > {TOL_BF16_MAXABS}"
    return maxabs, rel


def neighbour_lists(cfg, k, device):
    """Neighbour lists [L, k] int32 for the sparse-attention tests: the structured budget of the synthetic
    assembly's coordinates, built by the library's own dcp_knn_budget (itself bit-exact against oracle/knn_budget.py,
    tests/test_gpu_knn.py).  They are INPUTS of the attention under test: its oracle receives the same lists."""
    import paper_2607_05439_b200 as dcp
    x = syn.make_atom_coords(cfg, device)
    rid, cid, n_chains = syn.make_atom_topology(cfg, device)
    return dcp.dcp_knn_budget(x, rid, cid, min(k, cfg.I), n_chains)
