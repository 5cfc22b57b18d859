"""GPU parity of the pairwise SwiGLU transition (Eq. 6 / Algorithm 1) against the
fp64 oracle, through the C ABI.  bf16 storage: rel-L2 <= 1e-2 (BASELINE.json's bf16 bound) and, because the output is
z + update rounded to bf16 (half an ulp = 2^-9 |out|), elementwise |got - ref| <= 2e-2 + 2^-8 |ref|."""
import math

import numpy as np
import pytest
import torch

from oracle import pair_transition as pto
from tests import util

pytestmark = pytest.mark.gpu
DEV = "cuda:0"
C_Z = 128


def _dcp():
    import paper_2607_05439_b200 as dcp
    return dcp


def _weights(seed):
    g = torch.Generator(device="cpu").manual_seed(seed)
    n = lambda *s, std=1.0: (torch.randn(*s, generator=g) * std).to(torch.bfloat16).to(DEV)
    return (n(C_Z, 4 * C_Z, std=1 / math.sqrt(C_Z)), n(C_Z, 4 * C_Z, std=1 / math.sqrt(C_Z)),
            n(4 * C_Z, C_Z, std=1 / math.sqrt(4 * C_Z)), (1 + 0.1 * torch.randn(C_Z, generator=g)).to(torch.bfloat16).to(DEV),
            (0.1 * torch.randn(C_Z, generator=g)).to(torch.bfloat16).to(DEV))


def _check(got, z, w, what):
    ref = pto.pair_transition(util.np64(z), *[util.np64(t) for t in w])
    g = util.np64(got)
    assert np.all(np.isfinite(g)), what
    rel = np.linalg.norm(g - ref) / np.linalg.norm(ref)
    assert rel <= 1e-2, f"{what}: rel-L2 {rel:.3e}"
    assert np.all(np.abs(g - ref) <= 2e-2 + 2.0 ** -8 * np.abs(ref)), f"{what}: max-abs {np.abs(g - ref).max():.3e}"
    # the update itself (out - z) is what the kernel computes: it must carry signal, not just the residual
    upd_ref = ref - util.np64(z)
    upd = g - util.np64(z)
    assert np.linalg.norm(upd - upd_ref) / np.linalg.norm(upd_ref) <= 5e-2, what


@pytest.mark.parametrize("n_pairs", [1, 127, 128, 129, 1000, 148 * 128 * 2 + 77])
def test_transition_shapes(n_pairs):
    dcp = _dcp()
    g = torch.Generator(device="cpu").manual_seed(n_pairs)
    z = (torch.randn(n_pairs, C_Z, generator=g) * 1.4 + 0.2).to(torch.bfloat16).to(DEV)
    w = _weights(7)
    out = dcp.dcp_pair_transition(z, *w)
    _check(out, z, w, f"transition n_pairs={n_pairs}")
    again = dcp.dcp_pair_transition(z, *w)
    assert torch.equal(out, again)


def test_transition_in_place_and_3d():
    dcp = _dcp()
    import dcp_synth as syn
    cfg = syn.small_config("tr", I=120, c_s=64, c_z=C_Z, H=16, c=24, dtype="bf16", seed=3, structured=True, copies=60)
    z = syn.make_z(cfg, DEV)                                  # [I, I, c_z], icosahedral-structured values
    w = _weights(11)
    out = dcp.dcp_pair_transition(z, *w)
    _check(out.reshape(-1, C_Z), z.reshape(-1, C_Z), w, "transition [I, I, c_z]")
    zc = z.clone()
    dcp.dcp_pair_transition(zc, *w, out=zc)                   # in place
    assert torch.equal(zc, out)


def test_transition_special_weights():
    dcp = _dcp()
    g = torch.Generator(device="cpu").manual_seed(5)
    z = torch.randn(300, C_Z, generator=g).to(torch.bfloat16).to(DEV)
    w1, w2, w3, gamma, beta = _weights(13)
    assert torch.equal(dcp.dcp_pair_transition(z, w1, w2, torch.zeros_like(w3), gamma, beta), z)     # W3 = 0
    assert torch.equal(dcp.dcp_pair_transition(z, torch.zeros_like(w1), w2, w3, gamma, beta), z)     # SiLU(0) = 0


def test_transition_error_paths():
    dcp = _dcp()
    z = torch.zeros(10, 64, dtype=torch.bfloat16, device=DEV)
    w = _weights(1)
    with pytest.raises(dcp.DcpError) as e:
        dcp.dcp_pair_transition(z, *w)
    assert e.value.status == 2
    with pytest.raises(dcp.DcpError) as e:
        dcp.dcp_pair_transition(torch.zeros(10, C_Z, device=DEV), *[t.float() for t in w])
    assert e.value.status == 2


def test_transition_full_size_sampled():
    """C2's pair tensor (I = 3000, 9.0 M pairs), the launch configuration bench.py --workload T2 times: sampled pairs
    (first / last, both sides of tile and CTA-pair boundaries, seeded random ones) against the oracle, in place."""
    dcp = _dcp()
    import dcp_synth as syn
    cfg = syn.CONFIGS["C2"]
    z = syn.make_z(cfg, DEV)
    w = _weights(11)
    n_pairs = cfg.I * cfg.I
    g = torch.Generator(device="cpu").manual_seed(5)
    idx = torch.cat([torch.tensor([0, 1, 127, 128, 129, 255, 256, 148 * 128 - 1, 148 * 128, 148 * 128 + 1, n_pairs - 129,
                                   n_pairs - 128, n_pairs - 2, n_pairs - 1]),
                     torch.randint(0, n_pairs, (4000,), generator=g)]).to(DEV)
    zs = z.reshape(-1, C_Z).index_select(0, idx)
    dcp.dcp_pair_transition(z, *w, out=z)
    torch.cuda.synchronize()
    _check(z.reshape(-1, C_Z).index_select(0, idx), zs, w, "transition I=3000 sampled")
