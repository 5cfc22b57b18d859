"""GPU parity of dcp_knn against the oracle: index work, so BIT-EXACT."""
import numpy as np
import pytest
import torch

import dcp_synth as syn
from oracle import knn as ko

pytestmark = pytest.mark.gpu
DEV = "cuda:0"


def _dcp():
    import paper_2607_05439_b200 as dcp
    return dcp


@pytest.mark.parametrize("L,k", [(1, 1), (33, 33), (100, 7), (257, 32), (300, 128), (700, 160), (1000, 512), (64, 1)])
def test_knn_random_points_bit_exact(L, k):
    dcp = _dcp()
    g = torch.Generator(device="cpu").manual_seed(1000 + L)
    x = (torch.randn(L, 3, generator=g) * 9).to(DEV)
    got = dcp.dcp_knn(x, k).cpu().numpy()
    assert np.array_equal(got, ko.knn(x.cpu().numpy(), k))


def test_knn_ties_and_duplicates():
    """Integer lattice (many exactly equal distances) and duplicated points: order = (distance, index)."""
    dcp = _dcp()
    g = torch.Generator(device="cpu").manual_seed(7)
    x = torch.randint(0, 4, (500, 3), generator=g).float().to(DEV)     # 64 distinct sites, heavy ties
    got = dcp.dcp_knn(x, 96).cpu().numpy()
    assert np.array_equal(got, ko.knn(x.cpu().numpy(), 96))


def test_knn_dense_cluster_takes_the_exact_fallback():
    """3000 coincident points + a few others: far more than the select kernel's candidate buffer lie within the
    threshold, so every query takes the insertion fallback; the order is then purely by index."""
    dcp = _dcp()
    x = torch.zeros(3100, 3)
    x[3000:] = torch.arange(100, dtype=torch.float32)[:, None] + 5.0
    x = x.to(DEV)
    got = dcp.dcp_knn(x, 128).cpu().numpy()
    assert np.array_equal(got, ko.knn(x.cpu().numpy(), 128))
    assert np.array_equal(got[7], np.arange(128))


def test_knn_structured_atoms_sampled_rows():
    """C4's synthetic assembly (L = 24000), k = 128: sampled queries against the oracle, and against the torch
    cdist + topk lists the input generator builds (same sets wherever no near-tie decides)."""
    dcp = _dcp()
    cfg = syn.CONFIGS["C4"]
    x = syn.make_atom_coords(cfg, DEV)
    got = dcp.dcp_knn(x, 128)
    rows = syn.sample_rows(cfg.I, 300, boundaries=[400, 12000], seed=2)
    ref = ko.knn_rows(x.cpu().numpy(), 128, rows)
    assert np.array_equal(got[torch.as_tensor(rows, device=DEV)].cpu().numpy(), ref)
    assert torch.equal(got[:, 0].cpu(), torch.arange(cfg.I, dtype=torch.int32))
    again = dcp.dcp_knn(x, 128)
    assert torch.equal(got, again)


def test_knn_error_paths():
    dcp = _dcp()
    x = torch.zeros(10, 3, device=DEV)
    for k in (0, 11):
        with pytest.raises(dcp.DcpError) as e:
            dcp.dcp_knn(x, k)
        assert e.value.status == 1
    xl = torch.zeros(600, 3, device=DEV)
    with pytest.raises(dcp.DcpError) as e:
        dcp.dcp_knn(xl, 513)
    assert e.value.status == 2
