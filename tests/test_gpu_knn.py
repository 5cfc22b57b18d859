"""GPU parity of dcp_knn and dcp_knn_budget against their oracles: index
work, so BIT-EXACT."""
import numpy as np
import pytest
import torch

import dcp_synth as syn
from oracle import knn as ko
from oracle import knn_budget as kbo

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


def test_knn_dense_cluster_tightens_the_threshold():
    """A cluster of 1500 distinct points far denser than the queries' own tile: the bound from the own tile lets the whole
    cluster through, the candidate buffer (512) would overflow, and the kernel re-derives the bound from the buffer
    instead of falling back.  Queries inside the cluster, next to it and far from it."""
    dcp = _dcp()
    g = torch.Generator(device="cpu").manual_seed(11)
    x = torch.rand(9000, 3, generator=g) * 100.0
    centre = torch.tensor([50.0, 50.0, 50.0])
    x[4000:5500] = centre + (torch.rand(1500, 3, generator=g) - 0.5) * 2.0
    x[5] = centre
    x[6] = centre + 3.0
    x = x.to(DEV)
    for k in (128, 256, 40):
        got = dcp.dcp_knn(x, k).cpu().numpy()
        rows = [5, 6, 7, 100, 2047, 2048, 4000, 4700, 5499, 5500, 8999]
        assert np.array_equal(got[rows], ko.knn_rows(x.cpu().numpy(), k, rows))


def test_knn_structured_atoms_sampled_rows():
    """C4's synthetic assembly (L = 24000), k = 128: sampled queries against the oracle."""
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


# ------------------------------------------------------------------ the structured budget
def _topology(L, n_chains, atoms_per_residue, seed):
    g = torch.Generator(device="cpu").manual_seed(seed)
    cid = torch.sort(torch.randint(0, n_chains, (L,), generator=g)).values.to(torch.int32)
    rid = (torch.arange(L) // atoms_per_residue).to(torch.int32)
    return rid, cid, int(torch.unique(cid).numel())


@pytest.mark.parametrize("L,k,n_chains,apr,n_seq", [
    (300, 128, 6, 8, 2),      # the paper's defaults: k = 128, n_seq = 2, more than three chains: both quotas live
    (300, 128, 3, 8, 2),      # three chains: no split
    (200, 48, 5, 4, 2),       # q_out = 32 of 48
    (150, 33, 4, 5, 1),       # own residue only
    (257, 40, 7, 3, 0),       # no sequence-local atoms
    (90, 8, 5, 6, 2),         # the sequence-local set alone exceeds k; q_out = k - 1
    (64, 64, 4, 4, 2),        # k = L
    (700, 300, 9, 10, 2),     # NR = 16 lists
    (1000, 512, 5, 8, 2),     # the largest budget
    (40, 1, 4, 4, 2),         # k = 1: the query itself
    (5000, 128, 12, 8, 2),    # select kernel, 256-entry buffers re-bounded many times
    (3000, 200, 8, 8, 2),     # select kernel with 512-entry buffers
    (2500, 256, 3, 8, 2),     # no split, k = 256
])
def test_knn_budget_bit_exact(L, k, n_chains, apr, n_seq):
    dcp = _dcp()
    g = torch.Generator(device="cpu").manual_seed(2000 + L + k)
    x = (torch.randn(L, 3, generator=g) * 6)
    rid, cid, nch = _topology(L, n_chains, apr, L + k)
    got = dcp.dcp_knn_budget(x.to(DEV), rid.to(DEV), cid.to(DEV), k, nch, n_seq=n_seq).cpu().numpy()
    ref = kbo.knn_budget(x.numpy(), rid.numpy(), cid.numpy(), k, n_seq=n_seq)
    assert np.array_equal(got, ref)


def test_knn_budget_ties_and_short_chains():
    """Integer lattice (exact ties everywhere), one chain of 5 atoms and one of 2 among six: order = (distance, index)."""
    dcp = _dcp()
    g = torch.Generator(device="cpu").manual_seed(9)
    L = 400
    x = torch.randint(0, 4, (L, 3), generator=g).float()
    cid = torch.cat([torch.full((5,), 0), torch.full((2,), 1), torch.full((150,), 2), torch.full((100,), 3),
                     torch.full((100,), 4), torch.full((43,), 5)]).to(torch.int32)
    rid = (torch.arange(L) // 7).to(torch.int32)
    for k, n_seq in ((96, 2), (40, 1), (400, 2)):
        got = dcp.dcp_knn_budget(x.to(DEV), rid.to(DEV), cid.to(DEV), k, 6, n_seq=n_seq).cpu().numpy()
        assert np.array_equal(got, kbo.knn_budget(x.numpy(), rid.numpy(), cid.numpy(), k, n_seq=n_seq))


def test_knn_budget_interleaved_chains_and_clustered_space():
    """Chain and residue ids that are NOT contiguous in index (every 128-atom chunk straddles chains: the chunk test can
    neither skip on ids nor count whole chunks) over spatially clustered atoms (chunks far from a query are skipped on
    distance), L not a multiple of 128 or of the tile."""
    dcp = _dcp()
    g = torch.Generator(device="cpu").manual_seed(31)
    L = 4500
    centres = torch.rand(36, 3, generator=g) * 200.0
    x = centres[torch.arange(L) // 125] + torch.randn(L, 3, generator=g) * 3.0          # coherent in index, like an assembly
    cid = torch.randint(0, 7, (L,), generator=g).to(torch.int32)                        # interleaved chains
    rid = torch.randint(0, 40, (L,), generator=g).to(torch.int32)                       # arbitrary residue ids
    for k, n_seq in ((128, 2), (64, 1), (200, 2)):
        got = dcp.dcp_knn_budget(x.to(DEV), rid.to(DEV), cid.to(DEV), k, 7, n_seq=n_seq).cpu().numpy()
        rows = list(range(0, L, 97)) + [L - 1, 2047, 2048, 4095, 4096]
        assert np.array_equal(got[rows], kbo.knn_budget_rows(x.numpy(), rid.numpy(), cid.numpy(), k, rows, n_seq=n_seq))
    # the same atoms with contiguous chains: whole chunks are counted without a scan
    cid2 = (torch.arange(L) // 700).to(torch.int32)
    rid2 = (torch.arange(L) // 9).to(torch.int32)
    got = dcp.dcp_knn_budget(x.to(DEV), rid2.to(DEV), cid2.to(DEV), 128, 7, n_seq=2).cpu().numpy()
    rows = list(range(0, L, 61)) + [L - 1]
    assert np.array_equal(got[rows], kbo.knn_budget_rows(x.numpy(), rid2.numpy(), cid2.numpy(), 128, rows, n_seq=2))
    # and the plain lists on the clustered cloud (chunk skipping in knn_select_kernel)
    gk = dcp.dcp_knn(x.to(DEV), 128).cpu().numpy()
    assert np.array_equal(gk[rows], ko.knn_rows(x.numpy(), 128, rows))


def test_knn_budget_coincident_atoms_take_the_exact_fallback():
    """900 coincident atoms spread over four chains (+ a few others): more entries tie within a class bound than a
    candidate buffer holds, so the queries take the register-list fallback; order = (flag, distance, index)."""
    dcp = _dcp()
    L = 1000
    x = torch.zeros(L, 3)
    x[900:] = torch.arange(100, dtype=torch.float32)[:, None] * 0.5 + 2.0
    cid = (torch.arange(L) // 250).to(torch.int32)
    rid = (torch.arange(L) // 6).to(torch.int32)
    for k in (128, 200):
        got = dcp.dcp_knn_budget(x.to(DEV), rid.to(DEV), cid.to(DEV), k, 4, n_seq=2).cpu().numpy()
        assert np.array_equal(got, kbo.knn_budget(x.numpy(), rid.numpy(), cid.numpy(), k, n_seq=2))


def test_knn_budget_reduces_to_plain_knn_on_the_device():
    dcp = _dcp()
    g = torch.Generator(device="cpu").manual_seed(4)
    x = (torch.randn(500, 3, generator=g) * 5).to(DEV)
    rid = (torch.arange(500) // 8).to(torch.int32).to(DEV)
    cid = (torch.arange(500) // 200).to(torch.int32).to(DEV)          # three chains
    assert torch.equal(dcp.dcp_knn_budget(x, rid, cid, 100, 3, n_seq=0), dcp.dcp_knn(x, 100))


def test_knn_budget_structured_atoms_sampled_rows():
    """C4's synthetic assembly (L = 24000: 60 chains of 400 atoms, 8 atoms per residue), the paper's k = 128, n_seq = 2:
    sampled queries bit-exact against the oracle; every list keeps >= 32 atoms of other chains."""
    dcp = _dcp()
    cfg = syn.CONFIGS["C4"]
    x = syn.make_atom_coords(cfg, DEV)
    rid, cid, nch = syn.make_atom_topology(cfg, DEV)
    got = dcp.dcp_knn_budget(x, rid, cid, 128, nch)
    rows = syn.sample_rows(cfg.I, 300, boundaries=[400, 12000], seed=2)
    ref = kbo.knn_budget_rows(x.cpu().numpy(), rid.cpu().numpy(), cid.cpu().numpy(), 128, rows)
    assert np.array_equal(got[torch.as_tensor(rows, device=DEV)].cpu().numpy(), ref)
    foreign = (cid[got.long()] != cid[:, None]).sum(dim=1)
    assert int(foreign.min()) >= 32
    assert torch.equal(got[:, 0].cpu(), torch.arange(cfg.I, dtype=torch.int32))
    assert torch.equal(got, dcp.dcp_knn_budget(x, rid, cid, 128, nch))


def test_knn_budget_error_paths():
    dcp = _dcp()
    x = torch.zeros(10, 3, device=DEV)
    z = torch.zeros(10, dtype=torch.int32, device=DEV)
    for k, n_seq, nch in ((0, 2, 1), (11, 2, 1), (4, -1, 1), (4, 2, 0)):
        with pytest.raises(dcp.DcpError) as e:
            dcp.dcp_knn_budget(x, z, z, k, nch, n_seq=n_seq)
        assert e.value.status == 1
