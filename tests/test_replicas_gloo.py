"""N > 1 path of bench.py ("replicas only") on CPU: world_size 2, gloo.

Each rank gets its own seed (independent replica inputs), the reported time is the max over ranks, and the
whole-job value counts every rank's pairs.  The oracle stands in for the layer here (test infrastructure; no GPU)."""
import os
import socket
import sys

import numpy as np
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, q):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    import bench
    import dcp_synth as syn
    from oracle import pair_bias_attention as orc
    cfg = bench.replica_config(syn.small_config("rep", I=24, c_s=16, c_z=8, H=2, c=8, seed=5), rank, world)
    w = syn.make_weights(cfg, "cpu")
    s = syn.make_s(cfg, "cpu")
    z = syn.make_z(cfg, "cpu")
    f64 = lambda t: t.double().numpy()
    out = orc.pair_bias_attention(f64(s), z.float().numpy(), {k: f64(v) for k, v in w.items()}, cfg.H, cfg.c)
    my_ms = 10.0 * (rank + 1)                       # rank 1 is the slow one
    ms = bench.max_over_ranks_ms(my_ms, world, "cpu")
    dist.barrier()
    q.put((rank, cfg.seed, float(np.abs(out).sum()), ms, bench.aggregate_gpairs(cfg.I, 3, world, ms)))
    dist.destroy_process_group()


def test_replicas_world2_gloo():
    world, port = 2, _free_port()
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=_worker, args=(r, world, port, q)) for r in range(world)]
    for p in procs:
        p.start()
    res = sorted(q.get(timeout=120) for _ in range(world))
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    (r0, seed0, sum0, ms0, v0), (r1, seed1, sum1, ms1, v1) = res
    assert seed1 == seed0 + 1000 and sum0 != sum1          # independent replicas: different inputs, different outputs
    assert ms0 == ms1 == 20.0                               # max over ranks, identical on every rank
    assert v0 == v1 == 24.0 * 24 * 3 * 2 / 20e-3 / 1e9     # whole-job pairs / max time


def test_single_rank_is_identity():
    import bench
    import dcp_synth as syn
    cfg = syn.small_config("rep", I=24, c_s=16, c_z=8, H=2, c=8, seed=5)
    assert bench.replica_config(cfg, 0, 1) is cfg
    assert bench.max_over_ranks_ms(3.5, 1, "cpu") == 3.5
