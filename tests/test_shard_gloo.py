"""N > 1 plumbing on CPU: world_size-2 gloo process group."""
import os
import socket

import torch
import torch.distributed as dist
import torch.multiprocessing as mp


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, q):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    from paper_2507_00129_b200 import gen, shard
    # every rank builds its own shaped catalogue (independent seeds), as bench.py does
    seed = shard.rank_seed(gen.SEED_BASE + 1, rank)
    f = gen.make_config(1, n_forest=200, seed=seed)
    ms = 10.0 * (rank + 1)               # rank 1 is the slow one
    units = float(f.n_pix)
    m, u = shard.aggregate(ms, units)
    v = shard.throughput(ms, units)
    q.put((rank, f.n_pix, float(f.chi[0]), m, u, v))
    dist.barrier()
    dist.destroy_process_group()


def test_world_size_2_weak_scaling_aggregation():
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    out = sorted(q.get(timeout=120) for _ in range(2))
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    (r0, n0, c0, m0, u0, v0), (r1, n1, c1, m1, u1, v1) = out
    assert c0 != c1                                  # independent catalogues
    assert m0 == m1 == 20.0                          # max over ranks
    assert u0 == u1 == float(n0 + n1)                # whole-job units
    assert abs(v0 - (n0 + n1) / 20e-3) < 1e-6 and v0 == v1


def test_single_process_passthrough():
    from paper_2507_00129_b200 import shard
    assert shard.aggregate(5.0, 7.0) == (5.0, 7.0)
    assert shard.rank_seed(100, 0) is None and shard.rank_seed(100, 3) == 3100
