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


# ---------------------------------------------------------------- section 8(e): one catalogue, split list
def _split_worker(rank, world, port, q):
    import numpy as np
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    from oracle import oracle as orc
    from paper_2507_00129_b200 import gen, shard
    f = gen.make_config(1, n_forest=220, density_scale=3.0)          # the SAME catalogue on every rank
    cat = orc.Catalogue(f)
    pq = orc.pairs_window(cat)
    lens = torch.from_numpy(np.diff(f.pix_off))
    mine = shard.split_pairs(torch.from_numpy(pq), lens, rank, world).numpy()
    seed = gen.mask_seed(1)
    x = orc.xi(cat, mine)
    d = orc.dmat(cat, mine, 0.9, seed, want_D=False)
    S, W = torch.from_numpy(x["S"]), torch.from_numpy(x["W"])
    N = torch.from_numpy(x["N"].view(np.int64).copy())
    Dn, Wd = torch.from_numpy(d["Dn"]), torch.from_numpy(d["Wd"])
    nk = torch.tensor([d["n_kept"]], dtype=torch.int64)
    shard.allreduce_sum(S, W, N, Dn, Wd, nk)
    # reference: the un-split list on this rank
    x0 = orc.xi(cat, pq)
    d0 = orc.dmat(cat, pq, 0.9, seed, want_D=False)
    ok_N = bool(np.array_equal(N.numpy().view(np.uint64), x0["N"]))
    errS = float(np.max(np.abs(S.numpy() - x0["S"]) / np.maximum(np.abs(x0["S"]), 1e-4 * x0["Sabs"] + 1e-300)))
    errW = float(np.max(np.abs(W.numpy() - x0["W"]) / np.maximum(x0["W"], 1e-300)))
    errD = float(np.max(np.abs(Dn.numpy() - d0["Dn"])) / np.max(np.abs(d0["Dn"])))
    errWd = float(np.max(np.abs(Wd.numpy() - d0["Wd"]) / np.maximum(d0["Wd"], 1e-300)))
    cost = (lens[mine[:, 0]] * lens[mine[:, 1]]).sum().item() if len(mine) else 0
    q.put((rank, len(mine), len(pq), cost, ok_N, errS, errW, errD, errWd, int(nk[0]), d0["n_kept"]))
    dist.barrier()
    dist.destroy_process_group()


def test_world_size_2_split_list_and_allreduce():
    """chunks are disjoint, cover the list and are balanced by sum n_p n_q; after ONE
    all_reduce(SUM) N and n_kept equal the un-split values exactly and S, W, Dn, Wd to 1e-12."""
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_split_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    out = sorted(q.get(timeout=300) for _ in range(2))
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    n_total = out[0][2]
    assert out[0][1] + out[1][1] == n_total and min(out[0][1], out[1][1]) > 0
    c0, c1 = out[0][3], out[1][3]
    assert abs(c0 - c1) <= 0.02 * (c0 + c1)                     # balanced by visited pixel pairs
    for r in out:
        assert r[4], "N after the all-reduce differs from the un-split N"
        assert r[5] <= 1e-12 and r[6] <= 1e-12 and r[7] <= 1e-12 and r[8] <= 1e-12, r
        assert r[9] == r[10]                                    # n_kept independent of the split


def test_chunk_bounds_properties():
    from paper_2507_00129_b200 import shard
    g = torch.Generator().manual_seed(3)
    cost = torch.randint(0, 5000, (10007,), generator=g)
    for world in (1, 2, 3, 8):
        b = shard.chunk_bounds(cost, world)
        assert b[0] == 0 and b[-1] == len(cost) and all(b[i] <= b[i + 1] for i in range(world))
        sums = [int(cost[b[i]:b[i + 1]].sum()) for i in range(world)]
        assert sum(sums) == int(cost.sum()) and max(sums) - min(sums) <= 2 * 5000
    assert shard.chunk_bounds(torch.zeros(0, dtype=torch.int64), 4) == [0] * 5
    z = shard.chunk_bounds(torch.zeros(10, dtype=torch.int64), 2)        # all-zero cost: split by count
    assert z == [0, 5, 10]
