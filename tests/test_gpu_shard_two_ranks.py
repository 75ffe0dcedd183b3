"""SURVEY 8(e) end to end on the GPU with TWO ranks: two processes (gloo process group, both on cuda:0 -- there is
one GPU here; the ranks only meet in the host-side all-reduce, no kernel waits on another) run shard.sharded_step
on the same catalogue; the reduced outputs must equal the single-process run exactly in N and n_kept and to
rounding in S, W, Dn, Wd, and the divided xi / D must match the oracle."""
import os
import socket

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

pytestmark = pytest.mark.gpu


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, q):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    from paper_2507_00129_b200 import binding as B, gen, shard
    f = gen.make_config(4, n_forest=700, density_scale=2.0)
    ctx = B.Context("cuda:0")
    d = B.DeviceForests(f)
    r = shard.sharded_step(ctx, d, B.binning(), 0.9, gen.mask_seed(4), rank, world)
    out = {k: r[k].cpu().numpy() for k in ("S", "W", "N", "xi", "Dn", "Wd", "D")}
    out["n_kept"] = r["n_kept"]
    out["own_pairs"] = r["stats_xi"]["n_forest_pairs"]
    q.put((rank, out))
    dist.barrier()
    ctx.close()
    dist.destroy_process_group()


def test_two_ranks_one_catalogue():
    if not torch.cuda.is_available():
        pytest.skip("needs a GPU")
    from paper_2507_00129_b200 import binding as B, build, gen, shard
    from oracle import oracle as orc
    build.build()
    c = mp.get_context("spawn")
    q = c.Queue()
    port = _free_port()
    procs = [c.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    res = dict(q.get(timeout=600) for _ in range(2))
    for p in procs:
        p.join(timeout=120)
        assert p.exitcode == 0
    f = gen.make_config(4, n_forest=700, density_scale=2.0)
    ctx = B.Context("cuda:0")
    one = shard.sharded_step(ctx, B.DeviceForests(f), B.binning(), 0.9, gen.mask_seed(4), 0, 1)
    a, b = res[0], res[1]
    assert a["own_pairs"] + b["own_pairs"] == one["stats_xi"]["n_forest_pairs"] and min(a["own_pairs"], b["own_pairs"]) > 0
    for k in ("S", "W", "N", "xi", "Dn", "Wd", "D"):
        assert np.array_equal(a[k], b[k]), k                               # every rank holds the same reduced result
    assert np.array_equal(a["N"], one["N"].cpu().numpy()) and a["n_kept"] == one["n_kept"]
    assert np.allclose(a["S"], one["S"].cpu().numpy(), rtol=0, atol=1e-11 * np.abs(a["S"]).max())
    assert np.allclose(a["W"], one["W"].cpu().numpy(), rtol=1e-12)
    assert np.allclose(a["Dn"], one["Dn"].cpu().numpy(), rtol=0, atol=1e-11 * np.abs(a["Dn"]).max())
    ref = orc.pairs_window(f)
    od = orc.dmat(f, ref, 0.9, gen.mask_seed(4))
    ox = orc.xi(f, ref)
    assert np.array_equal(a["N"].view(np.uint64), ox["N"]) and a["n_kept"] == od["n_kept"]
    assert np.all(np.abs(a["D"] - od["D"]) <= 1e-7 * np.maximum(np.abs(od["D"]), 1e-6))
    nz = ox["W"] > 0
    assert np.all(np.abs(a["xi"][nz] - ox["xi"][nz]) <= 1e-9 * np.maximum(np.abs(ox["xi"][nz]), 1e-4 * ox["Sabs"][nz] / ox["W"][nz]))
    ctx.close()
