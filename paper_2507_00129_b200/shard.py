"""Multi-GPU plumbing of the hot path.

Forest pairs are independent units and every output is an additive accumulator before its final
division (S, W, N for xi; Dn, Wd, n_kept for D), so ONE catalogue shards over G ranks as the paper's
own work split does ("distribute the work load between different nodes", PAPER.md:134
two A100s): every rank holds the catalogue, takes one contiguous chunk of the forest-pair list
balanced by sum n_p n_q, runs lya_xi2pcf / lya_dmat on it, and ONE all-reduce(sum) of the numerators
follows; xi = S / W and D = Dn / Wd are taken AFTER the reduction (lya_xi_normalise,
lya_dmat_normalise).  The keep mask is keyed on pixel ids, so N and n_kept do not depend on G.

Nothing here touches the method's arithmetic: index slicing, torch.distributed collectives and the
(time, work) aggregation of the timing contract.  It works on any initialised process group (nccl
on GPUs, gloo on CPU -- the world_size-2 CPU test drives it with the oracle as the per-rank
compute).
"""
from __future__ import annotations


# ---------------------------------------------------------------- partition of the forest-pair list
def chunk_bounds(cost, world: int):
    """Boundaries k_0 = 0 <= k_1 <= ... <= k_world = n of `world` contiguous chunks of a list whose
    entries cost `cost[k]` (1-D integer torch tensor, any device), balanced by total cost: chunk r
    ends at the first entry where the running cost reaches (r + 1) / world of the total."""
    import torch
    n = int(cost.numel())
    if n == 0:
        return [0] * (world + 1)
    cum = torch.cumsum(cost.to(torch.int64), 0)
    total = int(cum[-1])
    targets = torch.tensor([(total * r) // world for r in range(1, world)], dtype=torch.int64, device=cum.device)
    cuts = torch.searchsorted(cum, targets, right=False).tolist() if world > 1 else []
    b = [0] + [min(int(c) + 1, n) if total > 0 else (n * (r + 1)) // world for r, c in enumerate(cuts)] + [n]
    for r in range(1, len(b)):                       # monotone
        b[r] = max(b[r], b[r - 1])
    return b


def split_pairs(pq, lens, rank: int, world: int):
    """Chunk `rank` of `world` of the forest-pair list pq (int tensor [n][2]); lens = pixels per
    forest (1-D integer tensor on pq's device).  The chunks are contiguous, disjoint, cover the
    list, and carry about equal sum n_p n_q."""
    if world == 1:
        return pq
    cost = lens[pq[:, 0].long()].to(pq.device).long() * lens[pq[:, 1].long()].to(pq.device).long()
    b = chunk_bounds(cost, world)
    return pq[b[rank]:b[rank + 1]]


# ---------------------------------------------------------------- collectives
def _dist():
    import torch.distributed as dist
    return dist if (dist.is_available() and dist.is_initialized() and dist.get_world_size() > 1) else None


def allreduce_sum(*tensors):
    """In-place all_reduce(SUM) of every tensor (fp64 numerators; int64 tensors carrying the u64
    pair counts -- two's-complement addition is the same operation).  No-op without a group."""
    dist = _dist()
    if dist is not None:
        for t in tensors:
            if t is not None:
                dist.all_reduce(t, op=dist.ReduceOp.SUM)
    return tensors


def rank_seed(base_seed: int, rank: int) -> int | None:
    """Catalogue seed of a rank for the independent-replica mode: rank 0 uses the config's own seed
    (None), others base + 1000 * rank."""
    return None if rank == 0 else int(base_seed) + 1000 * int(rank)


def aggregate(ms: float, units: float, device=None):
    """(max over ranks of ms, sum over ranks of units): the timing contract's reduction."""
    import torch
    dist = _dist()
    if dist is None:
        return float(ms), float(units)
    t = torch.tensor([float(ms), float(units)], dtype=torch.float64, device=device)
    tmax = t.clone()
    dist.all_reduce(tmax, op=dist.ReduceOp.MAX)
    tsum = t.clone()
    dist.all_reduce(tsum, op=dist.ReduceOp.SUM)
    return float(tmax[0]), float(tsum[1])


def throughput(ms: float, units: float, device=None) -> float:
    """Whole-job units per second: all ranks' units over the slowest rank's time."""
    m, u = aggregate(ms, units, device)
    return u / (m * 1e-3)


# ---------------------------------------------------------------- the sharded step (section 8(e))
def sharded_step(ctx, forests, b, reject_fraction: float, seed: int, rank: int, world: int,
                 do_dmat: bool = True, lens=None):
    """One pass of the hot path over ONE catalogue split across `world` ranks.

    Every rank: lya_neighbours (replicated: 0.5 % of the step) -> its chunk of the list -> one
    lya_plan -> lya_xi2pcf_plan (S, W, N) and lya_dmat_plan (Dn, Wd) -> all_reduce(SUM) -> lya_xi_normalise /
    lya_dmat_normalise.  Returns the reduced outputs (identical on every rank) plus this rank's
    stats.  `ctx`, `forests`, `b` are binding.Context / DeviceForests / CBinning."""
    import torch
    pairs = ctx.lya_neighbours(forests, b)
    if world > 1:
        pq = pairs.export()
        if lens is None:
            lens = (forests.pix_off[1:] - forests.pix_off[:-1])
        mine = split_pairs(pq, lens, rank, world).contiguous()
        pairs.free()
        pairs = ctx.lya_pairs_import(mine)
        del pq
    plan = ctx.lya_plan_create(forests, b, pairs, want_xi=True, want_dmat=do_dmat)     # prepared once for both stages
    pairs.free()
    x = ctx.lya_xi2pcf_plan(plan)
    dm = ctx.lya_dmat_plan(plan, reject_fraction, seed, want_Dn=True, want_D=False) if do_dmat else None
    plan.free()
    allreduce_sum(x["S"], x["W"], x["N"])
    out = dict(S=x["S"], W=x["W"], N=x["N"], xi=ctx.lya_xi_normalise(x["S"], x["W"]), stats_xi=x["stats"])
    if dm is not None:
        n_kept = torch.tensor([dm["stats"]["n_kept"]], dtype=torch.int64, device=dm["Dn"].device)
        allreduce_sum(dm["Dn"], dm["Wd"], n_kept)
        out.update(Dn=dm["Dn"], Wd=dm["Wd"], D=ctx.lya_dmat_normalise(b, dm["Dn"], dm["Wd"]),
                   n_kept=int(n_kept[0]), stats_dmat=dm["stats"])
    return out
