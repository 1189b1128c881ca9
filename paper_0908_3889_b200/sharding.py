"""Host-side plumbing of the multi-GPU path: the batch dimension is sharded, every rank
runs its own persistent grid, and the only exchange is the sum of the 3 x bins histogram counters.
Backend-agnostic (NCCL on GPUs, gloo in the CPU tests); holds no arithmetic of the method."""
from __future__ import annotations

from dataclasses import replace


def rank_config(cfg, rank: int):
    """Weak scaling: every rank integrates its own full-size batch with a rank-specific seed."""
    return replace(cfg, seed=cfg.seed + 1000 * int(rank))


def shard_range(n: int, rank: int, world: int):
    """Strong scaling: contiguous, balanced [lo, hi) slice of a batch of n systems for this rank."""
    base, rem = divmod(int(n), int(world))
    lo = rank * base + min(rank, rem)
    return lo, lo + base + (1 if rank < rem else 0)


def allreduce_counts(counts, dist=None):
    """In-place sum of the histogram counters over ranks (int64 tensor [3, bins]); no-op for one rank."""
    if dist is not None and dist.is_initialized() and dist.get_world_size() > 1:
        dist.all_reduce(counts)
    return counts


def max_over_ranks(value: float, device, dist=None) -> float:
    """A timing is the max over ranks, reduced on the device."""
    import torch

    t = torch.tensor([float(value)], dtype=torch.float64, device=device)
    if dist is not None and dist.is_initialized() and dist.get_world_size() > 1:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def allgather_moments(moments, dist=None):
    """Statistics over a sharded ensemble: gathers every rank's `moments` output of pn_statistics ([G, 3, 6]) into
    [world, G, 3, 6] in rank order, the input of pn_merge_statistics (which does the arithmetic on the device)."""
    import torch

    if dist is None or not dist.is_initialized() or dist.get_world_size() == 1:
        return moments.unsqueeze(0).contiguous()
    parts = [torch.empty_like(moments) for _ in range(dist.get_world_size())]
    dist.all_gather(parts, moments.contiguous())
    return torch.stack(parts).contiguous()


_COUNTERS = ("n_skipped", "hist1", "hist2")


def combine_statistics(local, dist=None, merge=None):
    """Ensemble statistics over a run that is sharded per section 8 of DESIGN.md: every rank holds the statistics of ITS
    slice [lo, hi) of every ensemble (pn_run_ensembles / pn_statistics outputs as tensors: 'moments' [G, 3, 6], and the
    integer counters 'n_skipped', 'hist1', 'hist2' where present).  The exchange: the counters are summed by an integer
    all-reduce; the moment records are all-gathered in rank order and merged by `merge(parts) -> (moments, pearson_r)`
    (pn_merge_statistics on the GPUs; the arithmetic stays in the library).  Returns a new dict; every rank gets the
    statistics of the whole run.  hist2_max is the largest cell of the summed bivariate histogram."""
    out = dict(local)
    for k in _COUNTERS:
        if out.get(k) is not None:
            out[k] = allreduce_counts(out[k].clone(), dist)
    out["moments"], out["pearson_r"] = merge(allgather_moments(local["moments"], dist))
    if out.get("hist2") is not None:
        out["hist2_max"] = out["hist2"].flatten(2).amax(dim=2)
    return out


def merge_shards(locals_in_rank_order, merge):
    """combine_statistics for shards that live in ONE process (tests; several shards run one after another on one GPU):
    same sums, same merge order."""
    import torch

    out = dict(locals_in_rank_order[0])
    for k in _COUNTERS:
        if out.get(k) is not None:
            out[k] = torch.stack([d[k] for d in locals_in_rank_order]).sum(dim=0)
    out["moments"], out["pearson_r"] = merge(torch.stack([d["moments"] for d in locals_in_rank_order]).contiguous())
    if out.get("hist2") is not None:
        out["hist2_max"] = out["hist2"].flatten(2).amax(dim=2)
    return out
