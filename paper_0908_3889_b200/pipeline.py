"""Seed in, statistics out on the current CUDA device, for one ensemble or a sweep of ensembles.

Orchestration only: every step is one call of the C ABI (include/pn.h) through binding.py; nothing is computed here.
fused=True (FP64): ONE call, pn_run_ensembles, no state arrays.  Otherwise the unfused chain
pn_generate -> pn_integrate -> pn_statistics (-> pn_selfcheck) on device buffers, which also serves FP32 / mixed
precision, the cross-check and keep_states.
"""
from __future__ import annotations

from . import binding as B


def _merge_on_device(parts):
    """pn_merge_statistics on the gathered moment records [R, G, 3, 6] -> (moments [G, 3, 6], pearson_r [G, 3])."""
    import torch

    mom = torch.zeros(parts.shape[1], 3, 6, dtype=torch.float64, device=parts.device)
    r = torch.zeros(parts.shape[1], 3, dtype=torch.float64, device=parts.device)
    B.pn_merge_statistics(parts, moments=mom, pearson_r=r)
    return mom, r


def run_ensembles(ensembles, n, omegaf, *, rtol=1e-10, atol=1e-12, precision=B.PN_FP64, bins1=50, bins2=79,
                  check_fraction=0.0, check_key=(0, 0), keep_states=False, fused=False, dist=None, shard=None):
    """ensembles: list of dicts for binding.make_ensemble (key, omega0, q, chi1, chi2, m1_fixed, s1_tilt_deg).

    Returns a dict of numpy arrays: pearson_r[G,3], moments[G,3,6], n_skipped[G,3], hist1[G,3,bins1],
    hist2[G,3,bins2,bins2], hist2_max[G,3], steps_mean[G], status, and, if check_fraction > 0, `check`
    (pn_selfcheck's report: the paper's random double-precision cross-check).

    Several GPUs ("embarrassingly parallel", 140-156): with `dist` (an initialised
    torch.distributed, one process per GPU) every rank takes the slice sharding.shard_range(n, rank, world) of EVERY
    ensemble's variate stream, runs it as below, and the statistics are combined over the ranks
    (sharding.combine_statistics: integer all-reduce of the counters, all-gather + pn_merge_statistics of the moments):
    every rank returns the statistics of the whole run, status = the worst over ranks.  `shard = (rank, world)` without
    `dist` returns this share's own statistics (tests, or a caller with its own exchange; sharding.merge_shards).
    A sharded run keeps no states and makes no cross-check."""
    import torch

    from . import sharding

    ens = ensembles if isinstance(ensembles, (list, tuple)) else [ensembles]
    if dist is not None and dist.is_initialized() and dist.get_world_size() > 1 and shard is None:
        shard = (dist.get_rank(), dist.get_world_size())
    if shard is not None:
        if check_fraction > 0 or keep_states:
            raise ValueError("a sharded run keeps no states and makes no cross-check")
        lo, hi = sharding.shard_range(int(n), int(shard[0]), int(shard[1]))
        local = _run_slice(ens, int(n), lo, hi - lo, omegaf, rtol, atol, precision, bins1, bins2, fused)
        if dist is not None and dist.is_initialized() and dist.get_world_size() > 1:
            status = torch.tensor([int(local.pop("status"))], dtype=torch.int64, device=local["moments"].device)
            dist.all_reduce(status, op=dist.ReduceOp.MAX)
            local.pop("steps_mean", None)
            res = {k: v.cpu().numpy() for k, v in sharding.combine_statistics(local, dist, _merge_on_device).items()}
            res.update(status=int(status.item()), steps_mean=None, shard=(lo, hi))
            return res
        local["shard"] = (lo, hi)
        return local                 # tensors on the device: the caller combines the shares (sharding.merge_shards)
    G, N = len(ens), len(ens) * int(n)
    dev = torch.device("cuda", torch.cuda.current_device())
    f64 = dict(dtype=torch.float64, device=dev)
    i64 = dict(dtype=torch.int64, device=dev)
    if fused:
        if precision != B.PN_FP64 or check_fraction > 0 or keep_states:
            raise ValueError("the fused mode is FP64 only and keeps no states (no cross-check, no keep_states)")
        out = dict(pearson_r=torch.zeros(G, 3, **f64), moments=torch.zeros(G, 3, 6, **f64), n_skipped=torch.zeros(G, 3, **i64))
        if bins1 > 0:
            out["hist1"] = torch.zeros(G, 3, bins1, **i64)
        if bins2 > 0:
            out["hist2"] = torch.zeros(G, 3, bins2, bins2, **i64)
            out["hist2_max"] = torch.zeros(G, 3, **i64)
        status = B.pn_run_ensembles([B.make_ensemble(**e) for e in ens], int(n), omegaf, rtol, atol, bins1=bins1, bins2=bins2,
                                    allow_failures=True, **out)
        res = {k: v.cpu().numpy() for k, v in out.items()}
        res["status"] = status
        res["steps_mean"] = None
        return res
    y0, m = torch.empty(N, 10, **f64), torch.empty(N, 2, **f64)
    B.pn_generate([B.make_ensemble(**e) for e in ens], int(n), y0, m)
    yf = torch.empty_like(y0)
    steps = torch.empty(N, dtype=torch.int32, device=dev)
    times = torch.empty(N, **f64)
    status = B.pn_integrate(y0, m, 0.0, omegaf, rtol, atol, precision, yf, steps, out_time=times, allow_failures=True)
    out = dict(pearson_r=torch.zeros(G, 3, **f64), moments=torch.zeros(G, 3, 6, **f64), n_skipped=torch.zeros(G, 3, **i64))
    if bins1 > 0:
        out["hist1"] = torch.zeros(G, 3, bins1, **i64)
    if bins2 > 0:
        out["hist2"] = torch.zeros(G, 3, bins2, bins2, **i64)
        out["hist2_max"] = torch.zeros(G, 3, **i64)
    B.pn_statistics(y0, yf, steps, group_size=int(n), bins1=bins1, bins2=bins2, **out)
    res = {k: v.cpu().numpy() for k, v in out.items()}
    res["status"] = status
    res["steps_mean"] = steps.view(G, int(n)).clamp(min=0).double().mean(dim=1).cpu().numpy()
    if check_fraction > 0:
        res["check"] = B.pn_selfcheck(y0, m, yf, omegaf, fraction=check_fraction, key=check_key, times=times, allow_failures=True)
    if keep_states:
        res.update(init_states=y0, masses=m, final_states=yf, steps=steps, times=times)
    return res


def _run_slice(ens, n_total, first, count, omegaf, rtol, atol, precision, bins1, bins2, fused):
    """The statistics of the systems [first, first + count) of every ensemble, as device tensors (one rank's share)."""
    import torch

    G = len(ens)
    dev = torch.device("cuda", torch.cuda.current_device())
    f64 = dict(dtype=torch.float64, device=dev)
    i64 = dict(dtype=torch.int64, device=dev)
    out = dict(pearson_r=torch.zeros(G, 3, **f64), moments=torch.zeros(G, 3, 6, **f64), n_skipped=torch.zeros(G, 3, **i64))
    if bins1 > 0:
        out["hist1"] = torch.zeros(G, 3, bins1, **i64)
    if bins2 > 0:
        out["hist2"] = torch.zeros(G, 3, bins2, bins2, **i64)
        out["hist2_max"] = torch.zeros(G, 3, **i64)
    specs = [B.make_ensemble(**e) for e in ens]
    status = B.PN_OK
    if count > 0 and fused:
        if precision != B.PN_FP64:
            raise ValueError("the fused mode is FP64 only")
        status = B.pn_run_ensembles(specs, n_total, omegaf, rtol, atol, first=first, count=count, bins1=bins1, bins2=bins2,
                                    allow_failures=True, **out)
    elif count > 0:
        y0, m = torch.empty(G * count, 10, **f64), torch.empty(G * count, 2, **f64)
        B.pn_generate(specs, n_total, y0, m, first=first, count=count)
        yf = torch.empty_like(y0)
        steps = torch.empty(G * count, dtype=torch.int32, device=dev)
        status = B.pn_integrate(y0, m, 0.0, omegaf, rtol, atol, precision, yf, steps, allow_failures=True)
        B.pn_statistics(y0, yf, steps, group_size=count, bins1=bins1, bins2=bins2, **out)
    out["status"] = status
    return out
