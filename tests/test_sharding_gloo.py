"""N > 1 host logic on CPU: world_size 2, gloo backend.  No GPU, no CUDA library call."""
import os
import socket

import numpy as np
import pytest

torch = pytest.importorskip("torch")
import torch.distributed as dist  # noqa: E402
import torch.multiprocessing as mp  # noqa: E402

from paper_0908_3889_b200 import sharding  # noqa: E402
from paper_0908_3889_b200 import workloads as W  # noqa: E402


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, out):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        cfg = W.with_size(W.CONFIGS["C3"], 2000)
        mine = sharding.rank_config(cfg, rank)
        y0, m = W.generate(mine)
        # stand-in for this rank's final dot products: something deterministic from ITS inputs
        d = y0[:, 4] / np.linalg.norm(y0[:, 4:7], axis=1)
        local = np.stack([np.histogram(d, bins=50, range=(-1, 1))[0]] * 3).astype(np.int64)
        counts = torch.from_numpy(local.copy())
        sharding.allreduce_counts(counts, dist)
        tmax = sharding.max_over_ranks(10.0 + rank, torch.device("cpu"), dist)
        lo, hi = sharding.shard_range(1001, rank, world)
        mom = torch.full((2, 3, 6), float(rank + 1), dtype=torch.float64)
        parts = sharding.allgather_moments(mom, dist)
        out.put((rank, local, counts.numpy(), tmax, lo, hi, float(y0[:, 1].sum()), parts.numpy()))
    finally:
        dist.destroy_process_group()


def test_two_rank_sharding_and_count_allreduce():
    world, port = 2, _free_port()
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=_worker, args=(r, world, port, q)) for r in range(world)]
    for p in procs:
        p.start()
    res = sorted([q.get(timeout=120) for _ in range(world)], key=lambda t: t[0])
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    total = res[0][1] + res[1][1]
    for rank, local, reduced, tmax, lo, hi, chk, parts in res:
        assert parts.shape == (2, 2, 3, 6) and np.all(parts[0] == 1.0) and np.all(parts[1] == 2.0)   # rank order
        assert np.array_equal(reduced, total)           # every rank holds the global histogram
        assert reduced.sum() == 3 * 2000 * world
        assert tmax == 11.0                             # max over ranks
    assert (res[0][4], res[0][5], res[1][4], res[1][5]) == (0, 501, 501, 1001)   # disjoint, covering
    assert res[0][6] != res[1][6]                       # ranks drew different batches


def _moment_record(x, y):
    """(n, xbar, ybar, M2x, M2y, Cxy) of paired samples, the record layout of pn_statistics (include/pn.h)"""
    if len(x) == 0:
        return np.array([0.0, np.nan, np.nan, 0.0, 0.0, 0.0])
    return np.array([len(x), x.mean(), y.mean(), ((x - x.mean()) ** 2).sum(), ((y - y.mean()) ** 2).sum(),
                     ((x - x.mean()) * (y - y.mean())).sum()])


def _merge_standin(parts):
    """Stand-in for pn_merge_statistics on the CPU (the library's kernel needs a GPU): the textbook pairwise update of
    (n, mean, M2, C), parts in rank order.  parts [R, G, 3, 6] -> (moments [G, 3, 6], r [G, 3])."""
    p = parts.numpy()
    R, G = p.shape[:2]
    mom = np.zeros((G, 3, 6))
    for g in range(G):
        for k in range(3):
            n = mx = my = m2x = m2y = c = 0.0
            for part in range(R):
                nb, bx, by, b2x, b2y, bc = p[part, g, k]
                if nb == 0:
                    continue
                t = n + nb
                dx, dy = bx - mx, by - my
                m2x += b2x + dx * dx * n * nb / t
                m2y += b2y + dy * dy * n * nb / t
                c += bc + dx * dy * n * nb / t
                mx += dx * nb / t
                my += dy * nb / t
                n = t
            mom[g, k] = [n, mx, my, m2x, m2y, c]
    with np.errstate(invalid="ignore", divide="ignore"):
        r = mom[..., 5] / np.sqrt(mom[..., 3] * mom[..., 4])
    return torch.from_numpy(mom), torch.from_numpy(r)


def _sweep_samples(G=3, n=1001):
    """stand-in for the (initial, final) dot products of G ensembles of n systems: correlated pairs, per dot product"""
    g = np.random.Generator(np.random.Philox(99))
    x = g.uniform(-1, 1, size=(G, 3, n))
    y = np.clip(x * np.linspace(0.2, 0.9, G)[:, None, None] + 0.3 * g.normal(size=(G, 3, n)), -1, 1)
    return x, y


def _local_statistics(x, y, lo, hi, bins=20):
    """what one rank would hold for its slice [lo, hi) of every ensemble (layouts of pn_statistics)"""
    G = x.shape[0]
    mom = np.array([[_moment_record(x[g, k, lo:hi], y[g, k, lo:hi]) for k in range(3)] for g in range(G)])
    h1 = np.array([[np.histogram(y[g, k, lo:hi], bins=bins, range=(-1, 1))[0] for k in range(3)] for g in range(G)])
    h2 = np.array([[np.histogram2d(x[g, k, lo:hi], y[g, k, lo:hi], bins=4, range=((-1, 1), (-1, 1)))[0] for k in range(3)] for g in range(G)])
    return dict(moments=torch.from_numpy(mom), hist1=torch.from_numpy(h1.astype(np.int64)), hist2=torch.from_numpy(h2.astype(np.int64)),
                n_skipped=torch.full((G, 3), lo, dtype=torch.int64))


def _sweep_worker(rank, world, port, out):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        x, y = _sweep_samples()
        lo, hi = sharding.shard_range(x.shape[2], rank, world)
        res = sharding.combine_statistics(_local_statistics(x, y, lo, hi), dist, _merge_standin)
        out.put((rank, {k: v.numpy() for k, v in res.items()}))
    finally:
        dist.destroy_process_group()


def test_two_rank_sharded_sweep_statistics():
    """SURVEY.md 8(f) NEXT-3 "sharded over GPUs per 8(e)", the exchange on CPU: two ranks each hold the statistics of
    their slice of every ensemble of a sweep; sharding.combine_statistics (integer all-reduce of the counters, all-gather
    of the moment records in rank order, merge) gives EVERY rank the statistics of the whole run: equal to the
    single-process combination of the same shares, and to the statistics of the unsplit samples."""
    world, port = 2, _free_port()
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=_sweep_worker, args=(r, world, port, q)) for r in range(world)]
    for p in procs:
        p.start()
    res = dict(q.get(timeout=120) for _ in range(world))
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    x, y = _sweep_samples()
    n = x.shape[2]
    shares = [_local_statistics(x, y, *sharding.shard_range(n, r, world)) for r in range(world)]
    single = {k: v.numpy() for k, v in sharding.merge_shards(shares, _merge_standin).items()}
    whole = _local_statistics(x, y, 0, n)
    for rank in range(world):
        got = res[rank]
        for k in single:
            assert np.array_equal(got[k], single[k]), (rank, k)            # same sums, same merge order: same bits
        assert np.array_equal(got["hist1"], whole["hist1"].numpy()) and np.array_equal(got["hist2"], whole["hist2"].numpy())
        assert np.array_equal(got["hist2_max"], whole["hist2"].numpy().reshape(3, 3, -1).max(axis=2))
        assert np.array_equal(got["n_skipped"], np.full((3, 3), 0 + 501))  # the sum of the ranks' counters
        assert np.array_equal(got["moments"][..., 0], np.full((3, 3), float(n)))
        assert np.abs(got["moments"][..., 1:] - whole["moments"].numpy()[..., 1:]).max() < 1e-10
        r_ref = np.array([[np.corrcoef(x[g, k], y[g, k])[0, 1] for k in range(3)] for g in range(3)])
        assert np.abs(got["pearson_r"] - r_ref).max() < 1e-12


def test_shard_range_partitions():
    for n in (0, 1, 7, 1000, 1 << 20):
        for world in (1, 2, 3, 8):
            r = [sharding.shard_range(n, k, world) for k in range(world)]
            assert r[0][0] == 0 and r[-1][1] == n
            assert all(r[k][1] == r[k + 1][0] for k in range(world - 1))
            sizes = [hi - lo for lo, hi in r]
            assert max(sizes) - min(sizes) <= 1


def test_single_process_is_a_noop():
    c = torch.ones(3, 5, dtype=torch.int64)
    assert sharding.allreduce_counts(c, dist).sum().item() == 15
    assert sharding.max_over_ranks(3.5, torch.device("cpu"), dist) == 3.5
    assert sharding.allgather_moments(torch.ones(4, 3, 6, dtype=torch.float64), dist).shape == (1, 4, 3, 6)


def _bench(*flags, env=None):
    import json
    import subprocess
    import sys

    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    e = {k: v for k, v in os.environ.items() if k not in ("RANK", "LOCAL_RANK", "WORLD_SIZE", "MASTER_ADDR", "MASTER_PORT")}
    e.update(env or {})
    r = subprocess.run([sys.executable, os.path.join(root, "bench.py"), *flags], capture_output=True, text=True, env=e, timeout=300)
    lines = [ln for ln in r.stdout.splitlines() if ln.startswith("{")]
    return r, (json.loads(lines[-1]) if lines else None)


def test_bench_spawns_its_own_ranks():
    """`python bench.py --gpus 2` (no torchrun environment) must run TWO ranks: bench.py re-executes itself under
    torch.distributed.run.  --dry keeps CUDA out of it: launch, sharding and the exchange step only (gloo)."""
    r, line = _bench("--gpus", "2", "--dry", "--workload", "C1")
    assert r.returncode == 0, r.stderr[-2000:]
    assert line["n_gpus"] == 2 and line["scaling"] == "weak"
    assert line["systems_all_ranks"] == line["systems_expected"] == 2 * 1024      # both ranks reached the all-reduce
    assert line["max_over_ranks"] == 2.0
    # strong scaling: one batch split over the ranks
    r, line = _bench("--gpus", "2", "--dry", "--workload", "C1", "--scaling", "strong")
    assert r.returncode == 0 and line["n_gpus"] == 2 and line["systems_rank0"] == 512 and line["systems_all_ranks"] == 1024
    # one rank: no spawn, same code path
    r, line = _bench("--dry", "--workload", "C1")
    assert r.returncode == 0 and line["n_gpus"] == 1 and line["systems_all_ranks"] == 1024


def test_bench_fused_mode_shards_the_variate_stream():
    """`bench.py --fused --gpus 2 --dry`: the exchange of a sharded fused ensemble run (sharding.combine_statistics) under
    bench.py's own launch path: both ranks' slices add up to the whole ensemble, weak and strong."""
    r, line = _bench("--gpus", "2", "--dry", "--fused", "--workload", "C1")
    assert r.returncode == 0, r.stderr[-2000:]
    assert line["fused"] == {"systems_all_ranks": 2048, "systems_expected": 2048, "hist1_cell": 2048, "slice_rank0": [0, 1024]}
    r, line = _bench("--gpus", "2", "--dry", "--fused", "--workload", "C1", "--scaling", "strong")
    assert r.returncode == 0 and line["fused"]["systems_all_ranks"] == 1024 and line["fused"]["slice_rank0"] == [0, 512]


def test_bench_refuses_a_mislabelled_world():
    r, line = _bench("--gpus", "8", "--dry", env={"WORLD_SIZE": "2", "RANK": "0"})
    assert r.returncode != 0 and line is None and "WORLD_SIZE=2" in r.stderr
