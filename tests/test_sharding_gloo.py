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


def test_bench_refuses_a_mislabelled_world():
    r, line = _bench("--gpus", "8", "--dry", env={"WORLD_SIZE": "2", "RANK": "0"})
    assert r.returncode != 0 and line is None and "WORLD_SIZE=2" in r.stderr
