#!/usr/bin/env python
"""bench.py -- throughput of the hot path (pn_integrate + pn_histogram) on N B200s of one node.

One "step" = one pass of the whole hot path over one batch of synthetic inspirals of the workload
(default: C2 of BASELINE.json, 2^20 equal-mass maximally spinning inspirals, FP64, omega 0.005->0.05,
rtol 1e-10): stage-in, persistent DP5(4) integrator, stage-out, histogram kernel.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload C2] [--impl ours|reference] [--scaling weak|strong] [--fused]

Prints ONE JSON line (see DESIGN.md 6 for every field).  Multi-GPU: one process per GPU.  Started
under torchrun (RANK / LOCAL_RANK / WORLD_SIZE / MASTER_* in the environment) it uses those ranks; started as
plain `python bench.py --gpus N` with N > 1 it re-executes itself under `python -m torch.distributed.run
--nproc-per-node N` on 127.0.0.1.  The batch dimension is sharded: weak scaling (default) gives every rank its own
seeded batch of the full workload size, strong scaling splits ONE batch into contiguous slices
(sharding.shard_range); the only exchange is the all-reduce of the 3 x bins histogram counters.
`--dry` runs the launch, sharding and exchange logic on the CPU (gloo, no CUDA, no kernels): for the CPU tests.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

from paper_0908_3889_b200 import workloads as W  # noqa: E402

# Algorithmic work per unit, counted on a constants-hoisted form of Eqs. (1)-(4) and the DP5(4) step
# (every add, mul, div, sqrt, cbrt, log, pow = 1 flop, an FMA = 2).  Conservative: the
# oracle's as-printed form counts 151 state-dependent flops per RHS and 1652 per trial step.
F_RHS = 99           # one right-hand-side evaluation
F_STEP = 1198        # one trial step = 6 RHS (594) + stage sums (420) + error vector (116) + norm/controller (68)
F_RHS_ORACLE, F_STEP_ORACLE = 151, 1652
FP64_LANES_PER_SM = 64
FP32_LANES_PER_SM = 128


class ClockSampler(threading.Thread):
    """Samples nvidia-smi clocks and throttle reasons during the timed region (B200_PROFILING.md)."""

    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        super().__init__(daemon=True)
        self.index, self.samples, self._stop_evt = index, [], threading.Event()

    def run(self):
        while not self._stop_evt.is_set():
            try:
                out = subprocess.check_output(["nvidia-smi", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits",
                                               "-i", str(self.index)], timeout=5).decode().strip()
                self.samples.append([t.strip() for t in out.split(",")])
            except Exception:
                pass
            self._stop_evt.wait(0.02)

    def stop(self):
        self._stop_evt.set()
        self.join(timeout=6)
        sm, mx, reasons, pw = [], [], set(), []
        for s in self.samples:
            try:
                sm.append(float(s[0])); mx.append(float(s[1])); pw.append(float(s[2]))
            except (ValueError, IndexError):
                continue
            for name, v in zip(("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"), s[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(name)
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "power_w_max": max(pw) if pw else None, "samples": len(sm), "reasons": sorted(reasons)}


def cpu_model():
    try:
        for ln in open("/proc/cpuinfo"):
            if ln.lower().startswith("model name"):
                return ln.split(":", 1)[1].strip()
    except OSError:
        pass
    return "unknown"


def oracle_throughput(cfg, target_seconds=15.0, n_threads=0, single_thread=False):
    """Times the CPU oracle, as it stands, on a bounded seeded sample of the workload: a random-permutation prefix of
    the batch (so the q / chi mix is the workload's), sized from a 256-system probe for about target_seconds."""
    from oracle import pn_oracle

    pn_oracle.build()
    # torchrun exports OMP_NUM_THREADS=1 to its ranks: ask for the host's cores explicitly
    n_threads = n_threads if n_threads > 0 else (os.cpu_count() or 1)
    y0, m = W.generate(W.with_size(cfg, min(cfg.n, 1 << 19)))
    perm = np.random.Generator(np.random.Philox(20090826)).permutation(y0.shape[0])
    y0, m = np.ascontiguousarray(y0[perm]), np.ascontiguousarray(m[perm])
    probe = min(256, y0.shape[0])
    t0 = time.perf_counter()
    pn_oracle.integrate(y0[:probe], m[:probe], cfg.omegaf, 1e-10, 1e-12, n_threads=n_threads)
    dt = max(time.perf_counter() - t0, 1e-4)
    k = int(min(y0.shape[0], max(probe, probe * target_seconds / dt)))
    t0 = time.perf_counter()
    r = pn_oracle.integrate(y0[:k], m[:k], cfg.omegaf, 1e-10, 1e-12, n_threads=n_threads)
    pn_oracle.histogram(r["final"], cfg.bins)
    dt = time.perf_counter() - t0
    out = {"value": k / dt, "unit": "inspirals/s", "cores": n_threads, "kind": "oracle", "cpu_model": cpu_model(),
           "sample": f"random-permutation prefix of {k} systems of the seeded {cfg.name} batch (FP64 oracle, rtol 1e-10, atol 1e-12), "
                     f"{dt:.1f} s wall on {n_threads} threads, {os.cpu_count()} logical CPUs",
           "rhs_evals_per_s": float((6 * r["steps"].astype(np.int64) + 1).sum() / dt), "seconds": dt,
           "mean_steps": float(r["steps"].mean())}
    if single_thread:
        # one thread on 256 systems: the figure comparable with the paper's single-core number
        t0 = time.perf_counter()
        pn_oracle.integrate(y0[:probe], m[:probe], cfg.omegaf, 1e-10, 1e-12, n_threads=1)
        out["single_thread"] = {"value": probe / (time.perf_counter() - t0), "unit": "inspirals/s", "systems": probe}
    return out


def run_reference(args, cfg):
    """--impl reference: the oracle on the host cores; rank 0 only."""
    if int(os.environ.get("RANK", "0")) != 0:
        return
    per_step = []
    last = None
    for i in range(args.warmup + args.steps):
        last = oracle_throughput(cfg, target_seconds=8.0 if i >= args.warmup else 2.0)
        if i >= args.warmup:
            per_step.append(last)
    value = float(np.mean([p["value"] for p in per_step]))
    line = {"impl": "reference", "metric": "inspirals_per_sec", "value": value, "unit": "inspirals/s", "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * float(np.mean([p["seconds"] for p in per_step])),
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": cfg.name, "n_inspirals": cfg.n, "n_inspirals_per_gpu": cfg.n, "omega0": cfg.omega0,
                       "omegaf": cfg.omegaf, "rtol": cfg.rtol, "atol": cfg.atol, "bins": cfg.bins,
                       "note": "each step is a bounded sample of the workload"},
            "cpu_baseline": {k: last[k] for k in ("value", "unit", "cores", "kind", "sample", "cpu_model")},
            "e2e": {"value": value, "unit": "inspirals/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "rhs_evals_per_sec": float(np.mean([p["rhs_evals_per_s"] for p in per_step])), "gpu_launches": 0}
    line["cpu_baseline"]["value"] = value
    print(json.dumps(line))


def spawn_ranks_if_needed(args):
    """`python bench.py --gpus N` (N > 1, no torchrun environment): re-execute under torch.distributed.run with N ranks on
    this node.  Under torchrun a WORLD_SIZE that disagrees with --gpus is an error, never a silently mislabelled run."""
    if "WORLD_SIZE" in os.environ:
        world = int(os.environ["WORLD_SIZE"])
        if args.gpus != world:
            raise SystemExit(f"bench.py: --gpus {args.gpus} but WORLD_SIZE={world}: launch with --nproc-per-node {args.gpus}")
        return
    if args.gpus <= 1:
        return
    import socket

    with socket.socket() as sk:
        sk.bind(("127.0.0.1", 0))
        port = sk.getsockname()[1]
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={args.gpus}",
           "--master-addr", "127.0.0.1", "--master-port", str(port), os.path.abspath(__file__)] + sys.argv[1:]
    raise SystemExit(subprocess.call(cmd))


def rank_shard(cfg, rank, world, scaling):
    """This rank's share of the workload: (config to generate, slice of the generated batch, systems of the whole job)."""
    from paper_0908_3889_b200 import sharding

    if scaling == "strong":
        lo, hi = sharding.shard_range(cfg.n, rank, world)          # one batch, contiguous balanced slices
        return cfg, slice(lo, hi), cfg.n
    return sharding.rank_config(cfg, rank), slice(0, cfg.n), cfg.n * world     # every rank its own full-size batch


def run_dry(args, cfg):
    """--dry: the multi-rank launch, sharding and exchange logic on the CPU with gloo; no CUDA, no kernels, no timing
    claims.  Every rank contributes its shard size to the same all-reduce and max-reduction the real run uses."""
    import torch
    import torch.distributed as dist

    from paper_0908_3889_b200 import sharding

    rank, world = int(os.environ.get("RANK", "0")), int(os.environ.get("WORLD_SIZE", "1"))
    if world > 1:
        dist.init_process_group("gloo")
    gen_cfg, sl, total = rank_shard(cfg, rank, world, args.scaling)
    n_mine = len(range(*sl.indices(gen_cfg.n)))
    counts = torch.zeros(3, cfg.bins, dtype=torch.int64)
    counts[:, rank % cfg.bins] = n_mine                          # stand-in for this rank's histogram
    sharding.allreduce_counts(counts, dist if world > 1 else None)
    slowest = sharding.max_over_ranks(float(rank + 1), torch.device("cpu"), dist if world > 1 else None)
    fused = None
    if args.fused:
        # --fused: the exchange of a sharded ensemble run (sharding.combine_statistics) with stand-in records: this rank's
        # slice of ONE ensemble of n_total systems; the stand-in merge only adds the counts n of the gathered records
        n_total = cfg.n * world if args.scaling == "weak" else cfg.n
        lo, hi = sharding.shard_range(n_total, rank, world)
        mom = torch.zeros(1, 3, 6, dtype=torch.float64)
        mom[..., 0] = hi - lo
        local = dict(moments=mom, hist1=torch.full((1, 3, cfg.bins), hi - lo, dtype=torch.int64))
        res = sharding.combine_statistics(local, dist if world > 1 else None, lambda parts: (parts.sum(dim=0), parts.sum(dim=0)[..., 0]))
        fused = {"systems_all_ranks": int(res["moments"][0, 0, 0].item()), "systems_expected": n_total,
                 "hist1_cell": int(res["hist1"][0, 0, 0].item()), "slice_rank0": [lo, hi]}
    if rank == 0:
        print(json.dumps({"dry": True, "n_gpus": world, "scaling": args.scaling, "seed_rank0": gen_cfg.seed,
                          "systems_rank0": n_mine, "systems_all_ranks": int(counts[0].sum().item()), "systems_expected": total,
                          "max_over_ranks": slowest, "fused": fused, "config": {"workload": cfg.name}}))
    if world > 1:
        dist.destroy_process_group()


def run_fused(args, cfg):
    """--fused: a step is ONE sharded fused ensemble run of the workload's ensemble (pipeline.run_ensembles(fused=True,
    dist=...): seed in, statistics out, no state arrays; SURVEY.md 8(f) NEXT-1..3).  Weak scaling: the
    ensemble has cfg.n systems per rank; strong: cfg.n in all.  Every rank integrates its slice of the variate stream;
    the exchange per step is an int64 all-reduce of the counters and an all-gather of 18 doubles per ensemble.  Not the
    BASELINE.json metric's configuration (that is the default mode): a line for the widened rows."""
    import torch
    import torch.distributed as dist

    import paper_0908_3889_b200 as pn
    from paper_0908_3889_b200 import sharding

    rank, world, local = int(os.environ.get("RANK", "0")), int(os.environ.get("WORLD_SIZE", "1")), int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device (there is no CPU fallback)")
    if cfg.precision not in ("fp64",):
        raise SystemExit("bench.py --fused: the fused mode is FP64 only")
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    if world > 1:
        dist.init_process_group("nccl", device_id=dev)
    d = dist if world > 1 else None
    n_total = cfg.n * world if args.scaling == "weak" else cfg.n
    spec = W.generator_spec(cfg)
    flush = torch.empty(256 << 20, dtype=torch.uint8, device=dev)
    stream = torch.cuda.current_stream()

    def step():
        return pn.run_ensembles([spec], n_total, cfg.omegaf, rtol=cfg.rtol, atol=cfg.atol, bins1=cfg.bins, bins2=79, fused=True,
                                dist=d, shard=(rank, world) if world > 1 else None)

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    for _ in range(args.warmup):
        step(); flush.zero_()
    sampler = ClockSampler(local)
    barrier()
    sampler.start()
    launches0 = pn.pn_launch_count()
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    kern_ms, trial_steps = [], []
    ev0.record(stream)
    for _ in range(args.steps):
        res = step()
        kern_ms.append(pn.pn_last_kernel_ms()["integrate"]); trial_steps.append(pn.pn_last_counters()["trial_steps"])
        flush.zero_()
    ev1.record(stream)
    barrier()
    clocks = sampler.stop()
    ms_step = sharding.max_over_ranks(ev0.elapsed_time(ev1), dev, d) / args.steps
    steps_all = torch.tensor([float(np.mean(trial_steps))], dtype=torch.float64, device=dev)
    if world > 1:
        dist.all_reduce(steps_all)
    if rank == 0:
        sms = torch.cuda.get_device_properties(dev).multi_processor_count
        peak = sms * FP64_LANES_PER_SM * 2 * float(clocks.get("sm_max_mhz") or 1965.0) * 1e6 / 1e12
        n_mine = n_total // world
        achieved = (float(np.mean(trial_steps)) * F_STEP + n_mine * F_RHS) / (float(np.mean(kern_ms)) * 1e-3) / 1e12
        G = 1
        print(json.dumps({
            "metric": "inspirals_per_sec", "value": n_total / (ms_step * 1e-3), "unit": "inspirals/s", "n_gpus": world,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": ms_step, "higher_is_better": True, "scaling": args.scaling,
            "vs_baseline": None, "dtype": "f64", "data": "synthetic (drawn on the device from the seed)",
            "comm": {"backend": "nccl" if world > 1 else None, "nranks": world,
                     "exchange": "per step: int64 all-reduce of n_skipped, hist1, hist2; all-gather of 18 doubles per ensemble; max of the status"},
            "config": {"workload": cfg.name, "mode": "fused ensemble run (pn_run_ensembles), sharded by slices of the variate stream",
                       "n_inspirals": n_total, "n_inspirals_per_gpu": n_mine, "omega0": cfg.omega0, "omegaf": cfg.omegaf, "rtol": cfg.rtol,
                       "atol": cfg.atol, "bins": cfg.bins, "bins2": 79, "parallelism": f"stream-sharded x{world}",
                       "l2": "256 MiB memset between steps"},
            "rhs_evals_per_sec": (6.0 * float(steps_all.item()) + n_total) / (ms_step * 1e-3),
            "kernel_ms": {"integrate": float(np.mean(kern_ms))},
            "roofline": {"bound": "alu", "kernel": "pn_integrate_adaptive_kernel<..., FUSED>", "achieved": achieved, "peak": peak,
                         "unit": "TFLOP/s", "frac": achieved / peak, "traffic": None,
                         "flops_basis": "fixed algorithmic count, independent of the implementation (DESIGN.md 6.2)"},
            # the call a user makes takes a seed and returns statistics: its end-to-end time IS the step
            "e2e": {"value": n_total / (ms_step * 1e-3), "unit": "inspirals/s", "h2d_bytes_per_step": 88 * G,
                    "d2h_bytes_per_step": int(8 * G * (3 + 18 + 3 + 3 * cfg.bins + 3 * 79 * 79 + 3)), "steps": args.steps},
            "pearson_r": [float(x) for x in res["pearson_r"][0]], "status": int(res["status"]),
            "gpu_launches": int(pn.pn_launch_count() - launches0), "clocks": clocks}))
    if world > 1:
        dist.destroy_process_group()


def run_ours(args, cfg):
    import torch
    import torch.distributed as dist

    import paper_0908_3889_b200 as pn

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device (there is no CPU fallback)")
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    if world > 1:
        dist.init_process_group("nccl", device_id=dev)
    prec = {"fp32": pn.PN_FP32, "mixed": pn.PN_MIXED}.get(cfg.precision, pn.PN_FP64)

    # weak scaling: every rank integrates its own seeded batch of the full workload size; strong: its slice of one batch
    from paper_0908_3889_b200 import sharding
    gen_cfg, sl, total_inspirals = rank_shard(cfg, rank, world, args.scaling)
    y0, m = W.generate(gen_cfg)
    y0, m = np.ascontiguousarray(y0[sl]), np.ascontiguousarray(m[sl])
    n = y0.shape[0]
    h_y0 = torch.from_numpy(y0).pin_memory(); h_m = torch.from_numpy(m).pin_memory()
    d_y0, d_m = h_y0.to(dev), h_m.to(dev)
    d_yf = torch.empty_like(d_y0)
    d_steps = torch.empty(n, dtype=torch.int32, device=dev)
    d_counts = torch.zeros(3, cfg.bins, dtype=torch.int64, device=dev)
    flush = torch.empty(256 << 20, dtype=torch.uint8, device=dev)       # > 126 MB L2
    stream = torch.cuda.current_stream()

    def step():
        pn.pn_integrate(d_y0, d_m, cfg.omega0, cfg.omegaf, cfg.rtol, cfg.atol, prec, d_yf, d_steps,
                        input_order=bool(args.input_order), variant=args.variant)
        pn.pn_histogram(d_yf, cfg.bins, d_counts)
        sharding.allreduce_counts(d_counts, dist if world > 1 else None)   # the one exchange step

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    for _ in range(args.warmup):
        step(); flush.zero_()
    sampler = ClockSampler(local)
    barrier()
    sampler.start()
    launches0 = pn.pn_launch_count()
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    kern_ms, hist_ms, trial_steps = [], [], []
    ev0.record(stream)
    for _ in range(args.steps):
        step()
        k = pn.pn_last_kernel_ms(); kern_ms.append(k["integrate"]); hist_ms.append(k["histogram"])
        trial_steps.append(pn.pn_last_counters()["trial_steps"])
        flush.zero_()
    ev1.record(stream)
    barrier()
    clocks = sampler.stop()
    launches = pn.pn_launch_count() - launches0
    ms_total = ev0.elapsed_time(ev1)
    ms_step = sharding.max_over_ranks(ms_total, dev, dist if world > 1 else None) / args.steps
    counters = pn.pn_last_counters()
    # RHS evaluations of the whole job per step (6 per trial step + the seed evaluation), summed over ranks on the device
    rhs_mine = torch.tensor([6.0 * float(np.mean(trial_steps)) + n], dtype=torch.float64, device=dev)
    if world > 1:
        dist.all_reduce(rhs_mine)
    rhs_all_ranks = float(rhs_mine.item())

    # end to end through the C ABI with HOST buffers: H2D of inputs and D2H of results inside the timed region
    h_yf = torch.empty(n, 10, dtype=torch.float64).pin_memory()
    h_steps = torch.empty(n, dtype=torch.int32).pin_memory()
    h_counts = np.zeros((3, cfg.bins), dtype=np.int64)
    e2e_steps = max(1, args.steps)

    def e2e_step():
        # ONE host-buffer call: the library bins the final states while they are on the device (pn_options.hist_counts)
        pn.pn_integrate(h_y0, h_m, cfg.omega0, cfg.omegaf, cfg.rtol, cfg.atol, prec, h_yf, h_steps,
                        input_order=bool(args.input_order), variant=args.variant, hist_bins=cfg.bins, hist_counts=h_counts)

    e2e_step()
    barrier()
    t0 = time.perf_counter()
    for _ in range(e2e_steps):
        e2e_step()
    barrier()
    e2e_s = sharding.max_over_ranks((time.perf_counter() - t0) / e2e_steps, dev, dist if world > 1 else None)
    h2d = (10 + 2) * 8 * n                       # states + masses; the final states are binned on the device (r2: + 80 n)
    d2h = 10 * 8 * n + 4 * n + 3 * cfg.bins * 8

    # rows beyond the hot path, timed outside the step: on-device statistics of
    # (initial, final) states and on-device generation of the same batch; both HBM-bound
    widened = None
    if world == 1:
        hbm = None
        pk = os.path.join(ROOT, "MEASURED_PEAKS.json")
        if os.path.exists(pk):
            hbm = json.load(open(pk)).get("hbm_gbs")
        hbm_src = "MEASURED_PEAKS.json hbm_gbs" if hbm else "fallback 6500 GB/s (B200_PROFILING.md)"
        hbm = float(hbm or 6500.0)
        out = dict(pearson_r=torch.zeros(1, 3, dtype=torch.float64, device=dev),
                   moments=torch.zeros(1, 3, 6, dtype=torch.float64, device=dev),
                   hist1=torch.zeros(1, 3, cfg.bins, dtype=torch.int64, device=dev),
                   hist2=torch.zeros(1, 3, 79, 79, dtype=torch.int64, device=dev),
                   hist2_max=torch.zeros(1, 3, dtype=torch.int64, device=dev))
        st_ms, gen_ms = [], []
        g_y0, g_m = torch.empty_like(d_y0), torch.empty_like(d_m)
        ens = pn.make_ensemble(**W.generator_spec(cfg))
        for i in range(4):
            flush.zero_()
            pn.pn_statistics(d_y0, d_yf, d_steps, bins1=cfg.bins, bins2=79, **out)
            st_ms.append(pn.pn_last_kernel_ms()["histogram"])
            flush.zero_()
            pn.pn_generate(ens, n, g_y0, g_m)
            gen_ms.append(pn.pn_last_kernel_ms()["stage_in"])
        st, ge = float(np.median(st_ms[1:])), float(np.median(gen_ms[1:]))
        widened = {"statistics": {"ms": st, "bytes_per_system": 164, "achieved_gbs": 164 * n / st / 1e6,
                                  "frac_of_hbm": 164 * n / st / 1e6 / hbm, "pearson_r": out["pearson_r"].cpu().numpy()[0].tolist(),
                                  "bins2": 79},
                   "generate": {"ms": ge, "bytes_per_system": 96, "achieved_gbs": 96 * n / ge / 1e6,
                                "frac_of_hbm": 96 * n / ge / 1e6 / hbm,
                                "max_abs_diff_vs_host_recipe": float((g_y0 - d_y0).abs().max().item())},
                   "hbm_peak_gbs": hbm, "hbm_peak_source": hbm_src}
        # the same workload as ONE fused call (pn_run_ensembles: seed in, statistics out, no state arrays; FP64 only),
        # next to the unfused chain generate -> integrate -> statistics on the same ensemble
        if prec == pn.PN_FP64:
            fo = dict(pearson_r=torch.zeros(1, 3, dtype=torch.float64, device=dev), hist1=torch.zeros(1, 3, cfg.bins, dtype=torch.int64, device=dev),
                      hist2=torch.zeros(1, 3, 79, 79, dtype=torch.int64, device=dev))
            fu_ms, fu_wall = [], []
            for i in range(3):
                flush.zero_(); torch.cuda.synchronize()
                t0 = time.perf_counter()
                pn.pn_run_ensembles(ens, n, cfg.omegaf, cfg.rtol, cfg.atol, bins1=cfg.bins, bins2=79, **fo)
                fu_wall.append((time.perf_counter() - t0) * 1e3); fu_ms.append(pn.pn_last_kernel_ms()["integrate"])
            chain_ms = ge + float(np.mean(kern_ms)) + st
            widened["fused"] = {"ms_kernels": float(np.median(fu_ms[1:])), "ms_call": float(np.median(fu_wall[1:])),
                                "inspirals_per_sec": n / (float(np.median(fu_wall[1:])) * 1e-3),
                                "unfused_chain_ms_kernels": chain_ms, "pearson_r": fo["pearson_r"].cpu().numpy()[0].tolist(),
                                "hist1_equals_unfused": bool(torch.equal(fo["hist1"], out["hist1"])),
                                "hist2_equals_unfused": bool(torch.equal(fo["hist2"], out["hist2"]))}
            # a sweep of 16 ensembles in ONE fused call (r against chi at equal masses), n/16 systems each:
            # the default queue order for more than 4 ensembles (index order) next to the cost order it replaces
            # (pn_options.variant bit 2; interleaved ensembles thrash the blocks' moment tables)
            ns = max(n // 16, 1)
            sweep = [pn.make_ensemble((20090826, k), cfg.omega0, q=(1.0, 1.0), chi1=((k + 1) / 16,) * 2, chi2=((k + 1) / 16,) * 2,
                                      m1_fixed=0.5) for k in range(16)]
            so = dict(pearson_r=torch.zeros(16, 3, dtype=torch.float64, device=dev), hist1=torch.zeros(16, 3, cfg.bins, dtype=torch.int64, device=dev))
            sw = {}
            for name, var in (("ms_kernels", 0), ("ms_kernels_cost_order", 4)):
                t = []
                for i in range(2):
                    pn.pn_run_ensembles(sweep, ns, cfg.omegaf, cfg.rtol, cfg.atol, bins1=cfg.bins, variant=var, **so)
                    t.append(pn.pn_last_kernel_ms()["integrate"])
                sw[name] = float(min(t))
            sw.update(ensembles=16, systems_per_ensemble=ns, inspirals_per_sec=16 * ns / (sw["ms_kernels"] * 1e-3),
                      pearson_r_s1s2=[float(x) for x in so["pearson_r"][:, 0].cpu().numpy()])
            widened["fused_sweep"] = sw
    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return
    # roofline of the dominant kernel (the integrator): algorithmic flops / CUDA-event duration
    lanes = FP64_LANES_PER_SM if prec == pn.PN_FP64 else FP32_LANES_PER_SM
    sms = torch.cuda.get_device_properties(dev).multi_processor_count
    peaks = json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json"))) if os.path.exists(os.path.join(ROOT, "MEASURED_PEAKS.json")) else {}
    sm_max = float(peaks.get("sm_max_mhz") or clocks.get("sm_max_mhz") or 1965.0)
    peak_nominal = sms * lanes * 2 * sm_max * 1e6 / 1e12
    peak_prec = pn.PN_FP64 if prec == pn.PN_FP64 else pn.PN_FP32       # the pipe the slopes are computed on
    peak_meas, peak_mhz = pn.pn_measure_fma_peak(peak_prec, 0.5)
    traffic, traffic_src, executed = None, None, None
    tj = os.path.join(ROOT, "profiles", "traffic.json")
    if os.path.exists(tj):
        ent = json.load(open(tj)).get(f"{cfg.name}:{n}")
        if ent:
            traffic, traffic_src = float(ent["dram_bytes_read"]) + float(ent["dram_bytes_write"]), ent["source"]
            ex = ent.get("fp64_inst_per_trial_step")
            if ex:       # what the captured kernel executes per trial step, in flops (FMA = 2), next to the fixed F_STEP
                executed = dict(ex, flops=2 * ex["dfma"] + ex["dmul"] + ex["dadd"], source=ent["source"])
    flops_launch = float(np.mean(trial_steps)) * F_STEP + n * F_RHS
    k_ms = float(np.mean(kern_ms))
    achieved = flops_launch / (k_ms * 1e-3) / 1e12
    line = {
        "metric": "inspirals_per_sec", "value": total_inspirals / (ms_step * 1e-3), "unit": "inspirals/s",
        "n_gpus": world, "steps": args.steps, "warmup": args.warmup, "ms_per_step": ms_step,
        "higher_is_better": True, "scaling": args.scaling, "vs_baseline": None,
        "dtype": {pn.PN_FP32: "f32", pn.PN_MIXED: "f32 slopes + f64 state"}.get(prec, "f64"), "data": "synthetic",
        "comm": {"backend": "nccl" if world > 1 else None, "nranks": world, "exchange": "all-reduce of 3 x bins int64 counters per step"},
        "config": {"workload": cfg.name, "n_inspirals": cfg.n, "n_inspirals_per_gpu": n, "omega0": cfg.omega0, "omegaf": cfg.omegaf,
                   "rtol": cfg.rtol, "atol": cfg.atol, "bins": cfg.bins, "queue": "input order" if args.input_order else "longest-expected-first", "variant": args.variant, "parallelism": f"batch-sharded x{world}",
                   "l2": "256 MiB memset between steps, inside the timed region (<0.1 % of a step)"},
        "rhs_evals_per_sec": rhs_all_ranks / (ms_step * 1e-3),
        "trial_steps_per_inspiral": float(np.mean(trial_steps)) / n,
        "counters_last_step": counters,
        "kernel_ms": {"integrate": k_ms, "histogram": float(np.mean(hist_ms))},
        "roofline": {"bound": "alu", "kernel": "pn_integrate_adaptive_kernel", "achieved": achieved, "peak": peak_nominal,
                     "unit": "TFLOP/s", "frac": achieved / peak_nominal,
                     # dram__bytes_read + dram__bytes_write of this kernel per launch, from the committed ncu --set full
                     # capture of the same workload and size (profiles/traffic.json names the capture); null if none.
                     # algorithmic bytes: 96 B in + 100 B out (state, steps, time) per inspiral
                     "traffic": traffic, "traffic_unit": "bytes/launch", "traffic_source": traffic_src,
                     "algorithmic_bytes": 196 * n,
                     "peak_source": f"nominal {sms} SMs x {lanes} FMA lanes x 2 x {sm_max:.0f} MHz (DESIGN.md 6.3)",
                     "peak_measured_fma": peak_meas, "peak_measured_sm_mhz": peak_mhz,
                     "peak_measured_ffma2": pn.pn_measure_fma_peak(3, 0.25)[0] if peak_prec == pn.PN_FP32 else None,
                     "frac_of_measured_fma": achieved / peak_meas if peak_meas > 0 else None,
                     "flops_per_trial_step": F_STEP, "flops_per_rhs": F_RHS,
                     # F_STEP / F_RHS are a FIXED algorithmic count of the method, not a count of what this
                     # kernel executes: they have not moved since r1 although the kernel now does less arithmetic per RHS
                     # (folded constants, shared products) and more for cbrt / log than the count books (2 per stage).
                     "flops_basis": "fixed algorithmic count, independent of the implementation (DESIGN.md 6.2)",
                     "executed_fp64_per_trial_step": executed,
                     "frac_with_oracle_as_printed_count": (float(np.mean(trial_steps)) * F_STEP_ORACLE + n * F_RHS_ORACLE)
                     / (k_ms * 1e-3) / 1e12 / peak_nominal,
                     "fma_issue_cycles_by_register_sources": {str(k): pn.pn_measure_fma_operands(peak_prec, k) for k in (1, 2, 3)},
                     # a two-source FMA + two independent integer instructions: 2 cycles if they issued in the FMA's
                     # shadow, 4 if every instruction takes its own issue cycles
                     "fma_plus_two_alu_issue_cycles": pn.pn_measure_fma_operands(peak_prec, 4)},
        "e2e": {"value": total_inspirals / e2e_s, "unit": "inspirals/s", "h2d_bytes_per_step": h2d,
                "d2h_bytes_per_step": d2h, "steps": e2e_steps},
        "gpu_launches": int(launches), "clocks": clocks,
    }
    if widened:
        line["widened"] = widened
    if world == 1 and not args.no_cpu_baseline:
        cb = oracle_throughput(cfg, target_seconds=args.cpu_seconds, single_thread=True)
        line["cpu_baseline"] = {k: cb[k] for k in ("value", "unit", "cores", "kind", "sample", "cpu_model", "single_thread")}
        line["cpu_baseline"]["rhs_evals_per_s"] = cb["rhs_evals_per_s"]
        line["paper_context"] = "paper: 0.057 inspirals/ms on 1 Xeon E5410 core (double) vs 2.7 inspirals/ms on 1 Tesla S1070 GPU (single), 'factor 50' (PAPER.md:86-96)"
    print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--workload", default="C2", choices=sorted(W.CONFIGS))
    ap.add_argument("--n", type=int, default=0, help="override the batch size (not a bench line)")
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--input-order", type=int, default=0, help="1: issue the work queue in input order instead of longest-expected-first")
    ap.add_argument("--cpu-seconds", type=float, default=15.0)
    ap.add_argument("--variant", type=int, default=0, help="pn_options.variant (kernel selection bits; not a bench line unless 0)")
    ap.add_argument("--scaling", default="weak", choices=["weak", "strong"],
                    help="weak: every rank its own full-size batch; strong: one batch split over the ranks")
    ap.add_argument("--fused", action="store_true",
                    help="a step is one sharded fused ensemble run (pn_run_ensembles through pipeline.run_ensembles): widened rows")
    ap.add_argument("--dry", action="store_true", help="launch / sharding / exchange logic only, on the CPU with gloo (tests)")
    args = ap.parse_args()
    cfg = W.CONFIGS[args.workload]
    if args.n > 0:
        cfg = W.with_size(cfg, args.n)
    spawn_ranks_if_needed(args)
    if args.dry:
        run_dry(args, cfg)
    elif args.impl == "reference":
        run_reference(args, cfg)
    elif args.fused:
        run_fused(args, cfg)
    else:
        run_ours(args, cfg)


if __name__ == "__main__":
    main()
