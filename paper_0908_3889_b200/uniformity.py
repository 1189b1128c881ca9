"""The paper's large uniformity run (Fig. 3) on one GPU: equal masses, chi_1 = chi_2 = 0.7, isotropic
spins, omega 0.00395 -> 0.05, N = 362,799,815 inspirals, 100 bins.  A demo of the library calls, not part of the hot path
(SURVEY.md marks the experiment out of scope).

    python -m paper_0908_3889_b200.uniformity [--n N] [--precision fp64|fp32|mixed] [--tol T] [--unfused] [--chunk C]

FP64 (default): ONE fused call, pn_run_ensembles -- the key goes in, 3 x 100 counters come out, no state array exists
(DESIGN.md 14).  --unfused, or FP32 / mixed (which have no fused kernel): the chunked reference loop, every chunk
pn_generate(first, count) -> pn_integrate -> pn_statistics(final-only histogram) on device buffers allocated once.  Prints one JSON line with
the histogram of the final S1^.S2^, its flatness (largest deviation of the binned CDF from the uniform CDF and the
chi-square statistic against equal bin contents) and the throughput.  The paper quotes a K-S "p-value of 5.17e-5";
the K-S statistic itself needs the unbinned sample and is analysis outside this library.
"""
from __future__ import annotations

import argparse
import json
import time


def main():
    import numpy as np
    import torch

    import paper_0908_3889_b200 as pn

    ap = argparse.ArgumentParser()
    ap.add_argument("--n", type=int, default=362_799_815)
    ap.add_argument("--chunk", type=int, default=1 << 22)
    ap.add_argument("--precision", default="fp64", choices=["fp64", "fp32", "mixed"])
    ap.add_argument("--tol", type=float, default=5e-7, help="rtol = atol (PAPER.md:66: 5e-7)")
    ap.add_argument("--chi", type=float, default=0.7)
    ap.add_argument("--bins", type=int, default=100)
    ap.add_argument("--key", type=int, nargs=2, default=(908, 3889))
    ap.add_argument("--unfused", action="store_true", help="the chunked generate -> integrate -> statistics loop")
    a = ap.parse_args()
    prec = {"fp64": pn.PN_FP64, "fp32": pn.PN_FP32, "mixed": pn.PN_MIXED}[a.precision]
    dev = torch.device("cuda:0")
    c = min(a.chunk, a.n)
    h1 = torch.zeros(1, 3, a.bins, dtype=torch.int64, device=dev)
    skipped = torch.zeros(1, 3, dtype=torch.int64, device=dev)
    total = torch.zeros(3, a.bins, dtype=torch.int64, device=dev)
    ens = pn.make_ensemble(tuple(a.key), 0.00395, q=(1.0, 1.0), chi1=(a.chi, a.chi), chi2=(a.chi, a.chi))
    n_skipped = n_failed = trial_steps = 0
    fused = prec == pn.PN_FP64 and not a.unfused
    if not fused:
        y0 = torch.empty(c, 10, dtype=torch.float64, device=dev)
        m = torch.empty(c, 2, dtype=torch.float64, device=dev)
        yf = torch.empty_like(y0)
        steps = torch.empty(c, dtype=torch.int32, device=dev)
    torch.cuda.synchronize()
    t0 = time.perf_counter()
    if fused:
        pn.pn_run_ensembles(ens, a.n, 0.05, a.tol, a.tol, bins1=a.bins, hist1=h1, n_skipped=skipped, allow_failures=True)
        k = pn.pn_last_counters()
        n_failed, trial_steps = k["failed"], k["trial_steps"]
        total += h1[0]
        n_skipped = int(skipped[0, 0].item())
    for first in (() if fused else range(0, a.n, c)):
        cnt = min(c, a.n - first)
        pn.pn_generate(ens, a.n, y0[:cnt], m[:cnt], first=first, count=cnt)
        st = pn.pn_integrate(y0[:cnt], m[:cnt], 0.00395, 0.05, a.tol, a.tol, prec, yf[:cnt], steps[:cnt], allow_failures=True)
        k = pn.pn_last_counters()
        n_failed += k["failed"]; trial_steps += k["trial_steps"]
        pn.pn_statistics(None, yf[:cnt], steps[:cnt], bins1=a.bins, hist1=h1, n_skipped=skipped)
        total += h1[0]
        n_skipped += int(skipped[0, 0].item())
    torch.cuda.synchronize()
    dt = time.perf_counter() - t0
    h = total.cpu().numpy()
    n_ok = int(h[0].sum())
    cdf = np.cumsum(h[0]) / n_ok
    d_binned = float(np.abs(cdf - np.arange(1, a.bins + 1) / a.bins).max())
    chi2 = float(((h[0] - n_ok / a.bins) ** 2 / (n_ok / a.bins)).sum())
    print(json.dumps({"n": a.n, "mode": "fused pn_run_ensembles" if fused else f"unfused, chunks of {c}", "precision": a.precision, "tol": a.tol, "chi": a.chi, "seconds": dt,
                      "inspirals_per_sec": a.n / dt, "trial_steps_per_inspiral": trial_steps / a.n, "failed": n_failed,
                      "skipped": n_skipped, "binned_ks_distance": d_binned, "chi2": chi2, "chi2_dof": a.bins - 1,
                      "relative_spread_of_bins": float(h[0].std() / h[0].mean()),
                      "poisson_relative_spread": float(1.0 / np.sqrt(n_ok / a.bins)),
                      "hist_S1S2": h[0].tolist()}))


if __name__ == "__main__":
    main()
