"""CPU oracle of the ensemble statistics.  TEST INFRASTRUCTURE, NOT THE PRODUCT.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may import this
module.  It imports nothing from paper_0908_3889_b200, and shares no code with the CUDA path or with
oracle/pn_oracle.c (whose C histogram is used by the tests as an independent cross-check of `unit_dots`
and of the marginals of `histogram2d`).

What it computes, each as the plain definition in float64 numpy (two passes, no blocking, no merging):

  unit_dots     d = (A.B)/(|A||B|) for (S1,S2), (S1,L^), (S2,L^); norms from the state itself
                (R14).  A zero norm or a non-finite quotient -> NaN (skipped).
  pearson_r     r = 1/(N-1) sum_i ((x_i - xbar)/sigma_x) ((y_i - ybar)/sigma_y), xbar, ybar the sample
                means, sigma the standard deviations (typed as printed).  Reading R18
                (DESIGN.md 3): sigma is the SAMPLE standard deviation (divisor N-1), so |r| <= 1.
  moments       n, xbar, ybar, M2x = sum (x-xbar)^2, M2y, Cxy = sum (x-xbar)(y-ybar).
  histogram2d   bivariate counts of (x, y) = (initial, final) dot product on bins x bins equal cells of
                [-1,1]^2, bin rule of R14 on each axis (floor((d+1) bins/2), clamped, d = +1 in the last
                bin); `normalised` = counts / max(counts) ("normalized such that the maximum
                value is 1").
  statistics    all of the above per ensemble ("group"): group g = systems [g*group_size, (g+1)*group_size)
                (parameter sweeps, Figs. 6-7), x from init_states, y from final_states;
                a system is left out of a dot product's statistics if either of its two values is NaN, and
                out of everything if steps[i] < 0 (failed integration).

Parity unpinned: none.  Pins: tests/test_oracle_stats.py (hand-computed r, closed forms, invariances,
scipy.stats.pearsonr, numpy.histogram2d, marginals against the C oracle's 1-D histogram).
"""
from __future__ import annotations

import numpy as np

NAMES = ("S1S2", "S1L", "S2L")


def unit_dots(states) -> np.ndarray:
    """dots[n,3] = S1^.S2^, S1^.L^, S2^.L^ of states[n,10] (NaN where undefined)."""
    y = np.atleast_2d(np.asarray(states, dtype=np.float64))
    S1, S2, L = y[:, 1:4], y[:, 4:7], y[:, 7:10]
    n1 = np.sqrt(np.sum(S1 * S1, axis=1))
    n2 = np.sqrt(np.sum(S2 * S2, axis=1))
    nl = np.sqrt(np.sum(L * L, axis=1))
    out = np.full((y.shape[0], 3), np.nan)
    with np.errstate(divide="ignore", invalid="ignore"):
        pairs = ((S1, S2, n1, n2), (S1, L, n1, nl), (S2, L, n2, nl))
        for k, (A, B, na, nb) in enumerate(pairs):
            d = np.sum(A * B, axis=1) / (na * nb)
            ok = (na > 0) & (nb > 0) & np.isfinite(d)
            out[ok, k] = d[ok]
    return out


def moments(x, y) -> dict:
    """Two-pass sample moments of the pairs (x_i, y_i)."""
    x = np.asarray(x, dtype=np.float64)
    y = np.asarray(y, dtype=np.float64)
    n = x.size
    if n == 0:
        return dict(n=0, mean_x=np.nan, mean_y=np.nan, M2x=0.0, M2y=0.0, Cxy=0.0)
    xbar = np.sum(x) / n
    ybar = np.sum(y) / n
    dx, dy = x - xbar, y - ybar
    return dict(n=n, mean_x=xbar, mean_y=ybar, M2x=float(np.sum(dx * dx)), M2y=float(np.sum(dy * dy)),
                Cxy=float(np.sum(dx * dy)))


def pearson_r(x, y) -> float:
    """PAPER.md:138 as printed: r = 1/(N-1) sum ((x_i - xbar)/sigma_x)((y_i - ybar)/sigma_y)."""
    x = np.asarray(x, dtype=np.float64)
    y = np.asarray(y, dtype=np.float64)
    N = x.size
    if N < 2:
        return float("nan")
    xbar = np.sum(x) / N
    ybar = np.sum(y) / N
    sigma_x = np.sqrt(np.sum((x - xbar) ** 2) / (N - 1))       # R18: sample standard deviation
    sigma_y = np.sqrt(np.sum((y - ybar) ** 2) / (N - 1))
    with np.errstate(divide="ignore", invalid="ignore"):
        return float(np.sum(((x - xbar) / sigma_x) * ((y - ybar) / sigma_y)) / (N - 1))


def bin_index(d, bins: int) -> np.ndarray:
    """R14: bin = clamp(floor((d+1) bins/2), 0, bins-1)."""
    b = np.floor((np.asarray(d, dtype=np.float64) + 1.0) * float(bins) / 2.0)
    return np.clip(b, 0, bins - 1).astype(np.int64)


def histogram1d(d, bins: int) -> np.ndarray:
    counts = np.zeros(bins, dtype=np.uint64)
    np.add.at(counts, bin_index(d, bins), 1)
    return counts


def histogram2d(x, y, bins: int):
    """counts[bins,bins] with row = bin of x (initial), column = bin of y (final); and counts/max."""
    counts = np.zeros((bins, bins), dtype=np.uint64)
    if np.size(x):
        np.add.at(counts, (bin_index(x, bins), bin_index(y, bins)), 1)
    mx = counts.max() if counts.size else 0
    norm = counts.astype(np.float64) / float(mx) if mx > 0 else np.zeros((bins, bins))
    return counts, norm


def statistics(init_states, final_states, steps=None, group_size: int | None = None, bins1: int = 0,
               bins2: int = 0) -> dict:
    """Per-group Pearson r, moments, 1-D histograms of the final dots and bivariate histograms.

    Returns dict of arrays with leading dimension G = N / group_size:
      r[G,3], moments[G,3,6] (n, mean_x, mean_y, M2x, M2y, Cxy), skipped[G,3],
      hist1[G,3,bins1] (final dots), hist2[G,3,bins2,bins2], hist2_max[G,3], hist2_norm[G,3,bins2,bins2].
    """
    d0 = unit_dots(init_states)
    d1 = unit_dots(final_states)
    N = d0.shape[0]
    assert d1.shape[0] == N
    gs = N if not group_size else int(group_size)
    assert gs > 0 and N % gs == 0
    G = N // gs if N else 0
    failed = np.zeros(N, dtype=bool) if steps is None else (np.asarray(steps) < 0)
    out = dict(r=np.full((G, 3), np.nan), moments=np.zeros((G, 3, 6)), skipped=np.zeros((G, 3), dtype=np.uint64),
               hist1=np.zeros((G, 3, bins1), dtype=np.uint64), hist2=np.zeros((G, 3, bins2, bins2), dtype=np.uint64),
               hist2_max=np.zeros((G, 3), dtype=np.uint64), hist2_norm=np.zeros((G, 3, bins2, bins2)))
    for g in range(G):
        sl = slice(g * gs, (g + 1) * gs)
        for k in range(3):
            x, y = d0[sl, k], d1[sl, k]
            ok = np.isfinite(x) & np.isfinite(y) & ~failed[sl]
            out["skipped"][g, k] = np.count_nonzero(~ok)
            x, y = x[ok], y[ok]
            m = moments(x, y)
            out["moments"][g, k] = [m["n"], m["mean_x"], m["mean_y"], m["M2x"], m["M2y"], m["Cxy"]]
            out["r"][g, k] = pearson_r(x, y)
            if bins1:
                out["hist1"][g, k] = histogram1d(y, bins1)
            if bins2:
                c, nrm = histogram2d(x, y, bins2)
                out["hist2"][g, k] = c
                out["hist2_max"][g, k] = c.max()
                out["hist2_norm"][g, k] = nrm
    return out
