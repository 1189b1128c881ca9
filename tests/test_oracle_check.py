"""Pins of the cross-check oracle (oracle/pn_check_oracle.py)."""
import numpy as np

from oracle import pn_check_oracle as C
from paper_0908_3889_b200 import workloads as W


def test_selection_against_numpy_generator():
    for seed, n, frac in ((0, 10000, 0.01), (5, 77777, 0.013), (9, 1000, 0.5), (2, 100, 0.0), (2, 100, 1.0)):
        key = W.philox_key(seed)
        u = np.random.Generator(np.random.Philox(seed)).random(n)          # numpy's own Philox, same stream
        assert np.array_equal(C.selection(n, frac, key), np.nonzero(u < frac)[0])
    # size follows the binomial law: n p +- 5 sigma
    idx = C.selection(1_000_000, 0.01, (123, 456))
    assert abs(idx.size - 10000) < 5 * np.sqrt(10000 * 0.99)
    assert np.all(np.diff(idx) > 0) and idx.min() >= 0 and idx.max() < 1_000_000
    # roughly evenly spread: no decile of the index range is starved
    assert np.histogram(idx, bins=10, range=(0, 1_000_000))[0].min() > 800


def test_selfcheck_zero_and_planted_deviation(oracle):
    cfg = W.with_size(W.CONFIGS["C1"], 600)
    y0, m = W.generate(cfg)
    full = oracle.integrate(y0, m, cfg.omegaf, 1e-10, 1e-12)
    key = (42, 43)
    r = C.selfcheck(y0, m, full["final"], full["time"], cfg.omegaf, 0.1, key)
    assert r["n_checked"] == C.selection(600, 0.1, key).size > 30 and r["n_failed_ref"] == 0
    assert r["max_dot_dev"].max() == 0.0 and r["max_time_rel_dev"] == 0.0      # the same integrator on the same inputs
    # plant a rotation of S1 about z by 1e-3 rad in one selected system: S1^.S2^ moves, S1^.L^ does not (L^ ~ z? no: use exact algebra)
    j = int(r["indices"][7])
    bad = full["final"].copy()
    s1 = bad[j, 1:4].copy()
    ax = bad[j, 7:10] / np.linalg.norm(bad[j, 7:10])                         # rotate about L^: S1^.L^ is unchanged
    th = 1e-3
    bad[j, 1:4] = s1 * np.cos(th) + np.cross(ax, s1) * np.sin(th) + ax * np.dot(ax, s1) * (1 - np.cos(th))
    r2 = C.selfcheck(y0, m, bad, full["time"], cfg.omegaf, 0.1, key)
    s2 = bad[j, 4:7]
    want = abs(np.dot(bad[j, 1:4], s2) - np.dot(s1, s2)) / (np.linalg.norm(s1) * np.linalg.norm(s2))
    assert r2["worst_index"][0] == j and abs(r2["max_dot_dev"][0] - want) < 1e-15
    assert r2["max_dot_dev"][1] < 1e-15 and r2["max_dot_dev"][2] == 0.0
    # a system outside the subset is not looked at
    out = int(np.setdiff1d(np.arange(600), r["indices"])[0])
    bad2 = full["final"].copy(); bad2[out, 1:4] *= -1.0
    assert C.selfcheck(y0, m, bad2, None, cfg.omegaf, 0.1, key)["max_dot_dev"].max() == 0.0
