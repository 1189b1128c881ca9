"""Pins of the statistics oracle (oracle/pn_stats_oracle.py) against what the paper and the mathematics
fix: hand-computed values, closed forms, invariances, and independent library routines."""
import numpy as np
import pytest
from scipy.stats import pearsonr

from oracle import pn_stats_oracle as S
from paper_0908_3889_b200 import workloads as W


def rng(seed):
    return np.random.Generator(np.random.Philox(seed))


def test_pearson_hand_computed():
    # x = 1..5, y = (2,1,4,3,5): xbar = ybar = 3, sum dx dy = 8, sum dx^2 = sum dy^2 = 10 -> r = 0.8 (by hand)
    assert S.pearson_r([1, 2, 3, 4, 5], [2, 1, 4, 3, 5]) == pytest.approx(0.8, abs=1e-15)
    # orthogonal contrasts: x = (-1,0,1), y = (1,-2,1) -> sum dx dy = 0 -> r = 0
    assert S.pearson_r([-1, 0, 1], [1, -2, 1]) == pytest.approx(0.0, abs=1e-16)
    # x = (0,0,1,1), y = (0,1,0,1): independent 2x2 design -> r = 0; y = x -> 1
    assert S.pearson_r([0, 0, 1, 1], [0, 1, 0, 1]) == pytest.approx(0.0, abs=1e-16)
    # (1,2,3) vs (1,2,4): dx = (-1,0,1), dy = (-4/3,-1/3,5/3): sum dxdy = 3, M2x = 2, M2y = 42/9 -> r = 3/sqrt(28/3)
    assert S.pearson_r([1, 2, 3], [1, 2, 4]) == pytest.approx(3.0 / np.sqrt(28.0 / 3.0), abs=1e-15)


def test_pearson_closed_forms_and_invariances():
    g = rng(1)
    x = g.uniform(-1, 1, 5000)
    y = 0.3 * x + g.normal(0, 0.2, 5000)
    r = S.pearson_r(x, y)
    assert S.pearson_r(x, 2.5 * x - 7.0) == pytest.approx(1.0, abs=1e-14)        # exact linear dependence
    assert S.pearson_r(x, -0.1 * x + 3.0) == pytest.approx(-1.0, abs=1e-14)
    assert S.pearson_r(y, x) == pytest.approx(r, abs=1e-15)                      # symmetry
    assert S.pearson_r(4 * x + 1, 0.5 * y - 2) == pytest.approx(r, abs=1e-13)    # affine invariance
    assert S.pearson_r(-x, y) == pytest.approx(-r, abs=1e-15)
    assert abs(r) <= 1.0
    # population model: r -> a sx / sqrt(a^2 sx^2 + s^2) = 0.3 sqrt(1/3) / sqrt(0.09/3 + 0.04)
    assert r == pytest.approx(0.3 * np.sqrt(1 / 3) / np.sqrt(0.03 + 0.04), abs=0.02)
    # reading R18: sample standard deviations (N-1): r equals Cxy / sqrt(M2x M2y) of the moments
    m = S.moments(x, y)
    assert r == pytest.approx(m["Cxy"] / np.sqrt(m["M2x"] * m["M2y"]), abs=1e-14)
    # the population-sigma reading would differ by the factor N/(N-1); make sure we are not on it
    assert abs(r * 5000 / 4999 - r) > 1e-6


def test_pearson_against_scipy():
    g = rng(2)
    for n in (2, 3, 17, 1000, 100000):
        x = g.uniform(-1, 1, n)
        y = np.clip(x + g.normal(0, 0.5, n), -1, 1)
        assert S.pearson_r(x, y) == pytest.approx(pearsonr(x, y)[0], abs=1e-13)
        assert S.pearson_r(x, y) == pytest.approx(np.corrcoef(x, y)[0, 1], abs=1e-13)
    # large offset, small spread: the two-pass definition does not lose digits
    x = 0.5 + 1e-6 * g.normal(size=4000)
    y = 0.25 + 1e-6 * (x - 0.5) * 1e6 * 0.7 + 1e-6 * g.normal(size=4000)
    assert S.pearson_r(x, y) == pytest.approx(pearsonr(x, y)[0], abs=1e-10)
    assert np.isnan(S.pearson_r([0.5, 0.5, 0.5], [0.1, 0.2, 0.3]))               # sigma_x = 0: undefined
    assert np.isnan(S.pearson_r([0.5], [0.1]))


def test_moments_definition():
    x = np.array([1.0, 2.0, 4.0, 7.0])
    y = np.array([1.0, 3.0, 2.0, 6.0])
    m = S.moments(x, y)
    assert m["n"] == 4 and m["mean_x"] == 3.5 and m["mean_y"] == 3.0
    assert m["M2x"] == pytest.approx(21.0) and m["M2y"] == pytest.approx(14.0)   # by hand
    assert m["Cxy"] == pytest.approx(2.5 * 2 + 1.5 * 0 + 0.5 * -1 + 3.5 * 3)     # = 15


def test_bin_rule_by_hand():
    # R14 on 4 bins: edges -1, -0.5, 0, 0.5, 1; d = +1 in the last bin, d = -1 in the first
    d = np.array([-1.0, -0.75, -0.5, -1e-9, 0.0, 0.49999, 0.5, 1.0, np.nextafter(1.0, 0)])
    assert list(S.bin_index(d, 4)) == [0, 0, 1, 1, 2, 2, 3, 3, 3]
    assert list(S.bin_index([-1.0, 1.0, 0.3], 1)) == [0, 0, 0]
    assert list(S.histogram1d(d, 4)) == [2, 2, 2, 3]


def test_histogram2d_by_hand_and_numpy():
    x = np.array([-0.9, -0.9, 0.1, 0.9, 1.0, -1.0])
    y = np.array([-0.9, 0.9, 0.1, 0.9, 1.0, 1.0])
    c, nrm = S.histogram2d(x, y, 2)
    # bins: [-1,0) -> 0, [0,1] -> 1.  pairs: (0,0), (0,1), (1,1), (1,1), (1,1), (0,1)
    assert c.tolist() == [[1, 2], [0, 3]]
    assert nrm.tolist() == [[1 / 3, 2 / 3], [0.0, 1.0]]           # maximum normalised to 1
    g = rng(3)
    for bins in (1, 7, 79, 200):
        x = g.uniform(-1, 1, 20000)
        y = np.clip(0.9 * x + g.normal(0, 0.2, 20000), -1, 1)
        c, nrm = S.histogram2d(x, y, bins)
        edges = np.linspace(-1.0, 1.0, bins + 1)
        ref, _, _ = np.histogram2d(x, y, bins=[edges, edges])
        # numpy computes bin edges differently; samples within 1e-12 of an edge may fall either side
        frac = (np.stack([x, y]) + 1.0) * bins / 2.0
        near = np.any(np.abs(frac - np.round(frac)) < 1e-9, axis=0)
        assert np.abs(c.astype(np.int64) - ref.astype(np.int64)).sum() <= 2 * np.count_nonzero(near)
        assert c.sum() == 20000
        assert nrm.max() == 1.0 and nrm.min() >= 0.0
        assert np.array_equal(c.sum(axis=0), S.histogram1d(y, bins))     # marginals
        assert np.array_equal(c.sum(axis=1), S.histogram1d(x, bins))


def test_unit_dots_against_c_oracle_and_geometry(oracle):
    cfg = W.with_size(W.CONFIGS["C3"], 3000)
    y0, _ = W.generate(cfg)
    y0[5, 1:4] = 0.0            # zero spin: undefined dots are skipped
    y0[9, 4:7] = 0.0
    d = S.unit_dots(y0)
    _, skipped, d_c = oracle.histogram(y0, 50)
    assert np.array_equal(np.isnan(d), np.isnan(d_c))
    assert np.nanmax(np.abs(d - d_c)) < 4e-16
    assert skipped.tolist() == [2, 1, 1]
    # L^ = z: S_i^.L^ is the z-component of the unit spin; hand-built vectors
    y = np.zeros((2, 10))
    y[:, 9] = 1.0
    y[0, 1:4] = [0.0, 0.0, 2.0]
    y[0, 4:7] = [3.0, 0.0, 0.0]
    y[1, 1:4] = [1.0, 1.0, 0.0]
    y[1, 4:7] = [0.0, 2.0, 2.0]
    assert np.allclose(S.unit_dots(y), [[0.0, 1.0, 0.0], [0.5, 0.0, np.sqrt(0.5)]], atol=1e-16)


def test_statistics_groups_and_marginals(oracle):
    # two ensembles in one batch (a sweep): each group's statistics equal those of the
    # group run alone, hist1 equals the C oracle's histogram of the same final states, hist2 marginals match
    cfg = W.with_size(W.CONFIGS["C3"], 4000)
    y0, _ = W.generate(cfg)
    g = rng(4)
    rot = g.normal(size=(4000, 10)) * 0.05
    yf = y0 + rot * np.abs(y0).max()            # any "final" states: the statistics do not care where they come from
    steps = np.full(4000, 100, dtype=np.int32)
    steps[[7, 2500]] = -3                        # failed systems are left out
    st = S.statistics(y0, yf, steps, group_size=2000, bins1=50, bins2=79)
    for grp in range(2):
        sl = slice(2000 * grp, 2000 * (grp + 1))
        alone = S.statistics(y0[sl], yf[sl], steps[sl], bins1=50, bins2=79)
        for k in ("r", "moments", "hist1", "hist2", "hist2_max", "skipped"):
            assert np.array_equal(st[k][grp], alone[k][0], equal_nan=True), k
        ok = steps[sl] >= 0
        c_ref, _, _ = oracle.histogram(yf[sl][ok], 50)
        assert np.array_equal(st["hist1"][grp], c_ref)
        assert np.array_equal(st["hist2"][grp].sum(axis=1), S.statistics(y0[sl], yf[sl], steps[sl], bins1=79)["hist1"][0])
        assert np.all(st["moments"][grp, :, 0] + st["skipped"][grp] == 2000)
        assert st["skipped"][grp].tolist() == [1, 1, 1]
        d0, d1 = S.unit_dots(y0[sl][ok]), S.unit_dots(yf[sl][ok])
        for k in range(3):
            assert st["r"][grp, k] == pytest.approx(pearsonr(d0[:, k], d1[:, k])[0], abs=1e-13)
