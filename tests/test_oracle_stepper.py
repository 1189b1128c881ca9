"""Pins of the oracle's Dormand-Prince stepper, landing rule and histogram
against closed forms, invariants and library routines.  CPU only, small batches."""
import math
from fractions import Fraction as Fr

import numpy as np
import pytest
from scipy.integrate import quad

from paper_0908_3889_b200 import workloads as W
from test_oracle_rhs import omega_dot_aligned, random_states


def test_P11_tableau_order_conditions(oracle):
    """Exact rational check of the 7-stage tableau: row sums, all 17 order conditions up to order 5
    for b (row 7), up to order 4 for b^, FSAL row, sum(e) = 0."""
    a, c, bh = oracle.tableau()
    b = a[6] + [Fr(0)]
    A = [row + [Fr(0)] for row in a]
    n = 7
    for s in range(n):
        assert sum(A[s]) == c[s]
        assert all(A[s][j] == 0 for j in range(s, n))
    assert c == [Fr(0), Fr(1, 5), Fr(3, 10), Fr(4, 5), Fr(8, 9), Fr(1), Fr(1)]
    Ac = [sum(A[i][j] * c[j] for j in range(n)) for i in range(n)]
    Ac2 = [sum(A[i][j] * c[j] ** 2 for j in range(n)) for i in range(n)]
    Ac3 = [sum(A[i][j] * c[j] ** 3 for j in range(n)) for i in range(n)]
    AAc = [sum(A[i][j] * Ac[j] for j in range(n)) for i in range(n)]
    AAc2 = [sum(A[i][j] * Ac2[j] for j in range(n)) for i in range(n)]
    AcAc = [sum(A[i][j] * c[j] * Ac[j] for j in range(n)) for i in range(n)]
    AAAc = [sum(A[i][j] * AAc[j] for j in range(n)) for i in range(n)]
    dot = lambda w, v: sum(wi * vi for wi, vi in zip(w, v))
    ones = [Fr(1)] * n
    cp = lambda p: [ci ** p for ci in c]
    mul = lambda u, v: [ui * vi for ui, vi in zip(u, v)]
    conds4 = [(ones, 1), (c, Fr(1, 2)), (cp(2), Fr(1, 3)), (Ac, Fr(1, 6)), (cp(3), Fr(1, 4)), (mul(c, Ac), Fr(1, 8)),
              (Ac2, Fr(1, 12)), (AAc, Fr(1, 24))]
    conds5 = [(cp(4), Fr(1, 5)), (mul(cp(2), Ac), Fr(1, 10)), (mul(Ac, Ac), Fr(1, 20)), (mul(c, Ac2), Fr(1, 15)),
              (Ac3, Fr(1, 20)), (mul(c, AAc), Fr(1, 30)), (AcAc, Fr(1, 40)), (AAc2, Fr(1, 60)), (AAAc, Fr(1, 120))]
    for vec, rhs in conds4 + conds5:
        assert dot(b, vec) == rhs
    for vec, rhs in conds4:
        assert dot(bh, vec) == rhs
    assert any(dot(bh, vec) != rhs for vec, rhs in conds5)   # b^ is genuinely 4th order
    assert sum(bi - bhi for bi, bhi in zip(b, bh)) == 0
    assert b[1] == 0 and bh[1] == 0


@pytest.mark.parametrize("m1", [0.5, 0.6, 0.8, 0.9])
def test_P1_leading_order_closed_form(oracle, m1):
    """Only the '1' of the brace, no spins: omega^{-8/3}(t) = omega0^{-8/3} - (256/5) eta M^{5/3} t
    (north_star), so t_f is known in closed form; also checks the landing on omega_f."""
    m2 = 1 - m1
    om0, omf = 0.005, 0.05
    y0 = np.array([[om0, 0, 0, 0, 0, 0, 0, 0, 0, 1.0]])
    r = oracle.integrate(y0, [[m1, m2]], omf, 1e-12, 1e-14, term_mask=1)
    tf = (om0 ** (-8 / 3) - omf ** (-8 / 3)) / (256 / 5 * m1 * m2)
    assert r["n_failed"] == 0
    assert abs(r["time"][0] - tf) <= 5e-12 * tf
    assert abs(r["final"][0, 0] - omf) <= 1e-13 * omf
    # same closed form at intermediate times through the fixed-step mode
    n, h = 400, tf / 800
    rf = oracle.integrate(y0, [[m1, m2]], omf, 0, 0, fixed_steps=n, h0=h, term_mask=1)
    om_half = (om0 ** (-8 / 3) - 256 / 5 * m1 * m2 * n * h) ** (-3 / 8)
    assert abs(rf["final"][0, 0] - om_half) <= 1e-12 * om_half


@pytest.mark.parametrize("m1", [0.5, 0.65, 0.9])
@pytest.mark.parametrize("c", [(1.0, 1.0), (0.7, -0.7), (-1.0, -1.0), (0.3, 0.0)])
def test_P4_aligned_spins_time_to_omega_f(oracle, m1, c):
    """Spins along +-L^: nothing precesses (state unchanged to the bit) and
    t_f = int_{omega0}^{omega_f} d omega / omega_dot(omega) with the retyped Eq. (1)."""
    m2 = 1 - m1
    om0, omf = 0.005, 0.05
    y0 = np.array([[om0, 0, 0, c[0] * m1 ** 2, 0, 0, c[1] * m2 ** 2, 0, 0, 1.0]])
    r = oracle.integrate(y0, [[m1, m2]], omf, 1e-12, 1e-14)
    assert np.array_equal(r["final"][0, 1:], y0[0, 1:])
    tq, _ = quad(lambda w: 1.0 / omega_dot_aligned(w, m1, m2, c[0], c[1]), om0, omf, epsabs=0, epsrel=1e-13, limit=200)
    assert abs(r["time"][0] - tq) <= 1e-11 * tq


def test_P2_invariants_and_landing_C1(oracle):
    """|S1|, |S2|, |L^| are conserved by Eqs. (2)-(4); every system lands on omega_f within tau."""
    cfg = W.CONFIGS["C1"]
    y0, m = W.generate(cfg)
    r = oracle.integrate(y0, m, cfg.omegaf, cfg.rtol, cfg.atol)
    assert r["n_failed"] == 0
    f = r["final"]
    assert np.abs(f[:, 0] - cfg.omegaf).max() <= 1e-13 * cfg.omegaf
    for s in (slice(1, 4), slice(4, 7), slice(7, 10)):
        n0 = np.linalg.norm(y0[:, s], axis=1)
        n1 = np.linalg.norm(f[:, s], axis=1)
        assert np.abs(n1 / n0 - 1).max() < 2e-9
    # ~10 % spread of run lengths between inspirals: sanity only
    assert 0.03 < r["steps"].std() / r["steps"].mean() < 0.3
    assert np.all(r["steps"] == r["steps"].astype(int)) and r["steps"].min() > 50


def test_P6_step_halving_order_5(oracle):
    """Fixed-step mode: the error against a fine reference falls by 2^5 per halving of h."""
    cfg = W.with_size(W.CONFIGS["C1"], 8)
    y0, m = W.generate(cfg)
    T = 1600.0
    ref = oracle.integrate(y0, m, 0, 0, 0, fixed_steps=3200, h0=T / 3200)["final"]
    errs = []
    for n in (25, 50, 100, 200):
        f = oracle.integrate(y0, m, 0, 0, 0, fixed_steps=n, h0=T / n)["final"]
        errs.append(np.abs(f - ref).max(axis=1))
    errs = np.array(errs)
    ratios = errs[:-1] / errs[1:]
    assert np.all(ratios > 24) and np.all(ratios < 45), ratios


def test_P12_tolerance_self_convergence(oracle):
    """rtol 1e-10 against rtol 1e-13 of the same oracle: the 1e-7 parity bars are attainable."""
    for name, nsys in (("C2", 32), ("C3", 32), ("C5", 8)):
        cfg = W.with_size(W.CONFIGS[name], nsys)
        y0, m = W.generate(cfg)
        a = oracle.integrate(y0, m, cfg.omegaf, 1e-10, 1e-12)
        b = oracle.integrate(y0, m, cfg.omegaf, 1e-13, 1e-15)
        assert a["n_failed"] == 0 and b["n_failed"] == 0
        da = oracle.histogram(a["final"], 50)[2]
        db = oracle.histogram(b["final"], 50)[2]
        ok = np.isfinite(da) & np.isfinite(db)
        assert np.abs(da - db)[ok].max() < 5e-8, name
        assert np.abs(a["time"] / b["time"] - 1).max() < 1e-9, name


def test_P5_P7_P8_through_the_stepper(oracle):
    cfg = W.with_size(W.CONFIGS["C3"], 12)
    y0, m = W.generate(cfg)
    kw = dict(rtol=1e-12, atol=1e-14)
    a = oracle.integrate(y0, m, cfg.omegaf, **kw)
    # P5: relabel 1<->2
    ys = y0.copy(); ys[:, 1:4], ys[:, 4:7] = y0[:, 4:7], y0[:, 1:4]
    b = oracle.integrate(ys, m[:, ::-1], cfg.omegaf, **kw)
    assert np.abs(b["time"] / a["time"] - 1).max() < 1e-11
    assert np.abs(b["final"][:, 7:10] - a["final"][:, 7:10]).max() < 1e-9
    assert np.abs(b["final"][:, 1:4] - a["final"][:, 4:7]).max() < 1e-9
    # P7: scale freedom
    lam = 2.0
    yl = y0.copy(); yl[:, 0] /= lam; yl[:, 1:7] *= lam ** 2
    c = oracle.integrate(yl, m * lam, cfg.omegaf / lam, 1e-12, 1e-14, h0=10 * lam)
    assert np.abs(c["time"] / (lam * a["time"]) - 1).max() < 1e-11
    assert np.abs(c["final"][:, 7:10] - a["final"][:, 7:10]).max() < 1e-9
    assert np.abs(c["final"][:, 1:7] / lam ** 2 - a["final"][:, 1:7]).max() < 1e-9
    # P8: rotation covariance
    from scipy.spatial.transform import Rotation
    R = Rotation.random(random_state=1).as_matrix()
    yr = y0.copy()
    for s in (slice(1, 4), slice(4, 7), slice(7, 10)):
        yr[:, s] = y0[:, s] @ R.T
    d = oracle.integrate(yr, m, cfg.omegaf, **kw)
    assert np.abs(d["time"] / a["time"] - 1).max() < 1e-11
    for s in (slice(1, 4), slice(4, 7), slice(7, 10)):
        assert np.abs(d["final"][:, s] @ R - a["final"][:, s]).max() < 1e-9


def test_equal_mass_exchange_symmetry(oracle):
    """north_star: exchange symmetry 1<->2 for equal masses (swap the spins only)."""
    cfg = W.with_size(W.CONFIGS["C1"], 16)
    y0, m = W.generate(cfg)
    a = oracle.integrate(y0, m, cfg.omegaf, 1e-12, 1e-14)
    ys = y0.copy(); ys[:, 1:4], ys[:, 4:7] = y0[:, 4:7], y0[:, 1:4]
    b = oracle.integrate(ys, m, cfg.omegaf, 1e-12, 1e-14)
    assert np.abs(b["final"][:, 1:4] - a["final"][:, 4:7]).max() < 1e-10
    assert np.abs(b["final"][:, 7:10] - a["final"][:, 7:10]).max() < 1e-10
    assert np.abs(b["time"] / a["time"] - 1).max() < 1e-12


def test_P14_histogram_against_numpy(oracle):
    rng = np.random.default_rng(0)
    n = 20000
    y = rng.normal(size=(n, 10))
    y[5, 1:4] = 0.0                       # |S1| = 0 -> skipped in the two histograms that use S1
    y[6, 7:10] = y[6, 1:4] * 2.5          # d = +1 exactly -> last bin
    y[7, 4:7] = -3 * y[7, 7:10]           # d = -1 -> first bin
    for bins in (1, 20, 50, 100):
        counts, skipped, dots = oracle.histogram(y, bins)
        S1, S2, L = y[:, 1:4], y[:, 4:7], y[:, 7:10]
        def ud(a, b):
            with np.errstate(invalid="ignore", divide="ignore"):
                return np.einsum("ij,ij->i", a, b) / (np.linalg.norm(a, axis=1) * np.linalg.norm(b, axis=1))
        for h, d in enumerate((ud(S1, S2), ud(S1, L), ud(S2, L))):
            ok = np.isfinite(d)
            assert skipped[h] == (~ok).sum()
            ref, _ = np.histogram(np.clip(d[ok], -1, 1), bins=bins, range=(-1, 1))
            # numpy and the oracle may disagree only for samples within a few ulp of a bin edge
            edges = np.linspace(-1, 1, bins + 1)[1:-1]
            near = (np.abs(d[ok][:, None] - edges[None, :]) < 1e-14).sum() if bins > 1 else 0
            assert np.abs(counts[h].astype(np.int64) - ref).sum() <= 2 * near
            assert counts[h].sum() == ok.sum()
            assert np.allclose(dots[ok, h], d[ok], rtol=0, atol=1e-15)
    c50 = oracle.histogram(y, 50)[0]
    assert c50[1, 49] >= 1 and c50[2, 0] >= 1


def test_failure_codes(oracle):
    y0 = np.array([[0.02, 0, 0, 0.1, 0, 0, 0.1, 0, 0, 1.0]])
    r = oracle.integrate(y0, [[0.5, 0.5]], 0.05, 1e-10, 1e-12, max_steps=5)
    assert r["steps"][0] == oracle.FAIL_MAXSTEPS and r["n_failed"] == 1
    r = oracle.integrate(y0, [[0.5, 0.5]], 0.01, 1e-10, 1e-12)          # omega_f below omega_0
    assert r["steps"][0] == oracle.FAIL_BADINPUT
    r = oracle.integrate(y0, [[0.5, -0.5]], 0.05, 1e-10, 1e-12)
    assert r["steps"][0] == oracle.FAIL_BADINPUT
