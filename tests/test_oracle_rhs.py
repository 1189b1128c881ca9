"""Pins of the oracle's right-hand side (Eqs. (1)-(4)) against what the paper and
the mathematics fix.  CPU only.  None of these re-types the oracle's own code path: Eq. (1) is
re-transcribed here in a different form (exact fractions, aligned-spin special case), the rest are
identities, symmetries and stored values of a second transcription."""
import math
import os
from fractions import Fraction as Fr

import numpy as np
import pytest

HERE = os.path.dirname(os.path.abspath(__file__))
PI = math.pi
GAMMA_E = 0.5772156649015329


def omega_dot_aligned(omega, m1, m2, c1, c2):
    """Independent transcription of Eq. (1) for spins (anti-)aligned with L^:
    c_i = chi_i * (L^.S^_i) in [-1, 1], so S^_1.S^_2 = sign(c1 c2) and chi_1 chi_2 S^_1.S^_2 = c1 c2."""
    M = m1 + m2
    eta = m1 * m2 / M ** 2
    x = M * omega
    th = float(Fr(1039, 4620))
    t0 = 1.0
    t2 = -float(Fr(743, 336)) - float(Fr(924, 336)) * eta
    t3 = -((c1 * (113 * m1 ** 2 / M ** 2 + 75 * eta) + c2 * (113 * m2 ** 2 / M ** 2 + 75 * eta)) / 12.0 - 4 * PI)
    t4 = float(Fr(34103, 18144)) + float(Fr(13661, 2016)) * eta + float(Fr(59, 18)) * eta ** 2
    t4s = -(eta / 48.0) * (247 * c1 * c2 - 721 * c1 * c2)
    t5 = -(4159 + 15876 * eta) * PI / 672.0
    t6 = (float(Fr(16447322263, 139708800)) - float(Fr(1712, 105)) * GAMMA_E + float(Fr(16, 3)) * PI ** 2
          + (-float(Fr(273811877, 1088640)) + float(Fr(451, 48)) * PI ** 2 - float(Fr(88, 3)) * th) * eta
          + float(Fr(541, 896)) * eta ** 2 - float(Fr(5605, 2592)) * eta ** 3
          - float(Fr(856, 105)) * math.log(16 * x ** (2 / 3)))
    t7 = (-float(Fr(4415, 4032)) + float(Fr(358675, 6048)) * eta + float(Fr(91495, 1512)) * eta ** 2) * PI
    brace = (t0 + t2 * x ** (2 / 3) + t3 * x + (t4 + t4s) * x ** (4 / 3) + t5 * x ** (5 / 3) + t6 * x ** 2
             + t7 * x ** (7 / 3))
    return omega ** 2 * 96 / 5 * eta * x ** (5 / 3) * brace


def random_states(n, seed, qlo=0.1, M=1.0):
    rng = np.random.default_rng(seed)
    q = rng.uniform(qlo, 1, n)
    m1 = M / (1 + q)
    m2 = M * q / (1 + q)
    def unit():
        v = rng.normal(size=(n, 3))
        return v / np.linalg.norm(v, axis=1, keepdims=True)
    y = np.empty((n, 10))
    y[:, 0] = rng.uniform(0.001, 0.1, n) / M
    y[:, 1:4] = (rng.uniform(0, 1, n) * m1 ** 2)[:, None] * unit()
    y[:, 4:7] = (rng.uniform(0, 1, n) * m2 ** 2)[:, None] * unit()
    y[:, 7:10] = unit()
    return y, np.stack([m1, m2], 1)


def test_P10_second_transcription(oracle):
    """Stored values of a second transcription (tests/golden/rhs_values.txt)."""
    for line in open(os.path.join(HERE, "golden", "rhs_values.txt")):
        if line.startswith("#") or not line.strip():
            continue
        head, ys, fs = line.split("|")
        m = np.array([[float(t) for t in head.split()[1:]]])
        y = np.array([[float(t) for t in ys.split()]])
        fexp = np.array([float(t) for t in fs.split()])
        f = oracle.rhs(y, m)[0]
        scale = np.array([abs(fexp[0])] + [np.abs(fexp[1:4]).max()] * 3 + [np.abs(fexp[4:7]).max()] * 3
                         + [np.abs(fexp[7:10]).max()] * 3)
        assert np.all(np.abs(f - fexp) <= 2e-13 * scale), (f, fexp)


@pytest.mark.parametrize("m1", [0.5, 0.6, 0.8, 0.9])
@pytest.mark.parametrize("c", [(1.0, 1.0), (0.7, -0.7), (-1.0, -1.0), (0.3, 0.0), (0.0, 0.0)])
def test_P4_aligned_rhs_matches_retyped_eq1(oracle, m1, c):
    """Aligned spins: no precession at all (S_dot = L_dot = 0 exactly) and omega_dot equals the
    independently retyped Eq. (1); covers every coefficient incl. spin-orbit, spin-spin and log terms."""
    m2 = 1.0 - m1
    for omega in [0.001, 0.005, 0.02, 0.05, 0.1]:
        y = np.array([[omega, 0, 0, c[0] * m1 ** 2, 0, 0, c[1] * m2 ** 2, 0, 0, 1.0]])
        f = oracle.rhs(y, np.array([[m1, m2]]))[0]
        assert np.all(f[1:] == 0.0)
        ref = omega_dot_aligned(omega, m1, m2, c[0], c[1])
        assert abs(f[0] - ref) <= 5e-14 * abs(ref)


def test_term_mask_isolates_each_power(oracle):
    """Each bit k of term_mask keeps exactly the (M omega)^{k/3} term: the masked evaluations sum to
    the full one, the k=0 one is the leading (quadrupole) term 96/5 eta M^{5/3} omega^{11/3}, and k=1
    is absent (there is no 0.5PN term in Eq. (1))."""
    y, m = random_states(50, 3)
    full = oracle.rhs(y, m)[:, 0]
    parts = [oracle.rhs(y, m, term_mask=(1 << k) | (1 << 16))[:, 0] for k in range(8)]
    assert np.allclose(sum(parts), full, rtol=1e-13, atol=0)
    M = m.sum(1)
    eta = m[:, 0] * m[:, 1] / M ** 2
    assert np.allclose(parts[0], 96 / 5 * eta * M ** (5 / 3) * y[:, 0] ** (11 / 3), rtol=1e-14, atol=0)
    assert np.all(parts[1] == 0.0)
    # spin bit off == spins set to zero in Eq. (1)
    nospin = oracle.rhs(y, m, term_mask=0xFF)[:, 0]
    y0 = y.copy(); y0[:, 1:7] = 0
    assert np.allclose(nospin, oracle.rhs(y0, m)[:, 0], rtol=1e-14, atol=0)


def test_P3_rhs_identities(oracle):
    """S_i.S_i_dot = 0, L^.L^_dot = 0 and |L| L^_dot + S1_dot + S2_dot = 0 with |L| = eta M^{5/3} omega^{-1/3}
    (PAPER.md:50-54): total angular momentum J = |L|L^ + S1 + S2 changes only along L^."""
    for M in (1.0, 2.5):
        y, m = random_states(20000, 11, M=M)
        f = oracle.rhs(y, m)
        S1, S2, L = y[:, 1:4], y[:, 4:7], y[:, 7:10]
        d1 = np.einsum("ij,ij->i", S1, f[:, 1:4])
        d2 = np.einsum("ij,ij->i", S2, f[:, 4:7])
        dl = np.einsum("ij,ij->i", L, f[:, 7:10])
        sc1 = np.linalg.norm(S1, axis=1) * np.linalg.norm(f[:, 1:4], axis=1) + 1e-300
        sc2 = np.linalg.norm(S2, axis=1) * np.linalg.norm(f[:, 4:7], axis=1) + 1e-300
        scl = np.linalg.norm(f[:, 7:10], axis=1) + 1e-300
        assert np.abs(d1 / sc1).max() < 1e-13 and np.abs(d2 / sc2).max() < 1e-13 and np.abs(dl / scl).max() < 1e-13
        eta = m[:, 0] * m[:, 1] / M ** 2
        Lmag = eta * M ** (5 / 3) * y[:, 0] ** (-1 / 3)
        res = Lmag[:, None] * f[:, 7:10] + f[:, 1:4] + f[:, 4:7]
        scale = np.linalg.norm(f[:, 1:4], axis=1) + np.linalg.norm(f[:, 4:7], axis=1)
        assert (np.linalg.norm(res, axis=1) / scale).max() < 1e-13
        assert np.all(f[:, 0] > 0)      # P13: omega_dot > 0, termination at omega_f is well defined


def test_P5_relabelling(oracle):
    """1<->2: swapping masses and spins leaves omega_dot and L_dot unchanged and swaps S_dot."""
    y, m = random_states(2000, 5)
    f = oracle.rhs(y, m)
    ys = y.copy(); ys[:, 1:4], ys[:, 4:7] = y[:, 4:7], y[:, 1:4]
    fs = oracle.rhs(ys, m[:, ::-1])
    assert np.allclose(fs[:, 0], f[:, 0], rtol=1e-13, atol=0)
    assert np.allclose(fs[:, 1:4], f[:, 4:7], rtol=1e-12, atol=1e-22)
    assert np.allclose(fs[:, 4:7], f[:, 1:4], rtol=1e-12, atol=1e-22)
    assert np.allclose(fs[:, 7:10], f[:, 7:10], rtol=1e-11, atol=1e-20)


def test_P7_scale_freedom_rhs(oracle):
    """(m, S, omega) -> (lam m, lam^2 S, omega/lam), t -> lam t:
    omega_dot -> omega_dot/lam^2, S_dot -> lam S_dot, L_dot -> L_dot/lam."""
    y, m = random_states(2000, 6)
    f = oracle.rhs(y, m)
    for lam in (2.0, 0.37):
        ys = y.copy(); ys[:, 0] /= lam; ys[:, 1:7] *= lam ** 2
        fs = oracle.rhs(ys, m * lam)
        assert np.allclose(fs[:, 0] * lam ** 2, f[:, 0], rtol=2e-13, atol=0)
        assert np.allclose(fs[:, 1:7] / lam, f[:, 1:7], rtol=1e-11, atol=1e-22)
        assert np.allclose(fs[:, 7:10] * lam, f[:, 7:10], rtol=1e-10, atol=1e-20)


def test_P8_rotation_covariance_rhs(oracle):
    """No hidden use of L^ = z ("without loss of generality")."""
    from scipy.spatial.transform import Rotation

    y, m = random_states(2000, 7)
    f = oracle.rhs(y, m)
    R = Rotation.random(random_state=3).as_matrix()
    yr, fr = y.copy(), f.copy()
    for s in (slice(1, 4), slice(4, 7), slice(7, 10)):
        yr[:, s] = y[:, s] @ R.T
        fr[:, s] = f[:, s] @ R.T
    f2 = oracle.rhs(yr, m)
    assert np.allclose(f2[:, 0], f[:, 0], rtol=1e-13, atol=0)
    for s in (slice(1, 4), slice(4, 7), slice(7, 10)):
        sc = np.linalg.norm(fr[:, s], axis=1, keepdims=True)
        assert (np.abs(f2[:, s] - fr[:, s]) / sc).max() < 1e-11


def test_P9_equal_mass_collapse(oracle):
    """Equal masses: the spin-orbit bracket of Eq. (1) depends on the spins only through
    L^.(S1+S2), with weight (113/4 + 75/4)/12 * 4 = 47/3 on L^.S/M^2."""
    rng = np.random.default_rng(1)
    n = 500
    y, _ = random_states(n, 8)
    m = np.full((n, 2), 0.5)
    so_only = (1 << 3) | (1 << 16)
    f = oracle.rhs(y, m, term_mask=so_only)[:, 0]
    LS = np.einsum("ij,ij->i", y[:, 7:10], y[:, 1:4] + y[:, 4:7])
    x = y[:, 0]
    expect = y[:, 0] ** 2 * 96 / 5 * 0.25 * x ** (5 / 3) * (-(47 / 3 * LS - 4 * PI) * x)
    assert np.allclose(f, expect, rtol=1e-12, atol=0)
    # moving spin from body 1 to body 2 changes nothing in omega_dot's spin-orbit term
    y2 = y.copy(); d = rng.normal(size=(n, 3)) * 0.01
    y2[:, 1:4] += d; y2[:, 4:7] -= d
    assert np.allclose(oracle.rhs(y2, m, term_mask=so_only)[:, 0], f, rtol=1e-11, atol=0)


def test_precession_leading_behaviour(oracle):
    """Eq. (2),(4) by hand for one spinning body (S2 = 0): S1 precesses about L^ with
    Omega_1 = (M omega)^2/(2M) eta (M omega)^{-1/3} (4 + 3 m2/m1), i.e. S1_dot = Omega_1 L^ x S1."""
    m1, m2, om = 0.7, 0.3, 0.013
    S1 = np.array([0.1, -0.2, 0.05]); L = np.array([0.0, 0.6, 0.8])
    y = np.concatenate([[om], S1, [0, 0, 0], L])[None]
    f = oracle.rhs(y, np.array([[m1, m2]]))[0]
    eta = m1 * m2
    Om = om ** 2 / 2 * eta * om ** (-1 / 3) * (4 + 3 * m2 / m1)
    assert np.allclose(f[1:4], Om * np.cross(L, S1), rtol=1e-13, atol=0)
    assert np.allclose(f[4:7], 0.0)
    assert np.allclose(f[7:10], -om ** (1 / 3) / eta * f[1:4], rtol=1e-13, atol=0)


def test_two_spin_precession_by_hand(oracle):
    """Eq. (4) with BOTH spins present, reduced by hand for a configuration whose numbers are exact
    (Omega_1 = (M omega)^2/(2M) [eta (M omega)^{-1/3} (4 + 3 m2/m1) L^ + 1/M^2 (S2 - 3 (S2.L^) L^)]).

    m = (1.2, 0.8): M = 2, eta = 0.24.  omega = 1/16: M omega = 1/8, (M omega)^{1/3} = 1/2, (M omega)^2/(2M) = 1/256.
    L^ = z, S1 = (0.5, 0, 0), S2 = (0, 0.25, 0.4).
      Omega_1: eta/v (4 + 3*0.8/1.2) = 0.48 * 6 = 2.88;  S2 - 3 (S2.L^) L^ = (0, 0.25, 0.4 - 1.2) = (0, 0.25, -0.8);
               Omega_1 = (0, 0.25/4, 2.88 - 0.8/4)/256 = (0, 0.0625, 2.68)/256
      S1_dot = Omega_1 x S1 = (0, 2.68*0.5, -0.0625*0.5)/256 = (0, 1.34, -0.03125)/256
      Omega_2: eta/v (4 + 3*1.2/0.8) = 0.48 * 8.5 = 4.08;  S1 - 3 (S1.L^) L^ = S1;  Omega_2 = (0.125, 0, 4.08)/256
      S2_dot = Omega_2 x S2 = (-4.08*0.25, -0.125*0.4, 0.125*0.25)/256 = (-1.02, -0.05, 0.03125)/256
      L^_dot = -(1/2)/(0.24*4) (S1_dot + S2_dot) = -(1/1.92) (-1.02, 1.29, 0)/256 = (0.53125, -0.671875, 0)/256
    The z-component of S1_dot is pure spin-spin (pins 1/M^2); the -0.8 = 0.4 - 3*0.4 pins the "3"."""
    y = np.array([[1 / 16, 0.5, 0, 0, 0, 0.25, 0.4, 0, 0, 1.0]])
    f = oracle.rhs(y, np.array([[1.2, 0.8]]))[0]
    expect = np.array([0, 1.34, -0.03125, -1.02, -0.05, 0.03125, 0.53125, -0.671875, 0]) / 256
    assert np.abs(f[1:] - expect).max() < 2e-17 + 1e-14 * np.abs(expect).max()
    # a wrong "3" (say 2) would move S1_dot_y by 0.5*0.4/4/256 = 1.95e-4; a missing 1/M^2 would quadruple S1_dot_z
    assert abs(f[2] * 256 - 1.34) < 1e-13 and abs(f[3] * 256 + 0.03125) < 1e-15


def test_spin_spin_term_of_eq1_by_hand(oracle):
    """The two numbers of the 2PN spin-spin term of Eq. (1), -(1/48) eta chi_1 chi_2 (247 S^_1.S^_2 - 721 (L^.S^_1)(L^.S^_2))
    (M omega)^{4/3}, each on its own (aligned spins only see 247 - 721, and the symmetries hold
    for any pair of numbers).  The term is isolated as the difference of the (M omega)^{4/3} piece with and without the
    spin terms (term_mask bit 4, bit 16), on states whose numbers are exact:

    m = (1.2, 0.8): M = 2, eta = 0.24, m_1^2 = 1.44, m_2^2 = 0.64.  omega = 1/16: M omega = 1/8, (M omega)^{5/3} = 1/32,
    (M omega)^{4/3} = 1/16.  Prefactor of the brace: omega^2 (96/5) eta (M omega)^{5/3} = (1/256)(19.2)(0.24)/32.
    chi_1 = chi_2 = 1/2 (chi_1 chi_2 = 1/4), L^ = z.
      (a) S^_1 = (0.6, 0, 0.8), S^_2 = (-0.8, 0, 0.6): S^_1.S^_2 = 0, (L^.S^_1)(L^.S^_2) = 0.48: only 721 survives,
          term = -(1/48)(0.24)(1/4)(-721 * 0.48)/16 = +0.00125 * 346.08 / 16
      (b) S^_1 = (1, 0, 0), S^_2 = (0.6, 0, 0.8): L^.S^_1 = 0, S^_1.S^_2 = 0.6: only 247 survives,
          term = -(1/48)(0.24)(1/4)(247 * 0.6)/16 = -0.00125 * 148.2 / 16"""
    m = np.array([[1.2, 0.8]])
    pre = (1 / 256) * 19.2 * 0.24 / 32
    with_spin, without = (1 << 4) | (1 << 16), (1 << 4)
    cases = [((0.6, 0.0, 0.8), (-0.8, 0.0, 0.6), +0.00125 * 346.08 / 16),
             ((1.0, 0.0, 0.0), (0.6, 0.0, 0.8), -0.00125 * 148.2 / 16)]
    for s1, s2, term in cases:
        y = np.concatenate([[1 / 16], 0.5 * 1.44 * np.array(s1), 0.5 * 0.64 * np.array(s2), [0, 0, 1.0]])[None]
        d = oracle.rhs(y, m, term_mask=with_spin)[0, 0] - oracle.rhs(y, m, term_mask=without)[0, 0]
        assert abs(d / (pre * term) - 1) < 1e-12, (d, pre * term)
    # what a slip would do: 247 <-> 721 swapped changes (a) by the factor 247/721 and (b) by 721/247; a wrong sign
    # between them leaves (a) and (b) with the wrong sign on one of the two; both are far outside 1e-12
    # the non-spin part of the same order, for scale: 34103/18144 + 13661/2016 eta + 59/18 eta^2 at eta = 0.24
    y = np.concatenate([[1 / 16], np.zeros(6), [0, 0, 1.0]])[None]
    t4 = 34103 / 18144 + 13661 / 2016 * 0.24 + 59 / 18 * 0.24 ** 2
    assert abs(oracle.rhs(y, m, term_mask=without)[0, 0] / (pre * t4 / 16) - 1) < 1e-12
