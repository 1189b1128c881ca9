"""Pins of the generator oracle (oracle/pn_gen_oracle.c): Philox4x64-10 against numpy's own implementation,
the variate layout against numpy.random.Generator, the full recipe against workloads.generate (numpy), and
the distributional properties the paper asks for (uniform on the sphere)."""
import numpy as np
import pytest

from oracle import pn_gen_oracle as G
from paper_0908_3889_b200 import workloads as W


def test_philox_raw_words_against_numpy():
    # numpy increments the counter before every block of four words
    for key, ctr in [((0, 0), (0, 0, 0, 0)), ((1, 2), (5, 0, 0, 0)), ((2**64 - 1, 2**63 + 12345), (2**64 - 2, 7, 0, 9)),
                     ((0x243F6A8885A308D3, 0x13198A2E03707344), (0xA4093822299F31D0, 0x082EFA98EC4E6C89, 3, 4))]:
        bg = np.random.Philox(key=np.array(key, dtype=np.uint64), counter=np.array(ctr, dtype=np.uint64))
        want = bg.random_raw(8)
        c = list(ctr)
        got = []
        for _ in range(2):
            c[0] += 1                      # carry into the next word when it wraps
            if c[0] == 2**64:
                c[0] = 0
                c[1] += 1
            got.append(G.philox4x64_10(c, key))
        assert np.array_equal(np.concatenate(got), want), (key, ctr)


def test_raw_stream_and_uniform_against_numpy_generator():
    for seed in (0, 1, 4, 12345):
        key = W.philox_key(seed)
        assert np.array_equal(G.raw(key, 0, 1001), np.random.Philox(seed).random_raw(1001))
        u = np.random.Generator(np.random.Philox(seed)).random(999)
        got = (G.raw(key, 0, 999) >> np.uint64(11)).astype(np.float64) * 2.0**-53
        assert np.array_equal(got, u)
        # random access: element e of the stream without generating the ones before it
        assert np.array_equal(G.raw(key, 777, 5), np.random.Philox(seed).random_raw(782)[777:])


@pytest.mark.parametrize("name", ["C1", "C2", "C3", "C4", "C5"])
def test_recipe_against_workloads_generate(name):
    cfg = W.with_size(W.CONFIGS[name], 5003)
    y0, m = W.generate(cfg)
    gy, gm = G.generate(G.make_spec(**W.generator_spec(cfg)), cfg.n)
    assert np.array_equal(gm, m)                        # masses: no transcendental involved
    assert np.abs(gy - y0).max() <= 4e-16               # sin/cos of two libraries: an ulp or two of a unit vector
    assert np.array_equal(gy[:, 0], y0[:, 0]) and np.array_equal(gy[:, 7:], y0[:, 7:])
    # chunked generation reproduces the same global stream
    cy, cm = G.generate(G.make_spec(**W.generator_spec(cfg)), cfg.n, first=1234, count=777)
    assert np.array_equal(cy, gy[1234:2011]) and np.array_equal(cm, gm[1234:2011])


def test_distribution_uniform_on_the_sphere():
    # spin orientations uniform on the sphere; moments of a uniform unit vector:
    # <n_i> = 0, <n_i n_j> = delta_ij / 3, <n_z^4> = 1/5; |n| = 1
    n = 200000
    y0, m = G.generate(G.make_spec((11, 22), 0.01, q=(0.1, 1.0), chi1=(0.0, 1.0), chi2=(0.0, 1.0)), n)
    q = m[:, 1] / m[:, 0]
    assert np.allclose(m.sum(axis=1), 1.0, atol=1e-15)
    assert 0.1 <= q.min() and q.max() <= 1.0 and abs(q.mean() - 0.55) < 3 * 0.26 / np.sqrt(n) * 1.5
    for a, mi in ((y0[:, 1:4], m[:, 0]), (y0[:, 4:7], m[:, 1])):
        norm = np.linalg.norm(a, axis=1)
        chi = norm / mi**2
        assert chi.max() <= 1.0 + 1e-15 and abs(chi.mean() - 0.5) < 4 * 0.29 / np.sqrt(n)
        u = a / norm[:, None]
        assert np.abs(u.mean(axis=0)).max() < 4 * np.sqrt(1 / 3 / n)
        cov = u.T @ u / n
        assert np.abs(cov - np.eye(3) / 3).max() < 4 * np.sqrt(4 / 45 / n) + 1e-3
        assert abs((u[:, 2] ** 4).mean() - 0.2) < 5e-3
    # the two spins are independent: <S1^.S2^> = 0, <(S1^.S2^)^2> = 1/3
    d = np.sum(y0[:, 1:4] * y0[:, 4:7], axis=1) / np.linalg.norm(y0[:, 1:4], axis=1) / np.linalg.norm(y0[:, 4:7], axis=1)
    assert abs(d.mean()) < 4 * np.sqrt(1 / 3 / n) and abs((d * d).mean() - 1 / 3) < 5e-3


def test_fixed_tilt_and_fixed_masses():
    y0, m = G.generate(G.make_spec((3, 4), 0.01, q=(2 / 3, 2 / 3), chi1=(0.9, 0.9), chi2=(1.0, 1.0), m1_fixed=0.6,
                                   s1_tilt_deg=60.0), 100)
    assert np.all(m[:, 0] == 0.6) and np.all(m[:, 1] == 0.4)
    s1 = 0.9 * 0.6 * 0.6 * np.array([np.sin(np.pi / 3), 0.0, np.cos(np.pi / 3)])
    assert np.abs(y0[:, 1:4] - s1).max() < 1e-16
    assert np.allclose(np.linalg.norm(y0[:, 4:7], axis=1), 0.16, atol=1e-16)
