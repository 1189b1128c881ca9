"""GPU parity of pn_generate (through the C ABI) against the generator oracle: integer work (Philox words ->
variates -> masses, magnitudes) is bit-exact; unit-vector components agree to 4e-16 (CUDA sincos vs libm)."""
import numpy as np
import pytest

from oracle import pn_gen_oracle as G
from oracle import pn_stats_oracle as S
from paper_0908_3889_b200 import workloads as W

pytestmark = pytest.mark.gpu
torch = pytest.importorskip("torch")


@pytest.fixture(scope="module")
def pn():
    assert torch.cuda.is_available(), "the gpu tests need a CUDA device"
    import paper_0908_3889_b200 as pkg

    return pkg


def gpu_generate(pn, specs, n_total, first=0, count=None, host=False):
    specs = specs if isinstance(specs, list) else [specs]
    count = n_total - first if count is None else count
    rows = len(specs) * count
    if host:
        y, m = np.full((rows, 10), np.nan), np.full((rows, 2), np.nan)
    else:
        y = torch.full((rows, 10), float("nan"), dtype=torch.float64, device="cuda")
        m = torch.full((rows, 2), float("nan"), dtype=torch.float64, device="cuda")
    pn.pn_generate([pn.make_ensemble(**s) for s in specs], n_total, y, m, first=first, count=count)
    return (y, m) if host else (y.cpu().numpy(), m.cpu().numpy())


def check(gy, gm, oy, om):
    assert np.array_equal(gm, om)                                         # masses: bit-exact
    assert np.array_equal(gy[:, 0], oy[:, 0]) and np.array_equal(gy[:, 7:], oy[:, 7:])
    assert np.array_equal(gy[:, 3], oy[:, 3]) or np.abs(gy[:, 3] - oy[:, 3]).max() <= 1e-16   # z components: no sin/cos
    assert np.array_equal(gy[:, 6], oy[:, 6])
    assert np.abs(gy - oy).max() <= 4e-16


@pytest.mark.parametrize("name,n", [("C1", 1024), ("C2", 5003), ("C3", 5003), ("C4", 777), ("C5", 1), ("C3", 255), ("C5", 257)])
def test_generate_parity_small(pn, name, n):
    cfg = W.with_size(W.CONFIGS[name], n)
    spec = W.generator_spec(cfg)
    gy, gm = gpu_generate(pn, spec, n)
    oy, om = G.generate(G.make_spec(**spec), n)
    check(gy, gm, oy, om)
    y0, m = W.generate(cfg)                                               # and the numpy recipe the other tests use
    assert np.array_equal(gm, m) and np.abs(gy - y0).max() <= 4e-16
    gy2, gm2 = gpu_generate(pn, spec, n)
    assert np.array_equal(gy, gy2) and np.array_equal(gm, gm2)            # bit-identical run to run


def test_generate_chunks_ensembles_host(pn):
    cfg = W.with_size(W.CONFIGS["C3"], 100000)
    spec = W.generator_spec(cfg)
    oy, om = G.generate(G.make_spec(**spec), cfg.n, first=33333, count=1025)
    gy, gm = gpu_generate(pn, spec, cfg.n, first=33333, count=1025)
    check(gy, gm, oy, om)
    hy, hm = gpu_generate(pn, spec, cfg.n, first=33333, count=1025, host=True)
    assert np.array_equal(hy, gy) and np.array_equal(hm, gm)
    # a sweep: three ensembles with different parameters and keys in one call
    specs = [dict(key=(7, 8 + e), omega0=0.00395, q=(qq, qq), chi1=(c, c), chi2=(c, c)) for e, (qq, c) in
             enumerate([(1.0, 1.0), (2 / 3, 1.0), (1.0, 0.05)])]
    gy, gm = gpu_generate(pn, specs, 3000, first=100, count=2000)
    for e, sp in enumerate(specs):
        oy, om = G.generate(G.make_spec(**sp), 3000, first=100, count=2000)
        check(gy[2000 * e:2000 * (e + 1)], gm[2000 * e:2000 * (e + 1)], oy, om)


def test_generate_full_size_sampled_and_errors(pn):
    for name in ("C2", "C4"):
        cfg = W.CONFIGS[name]
        spec = W.generator_spec(cfg)
        gy, gm = gpu_generate(pn, spec, cfg.n)
        for first in (0, 123456, cfg.n - 300):
            oy, om = G.generate(G.make_spec(**spec), cfg.n, first=first, count=300)
            check(gy[first:first + 300], gm[first:first + 300], oy, om)
        # properties that hold at any size: |S_i| = chi_i m_i^2, L^ = z, isotropy moments
        s2 = np.linalg.norm(gy[:, 4:7], axis=1)
        assert np.abs(s2 / gm[:, 1] ** 2 - 1.0).max() < 1e-15
        u = gy[:, 4:7] / s2[:, None]
        assert np.abs(u.mean(axis=0)).max() < 4 * np.sqrt(1 / 3 / cfg.n)
        assert np.abs(u.T @ u / cfg.n - np.eye(3) / 3).max() < 2e-3
    e = pn.make_ensemble((1, 2), 0.01)
    y = torch.zeros(10, 10, dtype=torch.float64, device="cuda")
    m = torch.zeros(10, 2, dtype=torch.float64, device="cuda")
    with pytest.raises(pn.PnError):
        pn.pn_generate(e, 5, y, m, first=0, count=10)            # chunk beyond the ensemble
    with pytest.raises(pn.PnError):
        pn.pn_generate(pn.make_ensemble((1, 2), -1.0), 10, y, m)  # omega0 <= 0
    assert pn.pn_generate(e, 10, y, m, first=10, count=0) == 0


def test_seed_in_statistics_out(pn, oracle):
    """NEXT-2 end to end: key in -> pn_generate -> pn_integrate -> pn_statistics, nothing but the key and the
    statistics crossing the host boundary; compared with the oracle chain on the same ensemble."""
    cfg = W.with_size(W.CONFIGS["C1"], 2048)
    spec = W.generator_spec(cfg)
    d_y0 = torch.empty(cfg.n, 10, dtype=torch.float64, device="cuda")
    d_m = torch.empty(cfg.n, 2, dtype=torch.float64, device="cuda")
    pn.pn_generate(pn.make_ensemble(**spec), cfg.n, d_y0, d_m)
    d_yf = torch.empty_like(d_y0)
    d_steps = torch.empty(cfg.n, dtype=torch.int32, device="cuda")
    pn.pn_integrate(d_y0, d_m, cfg.omega0, cfg.omegaf, cfg.rtol, cfg.atol, pn.PN_FP64, d_yf, d_steps)
    r = torch.zeros(1, 3, dtype=torch.float64, device="cuda")
    h1 = torch.zeros(1, 3, 50, dtype=torch.int64, device="cuda")
    pn.pn_statistics(d_y0, d_yf, d_steps, bins1=50, pearson_r=r, hist1=h1)
    oy, om = G.generate(G.make_spec(**spec), cfg.n)
    of = oracle.integrate(oy, om, cfg.omegaf, cfg.rtol, cfg.atol)
    ref = S.statistics(oy, of["final"], of["steps"], None, 50, 0)
    assert np.abs(r.cpu().numpy() - ref["r"]).max() < 1e-8
    assert np.abs(h1.cpu().numpy() - ref["hist1"].astype(np.int64)).sum() <= 4
