"""GPU parity of pn_statistics (through the C ABI) against the statistics oracle: Pearson r, moments, 1-D and
bivariate histograms, per-ensemble groups.  Tolerances: counts bit-exact except samples within 1e-9 bins of
an edge (both sides round the unit dot product, DESIGN.md 3 R14); n and skipped exact; means 1e-14 absolute;
M2x, M2y, Cxy 1e-11 relative to n; r 1e-12 absolute (two-pass definition vs pairwise merge, both float64)."""
import numpy as np
import pytest

from oracle import pn_stats_oracle as S
from paper_0908_3889_b200 import workloads as W

pytestmark = pytest.mark.gpu
torch = pytest.importorskip("torch")


@pytest.fixture(scope="module")
def pn():
    assert torch.cuda.is_available(), "the gpu tests need a CUDA device"
    import paper_0908_3889_b200 as pkg

    return pkg


def fake_final(y0, seed, spread=0.3):
    """Any 'final' states do: rotate / perturb the spins so that dots change but stay correlated."""
    g = np.random.Generator(np.random.Philox(seed))
    yf = y0.copy()
    yf[:, 1:10] += spread * np.abs(y0[:, 1:10]).max() * g.normal(size=(y0.shape[0], 9)) * (np.abs(y0[:, 1:10]) > 0).any(axis=1, keepdims=True)
    return yf


def gpu_stats(pn, y0, yf, steps=None, group_size=0, bins1=0, bins2=0, host=False, want_norm=True, init=True):
    n = yf.shape[0]
    G = n // (group_size if group_size > 0 else n)
    dev = "cpu" if host else "cuda"
    t = lambda a: None if a is None else (np.ascontiguousarray(a) if host else torch.from_numpy(np.ascontiguousarray(a)).cuda())
    mk = (lambda shape, dt: np.full(shape, -1, dtype=dt)) if host else \
        (lambda shape, dt: torch.full(shape, -1, dtype={np.float64: torch.float64, np.int64: torch.int64}[dt], device=dev))
    out = dict(pearson_r=mk((G, 3), np.float64), moments=mk((G, 3, 6), np.float64), n_skipped=mk((G, 3), np.int64))
    if bins1:
        out["hist1"] = mk((G, 3, bins1), np.int64)
    if bins2 and init:
        out["hist2"] = mk((G, 3, bins2, bins2), np.int64)
        out["hist2_max"] = mk((G, 3), np.int64)
        if want_norm:
            out["hist2_norm"] = mk((G, 3, bins2, bins2), np.float64)
    pn.pn_statistics(t(y0) if init else None, t(yf), t(steps), group_size=group_size, bins1=bins1, bins2=bins2, **out)
    return {k: (v if host else v.cpu().numpy()) for k, v in out.items()}


def near_edge_count(d, bins):
    frac = (d[np.isfinite(d)] + 1.0) * bins / 2.0
    return int(np.count_nonzero(np.abs(frac - np.round(frac)) < 1e-9))


def compare(got, ref, y0, yf, bins1, bins2):
    G = ref["r"].shape[0]
    assert np.array_equal(got["n_skipped"], ref["skipped"].astype(np.int64))
    assert np.array_equal(got["moments"][..., 0], ref["moments"][..., 0])
    n = np.maximum(ref["moments"][..., 0], 1.0)
    has = ref["moments"][..., 0] > 0
    assert np.abs(got["moments"][..., 1:3] - ref["moments"][..., 1:3])[has].max(initial=0) <= 1e-14
    assert (np.abs(got["moments"][..., 3:] - ref["moments"][..., 3:]) / n[..., None]).max() <= 1e-11
    defined = np.isfinite(ref["r"]) & (ref["moments"][..., 3] > 1e-12 * n) & (ref["moments"][..., 4] > 1e-12 * n)
    assert np.abs(got["pearson_r"] - ref["r"])[defined].max(initial=0) <= 1e-12
    assert np.all(np.isnan(got["pearson_r"][(ref["moments"][..., 0] < 2)]))
    d0, d1 = S.unit_dots(y0) if y0 is not None else None, S.unit_dots(yf)
    if bins1:
        slack = 2 * near_edge_count(d1, bins1)
        assert np.abs(got["hist1"] - ref["hist1"].astype(np.int64)).sum() <= slack
        assert np.array_equal(got["hist1"].sum(axis=2), ref["moments"][..., 0].astype(np.int64))
    if bins2 and "hist2" in got:
        slack = 2 * (near_edge_count(d0, bins2) + near_edge_count(d1, bins2))
        assert np.abs(got["hist2"] - ref["hist2"].astype(np.int64)).sum() <= slack
        assert np.array_equal(got["hist2"].sum(axis=(2, 3)), ref["moments"][..., 0].astype(np.int64))
        assert np.array_equal(got["hist2_max"], got["hist2"].reshape(G, 3, -1).max(axis=2))
        if "hist2_norm" in got:
            mx = np.maximum(got["hist2_max"], 1)[..., None, None].astype(np.float64)
            assert np.array_equal(got["hist2_norm"], got["hist2"] / mx)
            assert got["hist2_norm"].max() <= 1.0


@pytest.mark.parametrize("n,gs,bins1,bins2", [(1, 0, 50, 79), (31, 0, 50, 79), (257, 0, 20, 5), (5003, 0, 50, 79),
                                               (6 * 777, 777, 50, 79), (500 * 100, 100, 10, 8), (3 * 40000, 40000, 100, 79),
                                               (20000, 0, 1, 1), (20000, 10000, 8192, 300)])
def test_statistics_parity_synthetic(pn, n, gs, bins1, bins2):
    cfg = W.with_size(W.CONFIGS["C3"], n)
    y0, _ = W.generate(cfg)
    yf = fake_final(y0, n + 1)
    steps = np.full(n, 7, dtype=np.int32)
    if n > 40:
        steps[[3, n // 2, n - 1]] = [-1, -3, -5]
        y0[11, 1:4] = 0.0
        yf[17, 4:7] = 0.0
        yf[19, 7:10] = np.nan
    got = gpu_stats(pn, y0, yf, steps, gs, bins1, bins2)
    ref = S.statistics(y0, yf, steps, gs if gs else None, bins1, bins2)
    compare(got, ref, y0, yf, bins1, bins2)
    again = gpu_stats(pn, y0, yf, steps, gs, bins1, bins2)
    for k in got:                                # bit-identical run to run
        assert np.array_equal(got[k], again[k], equal_nan=True), k


def test_statistics_host_buffers_and_final_only(pn):
    cfg = W.with_size(W.CONFIGS["C5"], 7001)
    y0, _ = W.generate(cfg)
    yf = fake_final(y0, 5)
    ref = S.statistics(y0, yf, None, None, 50, 79)
    compare(gpu_stats(pn, y0, yf, None, 0, 50, 79, host=True), ref, y0, yf, 50, 79)
    # final-only mode: the 1-D histograms of pn_histogram, through the bulk-copy kernel
    got = gpu_stats(pn, y0, yf, None, 0, 50, 0, init=False)
    c_ref = np.stack([S.histogram1d(d[np.isfinite(d)], 50) for d in S.unit_dots(yf).T]).astype(np.int64)
    assert np.abs(got["hist1"][0] - c_ref).sum() <= 2 * near_edge_count(S.unit_dots(yf), 50)
    assert np.all(np.isnan(got["pearson_r"]))
    d_cnt = torch.zeros(3, 50, dtype=torch.int64, device="cuda")
    pn.pn_histogram(torch.from_numpy(yf).cuda(), 50, d_cnt)
    assert np.abs(d_cnt.cpu().numpy() - got["hist1"][0]).sum() <= 2 * near_edge_count(S.unit_dots(yf), 50)


def test_statistics_degenerate_and_errors(pn):
    # C4: S1 direction fixed -> x = S1^.L^ is the same for every system -> sigma_x = 0 -> r undefined (NaN)
    cfg = W.with_size(W.CONFIGS["C4"], 3000)
    y0, _ = W.generate(cfg)
    yf = fake_final(y0, 9)
    got = gpu_stats(pn, y0, yf, None, 0, 50, 79)
    assert np.isnan(got["pearson_r"][0, 1]) and got["moments"][0, 1, 3] == 0.0
    assert np.isfinite(got["pearson_r"][0, 0]) and np.isfinite(got["pearson_r"][0, 2])
    assert got["moments"][0, 1, 1] == pytest.approx(0.5, abs=1e-15)
    # exact linear relation: final = initial -> r = 1, hist2 diagonal
    got = gpu_stats(pn, y0, y0, None, 0, 50, 79)
    assert got["pearson_r"][0, 0] == pytest.approx(1.0, abs=1e-14)
    h = got["hist2"][0, 0]
    assert h.sum() == np.trace(h) == 3000
    # errors: N not a multiple of group_size, misaligned pointer, hist2_norm without hist2
    d = torch.from_numpy(y0).cuda()
    r = torch.zeros(3, 3, dtype=torch.float64, device="cuda")
    with pytest.raises(pn.PnError):
        pn.pn_statistics(d, d, group_size=999, pearson_r=r)
    flat = torch.zeros(10 * 100 + 1, dtype=torch.float64, device="cuda")
    with pytest.raises(pn.PnError):
        pn.pn_statistics(flat[1:].view(100, 10), flat[1:].view(100, 10), pearson_r=r)
    with pytest.raises(pn.PnError):
        pn.pn_statistics(d, d, bins2=8, hist2_norm=torch.zeros(3, 8, 8, dtype=torch.float64, device="cuda"))
    assert pn.pn_statistics(d[:0], d[:0], pearson_r=r) == 0      # N = 0 is a successful no-op


def test_statistics_C2_full_size_through_the_integrator(pn, oracle):
    """The C2 deliverable (BASELINE.json configs[1]): initial-vs-final S1^.S2^ correlation and histograms of the
    2^20-inspiral batch, statistics on the device vs the oracle's statistics of the SAME final states, plus
    the oracle-integrated sample for the end-to-end chain."""
    cfg = W.CONFIGS["C2"]
    y0, m = W.generate(cfg)
    d_y0, d_m = torch.from_numpy(y0).cuda(), torch.from_numpy(m).cuda()
    d_yf = torch.empty_like(d_y0)
    d_steps = torch.empty(cfg.n, dtype=torch.int32, device="cuda")
    pn.pn_integrate(d_y0, d_m, cfg.omega0, cfg.omegaf, cfg.rtol, cfg.atol, pn.PN_FP64, d_yf, d_steps)
    yf, steps = d_yf.cpu().numpy(), d_steps.cpu().numpy()
    G = 1
    out = dict(pearson_r=torch.zeros(G, 3, dtype=torch.float64, device="cuda"),
               moments=torch.zeros(G, 3, 6, dtype=torch.float64, device="cuda"),
               n_skipped=torch.zeros(G, 3, dtype=torch.int64, device="cuda"),
               hist1=torch.zeros(G, 3, 50, dtype=torch.int64, device="cuda"),
               hist2=torch.zeros(G, 3, 79, 79, dtype=torch.int64, device="cuda"),
               hist2_max=torch.zeros(G, 3, dtype=torch.int64, device="cuda"))
    pn.pn_statistics(d_y0, d_yf, d_steps, bins1=50, bins2=79, **out)
    got = {k: v.cpu().numpy() for k, v in out.items()}
    ref = S.statistics(y0, yf, steps, None, 50, 79)
    compare(got, ref, y0, yf, 50, 79)
    # SURVEY probe for this config: r(S1^.S2^) ~ 0.986, r(S_i^.L^) ~ 0.63 (paper at omega0 = 0.00395: 0.99, 0.65)
    assert 0.975 < got["pearson_r"][0, 0] < 0.995
    assert 0.58 < got["pearson_r"][0, 1] < 0.68 and 0.58 < got["pearson_r"][0, 2] < 0.68
    # end-to-end against the oracle integrator on a sample: r of the sample from oracle finals vs GPU finals
    idx = W.sample_indices(cfg.n, 512)
    o = oracle.integrate(y0[idx], m[idx], cfg.omegaf, cfg.rtol, cfg.atol)
    r_o = S.statistics(y0[idx], o["final"])["r"]
    r_g = S.statistics(y0[idx], yf[idx])["r"]
    assert np.abs(r_o - r_g).max() < 1e-7


def test_merge_statistics_of_sharded_ensembles(pn):
    """The multi-GPU exchange step on one GPU: three ranks' shares (sharding.shard_range) of the same two ensembles,
    statistics per share, moments merged by pn_merge_statistics == statistics of the whole (oracle, 1e-12)."""
    from paper_0908_3889_b200 import sharding

    G, gs, world = 2, 3001, 3
    cfg = W.with_size(W.CONFIGS["C3"], G * gs)
    y0, _ = W.generate(cfg)
    yf = fake_final(y0, 77)
    ref = S.statistics(y0, yf, None, gs, 0, 0)
    parts = torch.zeros(world, G, 3, 6, dtype=torch.float64, device="cuda")
    counts = np.zeros((G, 3, 20), dtype=np.int64)
    for rank in range(world):
        lo, hi = sharding.shard_range(gs, rank, world)
        rows = np.concatenate([np.arange(g * gs + lo, g * gs + hi) for g in range(G)])      # this rank's slice of every ensemble
        got = gpu_stats(pn, y0[rows], yf[rows], None, hi - lo, 20, 0)
        parts[rank] = torch.from_numpy(got["moments"]).cuda()
        counts += got["hist1"]
    mom = torch.zeros(G, 3, 6, dtype=torch.float64, device="cuda")
    r = torch.zeros(G, 3, dtype=torch.float64, device="cuda")
    pn.pn_merge_statistics(parts, moments=mom, pearson_r=r)
    mom, r = mom.cpu().numpy(), r.cpu().numpy()
    assert np.array_equal(mom[..., 0], ref["moments"][..., 0])
    assert np.abs(mom[..., 1:3] - ref["moments"][..., 1:3]).max() <= 1e-14
    assert (np.abs(mom[..., 3:] - ref["moments"][..., 3:]) / gs).max() <= 1e-11
    assert np.abs(r - ref["r"]).max() <= 1e-12
    assert np.abs(counts - S.statistics(y0, yf, None, gs, 20, 0)["hist1"].astype(np.int64)).sum() <= 2 * near_edge_count(S.unit_dots(yf), 20)
    # an empty part (a rank with no systems) is neutral
    parts2 = torch.cat([parts, torch.zeros(1, G, 3, 6, dtype=torch.float64, device="cuda")])
    parts2[-1, :, :, 1:3] = float("nan")
    r2 = torch.zeros(G, 3, dtype=torch.float64, device="cuda")
    pn.pn_merge_statistics(parts2, pearson_r=r2)
    assert np.array_equal(r2.cpu().numpy(), r)
