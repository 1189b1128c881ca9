"""NEXT-3: parameter sweeps as one launch (Figs. 6-7).  G ensembles laid end to end:
one pn_generate, one pn_integrate, one pn_statistics(group_size).  Checked against the oracle chain
(generator oracle -> integrator oracle -> statistics oracle) per ensemble, and against what the paper says
about the curves (soft pins: two printed digits / qualitative statements)."""
import numpy as np
import pytest

from oracle import pn_gen_oracle as G
from oracle import pn_stats_oracle as S

pytestmark = pytest.mark.gpu
torch = pytest.importorskip("torch")

N_E = 20000
OMEGA0, OMEGAF, TOL = 0.00395, 0.05, 5e-7


def specs():
    out = []
    for e, m1 in enumerate((0.5, 0.45, 0.4, 0.3)):                     # Fig. 6: chi = 1, m1 varied
        q = (1 - m1) / m1
        out.append(dict(key=(2024, e), omega0=OMEGA0, q=(q, q), chi1=(1.0, 1.0), chi2=(1.0, 1.0)))
    for e, chi in enumerate((0.3, 0.5, 0.7)):                          # Fig. 7: m1 = m2, chi varied
        out.append(dict(key=(2025, e), omega0=OMEGA0, q=(1.0, 1.0), chi1=(chi, chi), chi2=(chi, chi)))
    return out


def test_sweep_one_launch_against_oracle_chain(oracle):
    import paper_0908_3889_b200 as pn

    sp = specs()
    n = N_E * len(sp)
    d_y0 = torch.empty(n, 10, dtype=torch.float64, device="cuda")
    d_m = torch.empty(n, 2, dtype=torch.float64, device="cuda")
    pn.pn_generate([pn.make_ensemble(**s) for s in sp], N_E, d_y0, d_m)
    d_yf = torch.empty_like(d_y0)
    d_steps = torch.empty(n, dtype=torch.int32, device="cuda")
    pn.pn_integrate(d_y0, d_m, OMEGA0, OMEGAF, TOL, TOL, pn.PN_FP64, d_yf, d_steps)
    r = torch.zeros(len(sp), 3, dtype=torch.float64, device="cuda")
    mom = torch.zeros(len(sp), 3, 6, dtype=torch.float64, device="cuda")
    h2 = torch.zeros(len(sp), 3, 79, 79, dtype=torch.int64, device="cuda")
    pn.pn_statistics(d_y0, d_yf, d_steps, group_size=N_E, bins2=79, pearson_r=r, moments=mom, hist2=h2)
    r, mom, h2 = r.cpu().numpy(), mom.cpu().numpy(), h2.cpu().numpy()
    assert np.all(mom[..., 0] == N_E) and np.all(h2.sum(axis=(2, 3)) == N_E)

    # oracle chain per ensemble (different step sequences at tol 5e-7: final dots differ by ~1e-5, r by less)
    r_ref = np.zeros_like(r)
    for e, s in enumerate(sp):
        y0, m = G.generate(G.make_spec(**s), N_E)
        assert np.abs(y0 - d_y0[e * N_E:(e + 1) * N_E].cpu().numpy()).max() <= 4e-16
        o = oracle.integrate(y0, m, OMEGAF, TOL, TOL)
        r_ref[e] = S.statistics(y0, o["final"], o["steps"])["r"][0]
    assert np.abs(r - r_ref).max() < 2e-4, np.abs(r - r_ref).max()

    # equal mass, maximal spin: 0.99 and 0.65
    assert 0.98 <= r[0, 0] <= 0.995 and 0.62 <= r[0, 1] <= 0.68 and 0.62 <= r[0, 2] <= 0.68
    # PAPER.md:148-150, Fig. 6: "the correlation drops quickly as the masses become uneven"
    assert r[0, 0] > r[1, 0] > r[2, 0] > r[3, 0] and r[3, 0] < 0.5 * r[0, 0]
    # PAPER.md:156, Fig. 7: r(S1^.S2^) > 0.98 for every chi at equal masses, while r(S_j^.L^) varies and is the
    # same for j = 1, 2 ("both BHs enter symmetrically")
    assert np.all(r[4:, 0] > 0.98)
    assert np.abs(r[4:, 1] - r[4:, 2]).max() < 0.03
    assert np.ptp(np.concatenate([r[4:, 1], r[:1, 1]])) > 0.05


def test_run_ensembles_pipeline(oracle):
    """The orchestration helper gives what the separate calls give, and its cross-check agrees with the FP32 bar."""
    import paper_0908_3889_b200 as pn

    sp = specs()[:2]
    res = pn.run_ensembles(sp, 4000, OMEGAF, rtol=1e-5, atol=1e-7, precision=pn.PN_FP32, bins1=20, bins2=16,
                           check_fraction=0.05, check_key=(5, 6))
    assert res["status"] == 0 and res["pearson_r"].shape == (2, 3) and res["hist2"].shape == (2, 3, 16, 16)
    assert np.all(res["moments"][..., 0] == 4000) and np.all(res["hist1"].sum(axis=2) == 4000)
    assert 0.97 < res["pearson_r"][0, 0] < 1.0 and res["pearson_r"][1, 0] < res["pearson_r"][0, 0]
    chk = res["check"]
    assert 300 < chk["n_checked"] < 500 and chk["n_failed_ref"] == 0 and 0 < max(chk["max_dot_dev"]) < 1e-2
    # the same ensembles through the oracle chain: r to the FP32 accuracy
    for e, s in enumerate(sp):
        y0, m = G.generate(G.make_spec(**s), 4000)
        o = oracle.integrate(y0, m, OMEGAF, 1e-10, 1e-12)
        assert np.abs(S.statistics(y0, o["final"])["r"][0] - res["pearson_r"][e]).max() < 5e-4


@pytest.mark.parametrize("fused", [False, True])
def test_sharded_sweep_equals_the_unsplit_call(fused):
    """NEXT-3 "sharded over GPUs per 8(e)" on one GPU: the seven ensembles of the sweep, every ensemble's variate stream
    split three ways (sharding.shard_range; what three ranks would run), each share through pipeline.run_ensembles, the
    shares combined as the ranks combine them (counters summed, moment records merged by pn_merge_statistics in rank order)
    == the unsplit call: every count exactly, means and r to rounding."""
    import paper_0908_3889_b200 as pn
    from paper_0908_3889_b200 import pipeline, sharding

    sp, n, world = specs(), 3001, 3
    kw = dict(rtol=1e-8, atol=1e-10, bins1=20, bins2=16, fused=fused)
    whole = pn.run_ensembles(sp, n, OMEGAF, **kw)
    shares = [pn.run_ensembles(sp, n, OMEGAF, shard=(k, world), **kw) for k in range(world)]
    assert [s["shard"] for s in shares] == [(0, 1001), (1001, 2001), (2001, 3001)]
    assert all(s["status"] == 0 for s in shares)
    got = {k: v.cpu().numpy() for k, v in sharding.merge_shards(shares, pipeline._merge_on_device).items() if hasattr(v, "cpu")}
    for k in ("n_skipped", "hist1", "hist2", "hist2_max"):
        assert np.array_equal(got[k], whole[k]), k
    assert np.array_equal(got["moments"][..., 0], whole["moments"][..., 0]) and np.all(got["moments"][..., 0] == n)
    assert np.abs(got["moments"][..., 1:3] - whole["moments"][..., 1:3]).max() <= 1e-13
    assert np.abs(got["moments"][..., 3:] - whole["moments"][..., 3:]).max() <= 1e-11 * n
    assert np.abs(got["pearson_r"] - whole["pearson_r"]).max() <= 1e-12
    # more ranks than systems: the empty shares are neutral
    tiny = [pn.run_ensembles(sp[:2], 2, OMEGAF, shard=(k, 4), **kw) for k in range(4)]
    assert [s["shard"] for s in tiny] == [(0, 1), (1, 2), (2, 2), (2, 2)]
    t = sharding.merge_shards(tiny, pipeline._merge_on_device)
    w = pn.run_ensembles(sp[:2], 2, OMEGAF, **kw)
    assert np.array_equal(t["hist1"].cpu().numpy(), w["hist1"]) and np.array_equal(t["moments"][..., 0].cpu().numpy(), w["moments"][..., 0])
    assert np.allclose(t["pearson_r"].cpu().numpy(), w["pearson_r"], rtol=0, atol=1e-12, equal_nan=True)
