"""The fused ensemble mode (pn_run_ensembles; SURVEY.md 8(f) NEXT-1/NEXT-2 as defined there): seed in,
statistics out, no state arrays.  Checked (a) against the unfused device chain pn_generate -> pn_integrate -> pn_statistics
on the same arguments (the per-system arithmetic is the same, so every count must agree exactly and the moments to
rounding), and (b) against the oracle chain (generator oracle -> integrator oracle -> statistics oracle)."""
import numpy as np
import pytest

from oracle import pn_gen_oracle as G
from oracle import pn_stats_oracle as S

pytestmark = pytest.mark.gpu
torch = pytest.importorskip("torch")


@pytest.fixture(scope="module")
def pn():
    import paper_0908_3889_b200 as pkg

    return pkg


def outputs(g, bins1, bins2, dev="cuda"):
    f64 = dict(dtype=torch.float64, device=dev)
    i64 = dict(dtype=torch.int64, device=dev)
    o = dict(pearson_r=torch.full((g, 3), -7.0, **f64), moments=torch.full((g, 3, 6), -7.0, **f64), n_skipped=torch.full((g, 3), -7, **i64))
    if bins1:
        o["hist1"] = torch.full((g, 3, bins1), -7, **i64)
    if bins2:
        o["hist2"] = torch.full((g, 3, bins2, bins2), -7, **i64)
        o["hist2_max"] = torch.full((g, 3), -7, **i64)
        o["hist2_norm"] = torch.full((g, 3, bins2, bins2), -7.0, **f64)
    return o


def chain(pn, specs, n_total, first, count, omegaf, rtol, atol, bins1, bins2, **iopts):
    g = len(specs)
    n = g * count
    y0 = torch.empty(n, 10, dtype=torch.float64, device="cuda")
    m = torch.empty(n, 2, dtype=torch.float64, device="cuda")
    pn.pn_generate([pn.make_ensemble(**s) for s in specs], n_total, y0, m, first=first, count=count)
    yf = torch.empty_like(y0)
    steps = torch.empty(n, dtype=torch.int32, device="cuda")
    st = pn.pn_integrate(y0, m, 0.0, omegaf, rtol, atol, pn.PN_FP64, yf, steps, allow_failures=True, **iopts)
    o = outputs(g, bins1, bins2)
    pn.pn_statistics(y0, yf, steps, group_size=count, bins1=bins1, bins2=bins2, **o)
    return st, {k: v.cpu().numpy() for k, v in o.items()}, pn.pn_last_counters()


def fused(pn, specs, n_total, first, count, omegaf, rtol, atol, bins1, bins2, **opts):
    o = outputs(len(specs), bins1, bins2)
    st = pn.pn_run_ensembles([pn.make_ensemble(**s) for s in specs], n_total, omegaf, rtol, atol, first=first, count=count,
                             bins1=bins1, bins2=bins2, allow_failures=True, **o, **opts)
    return st, {k: v.cpu().numpy() for k, v in o.items()}, pn.pn_last_counters()


def same(a, b, n_per):
    """fused vs chain: integer outputs exactly, moments to rounding"""
    for k in ("n_skipped", "hist1", "hist2", "hist2_max"):
        if k in a:
            assert np.array_equal(a[k], b[k]), k
    if "hist2_norm" in a:
        assert np.array_equal(a["hist2_norm"], b["hist2_norm"])
    assert np.array_equal(a["moments"][..., 0], b["moments"][..., 0])
    assert np.allclose(a["moments"][..., 1:3], b["moments"][..., 1:3], rtol=0, atol=1e-13, equal_nan=True)
    assert np.allclose(a["moments"][..., 3:], b["moments"][..., 3:], rtol=0, atol=1e-11 * n_per)
    assert np.allclose(a["pearson_r"], b["pearson_r"], rtol=0, atol=1e-12, equal_nan=True)


SWEEP = [dict(key=(11, 0), omega0=0.02, q=(1.0, 1.0), chi1=(1.0, 1.0), chi2=(1.0, 1.0)),
         dict(key=(11, 1), omega0=0.02, q=(0.3, 1.0), chi1=(0.0, 1.0), chi2=(0.0, 1.0)),
         dict(key=(11, 2), omega0=0.025, q=(2 / 3, 2 / 3), chi1=(0.9, 0.9), chi2=(1.0, 1.0), m1_fixed=0.6, s1_tilt_deg=60.0)]


def test_fused_equals_the_unfused_chain(pn):
    """Three ensembles (equal mass; mixed q and chi; C4's fixed tilted S1, whose x is constant: r = NaN, M2x = 0), a ragged
    chunk [first, first + count) whose size is not a multiple of the 32-system draws, 1-D and 2-D histograms."""
    n_total, first, count = 5000, 123, 4001
    st_c, c, kc = chain(pn, SWEEP, n_total, first, count, 0.05, 1e-10, 1e-12, 50, 79)
    st_f, f, kf = fused(pn, SWEEP, n_total, first, count, 0.05, 1e-10, 1e-12, 50, 79)
    assert st_c == st_f == 0
    same(f, c, count)
    assert kf["trial_steps"] == kc["trial_steps"] and kf["rejected"] == kc["rejected"] and kf["failed"] == 0
    assert np.all(f["moments"][..., 0] == count) and np.all(f["hist1"].sum(axis=2) == count) and np.all(f["hist2"].sum(axis=(2, 3)) == count)
    assert np.isnan(f["pearson_r"][2, 1]) and f["moments"][2, 1, 3] == 0.0       # constant x: exact zero variance
    # counts are reproducible run to run; moments to rounding
    st_g, g, _ = fused(pn, SWEEP, n_total, first, count, 0.05, 1e-10, 1e-12, 50, 79)
    same(g, f, count)
    # the queue is issued longest-expected-first inside every chunk (keys from a draw-only pass); the order changes nothing
    st_h, h, kh = fused(pn, SWEEP, n_total, first, count, 0.05, 1e-10, 1e-12, 50, 79, input_order=True)
    same(h, f, count)
    assert kh["trial_steps"] == kf["trial_steps"]
    # without histograms, without moments, tiny ensembles (fewer systems than one draw), one system
    for cnt in (1, 31, 33):
        _, c2, _ = chain(pn, SWEEP[:2], 64, 5, cnt, 0.05, 1e-10, 1e-12, 0, 0)
        _, f2, _ = fused(pn, SWEEP[:2], 64, 5, cnt, 0.05, 1e-10, 1e-12, 0, 0)
        same(f2, c2, cnt)


def test_fused_single_fixed_mass_ensemble_takes_the_uniform_mass_kernel(pn):
    """ONE ensemble with fixed masses (every ensemble of the paper's section V) runs the uniform-mass instantiation of the
    fused kernel (constants from the __constant__ table, brace constants folded).  The unfused chain
    takes the uniform-mass kernel for such a batch too, so the two still agree exactly; against the generic fused kernel
    (pn_options.variant bit 0) the arithmetic differs in rounding: same n, r to 1e-9, histogram counts off by a few
    systems next to a bin edge at most."""
    for spec in (SWEEP[0], SWEEP[2]):
        n = 6000 + 13
        st_c, c, kc = chain(pn, [spec], n, 0, n, 0.05, 1e-10, 1e-12, 50, 31)
        st_f, f, kf = fused(pn, [spec], n, 0, n, 0.05, 1e-10, 1e-12, 50, 31)
        st_g, g, kg = fused(pn, [spec], n, 0, n, 0.05, 1e-10, 1e-12, 50, 31, variant=1)
        assert st_c == st_f == st_g == 0
        same(f, c, n)
        assert kf["trial_steps"] == kc["trial_steps"] and kf["rejected"] == kc["rejected"]
        assert not np.array_equal(f["moments"], g["moments"])          # the uniform-mass kernel did run
        assert np.array_equal(f["moments"][..., 0], g["moments"][..., 0]) and np.array_equal(f["n_skipped"], g["n_skipped"])
        assert np.allclose(f["pearson_r"], g["pearson_r"], rtol=0, atol=1e-9, equal_nan=True)
        assert np.abs(f["hist1"] - g["hist1"]).sum() <= 4 and np.abs(f["hist2"] - g["hist2"]).sum() <= 8
        assert abs(kf["trial_steps"] / kg["trial_steps"] - 1) < 1e-3


def test_fused_equal_mass_sweep_takes_the_same_kernel_as_the_chain(pn):
    """Several ensembles that all have the SAME fixed masses (an equal-mass sweep over chi): the unfused
    chain's seed kernel finds the concatenated batch uniform and runs the uniform-mass kernel, so the fused call must take
    its uniform-mass instantiation too (it decides over ALL ensembles of the call), or step sequences and bin-edge counts
    could differ.  Exact agreement of every count and of the trial-step totals; and one ensemble with other
    masses in the call sends both sides to the generic kernel, again in exact agreement."""
    chis = (0.3, 0.7, 1.0)
    by_m1 = [dict(key=(21, k), omega0=0.02, q=(1.0, 1.0), chi1=(c, c), chi2=(c, c), m1_fixed=0.5) for k, c in enumerate(chis)]
    by_q = [dict(key=(22, k), omega0=0.02, q=(1.0, 1.0), chi1=(c, c), chi2=(c, c)) for k, c in enumerate(chis)]
    mixed = by_m1[:2] + [dict(key=(23, 0), omega0=0.02, q=(1.0, 1.0), chi1=(1.0, 1.0), chi2=(1.0, 1.0), m1_fixed=0.6)]
    n = 3000 + 7
    for specs, uniform in ((by_m1, True), (by_q, True), (by_m1[:1] + by_q[1:], True), (mixed, False)):
        st_c, c, kc = chain(pn, specs, n, 0, n, 0.05, 1e-10, 1e-12, 50, 31)
        st_f, f, kf = fused(pn, specs, n, 0, n, 0.05, 1e-10, 1e-12, 50, 31)
        assert st_c == st_f == 0
        same(f, c, n)
        assert kf["trial_steps"] == kc["trial_steps"] and kf["rejected"] == kc["rejected"] and kf["landing_trials"] == kc["landing_trials"]
        # the generic kernel (variant bit 0) rounds differently from the uniform-mass one: same n, r to 1e-9
        _, g, kg = fused(pn, specs, n, 0, n, 0.05, 1e-10, 1e-12, 50, 31, variant=1)
        if uniform:
            assert not np.array_equal(f["moments"], g["moments"])      # the uniform-mass kernel did run
        else:
            assert kg["trial_steps"] == kf["trial_steps"]              # both are the generic kernel
        assert np.array_equal(f["moments"][..., 0], g["moments"][..., 0])
        assert np.allclose(f["pearson_r"], g["pearson_r"], rtol=0, atol=1e-9, equal_nan=True)


def test_fused_against_the_oracle_chain(pn, oracle):
    specs = SWEEP[:2]
    n = 700
    _, f, _ = fused(pn, specs, n, 0, n, 0.05, 1e-10, 1e-12, 50, 20)
    for e, s in enumerate(specs):
        y0, m = G.generate(G.make_spec(**s), n)
        o = oracle.integrate(y0, m, 0.05, 1e-10, 1e-12)
        ref = S.statistics(y0, o["final"], o["steps"], None, 50, 20)
        assert np.abs(f["pearson_r"][e] - ref["r"][0]).max() < 1e-8
        assert np.abs(f["hist1"][e] - ref["hist1"][0].astype(np.int64)).sum() <= 4
        assert np.abs(f["hist2"][e] - ref["hist2"][0].astype(np.int64)).sum() <= 8
        assert np.array_equal(f["moments"][e, :, 0], ref["moments"][0, :, 0])
        assert np.abs(f["moments"][e, :, 1:3] - ref["moments"][0, :, 1:3]).max() < 1e-9


def test_fused_uniform_mass_kernel_against_the_oracle_chain(pn, oracle):
    """ONE fixed-mass ensemble selects the uniform-mass instantiation of the fused kernel (the one bench.py times as
    widened.fused): compared directly with the oracle chain (generator oracle -> integrator oracle -> statistics oracle),
    not through the unfused device chain.  4096 + 37 systems: several draws per warp and a ragged last one."""
    n = 4096 + 37
    for spec in (SWEEP[0], SWEEP[2]):
        _, f, kf = fused(pn, [spec], n, 0, n, 0.05, 1e-10, 1e-12, 50, 20)
        _, g, _ = fused(pn, [spec], n, 0, n, 0.05, 1e-10, 1e-12, 50, 20, variant=1)
        assert not np.array_equal(f["moments"], g["moments"])          # the uniform-mass kernel did run
        y0, m = G.generate(G.make_spec(**spec), n)
        o = oracle.integrate(y0, m, 0.05, 1e-10, 1e-12)
        ref = S.statistics(y0, o["final"], o["steps"], None, 50, 20)
        defined = np.isfinite(ref["r"][0])
        assert np.array_equal(defined, np.isfinite(f["pearson_r"][0]))
        assert np.abs(f["pearson_r"][0] - ref["r"][0])[defined].max() < 1e-8
        assert np.abs(f["hist1"][0] - ref["hist1"][0].astype(np.int64)).sum() <= 4
        assert np.abs(f["hist2"][0] - ref["hist2"][0].astype(np.int64)).sum() <= 8
        assert np.array_equal(f["moments"][0, :, 0], ref["moments"][0, :, 0])
        assert np.abs(f["moments"][0, :, 1:3] - ref["moments"][0, :, 1:3]).max() < 1e-9
        assert abs(kf["trial_steps"] / int(o["steps"].sum()) - 1) < 1e-3


def test_fused_redo_pass_failures_and_host_buffers(pn):
    # loose tolerance: steps leave the range of the cbrt/log series, such systems go through the redo pass of the fused mode too
    st_c, c, kc = chain(pn, SWEEP[:2], 3000, 0, 3000, 0.05, 1e-3, 1e-5, 40, 0)
    st_f, f, kf = fused(pn, SWEEP[:2], 3000, 0, 3000, 0.05, 1e-3, 1e-5, 40, 0)
    assert kf["redo"] > 0 and st_c == st_f
    same(f, c, 3000)
    # every system fails (max_steps): all skipped, nothing counted, status PN_ENOTCONVERGED
    st_f, f, kf = fused(pn, SWEEP[:2], 500, 0, 500, 0.05, 1e-10, 1e-12, 10, 0, max_steps=7)
    assert st_f == 3 and np.all(f["n_skipped"] == 500) and np.all(f["moments"][..., 0] == 0) and f["hist1"].sum() == 0
    assert np.all(np.isnan(f["pearson_r"])) and kf["failed"] == 1000 and kf["trial_steps"] == 7 * 1000
    # host buffers: numpy outputs
    o = {k: v.cpu().numpy() for k, v in outputs(2, 30, 12).items()}
    pn.pn_run_ensembles([pn.make_ensemble(**s) for s in SWEEP[:2]], 900, 0.05, 1e-10, 1e-12, bins1=30, bins2=12, **o)
    _, d, _ = fused(pn, SWEEP[:2], 900, 0, 900, 0.05, 1e-10, 1e-12, 30, 12)
    same(o, d, 900)
    # argument errors
    with pytest.raises(pn.PnError):
        pn.pn_run_ensembles(pn.make_ensemble((1, 1), 0.06), 100, 0.05, 1e-10, 1e-12, pearson_r=torch.zeros(1, 3, dtype=torch.float64, device="cuda"))
    with pytest.raises(pn.PnError):
        pn.pn_run_ensembles(pn.make_ensemble((1, 1), 0.02), 100, 0.05, 1e-5, 1e-7, precision=pn.PN_FP32,
                            pearson_r=torch.zeros(1, 3, dtype=torch.float64, device="cuda"))
    assert pn.pn_run_ensembles(pn.make_ensemble((1, 1), 0.02), 100, 0.05, 1e-10, 1e-12, count=0,
                               pearson_r=torch.zeros(1, 3, dtype=torch.float64, device="cuda")) == 0


def test_fused_large_run_needs_no_state_arrays(pn):
    """6.3 M short inspirals in two chunks of the launch loop (PN_FUSED_CHUNK = 2^22): device memory in use by the library
    stays small (no 96 + 80 + 320 B per system), and the counts equal the unfused chain's on the same ensemble."""
    spec = [dict(key=(77, 5), omega0=0.045, q=(0.5, 1.0), chi1=(0.2, 1.0), chi2=(0.2, 1.0))]
    n = 3 * (1 << 21) + 17
    pn.pn_shutdown()
    torch.cuda.synchronize(); torch.cuda.empty_cache()
    free0, _ = torch.cuda.mem_get_info()
    _, f, kf = fused(pn, spec, n, 0, n, 0.05, 1e-8, 1e-10, 50, 0)
    free1, _ = torch.cuda.mem_get_info()
    assert free0 - free1 < 256e6, (free0 - free1)                # the unfused chain holds ~600 B per system: 3.8 GB
    assert np.all(f["moments"][0, :, 0] == n) and np.all(f["hist1"][0].sum(axis=1) == n) and kf["failed"] == 0
    _, c, kc = chain(pn, spec, n, 0, n, 0.05, 1e-8, 1e-10, 50, 0)
    same(f, c, n)
    assert kc["trial_steps"] == kf["trial_steps"]
    pn.pn_shutdown()
    torch.cuda.empty_cache()
