"""GPU edge cases of the boundary: empty / tiny / ragged batches, failure codes, layouts, host buffers,
determinism, and the full-size launch configuration checked on sampled systems."""
import numpy as np
import pytest

from paper_0908_3889_b200 import workloads as W
from test_gpu_parity import check_adaptive, dots_of, gpu_integrate, pn  # noqa: F401

pytestmark = pytest.mark.gpu
torch = pytest.importorskip("torch")


def test_empty_and_tiny(pn, oracle):
    dev = "cuda:0"
    e10 = torch.empty(0, 10, dtype=torch.float64, device=dev)
    e2 = torch.empty(0, 2, dtype=torch.float64, device=dev)
    es = torch.empty(0, dtype=torch.int32, device=dev)
    assert pn.pn_integrate(e10, e2, 0.0, 0.05, 1e-10, 1e-12, 0, e10, es) == 0
    counts = torch.ones(3, 7, dtype=torch.int64, device=dev)
    pn.pn_histogram(e10, 7, counts, n=0)
    assert counts.sum().item() == 0
    for n in (1, 31, 33, 257):
        cfg = W.with_size(W.CONFIGS["C1"], n)
        y0, m = W.generate(cfg)
        check_adaptive(pn, oracle, cfg, y0, m)


def test_invalid_arguments(pn):
    from paper_0908_3889_b200 import PnError

    cfg = W.with_size(W.CONFIGS["C1"], 64)
    y0, m = W.generate(cfg)
    with pytest.raises(PnError) as e:
        gpu_integrate(pn, y0, m, cfg, rtol=0.0)
    assert e.value.status == 1
    with pytest.raises(PnError):
        gpu_integrate(pn, y0, m, cfg, omega0=0.06)            # omega0 >= omega_f
    with pytest.raises(PnError):
        gpu_integrate(pn, y0, m, cfg, precision=7)
    with pytest.raises(PnError):
        pn.pn_histogram(torch.zeros(4, 10, dtype=torch.float64, device="cuda:0"), 0,
                        torch.zeros(3, 1, dtype=torch.int64, device="cuda:0"))
    # wrong omega0 for one system -> that system is flagged, the call reports EINVAL, others complete
    y1 = y0.copy(); y1[5, 0] = 0.021
    g = gpu_integrate(pn, y1, m, cfg, omega0=0.02, allow_failures=True)
    assert g["status"] == 1 and g["steps"][5] == -5 and np.all(np.delete(g["steps"], 5) > 0)


def test_per_system_failures_do_not_stop_the_batch(pn):
    cfg = W.with_size(W.CONFIGS["C1"], 100)
    y0, m = W.generate(cfg)
    m[3, 1] = -0.5                      # bad mass
    y0[7, 0] = 0.07                     # already beyond omega_f
    g = gpu_integrate(pn, y0, m, cfg, allow_failures=True)
    assert g["status"] == 1
    assert g["steps"][3] == -5 and g["steps"][7] == -5
    good = np.ones(100, bool); good[[3, 7]] = False
    assert np.all(g["steps"][good] > 0)
    assert np.array_equal(g["final"][3], y0[3])
    # max_steps
    g = gpu_integrate(pn, y0[good], m[good], cfg, max_steps=20, allow_failures=True)
    assert g["status"] == 3 and np.all(g["steps"] == -1)
    c = pn.pn_last_counters()
    assert c["failed"] == good.sum() and c["trial_steps"] == 20 * good.sum()
    # non-finite state
    y2 = y0[good].copy(); y2[0, 2] = np.nan
    g = gpu_integrate(pn, y2, m[good], cfg, allow_failures=True)
    assert g["status"] == 4 and g["steps"][0] == -3 and np.all(g["steps"][1:] > 0)


def test_zero_spin_and_aligned_systems(pn, oracle):
    """Degenerate cases of the method: chi = 0 (no division by |S|), aligned spins (no precession)."""
    cfg = W.with_size(W.CONFIGS["C2"], 6)
    y0, m = W.generate(cfg)
    y0[0, 1:7] = 0.0
    y0[1, 1:4] = 0.0
    y0[2, 1:4] = [0, 0, 0.25]; y0[2, 4:7] = [0, 0, -0.25]
    g, r = check_adaptive(pn, oracle, cfg, y0, m)
    assert np.array_equal(g["final"][0, 1:], y0[0, 1:]) and np.array_equal(g["final"][2, 1:], y0[2, 1:])
    counts = torch.zeros(3, 10, dtype=torch.int64, device="cuda:0")
    skipped = torch.zeros(3, dtype=torch.int64, device="cuda:0")
    pn.pn_histogram(g["d_final"], 10, counts, skipped)
    assert skipped.cpu().tolist() == [2, 2, 1]


def test_layouts_host_buffers_and_determinism(pn, oracle):
    cfg = W.with_size(W.CONFIGS["C3"], 1000)
    y0, m = W.generate(cfg)
    a = gpu_integrate(pn, y0, m, cfg)
    b = gpu_integrate(pn, y0, m, cfg)
    assert np.array_equal(a["final"], b["final"]) and np.array_equal(a["steps"], b["steps"])   # queue order is irrelevant
    # SoA layout
    dev = "cuda:0"
    d_y0 = torch.from_numpy(y0.T.copy()).to(dev); d_m = torch.from_numpy(m.T.copy()).to(dev)
    d_yf = torch.empty_like(d_y0); d_steps = torch.empty(cfg.n, dtype=torch.int32, device=dev)
    pn.pn_integrate(d_y0, d_m, 0.0, cfg.omegaf, cfg.rtol, cfg.atol, 0, d_yf, d_steps, layout=1)
    assert np.array_equal(d_yf.cpu().numpy().T, a["final"]) and np.array_equal(d_steps.cpu().numpy(), a["steps"])
    # host buffers (numpy in, numpy out)
    h_yf = np.empty_like(y0); h_steps = np.empty(cfg.n, dtype=np.int32); h_t = np.empty(cfg.n)
    pn.pn_integrate(y0, m, 0.0, cfg.omegaf, cfg.rtol, cfg.atol, 0, h_yf, h_steps, out_time=h_t)
    assert np.array_equal(h_yf, a["final"]) and np.array_equal(h_steps, a["steps"]) and np.array_equal(h_t, a["time"])
    # queue order does not change any result: input order vs the default longest-expected-first
    d = gpu_integrate(pn, W.generate(W.with_size(cfg, 3000))[0], W.generate(W.with_size(cfg, 3000))[1], W.with_size(cfg, 3000))
    e = gpu_integrate(pn, W.generate(W.with_size(cfg, 3000))[0], W.generate(W.with_size(cfg, 3000))[1], W.with_size(cfg, 3000), input_order=True)
    assert np.array_equal(d["final"], e["final"]) and np.array_equal(d["steps"], e["steps"])
    d = gpu_integrate(pn, y0, m, cfg, input_order=True)
    assert np.array_equal(d["final"], a["final"]) and np.array_equal(d["steps"], a["steps"])
    # both block shapes agree bit for bit
    c = gpu_integrate(pn, y0, m, cfg, block_threads=256)
    assert np.array_equal(c["final"], a["final"])
    # a stream from torch, async enqueue, status collected afterwards
    s = torch.cuda.Stream()
    d_y0a = torch.from_numpy(y0).to(dev); d_ma = torch.from_numpy(m).to(dev)
    d_yfa = torch.empty_like(d_y0a); s.wait_stream(torch.cuda.current_stream())
    pn.pn_integrate(d_y0a, d_ma, 0.0, cfg.omegaf, cfg.rtol, cfg.atol, 0, d_yfa, d_steps, stream=s, async_=True)
    assert pn.pn_stream_status(s) == 0
    assert np.array_equal(d_yfa.cpu().numpy(), a["final"])


@pytest.mark.parametrize("name,nsample", [("C2", 768), ("C3", 768), ("C4", 1024), ("C5", 192)])
def test_full_size_launch_configuration_sampled(pn, oracle, name, nsample):
    """BASELINE.json's full sizes in the launch configuration bench.py times; outputs compared on a
    seeded sample the oracle can compute one by one, plus properties that hold at any size."""
    cfg = W.CONFIGS[name]
    y0, m = W.generate(cfg)
    idx = W.sample_indices(cfg.n, nsample)
    g, r = check_adaptive(pn, oracle, cfg, y0, m, idx=idx)
    f = g["final"]
    assert np.abs(f[:, 0] - cfg.omegaf).max() <= 1.01e-13 * cfg.omegaf
    for s in (slice(1, 4), slice(4, 7), slice(7, 10)):
        n0 = np.linalg.norm(y0[:, s], axis=1); n1 = np.linalg.norm(f[:, s], axis=1)
        ok = n0 > 0
        assert np.abs(n1[ok] / n0[ok] - 1).max() < 1e-7
    c = pn.pn_last_counters()
    assert c["trial_steps"] == g["steps"].sum() and c["failed"] == 0
    counts = torch.zeros(3, cfg.bins, dtype=torch.int64, device="cuda:0")
    skipped = torch.zeros(3, dtype=torch.int64, device="cuda:0")
    pn.pn_histogram(g["d_final"], cfg.bins, counts, skipped)
    c_ref = oracle.histogram(f, cfg.bins)[0].astype(np.int64)
    assert np.abs(counts.cpu().numpy() - c_ref).sum() <= 8
    assert counts.sum().item() + skipped.sum().item() == 3 * cfg.n


def test_fp32_full_size_C4_histograms(pn, oracle):
    cfg64, cfg32 = W.CONFIGS["C4"], W.CONFIGS["C4f"]
    y0, m = W.generate(cfg64)
    a = gpu_integrate(pn, y0, m, cfg64)
    b = gpu_integrate(pn, y0, m, cfg32, precision=1)
    da, db = dots_of(oracle, a["final"]), dots_of(oracle, b["final"])
    assert np.abs(da - db).max() <= 2e-3
    ca = oracle.histogram(a["final"], 50)[0].astype(np.int64); cb = oracle.histogram(b["final"], 50)[0].astype(np.int64)
    assert np.all(np.abs(ca - cb) <= 5 * np.sqrt(ca + cb + 1))


def test_loose_tolerance_uses_the_redo_pass(pn, oracle):
    """FP64 at a very loose tolerance: steps change omega by more than 3 %, which is outside the range of the
    in-step cbrt/log series; such systems are re-integrated by the wide-range redo kernel.  The result
    still tracks the oracle run with the same settings to tolerance level."""
    cfg = W.with_size(W.CONFIGS["C1"], 300)
    y0, m = W.generate(cfg)
    g = gpu_integrate(pn, y0, m, cfg, rtol=1e-3, atol=1e-5)
    assert g["status"] == 0 and np.all(g["steps"] > 0)
    assert pn.pn_last_counters()["redo"] > 0
    r = oracle.integrate(y0, m, cfg.omegaf, 1e-3, 1e-5)
    ref = oracle.integrate(y0, m, cfg.omegaf, 1e-10, 1e-12)
    dg, dr, dref = dots_of(oracle, g["final"]), dots_of(oracle, r["final"]), dots_of(oracle, ref["final"])
    err_oracle = np.abs(dr - dref).max()
    assert np.abs(dg - dref).max() <= 3 * err_oracle + 1e-6      # as accurate as the oracle at this tolerance
    assert np.abs(g["final"][:, 0] - cfg.omegaf).max() <= 1.01e-13 * cfg.omegaf
    assert abs(g["steps"].mean() / r["steps"].mean() - 1) < 0.1
    # fixed-step mode with a huge step goes through the fixed-step redo kernel and still matches the oracle
    g = gpu_integrate(pn, y0[:64], m[:64], cfg, fixed_steps=20, h0=100.0)
    r = oracle.integrate(y0[:64], m[:64], 0, 0, 0, fixed_steps=20, h0=100.0)
    assert pn.pn_last_counters()["redo"] > 0
    from test_gpu_parity import comp_scale
    assert (np.abs(g["final"] - r["final"]) / comp_scale(y0[:64])).max() <= 1e-11


def close_runs(a, b, frac_same_steps=0.999, rtol=1e-10):
    """Two FP64 runs of the same systems whose arithmetic differs only in rounding (constants folded differently).
    Bounds, with the measurement behind them (B200, uniform-mass vs generic kernel, rtol 1e-10: C4 x 200,000 systems,
    C2 x 20,000, C1 x 1024): the step sequence is the same unless an accept / reject decision with E within rounding of 1
    falls the other way, which happened to 6.5e-5 of the systems at worst (asserted: at most 1e-3); with the same step
    sequence the final states differ by accumulated rounding, 2.2e-13 at worst over ~1100 steps (asserted: 1e-2 rtol);
    with a different one both are solutions within the tolerance and differ by less than one step's allowed local
    error, measured 2.2e-13 (asserted: rtol); final times agreed to 2e-14 relative (asserted: 1e-2 rtol)."""
    same = a["steps"] == b["steps"]
    assert same.mean() >= frac_same_steps, same.mean()
    assert np.abs(a["final"][same] - b["final"][same]).max() <= 1e-2 * rtol
    assert np.abs(a["final"] - b["final"]).max() <= rtol
    assert np.abs(a["time"] / b["time"] - 1).max() <= 1e-2 * rtol


def test_uniform_mass_fast_path_matches_the_generic_kernel(pn):
    """FP64 batches whose systems all have the masses of system 0 run a kernel that takes the mass-dependent constants
    from a __constant__ table row, with the factor K0/Bc folded into the constants of the brace of Eq. (1)
    (one multiply fewer per evaluation), so its results equal the generic kernel's to rounding, not to the bit; one
    deviating system anywhere in the batch switches the whole launch to the generic kernel, bit for bit."""
    cfg = W.with_size(W.CONFIGS["C4"], 3000 + 17)
    y0, m = W.generate(cfg)
    a = gpu_integrate(pn, y0, m, cfg)
    b = gpu_integrate(pn, y0, m, cfg, variant=1)          # pn_options.variant bit 0: always the generic kernel
    assert not np.array_equal(a["final"], b["final"])     # the fast path did run
    close_runs(a, b)
    a2 = gpu_integrate(pn, y0, m, cfg)
    for k in ("final", "steps", "time", "rejected"):
        assert np.array_equal(a[k], a2[k]), k              # and is deterministic
    # a batch that is uniform except for its last system, and one whose system 0 is invalid: the generic kernel runs
    m2 = m.copy(); m2[-1] = [0.5, 0.5]
    c = gpu_integrate(pn, y0, m2, cfg)
    assert np.array_equal(c["final"][:-1], b["final"][:-1]) and not np.array_equal(c["final"][-1], b["final"][-1])
    m3 = m.copy(); m3[0, 0] = -1.0
    d = gpu_integrate(pn, y0, m3, cfg, allow_failures=True)
    assert d["steps"][0] == -5 and np.array_equal(d["final"][1:], b["final"][1:])


def test_large_batch_2_26_systems(pn):
    """Maximum sizes: 2^26 + 3 systems (67 M; ~36 GB of device memory with the library's scratch) generated on the
    device, integrated in FP32 over a short frequency range, reduced on the device.  Checked by properties that hold at
    any size and by re-integrating sampled rows in small batches (results do not depend on the batch they are in)."""
    n = (1 << 26) + 3
    free, _ = torch.cuda.mem_get_info()
    if free < 60e9:
        pytest.skip("needs ~40 GB of free device memory")
    ens = pn.make_ensemble((26, 3), 0.04, q=(0.5, 1.0), chi1=(0.2, 1.0), chi2=(0.2, 1.0))
    y0 = torch.empty(n, 10, dtype=torch.float64, device="cuda")
    m = torch.empty(n, 2, dtype=torch.float64, device="cuda")
    pn.pn_generate(ens, n, y0, m)
    yf = torch.empty_like(y0)
    st = torch.empty(n, dtype=torch.int32, device="cuda")
    assert pn.pn_integrate(y0, m, 0.04, 0.05, 1e-5, 1e-7, pn.PN_FP32, yf, st) == 0
    assert int(st.min().item()) > 0 and pn.pn_last_counters()["failed"] == 0
    mom = torch.zeros(1, 3, 6, dtype=torch.float64, device="cuda")
    h1 = torch.zeros(1, 3, 50, dtype=torch.int64, device="cuda")
    sk = torch.zeros(1, 3, dtype=torch.int64, device="cuda")
    pn.pn_statistics(y0, yf, st, bins1=50, moments=mom, hist1=h1, n_skipped=sk)
    mom, h1 = mom.cpu().numpy()[0], h1.cpu().numpy()[0]
    assert np.all(mom[:, 0] == n) and np.all(h1.sum(axis=1) == n) and int(sk.sum().item()) == 0
    # isotropic initial spins: <x> = 0, M2x / n = 1/3, to 5 sigma of 6.7e7 samples
    assert np.abs(mom[:, 1]).max() < 5 * np.sqrt(1 / 3 / n) and np.abs(mom[:, 3] / n - 1 / 3).max() < 5 * np.sqrt(4 / 45 / n)
    assert abs(float(yf[:, 0].max().item()) / 0.05 - 1) < 4e-7 and abs(float(yf[:, 0].min().item()) / 0.05 - 1) < 4e-7
    # the first, the last and a middle slice re-integrated alone give the same bits
    for lo in (0, n // 2 + 12345, n - 1000):
        a = torch.empty(1000, 10, dtype=torch.float64, device="cuda")
        s2 = torch.empty(1000, dtype=torch.int32, device="cuda")
        pn.pn_integrate(y0[lo:lo + 1000].contiguous(), m[lo:lo + 1000].contiguous(), 0.04, 0.05, 1e-5, 1e-7, pn.PN_FP32, a, s2)
        assert torch.equal(a, yf[lo:lo + 1000]) and torch.equal(s2, st[lo:lo + 1000])
    del y0, m, yf, st
    pn.pn_shutdown()                      # give the scratch back for the tests that follow
    torch.cuda.empty_cache()


@pytest.mark.parametrize("prec", [0, 1, 2])
def test_atol_zero_is_allowed(pn, oracle, prec):
    """atol = 0 with components that start at exactly 0 (L^_x = L^_y = 0): the error scale of such a component must not
    become 0 (0/0 in the norm); the run completes and agrees with the oracle at the same pure-relative tolerance."""
    cfg = W.with_size(W.CONFIGS["C1"], 257)
    y0, m = W.generate(cfg)
    rtol = [1e-9, 1e-5, 1e-7][prec]
    g = gpu_integrate(pn, y0, m, cfg, rtol=rtol, atol=0.0, precision=prec)
    assert g["status"] == 0 and np.all(g["steps"] > 0)
    r = oracle.integrate(y0, m, cfg.omegaf, 1e-10, 1e-12)
    dg, dr = dots_of(oracle, g["final"]), dots_of(oracle, r["final"])
    assert np.abs(dg - dr).max() <= [1e-6, 2e-3, 2e-4][prec]


def test_fp64_at_loose_tolerances_full_batch(pn, oracle):
    """FP64 at the paper's tolerance (5e-7) and looser, long inspirals (t_f ~ 2e5 M), 2^18 systems.
    (a) No system fails: a landing correction can be as small as one ulp of t, which the step-size-underflow test
    must not mistake for stagnation (the oracle's criterion is t + h == t).  (b) At 5e-7 the cbrt/log series range
    follows the tolerance, so almost no system needs the redo pass.  (c) Sampled systems agree with the oracle run at
    the same tolerance to the accuracy that tolerance buys."""
    cfg = W.with_size(W.CONFIGS["C2"], 1 << 18)
    y0, m = W.generate(cfg)
    y0[:, 0] = 0.00395
    idx = W.sample_indices(cfg.n, 256)
    ref = oracle.integrate(y0[idx], m[idx], cfg.omegaf, 1e-10, 1e-12)
    dref = dots_of(oracle, ref["final"])
    for tol, redo_max in ((5e-7, 0.01), (1e-5, 1.0)):
        g = gpu_integrate(pn, y0, m, cfg, rtol=tol, atol=tol, allow_failures=True)
        k = pn.pn_last_counters()
        assert g["status"] == 0 and k["failed"] == 0 and np.all(g["steps"] > 0)
        assert k["redo"] <= redo_max * cfg.n
        assert np.abs(g["final"][:, 0] / cfg.omegaf - 1).max() <= 1.01e-13
        o = oracle.integrate(y0[idx], m[idx], cfg.omegaf, tol, tol)
        err_o = np.abs(dots_of(oracle, o["final"]) - dref).max()
        err_g = np.abs(dots_of(oracle, g["final"][idx]) - dref).max()
        assert err_g <= 3 * err_o + 1e-6, (tol, err_g, err_o)
        assert abs(g["steps"][idx].mean() / o["steps"].mean() - 1) < 0.1
        assert np.abs(g["time"][idx] / o["time"] - 1).max() < 50 * tol


def test_async_calls_keep_their_status_and_scratch(pn):
    """The async contract of include/pn.h: pn_stream_status returns the worst status of ALL async calls enqueued on the
    stream since the last collection (a later call does not erase an earlier call's status), calls in flight on
    different streams do not share scratch, and async calls keep the uniform-mass fast path (decided on the device)."""
    dev = "cuda:0"
    cfg3 = W.with_size(W.CONFIGS["C3"], 3000 + 5)
    y3, m3 = W.generate(cfg3)
    cfg4 = W.with_size(W.CONFIGS["C4"], 4000 + 3)
    y4, m4 = W.generate(cfg4)
    ref3 = gpu_integrate(pn, y3, m3, cfg3)
    ref4 = gpu_integrate(pn, y4, m4, cfg4)
    ref4g = gpu_integrate(pn, y4, m4, cfg4, variant=1)
    close_runs(ref4, ref4g)

    def bufs(n):
        return (torch.full((n, 10), float("nan"), dtype=torch.float64, device=dev), torch.zeros(n, dtype=torch.int32, device=dev))

    m3_bad = m3.copy(); m3_bad[3, 1] = -0.5
    d_y3, d_m3, d_m3b = (torch.from_numpy(a).to(dev) for a in (y3, m3, m3_bad))
    d_y4, d_m4 = torch.from_numpy(y4).to(dev), torch.from_numpy(m4).to(dev)
    s1, s2 = torch.cuda.Stream(), torch.cuda.Stream()
    torch.cuda.synchronize()
    # (a) two calls back to back on ONE stream, the first with a bad-mass system
    f1, st1 = bufs(cfg3.n); f2, st2 = bufs(cfg3.n)
    assert pn.pn_integrate(d_y3, d_m3b, 0.0, cfg3.omegaf, cfg3.rtol, cfg3.atol, 0, f1, st1, stream=s1, async_=True) == 0
    assert pn.pn_integrate(d_y3, d_m3, 0.0, cfg3.omegaf, cfg3.rtol, cfg3.atol, 0, f2, st2, stream=s1, async_=True) == 0
    assert pn.pn_stream_status(s1) == 1                     # PN_EINVAL of the FIRST call survives the second
    assert pn.pn_stream_status(s1) == 0                     # collected: cleared
    good = np.ones(cfg3.n, bool); good[3] = False
    assert st1.cpu().numpy()[3] == -5
    assert np.array_equal(f1.cpu().numpy()[good], ref3["final"][good]) and np.array_equal(st1.cpu().numpy()[good], ref3["steps"][good])
    assert np.array_equal(f2.cpu().numpy(), ref3["final"]) and np.array_equal(st2.cpu().numpy(), ref3["steps"])
    # (b) two calls in flight on DIFFERENT streams (mixed-mass batch on one, uniform-mass batch on the other), twice
    for _ in range(2):
        fa, sa = bufs(cfg3.n); fb, sb = bufs(cfg4.n)
        pn.pn_integrate(d_y3, d_m3, 0.0, cfg3.omegaf, cfg3.rtol, cfg3.atol, 0, fa, sa, stream=s1, async_=True)
        pn.pn_integrate(d_y4, d_m4, 0.0, cfg4.omegaf, cfg4.rtol, cfg4.atol, 0, fb, sb, stream=s2, async_=True)
        assert pn.pn_stream_status(s2) == 0 and pn.pn_stream_status(s1) == 0
        assert np.array_equal(fa.cpu().numpy(), ref3["final"]) and np.array_equal(sa.cpu().numpy(), ref3["steps"])
        assert np.array_equal(fb.cpu().numpy(), ref4["final"]) and np.array_equal(sb.cpu().numpy(), ref4["steps"])
    # a sync call on the default stream is untouched by all that
    again = gpu_integrate(pn, y3, m3, cfg3)
    assert again["status"] == 0 and np.array_equal(again["final"], ref3["final"])


def test_integrate_with_the_histogram_in_the_same_call(pn):
    """pn_options.hist_counts (include/pn.h): pn_integrate_ex bins the final states it has just written while they are on
    the device, so a host-buffer caller uploads 96 bytes per system, not 176.  Ragged size; host buffers,
    device buffers and the SoA layout: states bit-identical to a call without the option, counts equal to pn_histogram
    of those states."""
    cfg = W.with_size(W.CONFIGS["C3"], 3001)
    y0, m = W.generate(cfg)
    ref = gpu_integrate(pn, y0, m, cfg)
    c_ref = torch.zeros(3, cfg.bins, dtype=torch.int64, device="cuda:0"); s_ref = torch.zeros(3, dtype=torch.int64, device="cuda:0")
    pn.pn_histogram(ref["d_final"], cfg.bins, c_ref, s_ref)
    c_ref, s_ref = c_ref.cpu().numpy(), s_ref.cpu().numpy()
    assert c_ref.sum() + s_ref.sum() == 3 * cfg.n
    # host buffers
    h_yf = np.full((cfg.n, 10), np.nan); h_steps = np.zeros(cfg.n, dtype=np.int32)
    h_c = np.full((3, cfg.bins), -1, dtype=np.int64); h_s = np.full(3, -1, dtype=np.int64)
    assert pn.pn_integrate(y0, m, 0.0, cfg.omegaf, cfg.rtol, cfg.atol, 0, h_yf, h_steps, hist_bins=cfg.bins, hist_counts=h_c, hist_skipped=h_s) == 0
    assert np.array_equal(h_yf, ref["final"]) and np.array_equal(h_steps, ref["steps"])
    assert np.array_equal(h_c, c_ref) and np.array_equal(h_s, s_ref)
    assert pn.pn_last_kernel_ms()["histogram"] > 0
    # device buffers, AoS and SoA
    for layout in (0, 1):
        t = (lambda a: torch.from_numpy(np.ascontiguousarray(a.T if layout else a)).cuda())
        d_yf = torch.empty((10, cfg.n) if layout else (cfg.n, 10), dtype=torch.float64, device="cuda:0")
        d_steps = torch.zeros(cfg.n, dtype=torch.int32, device="cuda:0")
        d_c = torch.full((3, cfg.bins), -1, dtype=torch.int64, device="cuda:0")
        assert pn.pn_integrate(t(y0), t(m), 0.0, cfg.omegaf, cfg.rtol, cfg.atol, 0, d_yf, d_steps, layout=layout, hist_bins=cfg.bins, hist_counts=d_c) == 0
        got = d_yf.cpu().numpy()
        assert np.array_equal(got.T if layout else got, ref["final"]) and np.array_equal(d_c.cpu().numpy(), c_ref)
    # N = 0: zero counts; a bad bin count is refused
    e10 = torch.zeros(0, 10, dtype=torch.float64, device="cuda:0"); e2 = torch.zeros(0, 2, dtype=torch.float64, device="cuda:0")
    d_c = torch.full((3, 7), -1, dtype=torch.int64, device="cuda:0")
    assert pn.pn_integrate(e10, e2, 0.0, 0.05, 1e-10, 1e-12, 0, e10, torch.zeros(0, dtype=torch.int32, device="cuda:0"), hist_bins=7, hist_counts=d_c) == 0
    assert d_c.sum().item() == 0
    with pytest.raises(pn.PnError):
        pn.pn_integrate(y0, m, 0.0, cfg.omegaf, cfg.rtol, cfg.atol, 0, h_yf, h_steps, hist_bins=0, hist_counts=h_c)


def test_stream_release_recycles_contexts_and_table_rows(pn):
    """pn_stream_release (include/pn.h): a device has 4 rows in the uniform-mass constant table, one per live stream
    context.  A 5th live stream runs the generic kernel (rounding differs); releasing a stream returns its row, so any
    number of short-lived streams keep the fast path, a released stream leaves no pending status behind, and a stream
    that was never used is a no-op."""
    dev = "cuda:0"
    cfg = W.with_size(W.CONFIGS["C4"], 2000 + 9)
    y, m = W.generate(cfg)
    pn.pn_shutdown()                                       # forget the contexts of earlier tests
    ref_u = gpu_integrate(pn, y, m, cfg)                   # default stream: row 0
    ref_g = gpu_integrate(pn, y, m, cfg, variant=1)
    assert not np.array_equal(ref_u["final"], ref_g["final"])          # the two kernels differ in rounding
    d_y, d_m = torch.from_numpy(y).to(dev), torch.from_numpy(m).to(dev)

    def run_on(s):
        f = torch.full((cfg.n, 10), float("nan"), dtype=torch.float64, device=dev)
        st = torch.zeros(cfg.n, dtype=torch.int32, device=dev)
        s.wait_stream(torch.cuda.current_stream())
        assert pn.pn_integrate(d_y, d_m, 0.0, cfg.omegaf, cfg.rtol, cfg.atol, 0, f, st, stream=s, async_=True) == 0
        assert pn.pn_stream_status(s) == 0
        return f.cpu().numpy()

    # ten streams one after another, each released: every one gets a table row
    for _ in range(10):
        s = torch.cuda.Stream()
        assert np.array_equal(run_on(s), ref_u["final"])
        assert pn.pn_stream_release(s) == 0
    # without release: rows 1-3 go to three streams, the next live stream has none and runs the generic kernel
    held = [torch.cuda.Stream() for _ in range(4)]
    for s in held[:3]:
        assert np.array_equal(run_on(s), ref_u["final"])
    assert np.array_equal(run_on(held[3]), ref_g["final"])
    # ... until a row is given back (the context of held[3] was created without one: release it too)
    assert pn.pn_stream_release(held[0]) == 0 and pn.pn_stream_release(held[3]) == 0
    assert np.array_equal(run_on(held[3]), ref_u["final"])
    # a pending async status dies with the context; an unused stream is a no-op
    m_bad = m.copy(); m_bad[1, 0] = -1.0
    f = torch.empty(cfg.n, 10, dtype=torch.float64, device=dev); st = torch.zeros(cfg.n, dtype=torch.int32, device=dev)
    pn.pn_integrate(d_y, torch.from_numpy(m_bad).to(dev), 0.0, cfg.omegaf, cfg.rtol, cfg.atol, 0, f, st, stream=held[1], async_=True)
    assert pn.pn_stream_release(held[1]) == 0 and pn.pn_stream_status(held[1]) == 0
    assert pn.pn_stream_release(torch.cuda.Stream()) == 0
    for s in held[2:]:
        pn.pn_stream_release(s)
    again = gpu_integrate(pn, y, m, cfg)
    assert np.array_equal(again["final"], ref_u["final"])


def test_fma_microbenchmark_is_self_consistent(pn):
    """The FP64 peak and operand-port micro-benchmarks behind the roofline denominator: the SM clock
    estimated from the longest per-block clock64() span agrees with nvidia-smi, the throughput with 64 FMA lanes per SM
    at that clock, and a DFMA issues every 2 cycles with <= 2 distinct register sources, every 3 with 3."""
    import subprocess

    tf, mhz = pn.pn_measure_fma_peak(pn.PN_FP64, 0.2)
    mx = float(subprocess.check_output(["nvidia-smi", "--query-gpu=clocks.max.sm", "--format=csv,noheader,nounits", "-i", "0"]).decode().split()[0])
    sms = torch.cuda.get_device_properties(0).multi_processor_count
    assert 0.9 * mx <= mhz <= 1.02 * mx, (mhz, mx)
    assert abs(tf / (sms * 64 * 2 * mhz * 1e6 / 1e12) - 1) < 0.03, (tf, mhz)
    cyc = [pn.pn_measure_fma_operands(pn.PN_FP64, k) for k in (1, 2, 3)]
    assert abs(cyc[0] - 2.0) < 0.25 and abs(cyc[1] - 2.0) < 0.1 and abs(cyc[2] - 3.0) < 0.15, cyc
    # the issue model of DESIGN.md 7.2: integer instructions do NOT issue in the shadow of a 2-cycle DFMA
    assert 3.3 < pn.pn_measure_fma_operands(pn.PN_FP64, 4) < 4.3        # 2 if they issued in the DFMA's shadow; measured 3.7
