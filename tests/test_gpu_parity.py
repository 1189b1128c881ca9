"""GPU parity: the CUDA path (through the C ABI) against the CPU oracle, element by element on the same
seeded inputs.  Tolerances are those of BASELINE.json's north_star:
  fixed-step FP64: 1e-11 relative (per component, relative to omega / |S_i| / 1, R15)
  adaptive FP64 rtol 1e-10: final dot products 1e-7 absolute, final time 1e-7 relative
  FP32 rtol 1e-5: final dot products 2e-3 absolute, histograms within binomial noise."""
import numpy as np
import pytest

from paper_0908_3889_b200 import workloads as W

pytestmark = pytest.mark.gpu
torch = pytest.importorskip("torch")


@pytest.fixture(scope="module")
def pn():
    assert torch.cuda.is_available(), "the gpu tests need a CUDA device"
    import paper_0908_3889_b200 as pkg

    return pkg


def gpu_integrate(pn, y0, m, cfg_or_none, *, omegaf=None, rtol=None, atol=None, precision=0, omega0=0.0, **opts):
    dev = torch.device("cuda:0")
    n = y0.shape[0]
    d_y0, d_m = torch.from_numpy(np.ascontiguousarray(y0)).to(dev), torch.from_numpy(np.ascontiguousarray(m)).to(dev)
    d_yf = torch.full((n, 10), float("nan"), dtype=torch.float64, device=dev)
    d_steps = torch.zeros(n, dtype=torch.int32, device=dev)
    d_time = torch.zeros(n, dtype=torch.float64, device=dev)
    d_rej = torch.zeros(n, dtype=torch.int32, device=dev)
    cfg = cfg_or_none
    st = pn.pn_integrate(d_y0, d_m, omega0, omegaf if omegaf is not None else cfg.omegaf,
                         rtol if rtol is not None else cfg.rtol, atol if atol is not None else cfg.atol, precision,
                         d_yf, d_steps, out_time=d_time, out_rejected=d_rej, **opts)
    return dict(final=d_yf.cpu().numpy(), steps=d_steps.cpu().numpy(), time=d_time.cpu().numpy(),
                rejected=d_rej.cpu().numpy(), status=st, d_final=d_yf)


def comp_scale(y0):
    s1 = np.linalg.norm(y0[:, 1:4], axis=1, keepdims=True)
    s2 = np.linalg.norm(y0[:, 4:7], axis=1, keepdims=True)
    one = np.ones_like(s1)
    return np.concatenate([y0[:, :1], s1, s1, s1, s2, s2, s2, one, one, one], axis=1)


def dots_of(oracle, final):
    return oracle.histogram(final, 50)[2]


def test_T1_fixed_step_fp64(pn, oracle):
    cfg = W.CONFIGS["C1"]
    y0, m = W.generate(cfg)
    g = gpu_integrate(pn, y0, m, cfg, fixed_steps=200, h0=8.0)
    r = oracle.integrate(y0, m, 0, 0, 0, fixed_steps=200, h0=8.0)
    assert np.all(g["steps"] == 200)
    rel = np.abs(g["final"] - r["final"]) / comp_scale(y0)
    assert rel.max() <= 1e-11, rel.max()
    assert np.allclose(g["time"], 1600.0)


def test_T1_fixed_step_unequal_masses(pn, oracle):
    cfg = W.with_size(W.CONFIGS["C3"], 777)     # ragged size, q in [0.1,1], chi in [0,1]
    y0, m = W.generate(cfg)
    g = gpu_integrate(pn, y0, m, cfg, fixed_steps=150, h0=40.0)
    r = oracle.integrate(y0, m, 0, 0, 0, fixed_steps=150, h0=40.0)
    rel = np.abs(g["final"] - r["final"]) / np.maximum(comp_scale(y0), 1e-3)
    assert rel.max() <= 1e-11, rel.max()


def check_adaptive(pn, oracle, cfg, y0, m, idx=None, tol_dot=1e-7, tol_t=1e-7, **opts):
    g = gpu_integrate(pn, y0, m, cfg, **opts)
    assert g["status"] == 0 and np.all(g["steps"] > 0)
    sel = np.arange(y0.shape[0]) if idx is None else idx
    r = oracle.integrate(y0[sel], m[sel], cfg.omegaf, cfg.rtol, cfg.atol)
    assert r["n_failed"] == 0
    dg, dr = dots_of(oracle, g["final"][sel]), dots_of(oracle, r["final"])
    ok = np.isfinite(dr)
    assert np.array_equal(ok, np.isfinite(dg))
    assert np.abs(dg - dr)[ok].max() <= tol_dot, np.abs(dg - dr)[ok].max()
    assert np.abs(g["time"][sel] / r["time"] - 1).max() <= tol_t
    assert np.abs(g["final"][sel, 0] - cfg.omegaf).max() <= 1.01e-13 * cfg.omegaf
    # same algorithm on both sides: step counts agree except where an accept/reject decision flipped
    assert np.mean(g["steps"][sel] == r["steps"]) > 0.5
    assert abs(g["steps"][sel].mean() / r["steps"].mean() - 1) < 0.01
    return g, r


def test_T2_adaptive_C1_full(pn, oracle):
    cfg = W.CONFIGS["C1"]
    y0, m = W.generate(cfg)
    g, r = check_adaptive(pn, oracle, cfg, y0, m, omega0=cfg.omega0)
    # histograms: GPU kernel on GPU final states vs oracle histogram of oracle final states
    counts = torch.zeros(3, cfg.bins, dtype=torch.int64, device="cuda:0")
    skipped = torch.zeros(3, dtype=torch.int64, device="cuda:0")
    pn.pn_histogram(g["d_final"], cfg.bins, counts, skipped)
    c_ref, s_ref, d_ref = oracle.histogram(r["final"], cfg.bins)
    edges = np.linspace(-1, 1, cfg.bins + 1)
    near = (np.abs(d_ref[:, :, None] - edges[None, None, :]) < 1e-7).sum()
    assert np.abs(counts.cpu().numpy() - c_ref.astype(np.int64)).sum() <= 2 * near
    assert counts.sum().item() == 3 * cfg.n and skipped.sum().item() == 0


@pytest.mark.parametrize("name,nsub", [("C2", 1536), ("C3", 1536), ("C4", 2048), ("C5", 384)])
def test_T2_adaptive_small_batches(pn, oracle, name, nsub):
    """Sizes the oracle finishes in seconds that still span several warps/blocks and a ragged tail."""
    cfg = W.with_size(W.CONFIGS[name], nsub + 37)
    y0, m = W.generate(cfg)
    check_adaptive(pn, oracle, cfg, y0, m)


def test_histogram_kernel_bit_exact_on_same_states(pn, oracle):
    """Integer work: on IDENTICAL final states the GPU histogram equals the oracle's, except for samples
    within a few ulp of a bin edge (FMA contraction of the dot product)."""
    rng = np.random.default_rng(5)
    n = 100003
    y = rng.normal(size=(n, 10))
    y[11, 1:4] = 0.0
    y[12, 7:10] = 2.0 * y[12, 1:4]
    y[13, 4:7] = -0.5 * y[13, 7:10]
    y[14, 4] = np.nan
    d_y = torch.from_numpy(y).cuda()
    for bins in (1, 2, 20, 50, 100, 79 * 79, 50000):
        counts = torch.zeros(3, bins, dtype=torch.int64, device="cuda:0")
        skipped = torch.zeros(3, dtype=torch.int64, device="cuda:0")
        pn.pn_histogram(d_y, bins, counts, skipped)
        c_ref, s_ref, d_ref = oracle.histogram(y, bins)
        assert np.array_equal(skipped.cpu().numpy(), s_ref.astype(np.int64))
        diff = np.abs(counts.cpu().numpy() - c_ref.astype(np.int64)).sum()
        scaled = (d_ref + 1) * bins / 2
        near = (np.abs(scaled - np.round(scaled)) < 1e-9 * bins).sum()
        assert diff <= 2 * near, (bins, diff, near)
        assert counts.sum().item() + skipped.sum().item() == 3 * n
    # SoA layout and host buffers give the same counts
    bins = 50
    c_ref = oracle.histogram(y, bins)[0].astype(np.int64)
    counts = torch.zeros(3, bins, dtype=torch.int64, device="cuda:0")
    pn.pn_histogram(d_y.t().contiguous(), bins, counts, None, layout=1, n=n)
    assert np.abs(counts.cpu().numpy() - c_ref).sum() <= 2
    hc = np.zeros((3, bins), dtype=np.uint64)
    hs = np.zeros(3, dtype=np.uint64)
    pn.pn_histogram(y, bins, hc, hs)
    assert np.abs(hc.astype(np.int64) - c_ref).sum() <= 2 and hs.sum() == 4


def test_fp32_C4_against_oracle(pn, oracle):
    cfg = W.with_size(W.CONFIGS["C4f"], 8192 + 5)
    y0, m = W.generate(cfg)
    g = gpu_integrate(pn, y0, m, cfg, precision=1)
    assert g["status"] == 0 and np.all(g["steps"] > 0)
    r = oracle.integrate(y0, m, cfg.omegaf, 1e-10, 1e-12)
    dg, dr = dots_of(oracle, g["final"]), dots_of(oracle, r["final"])
    assert np.abs(dg - dr).max() <= 2e-3, np.abs(dg - dr).max()
    assert np.abs(g["time"] / r["time"] - 1).max() <= 1e-3
    assert np.abs(g["final"][:, 0] / cfg.omegaf - 1).max() <= 4e-7
    # histograms within binomial noise: |ca - cb| <= 5 sqrt(ca + cb + 1) per bin
    counts = torch.zeros(3, cfg.bins, dtype=torch.int64, device="cuda:0")
    pn.pn_histogram(g["d_final"], cfg.bins, counts)
    ca, cb = counts.cpu().numpy(), oracle.histogram(r["final"], cfg.bins)[0].astype(np.int64)
    assert np.all(np.abs(ca - cb) <= 5 * np.sqrt(ca + cb + 1))
    # FP32 takes far fewer steps at its looser tolerance
    assert g["steps"].mean() < 0.3 * r["steps"].mean()


def test_leading_order_closed_form_on_gpu(pn):
    """P1 through the CUDA path: omega^{-8/3}(t) = omega0^{-8/3} - (256/5) eta M^{5/3} t."""
    m1 = np.array([0.5, 0.6, 0.8, 0.9])
    m = np.stack([m1, 1 - m1], 1)
    y0 = np.zeros((4, 10)); y0[:, 0] = 0.005; y0[:, 9] = 1.0
    g = gpu_integrate(pn, y0, m, None, omegaf=0.05, rtol=1e-12, atol=1e-14, term_mask=1)
    tf = (0.005 ** (-8 / 3) - 0.05 ** (-8 / 3)) / (256 / 5 * m1 * (1 - m1))
    assert np.abs(g["time"] / tf - 1).max() < 5e-12
    assert np.array_equal(g["final"][:, 1:], y0[:, 1:])      # nothing precesses


def test_packed_fp32_kernel_is_bit_identical_to_the_scalar_one(pn):
    """PN_FP32 keeps the ten components of a system in five register pairs and uses packed f32x2 arithmetic (FFMA2 /
    FMUL2 / FADD2) for the stage sums, the error vector and the x / y halves of the RHS's vector operations, and it
    prefetches seed records through shared memory.  Per component it performs the same IEEE operations
    in the same order as the plain scalar kernel (pn_options.variant bit 1 selects that one), so every output must agree
    bit for bit: ragged batch sizes, mixed masses, bad inputs, max_steps failures, tight and loose tolerances."""
    for name, n, tol in (("C4f", 5003, None), ("C3", 4097, (1e-5, 1e-7)), ("C3", 1, (1e-6, 1e-8)), ("C2", 2, (1e-4, 1e-6)),
                         ("C5", 63, (1e-5, 1e-7)), ("C1", 257, (1e-7, 1e-9))):
        cfg = W.with_size(W.CONFIGS[name], n)
        y0, m = W.generate(cfg)
        rtol, atol = tol if tol else (cfg.rtol, cfg.atol)
        a = gpu_integrate(pn, y0, m, cfg, rtol=rtol, atol=atol, precision=1)
        b = gpu_integrate(pn, y0, m, cfg, rtol=rtol, atol=atol, precision=1, variant=2)
        assert a["status"] == 0 and np.all(a["steps"] > 0)
        for k in ("final", "steps", "time", "rejected"):
            assert np.array_equal(a[k], b[k]), (name, n, k)
    # batches large enough for every lane to run through the prefetch pipeline many times, in both queue orders
    cfg = W.with_size(W.CONFIGS["C4f"], 300000 + 11)
    y0, m = W.generate(cfg)
    for io in (False, True):
        a = gpu_integrate(pn, y0, m, cfg, precision=1, input_order=io)
        b = gpu_integrate(pn, y0, m, cfg, precision=1, variant=2, input_order=io)
        for k in ("final", "steps", "time", "rejected"):
            assert np.array_equal(a[k], b[k]), (io, k)
    # C4f is a uniform-mass batch: the default run above took the uniform-mass instantiation (constants from the
    # __constant__ table: the very floats of system 0's record); the generic one (variant bit 0) gives the same bits, and
    # one deviating system sends the whole launch to the generic instantiation
    c = gpu_integrate(pn, y0, m, cfg, precision=1, variant=1)
    m2 = m.copy(); m2[-1] = [0.5, 0.5]
    d = gpu_integrate(pn, y0, m2, cfg, precision=1)
    for k in ("final", "steps", "time", "rejected"):
        assert np.array_equal(a[k], c[k]), k
        assert np.array_equal(a[k][:-1], d[k][:-1]), k
    assert not np.array_equal(a["final"][-1], d["final"][-1])
    # failures and bad inputs land in the same slots with the same codes
    cfg = W.with_size(W.CONFIGS["C3"], 777)
    y0, m = W.generate(cfg)
    m[5, 0] = -1.0; y0[6, 0] = 0.07; y0[9, 2] = np.nan
    for extra in ({}, {"max_steps": 15}):
        a = gpu_integrate(pn, y0, m, cfg, rtol=1e-5, atol=1e-7, precision=1, allow_failures=True, **extra)
        b = gpu_integrate(pn, y0, m, cfg, rtol=1e-5, atol=1e-7, precision=1, variant=2, allow_failures=True, **extra)
        assert a["status"] == b["status"] != 0
        assert a["steps"][5] == a["steps"][6] == -5 and a["steps"][9] == -3
        for k in ("steps", "time", "rejected"):
            assert np.array_equal(a[k], b[k]), k
        assert np.array_equal(a["final"], b["final"], equal_nan=True)
