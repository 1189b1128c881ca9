"""GPU parity of the mixed-precision variant (PN_MIXED: float slopes, double state) against the FP64
oracle at rtol 1e-10.  Bars (derived from the arithmetic: the floor is the float RHS, 6e-8 relative
per evaluation, accumulated over ~500 steps and amplified by the precession dynamics): at rtol 1e-7, atol 1e-9
final dot products within 2e-4 absolute (99 % within 2e-5, median within 2e-6), final time within 1e-6 relative,
omega landed on omega_f within 1.5e-8 relative; and strictly better than PN_FP32 at the same tolerance."""
import numpy as np
import pytest

from paper_0908_3889_b200 import workloads as W

pytestmark = pytest.mark.gpu
torch = pytest.importorskip("torch")


def run(pn, y0, m, cfg, prec, rtol, atol, **opts):
    d0, dm = torch.from_numpy(y0).cuda(), torch.from_numpy(m).cuda()
    yf = torch.full_like(d0, float("nan"))
    st = torch.zeros(cfg.n, dtype=torch.int32, device="cuda")
    tt = torch.zeros(cfg.n, dtype=torch.float64, device="cuda")
    rc = pn.pn_integrate(d0, dm, cfg.omega0, cfg.omegaf, rtol, atol, prec, yf, st, out_time=tt, **opts)
    return rc, yf.cpu().numpy(), st.cpu().numpy(), tt.cpu().numpy()


@pytest.mark.parametrize("name,n", [("C2", 2048 + 37), ("C3", 2048 + 37), ("C4", 4096 + 5), ("C1", 1024)])
def test_mixed_against_fp64_oracle(oracle, name, n):
    import paper_0908_3889_b200 as pn

    cfg = W.with_size(W.CONFIGS[name], n)
    y0, m = W.generate(cfg)
    ref = oracle.integrate(y0, m, cfg.omegaf, 1e-10, 1e-12)
    dr = oracle.histogram(ref["final"], 50)[2]
    rc, yf, st, tt = run(pn, y0, m, cfg, pn.PN_MIXED, 1e-7, 1e-9)
    assert rc == 0 and np.all(st > 0)
    err = np.abs(oracle.histogram(yf, 50)[2] - dr)
    assert err.max() <= 2e-4 and np.quantile(err, 0.99) <= 2e-5 and np.median(err) <= 2e-6, (err.max(), np.median(err))
    assert np.abs(tt / ref["time"] - 1).max() <= 1e-6
    assert np.abs(yf[:, 0] / cfg.omegaf - 1).max() <= 1.5e-8
    # the double state keeps the conserved norms two orders better than float can hold them
    for sl in (slice(1, 4), slice(4, 7), slice(7, 10)):
        n0, n1 = np.linalg.norm(y0[:, sl], axis=1), np.linalg.norm(yf[:, sl], axis=1)
        assert np.abs(n1 / n0 - 1).max() < 5e-6
    # same tolerance in plain FP32: state rounding dominates; mixed is better in the median and at the 99th percentile
    rc32, yf32, st32, tt32 = run(pn, y0, m, cfg, pn.PN_FP32, 1e-7, 1e-9)
    err32 = np.abs(oracle.histogram(yf32, 50)[2] - dr)
    assert np.median(err) < 0.8 * np.median(err32) and np.quantile(err, 0.99) < np.quantile(err32, 0.99)
    assert np.abs(tt / ref["time"] - 1).max() < 0.2 * np.abs(tt32 / ref["time"] - 1).max()
    # far fewer steps than FP64 at 1e-10
    assert st.mean() < 0.45 * ref["steps"].mean()


def test_mixed_edges(oracle):
    import paper_0908_3889_b200 as pn

    cfg = W.with_size(W.CONFIGS["C3"], 333)
    y0, m = W.generate(cfg)
    y0[5, 1:7] = 0.0                 # non-spinning system: nothing precesses
    m[7, 0] = -1.0                   # bad input
    rc, yf, st, tt = run(pn, y0, m, cfg, pn.PN_MIXED, 1e-7, 1e-9, allow_failures=True)
    assert rc == 1 and st[7] == -5 and np.all(np.delete(st, 7) > 0)
    assert np.array_equal(yf[5, 1:], y0[5, 1:])
    # run-to-run bit identity, and independence of the queue order
    rc2, yf2, st2, tt2 = run(pn, y0, m, cfg, pn.PN_MIXED, 1e-7, 1e-9, allow_failures=True, input_order=True)
    assert np.array_equal(yf, yf2, equal_nan=True) and np.array_equal(st, st2) and np.array_equal(tt, tt2)
    # host buffers
    hy = np.empty_like(y0); hs = np.empty(cfg.n, dtype=np.int32)
    pn.pn_integrate(y0, m, cfg.omega0, cfg.omegaf, 1e-7, 1e-9, pn.PN_MIXED, hy, hs, allow_failures=True)
    assert np.array_equal(hy, yf, equal_nan=True) and np.array_equal(hs, st)
