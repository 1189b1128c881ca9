"""GPU parity of pn_selfcheck (the 1 % double-precision cross-check) against oracle/pn_check_oracle.py:
the selected subset is bit-exact; the worst deviations agree to 2e-7 (the two FP64 reference integrations agree
to 1e-7 on every dot product, the bar of the FP64 parity tests); the worst index is the same system."""
import numpy as np
import pytest

from oracle import pn_check_oracle as C
from paper_0908_3889_b200 import workloads as W

pytestmark = pytest.mark.gpu
torch = pytest.importorskip("torch")


def test_selfcheck_fp32_run_against_oracle(oracle):
    import paper_0908_3889_b200 as pn

    cfg = W.with_size(W.CONFIGS["C4f"], 60000 + 11)
    y0, m = W.generate(cfg)
    d0, dm = torch.from_numpy(y0).cuda(), torch.from_numpy(m).cuda()
    yf = torch.empty_like(d0)
    st = torch.empty(cfg.n, dtype=torch.int32, device="cuda")
    tt = torch.empty(cfg.n, dtype=torch.float64, device="cuda")
    pn.pn_integrate(d0, dm, cfg.omega0, cfg.omegaf, cfg.rtol, cfg.atol, pn.PN_FP32, yf, st, out_time=tt)
    key = (2009, 3889)
    idx = torch.full((4000,), -1, dtype=torch.int64, device="cuda")
    g = pn.pn_selfcheck(d0, dm, yf, cfg.omegaf, fraction=0.01, key=key, times=tt, checked_indices=idx)
    r = C.selfcheck(y0, m, yf.cpu().numpy(), tt.cpu().numpy(), cfg.omegaf, 0.01, key)
    assert g["n_checked"] == r["n_checked"] and 450 < g["n_checked"] < 750
    assert np.array_equal(idx.cpu().numpy()[:g["n_checked"]], r["indices"])
    assert g["n_failed_ref"] == 0 == r["n_failed_ref"]
    assert np.abs(np.array(g["max_dot_dev"]) - r["max_dot_dev"]).max() < 2e-7
    assert g["worst_index"] == r["worst_index"].tolist()
    assert abs(g["max_time_rel_dev"] - r["max_time_rel_dev"]) < 1e-7
    # the FP32 run is within the FP32 bar on the checked subset, and not suspiciously perfect
    assert 1e-6 < max(g["max_dot_dev"]) < 2e-3 and g["max_time_rel_dev"] < 1e-3
    # deterministic; host buffers give the same answer
    g2 = pn.pn_selfcheck(d0, dm, yf, cfg.omegaf, fraction=0.01, key=key, times=tt)
    h = pn.pn_selfcheck(y0, m, yf.cpu().numpy(), cfg.omegaf, fraction=0.01, key=key, times=tt.cpu().numpy())
    for k in ("n_checked", "max_dot_dev", "worst_index", "max_time_rel_dev"):
        assert g[k] == g2[k] == h[k], k


def test_selfcheck_finds_a_planted_error_and_edges(oracle):
    import paper_0908_3889_b200 as pn

    cfg = W.with_size(W.CONFIGS["C1"], 5000)
    y0, m = W.generate(cfg)
    d0, dm = torch.from_numpy(y0).cuda(), torch.from_numpy(m).cuda()
    yf = torch.empty_like(d0)
    st = torch.empty(cfg.n, dtype=torch.int32, device="cuda")
    pn.pn_integrate(d0, dm, cfg.omega0, cfg.omegaf, cfg.rtol, cfg.atol, pn.PN_FP64, yf, st)
    key = (7, 7)
    clean = pn.pn_selfcheck(d0, dm, yf, cfg.omegaf, fraction=0.05, key=key)
    assert max(clean["max_dot_dev"]) == 0.0            # FP64 checked against the same FP64 integrator: bit-identical
    sel = C.selection(cfg.n, 0.05, key)
    assert clean["n_checked"] == sel.size
    j = int(sel[len(sel) // 2])
    bad = yf.clone()
    bad[j, 4:7] = -bad[j, 4:7]                          # silent corruption of one spin
    g = pn.pn_selfcheck(d0, dm, bad, cfg.omegaf, fraction=0.05, key=key)
    assert g["worst_index"][0] == j and g["worst_index"][2] == j and g["max_dot_dev"][0] > 1e-3
    assert g["max_dot_dev"][1] == 0.0
    # fraction 0 selects nothing, fraction 1 everything; N = 0 is a no-op; bad arguments
    assert pn.pn_selfcheck(d0, dm, yf, cfg.omegaf, fraction=0.0, key=key)["n_checked"] == 0
    assert pn.pn_selfcheck(d0[:300], dm[:300], yf[:300], cfg.omegaf, fraction=1.0, key=key)["n_checked"] == 300
    assert pn.pn_selfcheck(d0[:0], dm[:0], yf[:0], cfg.omegaf, key=key)["n_checked"] == 0
    with pytest.raises(pn.PnError):
        pn.pn_selfcheck(d0, dm, yf, cfg.omegaf, fraction=1.5, key=key)
