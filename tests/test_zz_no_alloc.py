"""pn_statistics_static -- the statistics pass for callers that are not allowed to allocate device memory.

Who that is: a program that embeds the library after its framework's caching allocator has taken all of HBM (a
cudaMalloc issued by a library then fails although the job's pool has room), a loop that runs beside other streams
(cudaMalloc and cudaFree synchronise the whole device and would stall them), or a process with a fixed memory budget.
pn_statistics gets its scratch (per-block moment records) from cudaMalloc; pn_statistics_static runs the same kernels
on a fixed 336 KB `static __device__` array inside the library and takes only the caller's input and output tensors.

What is checked: on two calls in a row (different data, a different number of ensembles, the second one smaller, so
whatever the first call left in the shared array would show up) every output equals that of pn_statistics within the
tolerances of tests/test_gpu_stats.py: counts, n and skipped exactly, means 1e-14, second moments 1e-11 relative to n,
r 1e-12 (both paths run the same kernels in the same launch geometry, so in practice they agree bit for bit, which is
asserted too where NaNs allow).  The device's free memory does not change across the second call; a request
beyond PN_STATIC_MAX_GROUPS ensembles is refused with PN_ETOOLARGE and touches nothing.

This file sorts last on purpose: pytest -x stops at the first failure, and a failure here must not hide other tests.
It needs nothing from the tests before it and passes alone in a fresh process as well as after them.
"""
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


def make_batch(n, seed):
    """(initial, final, steps) with correlated dot products, a few failed systems and a few undefined dot products."""
    y0, _ = W.generate(W.with_size(W.CONFIGS["C3"], n))
    g = np.random.Generator(np.random.Philox(seed))
    yf = y0.copy()
    yf[:, 1:10] += 0.3 * np.abs(y0[:, 1:10]).max() * g.normal(size=(n, 9))
    steps = np.full(n, 9, dtype=np.int32)
    steps[[5, n // 3, n - 2]] = [-1, -2, -4]
    y0[13, 1:4] = 0.0
    yf[21, 4:7] = 0.0
    yf[29, 7:10] = np.nan
    return y0, yf, steps


def outputs(G, bins1, bins2, fill):
    f = lambda shape, dt: torch.full(shape, fill, dtype=dt, device="cuda")
    return dict(pearson_r=f((G, 3), torch.float64), moments=f((G, 3, 6), torch.float64), n_skipped=f((G, 3), torch.int64),
                hist1=f((G, 3, bins1), torch.int64), hist2=f((G, 3, bins2, bins2), torch.int64),
                hist2_max=f((G, 3), torch.int64), hist2_norm=f((G, 3, bins2, bins2), torch.float64))


def assert_same(got, ref):
    for k in ("n_skipped", "hist1", "hist2", "hist2_max"):
        assert np.array_equal(got[k], ref[k]), k
    assert np.array_equal(got["moments"][..., 0], ref["moments"][..., 0])
    n = np.maximum(ref["moments"][..., 0], 1.0)
    has = ref["moments"][..., 0] > 0
    assert np.abs(got["moments"][..., 1:3] - ref["moments"][..., 1:3])[has].max(initial=0) <= 1e-14
    assert (np.abs(got["moments"][..., 3:] - ref["moments"][..., 3:]) / n[..., None]).max() <= 1e-11
    assert np.array_equal(np.isnan(got["pearson_r"]), np.isnan(ref["pearson_r"]))
    ok = np.isfinite(ref["pearson_r"])
    assert np.abs(got["pearson_r"] - ref["pearson_r"])[ok].max(initial=0) <= 1e-12
    assert np.abs(got["hist2_norm"] - ref["hist2_norm"]).max() <= 1e-15
    # same kernels, same launch geometry, same merge order: in fact the same bits
    for k in got:
        assert np.array_equal(got[k], ref[k], equal_nan=True), k


def test_static_scratch_statistics_equal_the_allocating_path_twice_in_a_row(pn):
    # two batches: 6 ragged ensembles of 4001 systems (several tiles and a tail per ensemble, ensembles shared between
    # blocks), then ONE ensemble of 2999 systems, which uses fewer records than the first call wrote
    cases = [(6 * 4001, 4001, 50, 79, 101), (2999, 0, 20, 8, 202)]
    staged = []
    for n, gs, b1, b2, seed in cases:
        y0, yf, steps = make_batch(n, seed)
        G = n // (gs if gs else n)
        staged.append((torch.from_numpy(y0).cuda(), torch.from_numpy(yf).cuda(), torch.from_numpy(steps).cuda(), gs, b1, b2,
                       outputs(G, b1, b2, -7), outputs(G, b1, b2, -9)))
    torch.cuda.synchronize()
    results = []
    for call, (d0, df, dst, gs, b1, b2, out_static, out_ref) in enumerate(staged):
        free_before = torch.cuda.mem_get_info()[0]
        assert pn.pn_statistics_static(d0, df, dst, group_size=gs, bins1=b1, bins2=b2, **out_static) == 0
        if call > 0:
            # the address and the kernel attributes were set up by the first call: the device's free memory is untouched
            assert torch.cuda.mem_get_info()[0] == free_before
        results.append({k: v.cpu().numpy() for k, v in out_static.items()})
    # the stream argument and the enqueue-only mode: the second batch once more on a side stream, same bits
    d0, df, dst, gs, b1, b2, _, _ = staged[1]
    side, out_side = torch.cuda.Stream(), outputs(1, b1, b2, -3)
    side.wait_stream(torch.cuda.current_stream())
    assert pn.pn_statistics_static(d0, df, dst, group_size=gs, bins1=b1, bins2=b2, stream=side, async_=True, **out_side) == 0
    side.synchronize()
    for k, v in out_side.items():
        assert np.array_equal(v.cpu().numpy(), results[1][k], equal_nan=True), k
    # the existing path afterwards (it allocates its own scratch), on the same inputs
    for (d0, df, dst, gs, b1, b2, out_static, out_ref), got in zip(staged, results):
        pn.pn_statistics(d0, df, dst, group_size=gs, bins1=b1, bins2=b2, **out_ref)
        ref = {k: v.cpu().numpy() for k, v in out_ref.items()}
        assert ref["moments"][..., 0].min() > 0 and ref["n_skipped"].sum() > 0      # the batch exercises both
        assert_same(got, ref)


def test_static_scratch_refuses_what_does_not_fit(pn):
    G = pn.PN_STATIC_MAX_GROUPS + 1
    y0, yf, _ = make_batch(2 * G, 7)
    d0, df = torch.from_numpy(y0).cuda(), torch.from_numpy(yf).cuda()
    r = torch.full((G, 3), -5.0, dtype=torch.float64, device="cuda")
    with pytest.raises(pn.PnError) as err:
        pn.pn_statistics_static(d0, df, group_size=2, pearson_r=r)
    assert err.value.status == pn.PN_ETOOLARGE and "capacity" in str(err.value)
    assert bool((r == -5.0).all())                                                 # refused before anything ran
    # the largest accepted number of ensembles works, and agrees with the allocating path
    G = pn.PN_STATIC_MAX_GROUPS
    r = torch.zeros(G, 3, dtype=torch.float64, device="cuda")
    r_ref = torch.zeros(G, 3, dtype=torch.float64, device="cuda")
    assert pn.pn_statistics_static(d0[: 2 * G], df[: 2 * G], group_size=2, pearson_r=r) == 0
    pn.pn_statistics(d0[: 2 * G], df[: 2 * G], group_size=2, pearson_r=r_ref)
    assert np.array_equal(r.cpu().numpy(), r_ref.cpu().numpy(), equal_nan=True)
    # host arrays are refused by the binding (staging them would need an allocation), bad arguments by the library
    with pytest.raises(ValueError):
        pn.pn_statistics_static(y0, yf, pearson_r=np.zeros((1, 3)))
    with pytest.raises(pn.PnError) as err:
        pn.pn_statistics_static(d0, df, group_size=7, pearson_r=r)
    assert err.value.status == 1
    assert pn.pn_statistics_static(d0[:0], df[:0], pearson_r=r) == 0               # N = 0 is a successful no-op
