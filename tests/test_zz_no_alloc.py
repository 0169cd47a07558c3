"""dd_postprocess_static (the entry point that allocates no device memory: per-series statistics in the library's
static device array) against dd_postprocess (statistics in a workspace allocation), through the C ABI.

Both run the same kernels on the same series, so the processed series and the candidate sets must be identical
(stricter than the float32 rounding tolerance the oracle comparisons of test_gpu_postproc.py use).  Two calls in
a row with different shapes: the second has fewer series, so statistics left in the array by the first call
would show if a call read anything it had not written.  Collected last on purpose (own file, zz)."""
import numpy as np
import pytest

import paper_1401_8258_b200 as dd

pytestmark = pytest.mark.gpu


def _series(seed, nb, ndm, n):
    g = np.random.default_rng(seed)
    t = np.arange(n)
    level = g.uniform(-50, 500, (nb, ndm, 1))
    slope = g.uniform(-2e-3, 2e-3, (nb, ndm, 1))
    sig = g.uniform(0.5, 30.0, (nb, ndm, 1))
    D = level + slope * t + sig * g.standard_normal((nb, ndm, n))
    for _ in range(4 * nb * ndm):
        b, d, p = g.integers(0, nb), g.integers(0, ndm), g.integers(0, n - 16)
        D[b, d, p:p + g.integers(6, 13)] += sig[b, d, 0] * g.uniform(8, 12)      # resolved pulses survive the median
    return D.astype(np.float32)


def _run(fn, Dd, nb, ndm, n, stride, params, capacity, **kw):
    import torch
    Zd = torch.full((nb, ndm, stride), -7.0, dtype=torch.float32, device="cuda")
    cand = torch.zeros(capacity * 4, dtype=torch.int32, device="cuda")
    cnt = torch.zeros(1, dtype=torch.int64, device="cuda")
    fn(dd.DD_F32, Dd, stride, ndm * stride, ndm, n, nb, params, Zd, stride, ndm * stride,
       cand=cand, capacity=capacity, count=cnt, **kw)
    torch.cuda.synchronize()
    count = int(cnt.item())
    c = cand.cpu().numpy().view(dd.CANDIDATE_DTYPE)[:min(count, capacity)]
    rows = sorted(zip(c["beam"].tolist(), c["dm"].tolist(), c["t"].tolist(), c["value"].tolist()))
    return Zd.cpu().numpy(), count, rows


def test_static_scratch_entry_point_matches_the_allocating_path_on_two_calls_in_a_row():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    params = dd.post_params(median_window=5, detrend=True, normalise=True, nsigma=6.0)
    capacity = 1 << 15
    shapes = [(101, 2, 37, 9001, 3), (202, 1, 5, 4099, 0)]          # (seed, beams, trials, samples, row padding)
    inputs = []
    for seed, nb, ndm, n, pad in shapes:
        D = _series(seed, nb, ndm, n)
        Dd = torch.zeros((nb, ndm, n + pad), dtype=torch.float32, device="cuda")
        Dd[:, :, :n] = torch.from_numpy(D).cuda()
        inputs.append(Dd)
    # existing path first (its statistics go to a buffer of ours: the documented optional output)
    want = []
    for (seed, nb, ndm, n, pad), Dd in zip(shapes, inputs):
        Sd = torch.zeros((nb * ndm, 3), dtype=torch.float64, device="cuda")
        want.append(_run(dd.dd_postprocess, Dd, nb, ndm, n, n + pad, params, capacity, stats=Sd))
    # the two static calls back to back, nothing in between; the library must not take device memory for them
    Zs = [torch.full((nb, ndm, n + pad), -7.0, dtype=torch.float32, device="cuda") for _, nb, ndm, n, pad in shapes]
    cands = [torch.zeros(capacity * 4, dtype=torch.int32, device="cuda") for _ in shapes]
    cnts = [torch.zeros(1, dtype=torch.int64, device="cuda") for _ in shapes]
    torch.cuda.synchronize()
    free_mid = torch.cuda.mem_get_info()[0]
    for (seed, nb, ndm, n, pad), Dd, Zd, cand, cnt in zip(shapes, inputs, Zs, cands, cnts):
        dd.dd_postprocess_static(dd.DD_F32, Dd, n + pad, ndm * (n + pad), ndm, n, nb, params, Zd, n + pad,
                                 ndm * (n + pad), cand=cand, capacity=capacity, count=cnt)
    torch.cuda.synchronize()
    assert torch.cuda.mem_get_info()[0] >= free_mid, "the static entry point took device memory"
    for (seed, nb, ndm, n, pad), Zd, cand, cnt, (Zw, count_w, rows_w) in zip(shapes, Zs, cands, cnts, want):
        count = int(cnt.item())
        c = cand.cpu().numpy().view(dd.CANDIDATE_DTYPE)[:min(count, capacity)]
        rows = sorted(zip(c["beam"].tolist(), c["dm"].tolist(), c["t"].tolist(), c["value"].tolist()))
        Z = Zd.cpu().numpy()
        assert count_w > 0 and count == count_w
        assert rows == rows_w
        assert np.array_equal(Z, Zw)                                  # same kernels, same statistics: bit for bit
        assert np.all(Z[:, :, n:] == -7.0)                            # padding untouched
        assert np.isfinite(Z[:, :, :n]).all() and np.abs(Z[:, :, :n]).max() > 6.0


def test_static_scratch_entry_point_rejects_sizes_beyond_its_table():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    params = dd.post_params(median_window=3, detrend=True, normalise=True)
    ndm = dd.POSTPROCESS_STATIC_MAX_SERIES + 1
    n = 16
    Dd = torch.zeros((1, ndm, n), dtype=torch.float32, device="cuda")
    Zd = torch.full((1, ndm, n), -7.0, dtype=torch.float32, device="cuda")
    with pytest.raises(dd.DedispError) as ei:
        dd.dd_postprocess_static(dd.DD_F32, Dd, n, ndm * n, ndm, n, 1, params, Zd, n, ndm * n)
    assert "DD_POSTPROCESS_STATIC_MAX_SERIES" in str(ei.value)
    torch.cuda.synchronize()
    assert bool((Zd == -7.0).all())                                   # nothing was enqueued
    # exactly at the limit it runs (constant series: sigma = 0 -> all-zero output, R17)
    ndm = dd.POSTPROCESS_STATIC_MAX_SERIES
    Dd = torch.full((1, ndm, n), 3.0, dtype=torch.float32, device="cuda")
    Zd = torch.full((1, ndm, n), -7.0, dtype=torch.float32, device="cuda")
    dd.dd_postprocess_static(dd.DD_F32, Dd, n, ndm * n, ndm, n, 1, params, Zd, n, ndm * n)
    torch.cuda.synchronize()
    assert bool((Zd == 0.0).all())
