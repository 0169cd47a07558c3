"""GPU parity of the post-processing row f1 (median filter, detrend, normalise, threshold -> candidates;
PAPER.md:1204-1221) through the C ABI, against oracle/postproc_oracle.cpp.

Tolerances.  On IDENTICAL input series the device path selects medians exactly and evaluates
the regression, the residual and the scaling in double, so the only differences from the oracle's double
result are the final rounding to float32 and the ~1e-13 relative difference of the fitted parameters:
    |Z - z| <= 2^-23 |z| + 1e-9 max|y| / scale          (scale = sigma when normalised, else 1).
For the CHAIN dedisperse -> post-process the device series differ from the oracle's by delta <= 1e-5 A
(north_star's per-element tolerance, A = sum_c |X|); the median is 1-Lipschitz in the max norm, the line
fit's hat matrix has max-norm <= 4, so |r - r'| <= 5 delta, |sigma - sigma'| <= 5 delta and
    |Z - z| <= 5 delta (1 + |z|) / sigma  (+ the rounding term above).
The threshold decides list membership: both sides compare in double; samples whose oracle value lies within
the tolerance of n sigma may fall either way, every other sample must agree, and listed values must match."""
import numpy as np
import pytest

import oracle
import paper_1401_8258_b200 as dd
from paper_1401_8258_b200 import synth

from _util import dd_dtype, make_case, small

pytestmark = pytest.mark.gpu

EPS32 = 2.0 ** -23


@pytest.fixture(scope="module", autouse=True)
def _need_gpu():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"


def series(seed, nb, ndm, n, dtype=np.float32):
    """Synthetic dedispersed series: per-row level, slope and noise scale, isolated spikes, a few wide pulses."""
    g = np.random.default_rng(seed)
    t = np.arange(n)
    level = g.uniform(-50, 500, (nb, ndm, 1))
    slope = g.uniform(-2e-3, 2e-3, (nb, ndm, 1))
    sig = g.uniform(0.5, 30.0, (nb, ndm, 1))
    D = level + slope * t + sig * g.standard_normal((nb, ndm, n))
    for _ in range(3 * nb * ndm):
        b, d, p = g.integers(0, nb), g.integers(0, ndm), g.integers(0, n)
        D[b, d, p] += sig[b, d, 0] * g.uniform(6, 12)                              # single-sample spikes
    for _ in range(nb * ndm):
        b, d, p, wd = g.integers(0, nb), g.integers(0, ndm), g.integers(0, max(1, n - 20)), g.integers(4, 16)
        D[b, d, p:p + wd] += sig[b, d, 0] * g.uniform(5, 9)                        # resolved pulses
    if dtype == np.int32:
        return np.rint(D * 100).astype(np.int32)
    return D.astype(np.float32)


def run_post(D, params, want_series=True, capacity=1 << 16, pad=0, stats=True):
    """dd_postprocess on a host array D [nb][ndm][n] -> (Z or None, stats or None, candidates (structured), count)."""
    import torch
    nb, ndm, n = D.shape
    stride = n + pad
    Dd = torch.zeros((nb, ndm, stride), dtype=torch.float32 if D.dtype == np.float32 else torch.int32, device="cuda")
    Dd[:, :, :n] = torch.from_numpy(D).cuda()
    Zd = torch.full((nb, ndm, stride), -7.0, dtype=torch.float32, device="cuda") if want_series else None
    Sd = torch.zeros((nb * ndm, 3), dtype=torch.float64, device="cuda") if stats else None
    cand = torch.zeros(max(1, capacity) * 4, dtype=torch.int32, device="cuda")
    cnt = torch.zeros(1, dtype=torch.int64, device="cuda")
    dd.dd_postprocess(dd.DD_F32 if D.dtype == np.float32 else dd.DD_U8, Dd, stride, ndm * stride, ndm, n, nb, params,
                      Zd, stride, ndm * stride, Sd, cand if params.threshold_on else None, capacity,
                      cnt if params.threshold_on else None)
    torch.cuda.synchronize()
    count = int(cnt.item())
    c = cand.cpu().numpy().view(dd.CANDIDATE_DTYPE)[:min(count, capacity)]
    Z = None
    if Zd is not None:
        Zh = Zd.cpu().numpy()
        assert np.all(Zh[:, :, n:] == -7.0)                                        # padding untouched
        Z = Zh[:, :, :n]
    return Z, (Sd.cpu().numpy().reshape(nb, ndm, 3) if Sd is not None else None), c, count


def check_series(Z, z, stats, ymax, normalised, extra=0.0):
    scale = stats[..., 2:3] if normalised else np.ones_like(stats[..., 2:3])
    scale = np.where(scale > 0, scale, 1.0)
    tol = EPS32 * np.abs(z) + 1e-9 * ymax / scale + extra
    err = np.abs(Z.astype(np.float64) - z)
    assert np.all(err <= tol), "worst err/tol = %g" % (err / tol).max()


def check_candidates(c, count, z_snr, nsigma, tol):
    """c: structured candidates from the device; z_snr: the oracle's series in units of sigma [nb][ndm][n];
    tol: same shape or scalar."""
    assert count == len(c)
    tol = tol if np.isscalar(tol) else np.broadcast_to(tol, z_snr.shape)
    keys = set(zip(c["beam"].tolist(), c["dm"].tolist(), c["t"].tolist()))
    assert len(keys) == len(c), "duplicate candidates"
    must = np.argwhere(z_snr > nsigma + tol)
    may_not = z_snr < nsigma - tol
    for b, d, t in must:
        assert (int(b), int(d), int(t)) in keys, "missing candidate %s (S/N %g)" % ((b, d, t), z_snr[b, d, t])
    for k in c:
        b, d, t = int(k["beam"]), int(k["dm"]), int(k["t"])
        assert not may_not[b, d, t], "spurious candidate %s (S/N %g)" % ((b, d, t), z_snr[b, d, t])
        tt = tol if np.isscalar(tol) else tol[b, d, t]
        assert abs(float(k["value"]) - z_snr[b, d, t]) <= tt + EPS32 * abs(z_snr[b, d, t])
    return len(must)


# ------------------------------------------------------------------ identical input: every step and combination

@pytest.mark.parametrize("w", [0, 3, 5, 7, 9])
@pytest.mark.parametrize("mode", ["median_only", "detrend", "full"])
def test_steps_on_identical_series(w, mode):
    if mode == "median_only" and w == 0:
        pytest.skip("nothing to do")
    nb, ndm, n = 2, 7, 4096 * 2 + 333                      # several 2048-sample block steps and a ragged tail
    D = series(100 + w, nb, ndm, n)
    det, nrm = mode != "median_only", mode == "full"
    prm = dd.post_params(w, det, nrm, nsigma=5.0 if det else None)
    Z, st, c, count = run_post(D, prm, pad=5)
    z, stats = oracle.postprocess(D, median_window=w, detrend=det, normalise=nrm)
    ymax = np.abs(D).max()
    if det:
        assert np.all(np.abs(st - stats) <= 1e-10 * (1 + np.abs(stats)) + 1e-12 * ymax)
    check_series(Z, z, stats, ymax, nrm)
    if mode == "median_only":
        assert np.array_equal(Z.astype(np.float64), z)      # a selection: exact
    else:
        snr = z if nrm else z / stats[..., 2:3]
        assert check_candidates(c, count, snr, 5.0, 1e-9 * ymax / stats[..., 2:3] + 1e-12) > 10


def test_int32_series_from_the_uint8_path():
    D = series(7, 2, 5, 5000, dtype=np.int32)
    prm = dd.post_params(5, True, True, nsigma=6.0)
    Z, st, c, count = run_post(D, prm)
    z, stats = oracle.postprocess(D, median_window=5)
    check_series(Z, z, stats, np.abs(D).max(), True)
    check_candidates(c, count, z, 6.0, 1e-9 * np.abs(D).max() / stats[..., 2:3])


def test_edges_and_argument_errors():
    import torch
    # tiny series: n = 1, 2, shorter than the window; constant series (sigma = 0 -> zeros, no detections)
    for n in (1, 2, 3, 6):
        D = series(n, 1, 3, n)
        for w in (0, 3, 9):
            # two points always lie on their fitted line: the residual is rounding noise, which neither side can
            # normalise meaningfully (the device calls it sigma = 0); compare the detrended series there
            nrm = n != 2
            Z, st, c, count = run_post(D, dd.post_params(w, True, nrm, nsigma=0.5))
            z, stats = oracle.postprocess(D, median_window=w, normalise=nrm)
            check_series(Z, z, stats, np.abs(D).max(), nrm, extra=1e-6)
    D = np.full((1, 2, 3000), 42.5, dtype=np.float32)
    Z, st, c, count = run_post(D, dd.post_params(7, True, True, nsigma=1.0))
    assert not Z.any() and count == 0 and np.all(st[..., 2] == 0.0) and np.all(st[..., 0] == 42.5)
    # capacity overflow: the counter keeps counting, the buffer is not overrun
    D = series(11, 1, 4, 3000)
    z, stats = oracle.postprocess(D)
    total = int((z > 1.0).sum())
    Z, st, c, count = run_post(D, dd.post_params(0, True, True, nsigma=1.0), capacity=10)
    assert count == total and total > 100 and len(c) == 10
    for k in c:
        assert z[k["beam"], k["dm"], k["t"]] > 1.0
    # empty work writes nothing
    e = torch.full((4,), -7.0, device="cuda")
    dd.dd_postprocess(dd.DD_F32, e, 0, 0, 0, 100, 1, dd.post_params(0, True, True), e, 0, 0)
    dd.dd_postprocess(dd.DD_F32, e, 4, 0, 1, 0, 1, dd.post_params(0, True, True), e, 4, 0)
    torch.cuda.synchronize()
    assert bool((e == -7.0).all())
    # in place: allowed without a median window, refused with one
    Dd = torch.from_numpy(D[0]).cuda()
    dd.dd_postprocess(dd.DD_F32, Dd, 3000, 0, 4, 3000, 1, dd.post_params(0, True, True), Dd, 3000, 0)
    torch.cuda.synchronize()
    check_series(Dd.cpu().numpy()[None], z, stats, np.abs(D).max(), True)
    bad = [lambda: dd.dd_postprocess(dd.DD_F32, Dd, 3000, 0, 4, 3000, 1, dd.post_params(5, True, True), Dd, 3000, 0),
           lambda: dd.dd_postprocess(dd.DD_F32, Dd, 3000, 0, 4, 3000, 1, dd.post_params(4, True, True), None),
           lambda: dd.dd_postprocess(dd.DD_F32, Dd, 3000, 0, 4, 3000, 1, dd.post_params(0, False, True), None),
           lambda: dd.dd_postprocess(dd.DD_F32, Dd, 3000, 0, 4, 3000, 1, dd.post_params(0, True, True, nsigma=5.0), None),
           lambda: dd.dd_postprocess(dd.DD_F32, Dd, 100, 0, 4, 3000, 1, dd.post_params(0, True, True), None),
           lambda: dd.dd_postprocess(7, Dd, 3000, 0, 4, 3000, 1, dd.post_params(0, True, True), None)]
    for f in bad:
        with pytest.raises(dd.DedispError) as ei:
            f()
        assert ei.value.code == dd.DD_ERR_BAD_ARG


def test_threshold_only_calls_list_exactly_the_candidates_of_calls_with_series_output():
    """Without a series output the apply kernel screens samples in single precision before the double
    decision (post.cu); the candidate list must be exactly the one of the unscreened evaluation.  Cases that
    stress the screen: levels and slopes large against sigma (coarse float line), thresholds that many samples
    sit next to (n sigma = 0, 0.5), integer series, ragged lengths."""
    cases = []
    for seed, (nb, ndm, n) in enumerate([(1, 7, 10001), (2, 3, 2049), (1, 2, 40000), (1, 3, 5)]):
        cases.append((series(300 + seed, nb, ndm, n), "f32"))
    D = series(310, 1, 4, 30011)
    cases.append(((D + np.float32(3e6)).astype(np.float32), "level 3e6"))       # ulp(level) = 0.25 ~ sigma / 2 .. 100
    t = np.arange(30011, dtype=np.float64)
    cases.append(((D + 40.0 * t).astype(np.float32), "slope 40"))
    cases.append(((D - 55.0 * t - 1e5).astype(np.float32), "slope -55"))
    cases.append((series(311, 1, 3, 9000, dtype=np.int32), "i32"))
    cases.append((series(312, 1, 3, 9000, dtype=np.int32) + np.int32(2 ** 30), "i32 level 2^30"))
    cases.append((series(313, 1, 3, 9000, dtype=np.int32) - np.int32(2 ** 30), "i32 level -2^30"))
    checked = 0
    for D, name in cases:
        for w in (0, 5):
            for nsig in (0.0, 0.5, 3.0, 6.0):
                prm = dd.post_params(w, True, True, nsigma=nsig)
                cap = D.size + 1
                _, _, c1, n1 = run_post(D, prm, want_series=True, capacity=cap)
                _, _, c2, n2 = run_post(D, prm, want_series=False, capacity=cap, stats=False)
                assert n1 == n2, (name, w, nsig, n1, n2)
                k1 = sorted(zip(c1["beam"].tolist(), c1["dm"].tolist(), c1["t"].tolist(), c1["value"].tolist()))
                k2 = sorted(zip(c2["beam"].tolist(), c2["dm"].tolist(), c2["t"].tolist(), c2["value"].tolist()))
                assert k1 == k2, (name, w, nsig)
                checked += n1
        # un-normalised output compares against n * sigma with the same screen
        prm = dd.post_params(3, True, False, nsigma=4.0)
        _, _, c1, n1 = run_post(D, prm, want_series=True, capacity=D.size + 1)
        _, _, c2, n2 = run_post(D, prm, want_series=False, capacity=D.size + 1, stats=False)
        assert n1 == n2 and sorted(c1.tolist()) == sorted(c2.tolist()), name
    assert checked > 100000


@pytest.mark.parametrize("n", [1, 127, 128, 129, 2048 + 1, 3 * 2048 + 127, 70001])
def test_candidates_only_calls_find_detections_at_chunk_edges(n):
    """Candidates-only calls skip every 128-sample chunk whose largest median cannot pass (chunk maxima left by the
    statistics pass): single-sample detections at the first and last sample of chunks, of block steps and of the
    series (whose last chunk is partial) must all be listed, and nothing else."""
    g = np.random.default_rng(n)
    nb, ndm = 2, 3
    D = (100.0 + 0.25 * g.standard_normal((nb, ndm, n))).astype(np.float32)
    spots = sorted({t for t in (0, 1, 126, 127, 128, 129, 255, 256, 2047, 2048, 2049, 4095, 4096, n - 129, n - 128,
                                n - 2, n - 1) if 0 <= t < n})
    want = set()
    for b in range(nb):
        for d in range(ndm):
            for t in spots[(b + d) % 2::2]:                           # a different subset per series
                D[b, d, t] += 30.0 if n > 40 else 3.0
                want.add((b, d, t))
    # (the detections themselves inflate sigma of a short series: 30 / sigma is 5.6 at n = 127, 18 at n = 2049)
    prm = dd.post_params(0, True, True, nsigma=8.0 if n > 2000 else (4.0 if n > 40 else 1.2))
    _, _, c0, n0 = run_post(D, prm, want_series=True, capacity=1 << 12)
    _, _, c1, n1 = run_post(D, prm, want_series=False, capacity=1 << 12, stats=False)
    k0 = sorted(zip(c0["beam"].tolist(), c0["dm"].tolist(), c0["t"].tolist(), c0["value"].tolist()))
    k1 = sorted(zip(c1["beam"].tolist(), c1["dm"].tolist(), c1["t"].tolist(), c1["value"].tolist()))
    assert n0 == n1 and k0 == k1
    if n > 40:
        assert {(b, d, t) for b, d, t, _ in k1} == want


# ------------------------------------------------------------------ the chain: dedisperse -> post-process -> candidates

@pytest.mark.parametrize("idx,nchans,ndm,nsamp,w", [(3, 512, 50, 8192 + 100, 0), (2, 256, 70, 9000, 3), (4, 128, 40, 6000, 5)])
def test_chain_against_the_oracle_chain(idx, nchans, ndm, nsamp, w):
    import torch
    wl = small(idx, nchans, ndm, nsamp)
    X, ms = make_case(wl)
    tab = oracle.shift_table(wl.nchans, wl.fch1, wl.foff, wl.tsamp, wl.dm_list)
    amp = 0.6 if wl.dtype == "f32" else 10
    pulses = [(ndm // 3, nsamp // 4, 8), (ndm - 2, nsamp // 2, 16)]
    for d, t0, width in pulses:
        synth.inject_pulse(X, t0, width, amp, tab[d])
    nsigma = 6.0
    # device chain
    plan = dd.Plan(dd_dtype(wl), wl.nchans, wl.fch1, wl.foff, wl.tsamp, wl.dm_list)
    Xd = torch.from_numpy(X).cuda()
    Dd = torch.empty((wl.ndm, wl.nsamp), dtype=torch.float32 if wl.dtype == "f32" else torch.int32, device="cuda")
    plan.execute(Xd, X.shape[1], 0, Dd, wl.nsamp, 0, wl.nsamp, 1)
    Zd = torch.empty((wl.ndm, wl.nsamp), dtype=torch.float32, device="cuda")
    cand = torch.zeros(4 * 4096, dtype=torch.int32, device="cuda")
    cnt = torch.zeros(1, dtype=torch.int64, device="cuda")
    prm = dd.post_params(w, True, True, nsigma=nsigma)
    dd.dd_postprocess(dd_dtype(wl), Dd, wl.nsamp, 0, wl.ndm, wl.nsamp, 1, prm, Zd, wl.nsamp, 0, None, cand, 4096, cnt)
    torch.cuda.synchronize()
    count = int(cnt.item())
    c = cand.cpu().numpy().view(dd.CANDIDATE_DTYPE)[:count]
    # oracle chain: dedisperse in double, hand the series over in the product's output type, post-process in double
    if wl.dtype == "f32":
        D64, A = oracle.dedisperse_f32(X, wl.nsamp, wl.fch1, wl.foff, wl.tsamp, wl.dm_list, interchanged=True)
        Dor = D64.astype(np.float32)
        delta = 1e-5 * A.max()
    else:
        Dor = oracle.dedisperse_u8(X, wl.nsamp, wl.fch1, wl.foff, wl.tsamp, wl.dm_list, interchanged=True).astype(np.int32)
        delta = 0.0
    z, stats = oracle.postprocess(Dor[None], median_window=w)
    tol = 5.0 * delta * (1.0 + np.abs(z)) / stats[..., 2:3] + EPS32 * np.abs(z) + 1e-9 * np.abs(Dor).max() / stats[..., 2:3]
    err = np.abs(Zd.cpu().numpy()[None].astype(np.float64) - z)
    assert np.all(err <= tol), (err / tol).max()
    check_candidates(c, count, z, nsigma, tol)
    # the planted pulses are found at their trial and time (each has S/N ~ amp sqrt(nchans) / noise per sample)
    found = {(int(k["dm"]), int(k["t"])) for k in c}
    for d, t0, width in pulses:
        if w <= 1 or width > w:
            assert any(dd_ == d and t0 <= t < t0 + width for dd_, t in found), (d, t0)
    # dd_search_host: same candidates from host buffers, only the list comes back
    hc = np.zeros(4096, dtype=dd.CANDIDATE_DTYPE)
    n = plan.search_host(X, X.shape[1], 0, wl.nsamp, 1, prm, hc, 4096)
    assert n == count
    assert sorted(map(tuple, hc[:n].tolist())) == sorted(map(tuple, c.tolist()))
    plan.destroy()


def test_config3_full_size_postprocess_properties_and_rows():
    # the launch configuration bench.py's search leg times: the whole (DM, t) plane of BASELINE.json configs[2]
    # (4096 x 2^18 float32) post-processed on the device with w = 5, 6 sigma.  Properties that hold at any size:
    # every series has mean 0 and variance 1; the candidate list is exactly {Z > 6}; plus whole rows against the
    # oracle chain (oracle dedispersion rows -> float32 -> oracle post-processing) with the chain tolerance.
    import torch
    w = synth.WORKLOADS[3]
    tab = oracle.shift_table(w.nchans, w.fch1, w.foff, w.tsamp, w.dm_list)
    ms = int(tab.max())
    X = synth.make_input(w, w.nsamp + ms)
    pulses = synth.pulse_plan(w, 5)
    for d, t0, width in pulses:
        synth.inject_pulse(X, t0, max(width, 8), 0.25, tab[d])
    stride = (w.nsamp + ms + 63) // 64 * 64
    plan = dd.Plan(dd.DD_F32, w.nchans, w.fch1, w.foff, w.tsamp, w.dm_list)
    Xd = torch.zeros((w.nchans, stride), dtype=torch.float32, device="cuda")
    Xd[:, :w.nsamp + ms] = torch.from_numpy(X).cuda()
    Dd = torch.empty((w.ndm, w.nsamp), dtype=torch.float32, device="cuda")
    plan.execute(Xd, stride, 0, Dd, w.nsamp, 0, w.nsamp, 1)
    del Xd
    Zd = torch.empty((w.ndm, w.nsamp), dtype=torch.float32, device="cuda")
    cap = 1 << 20
    cand = torch.zeros(4 * cap, dtype=torch.int32, device="cuda")
    cnt = torch.zeros(1, dtype=torch.int64, device="cuda")
    prm = dd.post_params(5, True, True, nsigma=6.0)
    dd.dd_postprocess(dd.DD_F32, Dd, w.nsamp, 0, w.ndm, w.nsamp, 1, prm, Zd, w.nsamp, 0, None, cand, cap, cnt)
    torch.cuda.synchronize()
    count = int(cnt.item())
    assert 0 < count < cap
    c = cand.cpu().numpy().view(dd.CANDIDATE_DTYPE)[:count]
    mean = Zd.mean(dim=1, dtype=torch.float64).cpu().numpy()
    var = (Zd.double() ** 2).mean(dim=1).cpu().numpy()
    assert np.abs(mean).max() < 1e-6 and np.abs(var - 1.0).max() < 1e-5
    assert count == int((Zd > 6.0).sum().item())
    got = Zd[torch.from_numpy(c["dm"].astype(np.int64)).cuda(), torch.from_numpy(c["t"].astype(np.int64)).cuda()].cpu().numpy()
    assert np.array_equal(got, c["value"]) and np.all(c["value"] > 6.0) and np.all(c["beam"] == 0)
    # every pulse of width >= 8 survives the w = 5 median and is listed at its trial
    found = set(zip(c["dm"].tolist(), c["t"].tolist()))
    for d, t0, width in pulses:
        assert any((d, t) in found for t in range(t0, t0 + max(width, 8))), (d, t0, width)
    rows = np.array(sorted({0, w.ndm - 1, 1000} | {d for d, _, _ in pulses}), dtype=np.int32)
    D64, A = oracle.dedisperse_f32(X, w.nsamp, w.fch1, w.foff, w.tsamp, w.dm_list, rows=rows, interchanged=True)
    z, stats = oracle.postprocess(D64.astype(np.float32)[None], median_window=5)
    tol = 5e-5 * A.max() * (1.0 + np.abs(z)) / stats[..., 2:3] + EPS32 * np.abs(z) + 1e-9 * np.abs(D64).max() / stats[..., 2:3]
    err = np.abs(Zd[torch.from_numpy(rows).long().cuda()].cpu().numpy()[None].astype(np.float64) - z)
    assert np.all(err <= tol), (err / tol).max()
    print("post-processing rows: worst err/tol = %.3g, worst abs err = %.3g" % ((err / tol).max(), err.max()))
    plan.destroy()
