"""Pins for the post-processing oracle (oracle/postproc_oracle.cpp; §3.5-3.6), CPU only.
Each test anchors it to something other than itself: numpy library routines (median over edge-padded
sliding windows, polyfit), hand-worked windows, closed forms, invariants, and the thesis' own S/N recipe
(PAPER.md:995).  A plausible mistake (window off centre, wrong edge rule, sample instead of population
variance, slope/intercept swapped, >= instead of >, wrong triplet order) fails at least one of them."""
import numpy as np
import pytest

import oracle
from paper_1401_8258_b200 import synth


def np_median_filter(x, w):
    h = (w - 1) // 2
    xp = np.pad(np.asarray(x, dtype=np.float64), h, mode="edge")
    return np.median(np.lib.stride_tricks.sliding_window_view(xp, w), axis=1)


# ---------------------------------------------------------------- median filter (eq 3.4)

def test_median_by_hand():
    # w = 3: each output is the middle of (left, self, right), ends replicated (R15)
    x = [1, 9, 2, 8, 3, 7, 4]
    assert oracle.median_filter(x, 3).tolist() == [1, 2, 8, 3, 7, 4, 4]
    # w = 5 around an isolated spike: the spike disappears, the edges of the step survive
    x = [0, 0, 0, 50, 0, 0, 0, 5, 5, 5, 5, 5]
    assert oracle.median_filter(x, 5).tolist() == [0, 0, 0, 0, 0, 0, 0, 5, 5, 5, 5, 5]
    assert oracle.median_filter([4.0], 7).tolist() == [4.0]          # n = 1: all window entries are the sample
    assert oracle.median_filter([3, 1, 2], 1).tolist() == [3, 1, 2]  # w = 1: identity


@pytest.mark.parametrize("w", [3, 5, 7, 9])
def test_median_against_numpy_sliding_windows(w):
    g = np.random.default_rng(w)
    for n in (1, 2, w - 1, w, 40, 1001):
        x = g.standard_normal(n)
        x[g.integers(0, n, max(1, n // 10))] += 30.0              # outliers
        assert np.array_equal(oracle.median_filter(x, w), np_median_filter(x, w))
        xi = g.integers(-5, 5, n).astype(np.float64)              # many ties
        assert np.array_equal(oracle.median_filter(xi, w), np_median_filter(xi, w))


def test_median_invariants():
    g = np.random.default_rng(0)
    ramp = np.arange(100, dtype=np.float64) * 0.25 - 3
    for w in (3, 5, 7):
        assert np.array_equal(oracle.median_filter(ramp, w), ramp)                 # monotone series are fixed points
        assert np.array_equal(oracle.median_filter(ramp[::-1].copy(), w), ramp[::-1])
        x = g.standard_normal(500)
        y = oracle.median_filter(x, w)
        assert np.all(np.isin(y, x))                                               # a selection, never a new value
        assert np.array_equal(oracle.median_filter(-x, w), -y)                     # odd window: symmetric
        assert np.array_equal(oracle.median_filter(2.0 * x, w), 2.0 * y)           # scale covariance (exact: powers of 2)
    # "preserves the edges of the signal": a step stays a step
    step = np.r_[np.zeros(20), np.ones(20)]
    assert np.array_equal(oracle.median_filter(step, 7), step)


# ---------------------------------------------------------------- detrending and normalisation

def test_fit_line_against_polyfit_and_closed_forms():
    g = np.random.default_rng(1)
    t = np.arange(2000, dtype=np.float64)
    assert oracle.fit_line(3.0 + 0.5 * np.arange(10)) == (3.0, 0.5)               # exact line, exact arithmetic
    y = 100.0 - 0.01 * t + g.standard_normal(2000)
    a, b = oracle.fit_line(y)
    pb, pa = np.polyfit(t, y, 1)
    assert abs(a - pa) < 1e-9 and abs(b - pb) < 1e-12
    # residuals of a least-squares line are orthogonal to 1 and to t
    r, sigma = oracle.detrend(y, a, b)
    assert abs(r.sum()) < 1e-7 and abs((r * t).sum()) < 1e-4
    assert oracle.fit_line([5.0]) == (5.0, 0.0)                                    # n = 1
    a, b = oracle.fit_line([1.0, 3.0])
    assert (a, b) == (1.0, 2.0)


def test_detrend_and_sigma_closed_forms():
    t = np.arange(64, dtype=np.float64)
    r, sigma = oracle.detrend(7.0 - 2.0 * t, 7.0, -2.0)                            # an exact line -> zeros
    assert not r.any() and sigma == 0.0
    assert not oracle.normalise(r, sigma).any()                                    # R17: sigma = 0 -> zeros
    alt = np.where(t % 2 == 0, 1.0, -1.0)                                          # +-1: population sigma = 1
    r, sigma = oracle.detrend(alt, 0.0, 0.0)
    assert sigma == 1.0 and np.array_equal(r, alt)
    # population (1/n), not sample (1/(n-1)), variance: values {0, 2} -> mean 1, sigma 1 (sample form: sqrt 2)
    r, sigma = oracle.detrend(np.array([0.0, 2.0]), 1.0, 0.0)
    assert sigma == 1.0
    # the residual of a ramp about the WRONG line y = 0 has sigma^2 = mean(t^2) = (n-1)(2n-1)/6
    r, sigma = oracle.detrend(t, 0.0, 0.0)
    assert abs(sigma ** 2 - 63 * 127 / 6.0) < 1e-9


def test_postprocess_pipeline_properties():
    g = np.random.default_rng(2)
    n = 4096
    D = (50.0 + 0.003 * np.arange(n) + 4.0 * g.standard_normal((3, 5, n))).astype(np.float32)
    z, stats = oracle.postprocess(D, median_window=0, detrend=True, normalise=True)
    assert z.shape == D.shape and stats.shape == (3, 5, 3)
    assert np.all(np.abs(z.mean(axis=-1)) < 1e-12) and np.all(np.abs(z.std(axis=-1) - 1.0) < 1e-12)
    assert np.all(np.abs(stats[..., 1] - 0.003) < 1e-3) and np.all(np.abs(stats[..., 2] - 4.0) < 0.2)
    # the steps compose exactly as the single-step functions (same code path, checks the row plumbing / order R19)
    for w in (0, 5):
        z, stats = oracle.postprocess(D, median_window=w)
        x = D[1, 2].astype(np.float64)
        if w:
            x = np_median_filter(x, w)
        pb, pa = np.polyfit(np.arange(n, dtype=np.float64), x, 1)
        r = x - (pa + pb * np.arange(n))
        want = r / np.sqrt((r * r).mean())
        assert np.abs(z[1, 2] - want).max() < 1e-9
    # int32 input (the uint8 path's output) gives what its float64 copy gives
    Di = g.integers(100000, 140000, (2, 3, 500)).astype(np.int32)
    zi, _ = oracle.postprocess(Di, median_window=3)
    zf, _ = oracle.postprocess(Di.astype(np.float32), median_window=3)            # exact in float32 (< 2^24)
    assert np.array_equal(zi, zf)
    # partial pipelines
    z, stats = oracle.postprocess(D, median_window=7, detrend=False, normalise=False)
    assert np.array_equal(z[0, 0], np_median_filter(D[0, 0].astype(np.float64), 7)) and not stats.any()
    z, stats = oracle.postprocess(D, median_window=0, detrend=True, normalise=False)
    assert np.all(np.abs(z.std(axis=-1) - stats[..., 2]) < 1e-9)


# ---------------------------------------------------------------- thresholding

def test_threshold_triplets_order_and_strictness():
    z = np.zeros((2, 3, 10))
    z[0, 1, 4] = 6.0
    z[0, 1, 5] = 5.0            # == threshold: NOT a detection (strict >, R18)
    z[1, 2, 9] = 5.0000001
    z[1, 0, 0] = 100.0
    b, d, t, v, cnt = oracle.threshold(z, 5.0)
    assert cnt == 3
    assert list(zip(b.tolist(), d.tolist(), t.tolist(), v.tolist())) == [(0, 1, 4, 6.0), (1, 0, 0, 100.0), (1, 2, 9, 5.0000001)]
    # capacity smaller than the number found: the count keeps counting
    b, d, t, v, cnt = oracle.threshold(z, 5.0, capacity=2)
    assert cnt == 3 and len(b) == 2
    # un-normalised series: level = n * sigma(row)
    sig = np.full((2, 3), 2.0)
    sig[1, 0] = 60.0
    b, d, t, v, cnt = oracle.threshold(z, 2.75, sigma=sig)
    assert list(zip(b.tolist(), d.tolist(), t.tolist())) == [(0, 1, 4)]          # 6 > 5.5; 5 < 5.5; 100 < 165
    # brute force on random data
    g = np.random.default_rng(3)
    z = g.standard_normal((2, 4, 300))
    b, d, t, v, cnt = oracle.threshold(z, 2.0)
    want = np.argwhere(z > 2.0)
    assert cnt == len(want) and np.array_equal(np.stack([b, d, t], axis=1), want) and np.array_equal(v, z[z > 2.0])


def test_fig_2_6_recipe_gives_one_detection_at_the_injected_pulse():
    # noise mu = 0 sigma = 1, a pulse of amplitude 0.25 in each of 1024 channels ->
    # S/N = 0.25 * sqrt(1024) = 8 in the dedispersed series at the right DM.  Dedisperse with the (pinned)
    # dedispersion oracle, post-process, threshold at 6 sigma: the detections sit at the injected
    # (DM, t); Gaussian noise alone exceeds 6 sigma with probability 1e-9 per sample.
    w = synth.scaled(synth.WORKLOADS[2], dtype="f32", nchans=1024, ndm=24, nsamp=4096, seed=2601)
    tab = oracle.shift_table(w.nchans, w.fch1, w.foff, w.tsamp, w.dm_list)
    X = synth.make_input(w, w.nsamp + int(tab.max()))
    synth.inject_pulse(X, 1500, 1, 0.25, tab[17])
    D, _ = oracle.dedisperse_f32(X, w.nsamp, w.fch1, w.foff, w.tsamp, w.dm_list, interchanged=True)
    z, stats = oracle.postprocess(D.astype(np.float32)[None], median_window=0)
    assert np.all(np.abs(stats[0, :, 2] - 32.0) < 1.5)                             # sigma = sqrt(1024)
    assert abs(z[0, 17, 1500] - 8.0) < 2.5
    b, d, t, v, cnt = oracle.threshold(z, 6.0)
    assert cnt >= 1 and (0, 17, 1500) in set(zip(b.tolist(), d.tolist(), t.tolist()))
    assert all(abs(int(dd_) - 17) <= 1 and abs(int(tt) - 1500) <= 2 for dd_, tt in zip(d, t))
    # "median filtering will limit the detectability of short duration ... signals":
    # the single-sample pulse does not survive a w = 5 median filter
    z5, _ = oracle.postprocess(D.astype(np.float32)[None], median_window=5)
    assert oracle.threshold(z5, 6.0)[4] == 0
