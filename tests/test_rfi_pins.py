"""Pins for the RFI-mitigation oracle (oracle/rfi.py; §3.3), CPU only: numpy's own
polynomial fit, exact polynomials, hand-worked windows, closed-form statistics, and the thesis' §3.3.4 test
recipe: narrowband periodic RFI and a broadband pulse are removed, a dispersed pulse is
left untouched."""
import numpy as np

import oracle
from oracle import rfi
from paper_1401_8258_b200 import synth


def test_bandpass_fit_against_numpy_polynomial_and_exact_recovery():
    g = np.random.default_rng(0)
    nch = 200
    x = rfi.channel_abscissa(nch)
    assert x[0] == -1.0 and x[-1] == 1.0 and abs(x[1] - x[0] - 2.0 / (nch - 1)) < 1e-15
    truth = 5.0 + 2.0 * x - 3.0 * x ** 2 + 0.5 * x ** 3
    B, rmse = rfi.fit_bandpass(truth, 3)
    assert np.abs(B - truth).max() < 1e-12 and rmse < 1e-12                    # an exact cubic is recovered
    B5, _ = rfi.fit_bandpass(truth, 5)
    assert np.abs(B5 - truth).max() < 1e-11                                     # a higher order fits it too
    b = truth + 0.1 * g.standard_normal(nch)
    for order in (0, 1, 4, 8):
        B, rmse = rfi.fit_bandpass(b, order)
        want = np.polynomial.polynomial.polyval(x, np.polynomial.polynomial.polyfit(x, b, order))
        assert np.abs(B - want).max() < 1e-10
        assert abs(rmse - np.sqrt(np.mean((b - want) ** 2))) < 1e-12
        # least squares: the residual is orthogonal to every basis polynomial
        for k in range(order + 1):
            assert abs(((b - B) * x ** k).sum()) < 1e-8
    B0, rmse0 = rfi.fit_bandpass(b, 0)
    assert np.allclose(B0, b.mean()) and abs(rmse0 - b.std()) < 1e-12           # order 0: the mean; rmse = population std
    # the fitted values do not depend on how the abscissa is scaled (R21): compare with a fit in raw channel index
    raw = np.polynomial.polynomial.polyval(np.arange(nch), np.polynomial.polynomial.polyfit(np.arange(nch), b, 2))
    assert np.abs(rfi.fit_bandpass(b, 2)[0] - raw).max() < 1e-9
    # averaged bandpass = row means in double
    X = g.standard_normal((7, 1000)).astype(np.float32) + np.arange(7, dtype=np.float32)[:, None]
    assert np.abs(rfi.bandpass_mean(X) - X.astype(np.float64).sum(axis=1) / 1000).max() < 1e-15


def test_channel_windows_by_hand():
    # 2 channels, 10 samples, windows of 4 (the last has 2 samples); B = (1, 0), rmse = 0.5, T_c = 2 -> |M - B| > 1
    X = np.array([[1, 1, 1, 1, 5, 5, 5, 5, 1, 1],                # window means 1, 5, 1 -> own flag on window 1
                  [0, 0, 0, 0, 0, 0, 0, 0, -3, -3]], np.float32)  # means 0, 0, -3 -> own flag on window 2 (two-sided, R23)
    flags, own = rfi.channel_flags(X, np.array([1.0, 0.0]), 0.5, 4, 2.0)
    assert own.tolist() == [[False, True, False], [False, False, True]]
    assert flags.tolist() == [[True, True, True], [False, True, True]]          # neighbours k-1, k+1 (R24)
    Y = rfi.apply_channel_flags(X, np.array([1.0, 0.0]), flags, 4)
    assert Y.tolist() == [[1] * 10, [0, 0, 0, 0, 0, 0, 0, 0, 0, 0]]
    # a mean exactly at the threshold is not flagged (strict >)
    flags, own = rfi.channel_flags(np.full((1, 8), 2.0, np.float32), np.array([1.0]), 0.5, 4, 2.0)
    assert not own.any()
    # brute force on random data
    g = np.random.default_rng(1)
    X = g.standard_normal((5, 103)).astype(np.float32)
    B = g.standard_normal(5) * 0.1
    flags, own = rfi.channel_flags(X, B, 0.2, 10, 1.5)
    for c in range(5):
        for k in range(11):
            seg = X[c, 10 * k:10 * k + 10].astype(np.float64)
            assert own[c, k] == (abs(seg.sum() / len(seg) - B[c]) > 0.3)
            nb = own[c, max(0, k - 1):k + 2].any()
            assert flags[c, k] == nb


def test_spectrum_threshold_closed_forms():
    # 4 channels, 8 spectra; spectrum means m = (0,0,0,0,0,0,0,8): mu = 1, sigma^2 = (7*1 + 49)/8 = 7
    Y = np.zeros((4, 8))
    Y[:, 7] = [6.0, 8.0, 10.0, 8.0]
    m, mu, sigma = rfi.spectrum_stats(Y)
    assert m.tolist() == [0, 0, 0, 0, 0, 0, 0, 8] and mu == 1.0 and abs(sigma ** 2 - 7.0) < 1e-12
    B = np.array([1.0, 1.0, 1.0, 5.0])                                          # bandpass mean 2
    out, flagged, _ = rfi.apply_spectrum_threshold(Y, B, 2.0)                   # 8 - 1 = 7 > 2 sqrt 7 = 5.29
    assert flagged.tolist() == [False] * 7 + [True]
    assert out[:, 7].tolist() == [0.0, 2.0, 4.0, 2.0]                           # minus (8 - 2): the shape survives (R26)
    assert abs(out[:, 7].mean() - 2.0) < 1e-12                                  # its mean is now the bandpass mean
    out, flagged, _ = rfi.apply_spectrum_threshold(Y, B, 3.0)                   # 7 < 3 sqrt 7 = 7.94
    assert not flagged.any() and np.array_equal(out, Y)
    out, flagged, _ = rfi.apply_spectrum_threshold(-Y, B, 2.0)                  # one-sided (R25): dips are kept
    assert not flagged.any()


def rfi_test_buffer(seed=3304, nchans=512, nsamp=31250):
    """§3.3.4: 413 MHz centre, 10 MHz band, 512 channels, 1.6 s of N(0,1) noise (51.2 us sampling), a 10 ms
    dispersed pulse of S/N 10 at DM 120, narrowband RFI (78 kHz = 4 channels, period 6.5 ms), a broadband 2 ms
    pulse of S/N 10; multiplied by a smooth bandpass shape with a small ripple."""
    g = np.random.default_rng(seed)
    tsamp, fch1, foff = 51.2e-6, 418.0, -10.0 / nchans
    X = g.standard_normal((nchans, nsamp))
    w10 = int(round(10e-3 / tsamp))
    tab = oracle.shift_table(nchans, fch1, foff, tsamp, [120.0])[0]
    amp = 10.0 / np.sqrt(nchans * w10)
    for c in range(nchans):
        X[c, 8000 + tab[c]:8000 + tab[c] + w10] += amp
    per, t = int(round(6.5e-3 / tsamp)), np.arange(nsamp)
    on = (t % per) < per // 2
    X[300:304, on] += 3.0                                                       # narrowband, periodic
    w2 = int(round(2e-3 / tsamp))
    X[:, 20000:20000 + w2] += 10.0 / np.sqrt(nchans * w2) * 6.0                 # broadband pulse, strong per sample
    x = rfi.channel_abscissa(nchans)
    shape = 1.0 - 0.3 * x ** 2 + 0.1 * x + 0.01 * np.sin(40 * x)                 # smooth + ripple the cubic cannot follow
    X = (X + 20.0) * shape[:, None]
    return X.astype(np.float32), dict(tsamp=tsamp, fch1=fch1, foff=foff, pulse=(8000, w10, tab), nb=(300, 304),
                                      bb=(20000, w2), shape=shape)


def test_section_3_3_4_recipe():
    X, info = rfi_test_buffer()
    r = rfi.mitigate(X, order=4, window=512, t_chan=7.0, t_spec=5.0)
    out = r["out"]
    # the fit follows the bandpass, the RMSE is the size of the ripple the polynomial cannot follow
    assert np.abs(r["fit"] / (20.0 * info["shape"]) - 1.0).max() < 0.03 and 0.05 < r["rmse"] < 0.3
    # narrowband RFI: every window of the four channels is flagged and replaced (-> exactly 0 after correction)
    assert r["chan_flags"][300:304].all() and not out[300:304][:, ~r["spec_flags"]].any()
    clean = np.r_[0:298, 306:512]
    assert r["chan_flags"][clean].mean() < 0.01                                  # noise windows are rarely touched
    # broadband pulse: its spectra are flagged, nothing else is
    t0, w2 = info["bb"]
    assert r["spec_flags"][t0:t0 + w2].all() and r["spec_flags"].sum() == w2
    assert abs(out[clean][:, t0:t0 + w2].mean()) < 0.05                          # the excess is gone
    # the dispersed pulse "didn't trigger any thresholding mechanism": its samples are the input minus the fit
    p0, w10, tab = info["pulse"]
    for c in (0, 100, 250, 400, 511):
        seg = slice(p0 + tab[c], p0 + tab[c] + w10)
        k0, k1 = (p0 + tab[c]) // 512, (p0 + tab[c] + w10 - 1) // 512
        assert not r["chan_flags"][c, k0:k1 + 1].any() and not r["spec_flags"][seg].any()
        assert np.array_equal(out[c, seg], X[c, seg].astype(np.float64) - r["fit"][c])
    # corrected spectra sit at a mean of ~0
    assert abs(out[clean].mean()) < 0.02
