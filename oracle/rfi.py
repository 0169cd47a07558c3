"""ORACLE — test infrastructure only.  RFI mitigation front end of the thesis (§3.3),
plain numpy in float64, one function per stage, in the paper's order.  Shares no code with the CUDA
library and is never imported by the product.

Stages (§3.3.1-3.3.3):
  1. bandpass: average every frequency channel over the buffer ("a reduction sum ... resulting in N_c
     values"), fit a p-th order polynomial to the averaged bandpass by least squares, take the RMSE between
     fit and averaged bandpass;
  2. channel thresholding (eq 3.1): partition every channel into non-overlapping
     windows of W_c samples; a window whose mean is off the channel's fitted bandpass value by more than
     the channel threshold is flagged, "neighbouring blocks are also flagged", and flagged windows are
     replaced "with the frequency channel's fitted bandpass value";
  3. spectrum thresholding (eq 3.2): the mean of each full-band spectrum is compared
     with a spectrum threshold; a spectrum above it has its excess over the bandpass removed;
  4. the fitted bandpass is subtracted from all spectra ("moving the mean to, or near, 0").

Readings where the text is silent, garbled or at odds with itself (R20-R27):
  R20 layout: X [nchans][nsamp] float32, time fastest, processed in place;
  R21 the polynomial's abscissa is the channel index mapped linearly onto [-1, 1] (the fitted VALUES do not
      depend on this scaling; it only conditions the least-squares problem); all channels take part (the
      optional masking of known bad channels, is not built);
  R22 RMSE = sqrt(mean_c (b_c - B_c)^2), b the averaged and B the fitted bandpass;
  R23 eq 3.1 is printed as "M(c) < B_sigma => c_i = B_v"; the text ("if this threshold is exceeded",
      "the lower threshold is required for when input data are lost") makes the test two-sided:
      a window is flagged iff |M - B_v| > T_c * RMSE; the last, shorter window of a row counts with its own length;
  R24 neighbours: windows k-1 and k+1 of a window flagged by its own mean;
  R25 spectrum statistics: "the mean and standard deviation are used for the spectrum thresholding stage" --
      taken as the mean mu and population standard deviation sigma, over time, of the spectrum means m_t of
      the channel-clipped buffer; spectrum t is flagged iff m_t - mu > T_s * sigma (one-sided: "if the mean
      exceeds this threshold");
  R26 eq 3.2 as printed, S_c = S_c - (S_c - B_c), would erase the spectrum; §3.3.4 says the pulse "was
      replaced by the value of the noisy signal, its difference from the bandpass values subtracted": taken
      as S_c <- S_c - (m_t - mean_c B_c), the spectrum minus the excess of its mean over the bandpass mean;
  R27 order: channel thresholding, spectrum thresholding, then bandpass subtraction (§3.3.1 mentions the
      subtraction first, but then "replaced with the fitted bandpass value" could not hold; by linearity the
      two orders give the same corrected spectra: replaced samples end at exactly 0).

Pins (tests/test_rfi_pins.py): numpy.polynomial's own fit and an exact polynomial recovered; hand-worked
windows and neighbour flags; closed-form spectrum statistics; the §3.3.4 test recipe (512 channels, narrowband
periodic RFI, a broadband pulse, a dispersed pulse that must survive).  Nothing here is "parity unpinned".
"""
from __future__ import annotations

import numpy as np


def bandpass_mean(X) -> np.ndarray:
    """b_c = mean over time of channel c (float64)."""
    X = np.asarray(X)
    return X.astype(np.float64).mean(axis=1) if X.shape[1] else np.zeros(X.shape[0])


def channel_abscissa(nchans) -> np.ndarray:
    """channel index mapped linearly onto [-1, 1] (R21); a single channel sits at 0."""
    if nchans == 1:
        return np.zeros(1)
    return 2.0 * np.arange(nchans, dtype=np.float64) / (nchans - 1) - 1.0


def fit_bandpass(b, order):
    """Least-squares polynomial of the given order through (x_c, b_c) -> (B fitted values, rmse)  (R21, R22)."""
    b = np.asarray(b, dtype=np.float64)
    x = channel_abscissa(len(b))
    order = min(int(order), len(b) - 1)
    V = np.vander(x, order + 1, increasing=True)              # columns 1, x, x^2, ...
    coef, *_ = np.linalg.lstsq(V, b, rcond=None)
    B = V @ coef
    return B, float(np.sqrt(np.mean((b - B) ** 2)))


def channel_flags(X, B, rmse, window, t_chan):
    """Window flags [nchans][nwin] (bool) of eq 3.1 as read in R23/R24: own-mean test, then neighbours."""
    X = np.asarray(X)
    nchans, n = X.shape
    starts = np.arange(0, n, window)
    lengths = np.minimum(window, n - starts).astype(np.float64)
    # M(c) of every partition c: sum over the window / its length (np.add.reduceat sums [start_k, start_k+1))
    M = np.add.reduceat(X.astype(np.float64), starts, axis=1) / lengths[None, :]
    own = np.abs(M - np.asarray(B, dtype=np.float64)[:, None]) > t_chan * rmse
    flags = own.copy()
    flags[:, 1:] |= own[:, :-1]
    flags[:, :-1] |= own[:, 1:]
    return flags, own


def apply_channel_flags(X, B, flags, window):
    """Flagged windows take the channel's fitted bandpass value (float64 copy of X returned)."""
    Y = np.asarray(X).astype(np.float64)
    n = Y.shape[1]
    for c, k in zip(*np.nonzero(flags)):
        Y[c, k * window:min(n, (k + 1) * window)] = B[c]
    return Y


def spectrum_stats(Y):
    """m_t = mean over channels of spectrum t; mu, sigma = mean and population std of m over time (R25)."""
    m = np.asarray(Y, dtype=np.float64).mean(axis=0)
    return m, float(m.mean()), float(np.sqrt(np.mean((m - m.mean()) ** 2)))


def apply_spectrum_threshold(Y, B, t_spec):
    """Spectra whose mean exceeds mu + T_s sigma lose the excess of their mean over the bandpass mean (R25, R26)."""
    Y = np.asarray(Y, dtype=np.float64).copy()
    m, mu, sigma = spectrum_stats(Y)
    flagged = (m - mu) > t_spec * sigma
    Y[:, flagged] -= (m[flagged] - np.mean(B))[None, :]
    return Y, flagged, (mu, sigma)


def mitigate(X, order=4, window=512, t_chan=7.0, t_spec=5.0):
    """The whole of §3.3 on one buffer X [nchans][nsamp] (float32) -> dict with the corrected spectra (float64)
    and every intermediate (bandpass, fit, rmse, flags, spectrum statistics)."""
    X = np.asarray(X)
    b = bandpass_mean(X)
    B, rmse = fit_bandpass(b, order)
    flags, own = channel_flags(X, B, rmse, window, t_chan)
    Y = apply_channel_flags(X, B, flags, window)
    Y, sflag, (mu, sigma) = apply_spectrum_threshold(Y, B, t_spec)
    Y -= B[:, None]                                            # bandpass correction (R27)
    return {"out": Y, "bandpass": b, "fit": B, "rmse": rmse, "chan_flags": flags, "chan_own": own,
            "spec_flags": sflag, "spec_mu": mu, "spec_sigma": sigma}
