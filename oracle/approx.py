"""ORACLE — test infrastructure only.  The two approximate variants of direct dedispersion the thesis
describes next to the exact method, composed step by step from the pinned dedispersion oracle
(oracle/dedisp_oracle.cpp) in float64.  Shares no code with the CUDA library.

A. Time binning (PAPER.md:736 and the "downfactor" procedure): "reduce the sampling
   interval by a factor of 2 when the DM exceeds the diagonal, and then repeat the procedure at two times
   the diagonal, four times the diagonal, and so on"; the procedure list dedisperses 0..2 DM_diag at the full
   rate, then "downfactor[s] the time series by a factor of 2 by summing adjacent samples" before
   2..4 DM_diag, and repeats.
B. Subband dedispersion (§2.1.3): step 1 applies the direct method to subbands of N'_c channels
   at a reduced set of nominal DMs (one per N'_DM trials); step 2 applies the direct method to the reduced
   filterbank formed by the subband series (N_SB = N_c / N'_c channels) at each nominal DM, for the trials
   near it.

Readings (R28-R33):
  R28 diagonal DM: the DM at which the delay across ONE channel is ONE sample at the bottom of the band
      (where the smear is largest): DM_diag = tsamp / (4148.808 (f_last^-2 - f_secondlast^-2)); callers may
      pass their own value (eq 6.2, evaluates the same condition at the band centre);
  R29 level of a trial: k = 0 for DM < 2 DM_diag, else k = floor(log2(DM / DM_diag)) (so [2,4) DM_diag -> 1,
      [4,8) -> 2, ...), capped at max_level; level k runs on the input summed over 2^k adjacent samples, with
      sampling time 2^k tsamp in the delay formula; output sample i of such a trial covers full-rate samples
      [2^k i, 2^k (i+1)); a trailing incomplete group of samples is dropped;
  R30 trial lists are non-decreasing in DM (the levels / nominal groups are then contiguous row ranges);
  R31 subbands: consecutive blocks of N'_c channels (the last may be smaller); a subband is dedispersed as a
      filterbank of its own whose reference is its first (highest) channel, delays from the same formula;
  R32 nominal DMs: consecutive groups of N'_DM trials (the last may be smaller); the nominal DM of a group is
      its middle trial, index g N'_DM + (size - 1) // 2;
  R33 step 2: the subband series at a group's nominal DM form a filterbank of N_SB channels with
      fch1' = fch1, foff' = N'_c foff (the subbands' first channels); every trial of the group is dedispersed
      from it with the direct method at its own DM.
Pins (tests/test_approx_pins.py): pure-Python literal formulas on tiny inputs; the limits in which each
variant reduces to the exact method (one subband; one channel per subband; level 0 only); constant inputs;
hand-worked downsampling; pulse recovery.  Nothing here is "parity unpinned".
"""
from __future__ import annotations

import math

import numpy as np

from . import dedisperse_f32, max_shift, shift_table

K_DM = 4148.808


# ------------------------------------------------------------------ A. time binning

def diagonal_dm(nchans, fch1, foff, tsamp) -> float:
    """R28.  One channel: no smearing across channels, the diagonal is never reached (inf)."""
    if nchans < 2 or foff == 0.0:
        return math.inf
    f1, f2 = fch1 + (nchans - 1) * foff, fch1 + (nchans - 2) * foff
    return tsamp / (K_DM * (1.0 / (f1 * f1) - 1.0 / (f2 * f2)))


def timebin_levels(dms, dm_diag, max_level) -> np.ndarray:
    """R29: level k of every trial."""
    out = np.zeros(len(dms), dtype=np.int32)
    for i, dm in enumerate(dms):
        if dm >= 2.0 * dm_diag:
            out[i] = min(max_level, int(math.floor(math.log2(dm / dm_diag))))
    return out


def downsample2(X) -> np.ndarray:
    """Sum adjacent samples; a trailing odd sample is dropped.  float64."""
    X = np.asarray(X, dtype=np.float64)
    n2 = X.shape[-1] // 2
    return X[..., 0:2 * n2:2] + X[..., 1:2 * n2:2]


def _direct_f64(X, nsamp, fch1, foff, tsamp, dms):
    """Direct dedispersion (eq 2.1) of float64 rows with the oracle's own delay table: plain numpy loops."""
    tab = shift_table(X.shape[0], fch1, foff, tsamp, dms)
    D = np.zeros((len(dms), nsamp))
    for d in range(len(dms)):
        for c in range(X.shape[0]):
            D[d] += X[c, tab[d, c]:tab[d, c] + nsamp]
    return D


def timebin_input_samples(nchans, fch1, foff, tsamp, dms, nsamp_out, dm_diag, max_level) -> int:
    """Full-rate samples per channel needed to produce nsamp_out >> k outputs for every trial of every level."""
    lv = timebin_levels(dms, dm_diag, max_level)
    need = 0
    for k in sorted(set(lv.tolist())):
        sel = [dm for dm, l in zip(dms, lv) if l == k]
        ms = max_shift(nchans, fch1, foff, tsamp * 2 ** k, sel)
        need = max(need, ((nsamp_out >> k) + ms) << k)
    return need


def timebin_dedisperse(X, nsamp_out, fch1, foff, tsamp, dms, dm_diag=None, max_level=8):
    """X float32 [nchans][>= timebin_input_samples] -> list over trials of float64 arrays (nsamp_out >> level)
    and the levels.  Also returns the same computed on |X| (scale of the float tolerance)."""
    X = np.asarray(X)
    nchans = X.shape[0]
    dm_diag = diagonal_dm(nchans, fch1, foff, tsamp) if dm_diag is None else dm_diag
    lv = timebin_levels(dms, dm_diag, max_level)
    out, scale = [None] * len(dms), [None] * len(dms)
    Xk, Ak = X.astype(np.float64), np.abs(X.astype(np.float64))
    for k in range(int(lv.max()) + 1 if len(dms) else 0):
        if k > 0:
            Xk, Ak = downsample2(Xk), downsample2(Ak)
        idx = [i for i in range(len(dms)) if lv[i] == k]
        if not idx:
            continue
        sel = [dms[i] for i in idx]
        Dk = _direct_f64(Xk, nsamp_out >> k, fch1, foff, tsamp * 2 ** k, sel)
        Sk = _direct_f64(Ak, nsamp_out >> k, fch1, foff, tsamp * 2 ** k, sel)
        for j, i in enumerate(idx):
            out[i], scale[i] = Dk[j], Sk[j]
    return out, scale, lv


# ------------------------------------------------------------------ B. subband dedispersion

def subband_layout(nchans, ndm, chans_per_subband, dms_per_nominal):
    """(list of (c0, c1) channel ranges, list of (d0, d1, nominal index) trial groups)  (R31, R32)."""
    subs = [(c0, min(nchans, c0 + chans_per_subband)) for c0 in range(0, nchans, chans_per_subband)]
    groups = []
    for d0 in range(0, ndm, dms_per_nominal):
        d1 = min(ndm, d0 + dms_per_nominal)
        groups.append((d0, d1, d0 + (d1 - d0 - 1) // 2))
    return subs, groups


def subband_max_shifts(nchans, fch1, foff, tsamp, dms, chans_per_subband, dms_per_nominal):
    """(maxshift of step 1 over all subbands at the largest nominal DM, maxshift of step 2)."""
    subs, groups = subband_layout(nchans, len(dms), chans_per_subband, dms_per_nominal)
    noms = [dms[g[2]] for g in groups]
    ms1 = max(max_shift(c1 - c0, fch1 + c0 * foff, foff, tsamp, noms) for c0, c1 in subs)
    ms2 = max_shift(len(subs), fch1, chans_per_subband * foff, tsamp, dms)
    return ms1, ms2


def subband_dedisperse(X, nsamp_out, fch1, foff, tsamp, dms, chans_per_subband, dms_per_nominal):
    """X float32 [nchans][>= nsamp_out + ms1 + ms2] -> (D float64 [ndm][nsamp_out], A same shape: the same two
    steps applied to |X|, the scale of the float tolerance)."""
    X = np.ascontiguousarray(X, dtype=np.float32)
    nchans, ndm = X.shape[0], len(dms)
    subs, groups = subband_layout(nchans, ndm, chans_per_subband, dms_per_nominal)
    ms1, ms2 = subband_max_shifts(nchans, fch1, foff, tsamp, dms, chans_per_subband, dms_per_nominal)
    n1 = nsamp_out + ms2
    assert X.shape[1] >= n1 + ms1
    noms = np.array([dms[g[2]] for g in groups], dtype=np.float64)
    # step 1: every subband, as a filterbank of its own, at every nominal DM (the pinned C++ oracle)
    S = np.zeros((len(subs), len(groups), n1))
    SA = np.zeros_like(S)
    for sb, (c0, c1) in enumerate(subs):
        S[sb], SA[sb] = dedisperse_f32(np.ascontiguousarray(X[c0:c1]), n1, fch1 + c0 * foff, foff, tsamp, noms,
                                       interchanged=True)
    # step 2: the reduced filterbank of each nominal DM, at the DMs of its group
    D = np.zeros((ndm, nsamp_out))
    A = np.zeros_like(D)
    for g, (d0, d1, _) in enumerate(groups):
        D[d0:d1] = _direct_f64(S[:, g, :], nsamp_out, fch1, chans_per_subband * foff, tsamp, dms[d0:d1])
        A[d0:d1] = _direct_f64(SA[:, g, :], nsamp_out, fch1, chans_per_subband * foff, tsamp, dms[d0:d1])
    return D, A
