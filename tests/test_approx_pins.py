"""Pins for the oracle of the approximate variants (oracle/approx.py: time binning PAPER.md:736, 813-819;
subband dedispersion PAPER.md:823), CPU only: pure-Python literal formulas on tiny inputs, the limits in
which each variant reduces to the exact (pinned) direct method, constant inputs, hand-worked values, and
pulse recovery."""
import math

import numpy as np

import oracle
from oracle import approx
from paper_1401_8258_b200 import synth


def lit_shift(dm, c, fch1, foff, tsamp):
    fc = fch1 + c * foff
    return math.floor(4148.808 * dm * (1.0 / (fc * fc) - 1.0 / (fch1 * fch1)) / tsamp + 0.5)


# ------------------------------------------------------------------ time binning

def test_diagonal_dm_and_levels():
    # eq 6.2: DM_max = dt f0^3 / (8300 df) is the same unit-gradient condition in its
    # small-bandwidth form; at the bottom of a narrow band the two agree to a fraction of a per cent
    nch, fch1, foff, ts = 1024, 1400.0 + 10.24, -0.02, 50e-6
    fbot = fch1 + (nch - 1.5) * foff
    assert abs(approx.diagonal_dm(nch, fch1, foff, ts) / (ts * fbot ** 3 / (2 * 4148.808 * 0.02)) - 1.0) < 1e-3
    dd_ = approx.diagonal_dm(nch, fch1, foff, ts)
    # by definition: at DM_diag the last channel lags its neighbour by exactly one sample
    x = 4148.808 * dd_ * (1 / (fch1 + (nch - 1) * foff) ** 2 - 1 / (fch1 + (nch - 2) * foff) ** 2) / ts
    assert abs(x - 1.0) < 1e-12
    assert approx.diagonal_dm(1, 400.0, -1.0, 1e-3) == math.inf
    lv = approx.timebin_levels([0, 1.0, 1.99, 2.0, 3.99, 4.0, 7.9, 8.0, 100.0], 1.0, 3)
    assert lv.tolist() == [0, 0, 0, 1, 1, 2, 2, 3, 3]                                  # R29, capped at 3


def test_downsample_by_hand_and_constant_input():
    assert approx.downsample2([1, 2, 3, 4, 5]).tolist() == [3, 7]                       # odd tail dropped
    assert approx.downsample2([[1, 1, 1, 1], [0, 2, 4, 6]]).tolist() == [[2, 2], [2, 10]]
    # constant input: a level-k output sample is nchans * 2^k * const whatever the delays
    nch, fch1, foff, ts = 16, 400.0, -0.5, 1e-3
    dms = np.array([0.0, 5.0, 30.0, 61.0, 130.0])
    dg = 15.0
    n_in = approx.timebin_input_samples(nch, fch1, foff, ts, dms, 64, dg, 4)
    X = np.full((nch, n_in), 0.5, dtype=np.float32)
    out, scale, lv = approx.timebin_dedisperse(X, 64, fch1, foff, ts, dms, dm_diag=dg, max_level=4)
    assert lv.tolist() == [0, 0, 1, 2, 3]
    for o, k in zip(out, lv):
        assert len(o) == 64 >> k and np.all(o == nch * 2 ** k * 0.5)


def test_timebin_literal_formula_and_level0_is_exact():
    g = np.random.default_rng(4)
    nch, fch1, foff, ts = 6, 300.0, -2.0, 2e-3
    dms = np.array([0.0, 3.0, 9.0, 20.0, 45.0])
    dg = 4.0
    nout = 32
    n_in = approx.timebin_input_samples(nch, fch1, foff, ts, dms, nout, dg, 3)
    X = g.standard_normal((nch, n_in)).astype(np.float32)
    out, scale, lv = approx.timebin_dedisperse(X, nout, fch1, foff, ts, dms, dm_diag=dg, max_level=3)
    assert lv.tolist() == [0, 0, 1, 2, 3]
    for i, dm in enumerate(dms):
        k = int(lv[i])
        for t in range(nout >> k):
            # literal: sum over channels of the 2^k full-rate samples of binned sample t + s_k(d,c)
            want = 0.0
            for c in range(nch):
                s = lit_shift(dm, c, fch1, foff, ts * 2 ** k)
                want += math.fsum(float(v) for v in X[c, (t + s) << k:(t + s + 1) << k])
            assert abs(out[i][t] - want) < 1e-12
    # trials below 2 DM_diag are the exact direct method
    exact, _ = oracle.dedisperse_f32(X, nout, fch1, foff, ts, dms[:2])
    assert np.array_equal(np.stack(out[:2]), exact)


# ------------------------------------------------------------------ subband dedispersion

def test_subband_limits_reduce_to_the_exact_method():
    w = synth.scaled(synth.WORKLOADS[3], nchans=48, foff=-300.0 / 48, ndm=20, nsamp=400)
    dms = w.dm_list
    ms1, ms2 = approx.subband_max_shifts(w.nchans, w.fch1, w.foff, w.tsamp, dms, 48, 1)
    X = synth.make_input(w, w.nsamp + ms1 + ms2 + 8)
    exact, A = oracle.dedisperse_f32(X, w.nsamp, w.fch1, w.foff, w.tsamp, dms)
    # one subband holding the whole band, every trial its own nominal DM: step 1 IS the direct method
    D, SA = approx.subband_dedisperse(X, w.nsamp, w.fch1, w.foff, w.tsamp, dms, 48, 1)
    assert np.array_equal(D, exact) and np.array_equal(SA, A)
    # one channel per subband: step 1 is the identity, step 2 the direct method at every trial's own DM
    D, SA = approx.subband_dedisperse(X, w.nsamp, w.fch1, w.foff, w.tsamp, dms, 1, 7)
    assert np.array_equal(D, exact) and np.array_equal(SA, A)
    # DM = 0 is exact in any configuration whose nominal DM is 0 too
    D, _ = approx.subband_dedisperse(X, w.nsamp, w.fch1, w.foff, w.tsamp, dms, 8, 1)
    assert np.array_equal(D[0], exact[0])


def test_subband_literal_formula():
    g = np.random.default_rng(6)
    nch, fch1, foff, ts = 10, 350.0, -1.5, 1e-3
    dms = np.linspace(0.0, 40.0, 9)
    ncs, nds, nout = 4, 3, 24
    subs, groups = approx.subband_layout(nch, len(dms), ncs, nds)
    assert subs == [(0, 4), (4, 8), (8, 10)] and groups == [(0, 3, 1), (3, 6, 4), (6, 9, 7)]      # R31, R32
    ms1, ms2 = approx.subband_max_shifts(nch, fch1, foff, ts, dms, ncs, nds)
    X = g.standard_normal((nch, nout + ms1 + ms2)).astype(np.float32)
    D, A = approx.subband_dedisperse(X, nout, fch1, foff, ts, dms, ncs, nds)
    for d, dm in enumerate(dms):
        nom = dms[groups[d // nds][2]]
        for t in range(nout):
            want = 0.0
            for c0, c1 in subs:
                s2 = lit_shift(dm, c0, fch1, foff, ts)                         # subband's first channel, trial's DM
                for c in range(c0, c1):
                    s1 = lit_shift(nom, c - c0, fch1 + c0 * foff, foff, ts)    # inside the subband, nominal DM
                    want += float(X[c, t + s2 + s1])
            assert abs(D[d, t] - want) < 1e-12


def test_subband_recovers_a_pulse_near_its_dm():
    # a pulse dispersed at a nominal DM keeps (almost) all of its S/N; the delays differ from the exact ones
    # only through the two-stage rounding (<= 1 sample), "additional smearing" per PAPER.md:823
    w = synth.scaled(synth.WORKLOADS[2], dtype="f32", nchans=256, foff=-20.0 / 256, ndm=48, nsamp=2048, seed=77)
    dms = w.dm_list
    ms1, ms2 = approx.subband_max_shifts(w.nchans, w.fch1, w.foff, w.tsamp, dms, 16, 8)
    tab = oracle.shift_table(w.nchans, w.fch1, w.foff, w.tsamp, dms)
    X = synth.make_input(w, w.nsamp + ms1 + ms2 + 4)
    synth.inject_pulse(X, 700, 4, 1.0, tab[27])                                # trial 27 = nominal of group 3 (24..31)
    D, _ = approx.subband_dedisperse(X, w.nsamp, w.fch1, w.foff, w.tsamp, dms, 16, 8)
    exact, _ = oracle.dedisperse_f32(X, w.nsamp, w.fch1, w.foff, w.tsamp, dms)
    d, t = np.unravel_index(D.argmax(), D.shape)
    assert abs(d - 27) <= 1 and abs(t - 700) <= 4
    assert D.max() > 0.85 * exact.max() and exact.max() > 200
