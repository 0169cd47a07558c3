"""Pins for the oracle (CPU only).  Each test anchors oracle/ to something other
than itself: the paper's printed values (tests/golden/), exact rational
arithmetic, closed forms, special cases, or a literal brute force written
separately here in Python.  A plausible mistake in the oracle (dropped term,
wrong sign, t-s instead of t+s, transposed layout, wrong reference frequency)
fails at least one of them.
"""
import math
from fractions import Fraction

import numpy as np
import pytest

import oracle
from paper_1401_8258_b200 import synth


# ---------------------------------------------------------------- delay formula

def exact_shift(dm, c, fch1, foff, tsamp, const="4148.808"):
    """eq 2.2/2.3 in exact rational arithmetic on the decimal/binary inputs."""
    dm, fch1, foff, tsamp = (Fraction(v) for v in (dm, fch1, foff, tsamp))
    fc = fch1 + c * foff
    x = Fraction(const) * dm * (1 / (fc * fc) - 1 / (fch1 * fch1)) / tsamp
    return math.floor(x + Fraction(1, 2))


def test_constant_and_units_eq_1_14(paper_values):
    # eq 1.12/1.14: delay w.r.t. infinite frequency = D * DM / f^2,
    # D = 4.148808e3 MHz^2 pc^-1 cm^3 s  =>  DM=1 at 1000 MHz is 4.148808 ms.
    k = paper_values["dispersion_constant"]
    big = 1.0e12                        # "infinite" reference frequency, MHz
    foff = 1000.0 - big                 # channel 1 sits at 1000 MHz
    assert oracle.shift(1.0, 1, big, foff, 1e-6) == round(k)            # 4149 us
    assert oracle.shift(1.0, 1, big, foff, 1e-9) == round(k * 1000)     # 4148808 ns
    assert oracle.shift(10.0, 1, big, foff, 1e-6) == round(10 * k)      # linear in DM
    # f^-2 law: at 500 MHz the delay is 4x
    assert oracle.shift(1.0, 1, big, 500.0 - big, 1e-6) == round(4 * k)


def test_units_cross_check_eq_6_2(paper_values):
    # eq 6.2: DM_max = dt f0^3 / (8300 df) is the DM at which the delay
    # across ONE channel is ONE sample; Table 6.7 prints 827 for 50 us / 1400 MHz / 20 kHz.
    dt, f0, df = (paper_values[k] for k in ("dm_max_dt_s", "dm_max_f0_mhz", "dm_max_df_mhz"))
    dm_max = dt * f0 ** 3 / (8300.0 * df)
    assert round(dm_max) == paper_values["dm_max_table_6_7"]
    # two channels: fch1 = f0 + df (top), channel 1 = f0.  Delay ~ 1 sample at DM_max.
    assert oracle.shift(dm_max, 1, f0 + df, -df, dt) == 1
    assert oracle.shift(0.45 * dm_max, 1, f0 + df, -df, dt) == 0
    assert oracle.shift(1.55 * dm_max, 1, f0 + df, -df, dt) == 2
    assert oracle.shift(10.0 * dm_max, 1, f0 + df, -df, dt) == 10


def test_tiny_table_by_hand():
    # nchans=5 fch1=420 foff=-2 tsamp=1e-3 DM={0,3,6,9}: values checked in exact arithmetic
    tab = oracle.shift_table(5, 420.0, -2.0, 1e-3, [0.0, 3.0, 6.0, 9.0])
    want = [[exact_shift(dm, c, 420, -2, Fraction(1, 1000)) for c in range(5)] for dm in (0, 3, 6, 9)]
    assert tab.tolist() == want
    assert want == [[0, 0, 0, 0, 0], [0, 1, 1, 2, 3], [0, 1, 3, 4, 6], [0, 2, 4, 6, 8]]


@pytest.mark.parametrize("idx", [1, 2, 3, 4, 5])
def test_workload_tables_vs_exact_and_longdouble(idx):
    w = synth.WORKLOADS[idx]
    dms = w.dm_list
    tab = oracle.shift_table(w.nchans, w.fch1, w.foff, w.tsamp, dms)
    # (a) whole table against numpy longdouble (80-bit) evaluation
    ld = np.longdouble
    fc = ld(w.fch1) + np.arange(w.nchans, dtype=ld) * ld(w.foff)
    geo = (1 / (fc * fc) - 1 / (ld(w.fch1) * ld(w.fch1))) / ld(w.tsamp) * ld(4148.808)
    x = dms.astype(ld)[:, None] * geo[None, :]
    want = np.floor(x + ld(0.5)).astype(np.int64)
    assert np.array_equal(tab, want)
    # (b) sampled entries against exact rational arithmetic
    g = np.random.default_rng(idx)
    for d, c in zip(g.integers(0, w.ndm, 300), g.integers(0, w.nchans, 300)):
        assert tab[d, c] == exact_shift(float(dms[d]), int(c), w.fch1, w.foff, w.tsamp)
    # (c) invariants: reference channel has zero delay; monotone in DM and in c (1/f^2)
    assert np.all(tab[:, 0] == 0) and np.all(tab[0, :] == 0)
    assert np.all(np.diff(tab, axis=0) >= 0) and np.all(np.diff(tab, axis=1) >= 0)
    assert oracle.max_shift(w.nchans, w.fch1, w.foff, w.tsamp, dms) == tab[-1, -1] == tab.max()


def test_maxshift_values_of_the_survey_table():
    # maxshift of the five workloads (reproduced above in exact arithmetic)
    want = {1: 579, 2: 4883, 3: 14845, 4: 9760, 5: 37599}
    for i, m in want.items():
        w = synth.WORKLOADS[i]
        assert oracle.max_shift(w.nchans, w.fch1, w.foff, w.tsamp, w.dm_list) == m
        assert exact_shift(float(w.dm_list[-1]), w.nchans - 1, w.fch1, w.foff, w.tsamp) == m


# ---------------------------------------------------------------- the sum itself

def brute(X, nsamp, fch1, foff, tsamp, dms):
    """Literal eq 2.1 in pure Python: shift recomputed inline, exact Fractions for ints,
    math.fsum for floats."""
    nchans = X.shape[0]
    D = np.zeros((len(dms), nsamp), dtype=np.float64)
    for d, dm in enumerate(dms):
        for t in range(nsamp):
            vals = []
            for c in range(nchans):
                fc = fch1 + c * foff
                s = math.floor(4148.808 * dm * (1.0 / (fc * fc) - 1.0 / (fch1 * fch1)) / tsamp + 0.5)
                vals.append(float(X[c, t + s]))
            D[d, t] = math.fsum(vals)
    return D


@pytest.mark.parametrize("nchans,ndm,nsamp", [(1, 3, 17), (3, 4, 33), (8, 8, 64), (7, 5, 50)])
def test_brute_force_tiny(nchans, ndm, nsamp):
    fch1, foff, tsamp = 400.0, -3.0, 2e-4
    dms = np.linspace(0.0, 7.5, ndm)
    ms = oracle.max_shift(nchans, fch1, foff, tsamp, dms)
    g = np.random.default_rng(nchans * 100 + ndm)
    Xf = g.standard_normal((nchans, nsamp + ms)).astype(np.float32)
    Xu = g.integers(0, 256, (nchans, nsamp + ms), dtype=np.uint8)
    D, A = oracle.dedisperse_f32(Xf, nsamp, fch1, foff, tsamp, dms)
    want = brute(Xf, nsamp, fch1, foff, tsamp, dms)
    assert np.allclose(D, want, rtol=0, atol=1e-12)
    assert np.allclose(A, brute(np.abs(Xf), nsamp, fch1, foff, tsamp, dms), rtol=0, atol=1e-12)
    Du = oracle.dedisperse_u8(Xu, nsamp, fch1, foff, tsamp, dms)
    assert np.array_equal(Du, brute(Xu, nsamp, fch1, foff, tsamp, dms).astype(np.int64))
    # rows subset and sampled elements agree with the full pass
    rows = [ndm - 1, 0]
    Dr, _ = oracle.dedisperse_f32(Xf, nsamp, fch1, foff, tsamp, dms, rows=rows)
    assert np.array_equal(Dr, D[rows])
    di = g.integers(0, ndm, 40)
    ti = g.integers(0, nsamp, 40)
    De, Ae = oracle.elements(Xf, fch1, foff, tsamp, dms, di, ti)
    assert np.array_equal(De, D[di, ti]) and np.array_equal(Ae, A[di, ti])
    assert np.array_equal(oracle.elements(Xu, fch1, foff, tsamp, dms, di, ti), Du[di, ti])


def _small(idx, nchans=48, ndm=12, nsamp=700):
    w = synth.WORKLOADS[idx]
    return synth.scaled(w, nchans=nchans, ndm=ndm, nsamp=nsamp, nbeams=1,
                        foff=w.foff * w.nchans / nchans)


def test_dm0_row_is_channel_sum_and_nchans1_identity():
    w = _small(2)
    ms = oracle.max_shift(w.nchans, w.fch1, w.foff, w.tsamp, w.dm_list)
    X = synth.make_input(w, w.nsamp + ms)
    D = oracle.dedisperse_u8(X, w.nsamp, w.fch1, w.foff, w.tsamp, w.dm_list)
    assert np.array_equal(D[0], X[:, :w.nsamp].astype(np.int64).sum(axis=0))       # DM = 0
    X1 = X[:1].copy()
    D1 = oracle.dedisperse_u8(X1, w.nsamp, w.fch1, w.foff, w.tsamp, w.dm_list)
    assert np.array_equal(D1, np.broadcast_to(X1[0, :w.nsamp].astype(np.int64), D1.shape))
    # all-equal input: every output = nchans * value (no overflow, no dropped channel)
    X255 = np.full_like(X, 255)
    assert np.all(oracle.dedisperse_u8(X255, w.nsamp, w.fch1, w.foff, w.tsamp, w.dm_list) == 255 * w.nchans)


def test_impulse_response_fixes_gather_direction():
    # X = delta at (c0, u0)  =>  D[d][u0 - s(d,c0)] = 1, all else 0   (t + s, not t - s)
    w = _small(1, nchans=16, ndm=8, nsamp=400)
    dms = w.dm_list * 3.0
    tab = np.array([[exact_shift(float(dm), c, w.fch1, w.foff, w.tsamp) for c in range(w.nchans)]
                    for dm in dms])
    ms = int(tab.max())
    assert ms > 20
    c0, u0 = 11, 330
    assert 0 < tab[-1, c0] < u0          # every impulse lands inside the output range
    X = np.zeros((w.nchans, w.nsamp + ms), dtype=np.float32)
    X[c0, u0] = 1.0
    D, A = oracle.dedisperse_f32(X, w.nsamp, w.fch1, w.foff, w.tsamp, dms)
    want = np.zeros_like(D)
    for d in range(len(dms)):
        want[d, u0 - tab[d, c0]] = 1.0
    assert np.array_equal(D, want) and np.array_equal(A, want)


def test_linearity_and_time_shift_covariance():
    w = _small(2, nchans=32, ndm=9, nsamp=300)
    ms = oracle.max_shift(w.nchans, w.fch1, w.foff, w.tsamp, w.dm_list)
    g = np.random.default_rng(7)
    X1 = g.integers(0, 128, (w.nchans, w.nsamp + ms + 5), dtype=np.uint8)
    X2 = g.integers(0, 128, (w.nchans, w.nsamp + ms + 5), dtype=np.uint8)
    f = lambda X: oracle.dedisperse_u8(np.ascontiguousarray(X), w.nsamp, w.fch1, w.foff, w.tsamp, w.dm_list)
    assert np.array_equal(f(X1 + X2), f(X1) + f(X2))
    tau = 5
    Xs = np.zeros_like(X1)
    Xs[:, :-tau] = X1[:, tau:]
    assert np.array_equal(f(Xs)[:, :w.nsamp - tau], f(X1)[:, tau:w.nsamp])


def test_injected_pulse_snr_fig_2_6(paper_values):
    # top-hat of height 8/sqrt(1024) = 0.25 in N(0,1), 1024 channels -> S/N 8
    # at the true DM.  Here: config-1 shape scaled to 1024 channels, pulse at trial DM = 10.
    nch = int(paper_values["fig_2_6_nchans"])
    amp = paper_values["fig_2_6_amp"]
    w = synth.scaled(synth.WORKLOADS[1], nchans=nch, foff=-16.0 / nch, ndm=21, nsamp=2048)
    dms = w.dm_list
    tab = oracle.shift_table(w.nchans, w.fch1, w.foff, w.tsamp, dms)
    X = synth.make_input(w, w.nsamp + int(tab.max()))
    t0s = [300, 700, 1100, 1500, 1900]
    for t0 in t0s:
        synth.inject_pulse(X, t0, 1, amp, tab[10])
    D, _ = oracle.dedisperse_f32(X, w.nsamp, w.fch1, w.foff, w.tsamp, dms)
    sigma = math.sqrt(nch)                              # noise std of a sum of nch N(0,1)
    snr = D[10, t0s] / sigma
    assert abs(snr.mean() - paper_values["fig_2_6_snr"]) < 1.5      # 8 +- 1/sqrt(5)*3
    # the pulse peaks at the true trial: its S/N there beats every other trial at that time
    for t0 in t0s:
        col = D[:, t0] / sigma
        assert col.argmax() == 10
    # config 1 as stated: amplitude 3, 64 channels -> peak ~ 3*64 = 192 = 24 sigma at trial 10
    w1 = synth.WORKLOADS[1]
    tab1 = oracle.shift_table(w1.nchans, w1.fch1, w1.foff, w1.tsamp, w1.dm_list)
    X1 = synth.make_input(w1, w1.nsamp + int(tab1.max()))
    synth.inject_pulse(X1, 4000, 1, 3.0, tab1[10])
    D1, _ = oracle.dedisperse_f32(X1, w1.nsamp, w1.fch1, w1.foff, w1.tsamp, w1.dm_list)
    d, t = np.unravel_index(D1.argmax(), D1.shape)
    assert (d, t) == (10, 4000)
    assert abs(D1[10, 4000] / 8.0 - 24.0) < 4.0


def test_prefix_sum_row_checksum_identity():
    # sum_t D[d][t] = sum_c (P_c[nsamp + s] - P_c[s])  — independent O(nchans*(ndm+nsamp)) check
    w = _small(5, nchans=40, ndm=16, nsamp=900)
    tab = oracle.shift_table(w.nchans, w.fch1, w.foff, w.tsamp, w.dm_list)
    X = synth.make_input(w, w.nsamp + int(tab.max()))
    D = oracle.dedisperse_u8(X, w.nsamp, w.fch1, w.foff, w.tsamp, w.dm_list)
    P = np.concatenate([np.zeros((w.nchans, 1), np.int64), np.cumsum(X.astype(np.int64), axis=1)], axis=1)
    c = np.arange(w.nchans)
    for d in range(w.ndm):
        assert D[d].sum() == (P[c, w.nsamp + tab[d]] - P[c, tab[d]]).sum()


def test_generators_are_seeded_and_shaped():
    w = synth.WORKLOADS[2]
    a = synth.noise_u8(w.seed, 8, 5000)
    b = synth.noise_u8(w.seed, 8, 5000)
    assert np.array_equal(a, b) and a.dtype == np.uint8
    assert abs(a.mean() - 128) < 1 and abs(a.std() - 16) < 1
    f = synth.noise_f32(3, 4, 20000)
    assert abs(f.mean()) < 0.05 and abs(f.std() - 1) < 0.05
    assert not np.array_equal(synth.noise_f32(3, 4, 100), synth.noise_f32(4, 4, 100))
    assert [synth.WORKLOADS[i].adds for i in (1, 2)] == [64 * 32 * 8192, 1024 * 1024 * (1 << 17)]


# ---------------------------------------------------------------- the interchanged (d, c, t) nest

def test_interchanged_nest_is_bit_identical_to_the_literal_nest():
    """oracle_dedisperse_*_dct adds the channels of every element in the same order into a double
    that starts at zero, so its output must equal the literal (d, t, c) nest BIT FOR BIT -- on
    BASELINE.json config 1 in full, on config 2 (all channels and trials, time axis cut), on a
    row subset, and on a float32 case whose sums are inexact in double only through the order."""
    # config 1, full size, D and A
    w = synth.WORKLOADS[1]
    ms = oracle.max_shift(w.nchans, w.fch1, w.foff, w.tsamp, w.dm_list)
    X = synth.make_input(w, w.nsamp + ms)
    D1, A1 = oracle.dedisperse_f32(X, w.nsamp, w.fch1, w.foff, w.tsamp, w.dm_list)
    D2, A2 = oracle.dedisperse_f32(X, w.nsamp, w.fch1, w.foff, w.tsamp, w.dm_list, interchanged=True)
    assert np.array_equal(D1.view(np.int64), D2.view(np.int64))
    assert np.array_equal(A1.view(np.int64), A2.view(np.int64))
    # config 2: 1024 channels x 1024 trials, 3000 samples
    w = synth.scaled(synth.WORKLOADS[2], nsamp=3000)
    ms = oracle.max_shift(w.nchans, w.fch1, w.foff, w.tsamp, w.dm_list)
    X = synth.make_input(w, w.nsamp + ms)
    assert np.array_equal(oracle.dedisperse_u8(X, w.nsamp, w.fch1, w.foff, w.tsamp, w.dm_list),
                          oracle.dedisperse_u8(X, w.nsamp, w.fch1, w.foff, w.tsamp, w.dm_list, interchanged=True))
    # row subsets in arbitrary order, float32 data with a large dynamic range (order-sensitive sums)
    g = np.random.default_rng(77)
    w = synth.scaled(synth.WORKLOADS[3], nchans=300, foff=-300.0 / 300, ndm=90, nsamp=2001)
    ms = oracle.max_shift(w.nchans, w.fch1, w.foff, w.tsamp, w.dm_list)
    X = (g.standard_normal((w.nchans, w.nsamp + ms)) * 10.0 ** g.uniform(-6, 6, (w.nchans, 1))).astype(np.float32)
    rows = np.array([89, 0, 17, 17, 44], dtype=np.int32)
    D1, A1 = oracle.dedisperse_f32(X, w.nsamp, w.fch1, w.foff, w.tsamp, w.dm_list, rows=rows)
    D2, A2 = oracle.dedisperse_f32(X, w.nsamp, w.fch1, w.foff, w.tsamp, w.dm_list, rows=rows, interchanged=True)
    assert np.array_equal(D1.view(np.int64), D2.view(np.int64))
    assert np.array_equal(A1.view(np.int64), A2.view(np.int64))
    # and the interchanged nest against the separate pure-Python brute force on a tiny input
    fch1, foff, tsamp, dms = 400.0, -3.0, 2e-4, np.linspace(0.0, 7.5, 6)
    ms = oracle.max_shift(7, fch1, foff, tsamp, dms)
    Xf = g.standard_normal((7, 40 + ms)).astype(np.float32)
    D, _ = oracle.dedisperse_f32(Xf, 40, fch1, foff, tsamp, dms, interchanged=True)
    assert np.allclose(D, brute(Xf, 40, fch1, foff, tsamp, dms), rtol=0, atol=1e-12)
