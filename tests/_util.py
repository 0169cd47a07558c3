"""Helpers shared by the GPU parity tests (not collected by pytest)."""
import numpy as np

import oracle
import paper_1401_8258_b200 as dd
from paper_1401_8258_b200 import synth

F32_RTOL = 1e-5      # north_star: |D_gpu - D_oracle| <= 1e-5 * sum_c |X[c][t+s]| per element


def dd_dtype(w):
    return dd.DD_F32 if w.dtype == "f32" else dd.DD_U8


def small(idx, nchans, ndm, nsamp, **kw):
    """Workload `idx` shrunk to CPU-oracle size, keeping its band (foff rescaled) and DM step."""
    w = synth.WORKLOADS[idx]
    return synth.scaled(w, nchans=nchans, ndm=ndm, nsamp=nsamp, nbeams=kw.pop("nbeams", 1),
                        foff=w.foff * w.nchans / nchans, **kw)


def make_case(w, pulses=0, beam=0):
    """Host input of one beam: noise (+ optional injected pulses at trial DMs, delays from the oracle)."""
    ms = oracle.max_shift(w.nchans, w.fch1, w.foff, w.tsamp, w.dm_list)
    X = synth.make_input(w, w.nsamp + ms, beam=beam)
    if pulses:
        tab = oracle.shift_table(w.nchans, w.fch1, w.foff, w.tsamp, w.dm_list)
        for d, t0, width in synth.pulse_plan(w, pulses):
            synth.inject_pulse(X, t0, width, 3.0 if w.dtype == "f32" else 40, tab[d])
    return X, ms


def gpu_dedisperse(w, X, kernel=None, dms=None):
    """One beam through Plan.execute; returns D as numpy ([ndm][nsamp])."""
    import torch
    dms = w.dm_list if dms is None else dms
    plan = dd.Plan(dd_dtype(w), w.nchans, w.fch1, w.foff, w.tsamp, dms)
    if kernel is not None:
        plan.set_kernel(kernel)
    Xd = torch.from_numpy(X).cuda()
    Dd = torch.empty((len(dms), w.nsamp), dtype=torch.float32 if w.dtype == "f32" else torch.int32,
                     device="cuda")
    Dd.fill_(-7)
    plan.execute(Xd, X.shape[1], 0, Dd, w.nsamp, 0, w.nsamp, 1)
    torch.cuda.synchronize()
    out = Dd.cpu().numpy()
    plan.destroy()
    return out


def assert_parity(w, X, D_gpu, dms=None, rows=None):
    """Element-by-element comparison with the oracle (bit-exact for u8, 1e-5*sum|X| for f32)."""
    dms = w.dm_list if dms is None else dms
    if w.dtype == "u8":
        want = oracle.dedisperse_u8(X, w.nsamp, w.fch1, w.foff, w.tsamp, dms, rows=rows)
        got = D_gpu if rows is None else D_gpu[rows]
        assert got.dtype == np.int32
        assert np.array_equal(got.astype(np.int64), want), \
            "u8->i32 mismatch at %s" % (np.argwhere(got != want)[:5].tolist(),)
    else:
        want, A = oracle.dedisperse_f32(X, w.nsamp, w.fch1, w.foff, w.tsamp, dms, rows=rows)
        got = D_gpu if rows is None else D_gpu[rows]
        assert got.dtype == np.float32
        err = np.abs(got.astype(np.float64) - want)
        bad = err > F32_RTOL * A
        assert not bad.any(), "f32 mismatch: worst err/(1e-5*A) = %g at %s" % (
            (err / (F32_RTOL * A + 1e-300)).max(), np.argwhere(bad)[:5].tolist())


def assert_sampled_parity(w, X, D_gpu, n=200000, seed=0):
    g = np.random.default_rng(seed)
    di = g.integers(0, D_gpu.shape[0], n)
    ti = g.integers(0, w.nsamp, n)
    # always include the corners and the tile seams of both kernels
    di[:4] = [0, 0, D_gpu.shape[0] - 1, D_gpu.shape[0] - 1]
    ti[:4] = [0, w.nsamp - 1, 0, w.nsamp - 1]
    if w.dtype == "u8":
        want = oracle.elements(X, w.fch1, w.foff, w.tsamp, w.dm_list, di, ti)
        assert np.array_equal(D_gpu[di, ti].astype(np.int64), want)
    else:
        want, A = oracle.elements(X, w.fch1, w.foff, w.tsamp, w.dm_list, di, ti)
        err = np.abs(D_gpu[di, ti].astype(np.float64) - want)
        assert np.all(err <= F32_RTOL * A), (err / (F32_RTOL * A)).max()


def row_checksums(w, X, table):
    """P7: sum_t D[d][t] = sum_c (P_c[nsamp + s(d,c)] - P_c[s(d,c)]) for EVERY trial d, with
    P_c the prefix sum of channel row c -- O(nchans * (ndm + nsamp)), one channel in memory at a time.
    `table` is the ORACLE's delay table.  Returns (want, scale): exact int64 sums for uint8; for float32
    double sums and sum_t of the per-element tolerance scale sum_c |X|."""
    table = np.asarray(table)
    n = w.nsamp
    if w.dtype == "u8":
        want = np.zeros(len(table), dtype=np.int64)
        p = np.zeros(X.shape[1] + 1, dtype=np.int64)
        for c in range(w.nchans):
            np.cumsum(X[c], dtype=np.int64, out=p[1:])
            want += p[n + table[:, c]] - p[table[:, c]]
        return want, None
    want = np.zeros(len(table))
    scale = np.zeros(len(table))
    p = np.zeros(X.shape[1] + 1, dtype=np.float64)
    for c in range(w.nchans):
        np.cumsum(X[c], dtype=np.float64, out=p[1:])
        want += p[n + table[:, c]] - p[table[:, c]]
        np.cumsum(np.abs(X[c]), dtype=np.float64, out=p[1:])
        scale += p[n + table[:, c]] - p[table[:, c]]
    return want, scale


def assert_row_checksums(w, X, D_gpu, table):
    """P7 on a result held as numpy ([ndm][nsamp]) or as a torch tensor on the device (the row sums are
    then formed there in int64 / float64 -- a reduction by the checker, not by the product)."""
    want, scale = row_checksums(w, X, table)
    if isinstance(D_gpu, np.ndarray):
        got = D_gpu.sum(axis=1, dtype=np.int64 if w.dtype == "u8" else np.float64)
    else:
        import torch
        got = D_gpu.sum(dim=1, dtype=torch.int64 if w.dtype == "u8" else torch.float64).cpu().numpy()
    if w.dtype == "u8":
        assert np.array_equal(got, want), np.argwhere(got != want)[:5].tolist()
    else:
        # sum of the per-element tolerances, plus the rounding of the prefix-sum differences themselves
        tol = F32_RTOL * scale + 1e-9 * scale
        bad = np.abs(got - want) > tol
        assert not bad.any(), (np.argwhere(bad)[:5].tolist(), (np.abs(got - want) / tol).max())


def assert_whole_rows(w, X, D_rows_gpu, rows, dms=None):
    """P8: whole oracle rows (all nsamp samples) for the trials in `rows`; D_rows_gpu[i] is the product's
    row for trial rows[i] (numpy).  The oracle runs its interchanged nest (pinned bit-identical to the
    literal one in tests/test_oracle_pins.py)."""
    dms = w.dm_list if dms is None else dms
    rows = np.asarray(rows, dtype=np.int32)
    if w.dtype == "u8":
        want = oracle.dedisperse_u8(X, w.nsamp, w.fch1, w.foff, w.tsamp, dms, rows=rows, interchanged=True)
        assert np.array_equal(D_rows_gpu.astype(np.int64), want), np.argwhere(D_rows_gpu != want)[:5].tolist()
        return 0.0
    want, A = oracle.dedisperse_f32(X, w.nsamp, w.fch1, w.foff, w.tsamp, dms, rows=rows, interchanged=True)
    err = np.abs(D_rows_gpu.astype(np.float64) - want)
    worst = float((err / (F32_RTOL * A + 1e-300)).max())
    assert worst <= 1.0, "f32 mismatch: worst err/(1e-5*A) = %g at %s" % (worst, np.argwhere(err > F32_RTOL * A)[:5].tolist())
    return worst


def p8_rows(w, pulses=()):
    """first, last, every 64th trial, the tile seams around 63/64 and 127/128, and each injected-pulse DM"""
    r = set(range(0, w.ndm, 64)) | {w.ndm - 1, 63, 127, 128} | {d for d, _, _ in pulses}
    return np.array(sorted(x for x in r if 0 <= x < w.ndm), dtype=np.int32)
