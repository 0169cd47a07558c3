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


def assert_row_checksums(w, X, D_gpu, table):
    """P7: sum_t D[d][t] = sum_c (P_c[nsamp + s(d,c)] - P_c[s(d,c)]) for EVERY trial d, with
    P_c the prefix sum of channel row c.  `table` is the ORACLE's delay table."""
    nch = w.nchans
    if w.dtype == "u8":
        P = np.zeros((nch, X.shape[1] + 1), dtype=np.int64)
        np.cumsum(X, axis=1, dtype=np.int64, out=P[:, 1:])
        want = np.zeros(len(table), dtype=np.int64)
        for c in range(nch):
            want += P[c, w.nsamp + table[:, c]] - P[c, table[:, c]]
        got = D_gpu.sum(axis=1, dtype=np.int64)
        assert np.array_equal(got, want)
    else:
        P = np.zeros((nch, X.shape[1] + 1), dtype=np.float64)
        np.cumsum(X, axis=1, dtype=np.float64, out=P[:, 1:])
        PA = np.zeros((nch, X.shape[1] + 1), dtype=np.float64)
        np.cumsum(np.abs(X), axis=1, dtype=np.float64, out=PA[:, 1:])
        want = np.zeros(len(table)); scale = np.zeros(len(table))
        for c in range(nch):
            want += P[c, w.nsamp + table[:, c]] - P[c, table[:, c]]
            scale += PA[c, w.nsamp + table[:, c]] - PA[c, table[:, c]]
        got = D_gpu.sum(axis=1, dtype=np.float64)
        assert np.all(np.abs(got - want) <= F32_RTOL * scale + 1e-6 * np.abs(want))
