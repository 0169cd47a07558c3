"""ORACLE — test infrastructure only (see dedisp_oracle.cpp header).

Thin ctypes loader around ``oracle/dedisp_oracle.cpp`` (plain C++ ``(d, t, c)``
triple loop, double accumulation; eq 2.1-2.3).  It imports
nothing from ``paper_1401_8258_b200`` and the product never imports it.

``build()`` compiles ``libdedisp_oracle.so`` next to the source with
``g++ -O2 -ffp-contract=off -fopenmp``; every accessor below builds on demand.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
import threading

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "dedisp_oracle.cpp")
_SRC_POST = os.path.join(_HERE, "postproc_oracle.cpp")
_SO = os.path.join(_HERE, "libdedisp_oracle.so")
_lock = threading.Lock()
_lib = None


def build(force: bool = False) -> str:
    """Compile the oracle shared object (no CUDA involved)."""
    with _lock:
        if (not force and os.path.exists(_SO)
                and os.path.getmtime(_SO) >= max(os.path.getmtime(_SRC), os.path.getmtime(_SRC_POST))):
            return _SO
        tmp = _SO + ".tmp.%d" % os.getpid()
        cmd = ["g++", "-O2", "-ffp-contract=off", "-fopenmp", "-shared", "-fPIC",
               "-std=c++17", "-o", tmp, _SRC, _SRC_POST]
        subprocess.run(cmd, check=True)
        os.replace(tmp, _SO)
        return _SO


def _load():
    global _lib
    if _lib is not None:
        return _lib
    lib = C.CDLL(build())
    dp = C.POINTER(C.c_double)
    ip = C.POINTER(C.c_int)
    lp = C.POINTER(C.c_int64)
    lib.oracle_shift.restype = C.c_int64
    lib.oracle_shift.argtypes = [C.c_double, C.c_int, C.c_double, C.c_double, C.c_double]
    lib.oracle_shift_table.restype = None
    lib.oracle_shift_table.argtypes = [C.c_int, C.c_double, C.c_double, C.c_double, dp, C.c_int, lp]
    lib.oracle_max_shift.restype = C.c_int64
    lib.oracle_max_shift.argtypes = [C.c_int, C.c_double, C.c_double, C.c_double, dp, C.c_int]
    lib.oracle_dedisperse_f32.restype = None
    lib.oracle_dedisperse_f32.argtypes = [C.c_void_p, C.c_int, C.c_int64, C.c_int64, C.c_double,
                                          C.c_double, C.c_double, dp, C.c_int, ip, C.c_int,
                                          dp, dp]
    lib.oracle_dedisperse_u8.restype = None
    lib.oracle_dedisperse_u8.argtypes = [C.c_void_p, C.c_int, C.c_int64, C.c_int64, C.c_double,
                                         C.c_double, C.c_double, dp, C.c_int, ip, C.c_int, lp]
    lib.oracle_dedisperse_f32_dct.restype = None
    lib.oracle_dedisperse_f32_dct.argtypes = lib.oracle_dedisperse_f32.argtypes
    lib.oracle_dedisperse_u8_dct.restype = None
    lib.oracle_dedisperse_u8_dct.argtypes = lib.oracle_dedisperse_u8.argtypes
    lib.oracle_elements_f32.restype = None
    lib.oracle_elements_f32.argtypes = [C.c_void_p, C.c_int, C.c_int64, C.c_double, C.c_double,
                                        C.c_double, dp, ip, lp, C.c_int64, dp, dp]
    lib.oracle_elements_u8.restype = None
    lib.oracle_elements_u8.argtypes = [C.c_void_p, C.c_int, C.c_int64, C.c_double, C.c_double,
                                       C.c_double, dp, ip, lp, C.c_int64, lp]
    # post-processing (postproc_oracle.cpp)
    lib.oracle_median_filter.restype = None
    lib.oracle_median_filter.argtypes = [dp, C.c_int64, C.c_int, dp]
    lib.oracle_fit_line.restype = None
    lib.oracle_fit_line.argtypes = [dp, C.c_int64, dp, dp]
    lib.oracle_detrend.restype = None
    lib.oracle_detrend.argtypes = [dp, C.c_int64, C.c_double, C.c_double, dp, dp]
    lib.oracle_normalise.restype = None
    lib.oracle_normalise.argtypes = [dp, C.c_int64, C.c_double, dp]
    lib.oracle_postprocess_rows.restype = None
    lib.oracle_postprocess_rows.argtypes = [C.c_void_p, C.c_int, C.c_int64, C.c_int64, C.c_int64, C.c_int, C.c_int,
                                            C.c_int, dp, dp]
    lib.oracle_threshold.restype = C.c_int64
    lib.oracle_threshold.argtypes = [dp, C.c_int, C.c_int, C.c_int64, C.c_double, dp, C.POINTER(C.c_int32),
                                     C.POINTER(C.c_int32), lp, dp, C.c_int64]
    _lib = lib
    return lib


def _dp(a):
    return a.ctypes.data_as(C.POINTER(C.c_double))


def _ip(a):
    return a.ctypes.data_as(C.POINTER(C.c_int))


def _lp(a):
    return a.ctypes.data_as(C.POINTER(C.c_int64))


def _dms(dm_list):
    return np.ascontiguousarray(np.asarray(dm_list, dtype=np.float64))


def shift(dm, c, fch1, foff, tsamp) -> int:
    """s(d,c) of eq 2.2/2.3."""
    return int(_load().oracle_shift(float(dm), int(c), float(fch1), float(foff), float(tsamp)))


def shift_table(nchans, fch1, foff, tsamp, dm_list) -> np.ndarray:
    """int64 [ndm][nchans] delay table."""
    dms = _dms(dm_list)
    out = np.empty((len(dms), nchans), dtype=np.int64)
    _load().oracle_shift_table(nchans, fch1, foff, tsamp, _dp(dms), len(dms), _lp(out))
    return out


def max_shift(nchans, fch1, foff, tsamp, dm_list) -> int:
    dms = _dms(dm_list)
    return int(_load().oracle_max_shift(nchans, fch1, foff, tsamp, _dp(dms), len(dms)))


def _check_X(X, dtype, nsamp, maxshift):
    X = np.asarray(X)
    assert X.dtype == dtype and X.ndim == 2 and X.flags.c_contiguous, (X.dtype, X.shape)
    assert X.shape[1] >= nsamp + maxshift, "input rows must hold nsamp + maxshift samples"
    return X


def dedisperse_f32(X, nsamp, fch1, foff, tsamp, dm_list, rows=None, interchanged=False):
    """X float32 [nchans][>= nsamp+maxshift] -> (D, A) float64 [nrows][nsamp].

    D = eq 2.1 sums in double; A = sum_c |X| (scale of the float tolerance).
    interchanged=True runs the (d, c, t) nest (bit-identical results, see dedisp_oracle.cpp).
    """
    dms = _dms(dm_list)
    nchans = X.shape[0]
    X = _check_X(X, np.float32, nsamp, max_shift(nchans, fch1, foff, tsamp, dms))
    rws = None if rows is None else np.ascontiguousarray(np.asarray(rows, dtype=np.int32))
    nr = len(dms) if rws is None else len(rws)
    D = np.empty((nr, nsamp), dtype=np.float64)
    A = np.empty((nr, nsamp), dtype=np.float64)
    f = _load().oracle_dedisperse_f32_dct if interchanged else _load().oracle_dedisperse_f32
    f(X.ctypes.data, nchans, nsamp, X.shape[1], fch1, foff, tsamp,
      _dp(dms), len(dms), None if rws is None else _ip(rws), nr, _dp(D), _dp(A))
    return D, A


def dedisperse_u8(X, nsamp, fch1, foff, tsamp, dm_list, rows=None, interchanged=False):
    """X uint8 [nchans][>= nsamp+maxshift] -> D int64 [nrows][nsamp] (exact)."""
    dms = _dms(dm_list)
    nchans = X.shape[0]
    X = _check_X(X, np.uint8, nsamp, max_shift(nchans, fch1, foff, tsamp, dms))
    rws = None if rows is None else np.ascontiguousarray(np.asarray(rows, dtype=np.int32))
    nr = len(dms) if rws is None else len(rws)
    D = np.empty((nr, nsamp), dtype=np.int64)
    f = _load().oracle_dedisperse_u8_dct if interchanged else _load().oracle_dedisperse_u8
    f(X.ctypes.data, nchans, nsamp, X.shape[1], fch1, foff, tsamp,
      _dp(dms), len(dms), None if rws is None else _ip(rws), nr, _lp(D))
    return D


def elements(X, fch1, foff, tsamp, dm_list, d_idx, t_idx):
    """Sampled outputs D[d_idx[i]][t_idx[i]]; returns (D, A) for f32, D for u8."""
    dms = _dms(dm_list)
    X = np.asarray(X)
    assert X.ndim == 2 and X.flags.c_contiguous
    d_idx = np.ascontiguousarray(np.asarray(d_idx, dtype=np.int32))
    t_idx = np.ascontiguousarray(np.asarray(t_idx, dtype=np.int64))
    n = len(d_idx)
    assert len(t_idx) == n
    if X.dtype == np.float32:
        D = np.empty(n, dtype=np.float64)
        A = np.empty(n, dtype=np.float64)
        _load().oracle_elements_f32(X.ctypes.data, X.shape[0], X.shape[1], fch1, foff, tsamp,
                                    _dp(dms), _ip(d_idx), _lp(t_idx), n, _dp(D), _dp(A))
        return D, A
    assert X.dtype == np.uint8
    D = np.empty(n, dtype=np.int64)
    _load().oracle_elements_u8(X.ctypes.data, X.shape[0], X.shape[1], fch1, foff, tsamp,
                               _dp(dms), _ip(d_idx), _lp(t_idx), n, _lp(D))
    return D


def num_threads() -> int:
    """Threads the OpenMP loops will use (for the cpu_baseline report)."""
    n = os.environ.get("OMP_NUM_THREADS")
    if n:
        return int(n)
    try:
        return len(os.sched_getaffinity(0))
    except AttributeError:
        return os.cpu_count() or 1


# ------------------------------------------------------------------ post-processing

def _f64(a):
    return np.ascontiguousarray(np.asarray(a, dtype=np.float64))


def median_filter(x, w) -> np.ndarray:
    """eq 3.4 with the median, odd window w centred on each sample, ends clamped (R15)."""
    x = _f64(x)
    assert x.ndim == 1 and w >= 1 and w % 2 == 1
    y = np.empty_like(x)
    _load().oracle_median_filter(_dp(x), len(x), int(w), _dp(y))
    return y


def fit_line(y):
    """Least-squares line through (t, y_t), t = 0..n-1 -> (intercept, slope)."""
    y = _f64(y)
    a, b = C.c_double(0.0), C.c_double(0.0)
    _load().oracle_fit_line(_dp(y), len(y), C.byref(a), C.byref(b))
    return float(a.value), float(b.value)


def detrend(y, intercept, slope):
    """y_t - (intercept + slope t) and its population standard deviation (R17) -> (r, sigma)."""
    y = _f64(y)
    r = np.empty_like(y)
    s = C.c_double(0.0)
    _load().oracle_detrend(_dp(y), len(y), float(intercept), float(slope), _dp(r), C.byref(s))
    return r, float(s.value)


def normalise(r, sigma) -> np.ndarray:
    r = _f64(r)
    z = np.empty_like(r)
    _load().oracle_normalise(_dp(r), len(r), float(sigma), _dp(z))
    return z


def postprocess(D, median_window=0, detrend=True, normalise=True):
    """§3.5 on series D [..., n] (float32 or int32, the dedispersion output) -> (z float64 same shape,
    stats float64 [..., 3] = intercept, slope, sigma)."""
    D = np.ascontiguousarray(D)
    assert D.dtype in (np.float32, np.int32)
    assert detrend or not normalise
    n = D.shape[-1]
    nrows = D.size // n if n else 0
    z = np.empty(D.shape, dtype=np.float64)
    stats = np.empty(D.shape[:-1] + (3,), dtype=np.float64)
    _load().oracle_postprocess_rows(D.ctypes.data, int(D.dtype == np.int32), nrows, n, n, int(median_window),
                                    int(bool(detrend)), int(bool(normalise)), _dp(z), _dp(stats))
    return z, stats


def threshold(z, nsigma, sigma=None, capacity=None):
    """§3.6: samples of z [nbeams][ndm][n] above nsigma (times sigma [nbeams][ndm] when z is not normalised)
    -> (beam, dm, t, value) arrays in (beam, dm, t) order."""
    z = _f64(z)
    assert z.ndim == 3
    nb, ndm, n = z.shape
    sg = None if sigma is None else _f64(sigma)
    cap = int(capacity if capacity is not None else z.size)
    b = np.empty(cap, dtype=np.int32)
    d = np.empty(cap, dtype=np.int32)
    t = np.empty(cap, dtype=np.int64)
    v = np.empty(cap, dtype=np.float64)
    cnt = _load().oracle_threshold(_dp(z), nb, ndm, n, float(nsigma), None if sg is None else _dp(sg),
                                   b.ctypes.data_as(C.POINTER(C.c_int32)), d.ctypes.data_as(C.POINTER(C.c_int32)),
                                   _lp(t), _dp(v), cap)
    k = min(int(cnt), cap)
    return b[:k], d[:k], t[:k], v[:k], int(cnt)
