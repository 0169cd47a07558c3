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
_SO = os.path.join(_HERE, "libdedisp_oracle.so")
_lock = threading.Lock()
_lib = None


def build(force: bool = False) -> str:
    """Compile the oracle shared object (no CUDA involved)."""
    with _lock:
        if (not force and os.path.exists(_SO)
                and os.path.getmtime(_SO) >= os.path.getmtime(_SRC)):
            return _SO
        tmp = _SO + ".tmp.%d" % os.getpid()
        cmd = ["g++", "-O2", "-ffp-contract=off", "-fopenmp", "-shared", "-fPIC",
               "-std=c++17", "-o", tmp, _SRC]
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
