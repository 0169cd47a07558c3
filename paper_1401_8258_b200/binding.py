"""ctypes binding of ``include/dedisp_b200.h`` — argument marshalling only.

Every function here has the name and argument order of the C call it wraps; tensors / arrays are
turned into raw pointers and nothing else happens in Python.  All compute runs in the CUDA
library; if ``libdedisp_b200.so`` is missing and cannot be built, importing the library fails
loudly — there is no CPU path.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

from . import build as _build

DD_OK, DD_ERR_BAD_ARG, DD_ERR_UNSUPPORTED, DD_ERR_NOMEM, DD_ERR_CUDA, DD_ERR_STATE = 0, -1, -2, -3, -4, -5
DD_F32, DD_U8 = 0, 1
DD_KERNEL_AUTO, DD_KERNEL_GENERIC, DD_KERNEL_PS, DD_KERNEL_DIRECT = 0, 1, 2, 3

class dd_post_params(C.Structure):
    """Mirror of the C struct (include/dedisp_b200.h)."""
    _fields_ = [("median_window", C.c_int), ("detrend", C.c_int), ("normalise", C.c_int),
                ("threshold_on", C.c_int), ("nsigma", C.c_float)]


class dd_rfi_params(C.Structure):
    """Mirror of the C struct (include/dedisp_b200.h)."""
    _fields_ = [("poly_order", C.c_int), ("window", C.c_int), ("t_chan", C.c_float), ("t_spec", C.c_float)]


# numpy view of dd_candidate (16 bytes)
CANDIDATE_DTYPE = np.dtype([("beam", "<i4"), ("dm", "<i4"), ("t", "<i4"), ("value", "<f4")])

_dp = C.POINTER(C.c_double)
_vp = C.c_void_p
_i64 = C.c_int64

# name -> (restype, argtypes): one entry per function declared in include/dedisp_b200.h
SIGNATURES = {
    "dd_strerror": (C.c_char_p, [C.c_int]),
    "dd_last_error": (C.c_char_p, []),
    "dd_version": (C.c_char_p, []),
    "dd_max_shift": (_i64, [C.c_int, C.c_double, C.c_double, C.c_double, _dp, C.c_int]),
    "dd_shift_table": (C.c_int, [C.c_int, C.c_double, C.c_double, C.c_double, _dp, C.c_int, _vp]),
    "dd_dedisperse_f32": (C.c_int, [_vp, C.c_int, _i64, C.c_double, C.c_double, C.c_double, _dp, C.c_int, _vp]),
    "dd_dedisperse_u8_i32": (C.c_int, [_vp, C.c_int, _i64, C.c_double, C.c_double, C.c_double, _dp, C.c_int, _vp]),
    "dd_dedisperse_f32_host": (C.c_int, [_vp, C.c_int, _i64, C.c_double, C.c_double, C.c_double, _dp, C.c_int, _vp]),
    "dd_dedisperse_u8_i32_host": (C.c_int, [_vp, C.c_int, _i64, C.c_double, C.c_double, C.c_double, _dp, C.c_int, _vp]),
    "dd_plan_create": (C.c_int, [C.POINTER(_vp), C.c_int, C.c_int, C.c_double, C.c_double, C.c_double, _dp, C.c_int]),
    "dd_plan_destroy": (None, [_vp]),
    "dd_plan_max_shift": (_i64, [_vp]),
    "dd_plan_ndm": (C.c_int, [_vp]),
    "dd_plan_nchans": (C.c_int, [_vp]),
    "dd_plan_shift_table": (C.c_int, [_vp, _vp]),
    "dd_plan_set_kernel": (C.c_int, [_vp, C.c_int]),
    "dd_plan_kernel_for": (C.c_int, [_vp, _vp, _i64, _i64, _vp, _i64, _i64, _i64, C.c_int]),
    "dd_plan_launches_for": (C.c_int, [_vp, _vp, _i64, _i64, _vp, _i64, _i64, _i64, C.c_int]),
    "dd_plan_describe": (C.c_int, [_vp, C.c_char_p, C.c_int]),
    "dd_release_workspaces": (C.c_int, []),
    "dd_execute": (C.c_int, [_vp, _vp, _i64, _i64, _vp, _i64, _i64, _i64, C.c_int, _vp]),
    "dd_execute_host": (C.c_int, [_vp, _vp, _i64, _i64, _vp, _i64, _i64, _i64, C.c_int]),
    "dd_postprocess": (C.c_int, [C.c_int, _vp, _i64, _i64, C.c_int, _i64, C.c_int, C.POINTER(dd_post_params),
                                 _vp, _i64, _i64, _vp, _vp, _i64, _vp, _vp]),
    "dd_postprocess_static": (C.c_int, [C.c_int, _vp, _i64, _i64, C.c_int, _i64, C.c_int, C.POINTER(dd_post_params),
                                        _vp, _i64, _i64, _vp, _i64, _vp, _vp]),
    "dd_postprocess_launches": (C.c_int, [C.POINTER(dd_post_params), C.c_int]),
    "dd_search_host": (C.c_int, [_vp, _vp, _i64, _i64, _i64, C.c_int, C.POINTER(dd_post_params), _vp, _i64,
                                 C.POINTER(_i64)]),
    "dd_rfi_mitigate": (C.c_int, [_vp, C.c_int, _i64, _i64, _i64, C.c_int, C.POINTER(dd_rfi_params), _vp, _vp, _vp,
                                  _vp, _vp, _vp]),
    "dd_diagonal_dm": (C.c_double, [C.c_int, C.c_double, C.c_double, C.c_double]),
    "dd_downsample2_f32": (C.c_int, [_vp, _vp, _i64, _i64, _i64, _i64, _vp]),
    "dd_timebin_create": (C.c_int, [C.POINTER(_vp), C.c_int, C.c_double, C.c_double, C.c_double, _dp, C.c_int,
                                    C.c_double, C.c_int]),
    "dd_timebin_destroy": (None, [_vp]),
    "dd_timebin_levels": (C.c_int, [_vp, _vp]),
    "dd_timebin_input_samples": (_i64, [_vp, _i64]),
    "dd_timebin_execute": (C.c_int, [_vp, _vp, _i64, _i64, _vp, _i64, _i64, _vp]),
    "dd_subband_create": (C.c_int, [C.POINTER(_vp), C.c_int, C.c_double, C.c_double, C.c_double, _dp, C.c_int,
                                    C.c_int, C.c_int]),
    "dd_subband_destroy": (None, [_vp]),
    "dd_subband_max_shift": (_i64, [_vp]),
    "dd_subband_execute": (C.c_int, [_vp, _vp, _i64, _vp, _i64, _i64, _vp]),
    "dd_beamform_power_u4": (C.c_int, [_vp, C.c_int, C.c_int, _i64, _vp, C.c_int, _vp, _i64, _i64, _vp]),
    "dd_stream_create": (C.c_int, [C.POINTER(_vp), _vp, _i64, C.c_int]),
    "dd_stream_push": (C.c_int, [_vp, _vp, _i64, _i64, _i64, _vp, _i64, _i64, C.POINTER(_i64), _vp]),
    "dd_stream_reset": (C.c_int, [_vp]),
    "dd_stream_destroy": (None, [_vp]),
}

_lib = None


def lib() -> C.CDLL:
    """Load (building if stale and nvcc is present) the CUDA library.  Raises if impossible."""
    global _lib
    if _lib is not None:
        return _lib
    path = _build.LIB
    try:
        path = _build.build()
    except Exception:
        if not os.path.exists(path):
            raise RuntimeError(
                "libdedisp_b200.so is missing and could not be built with nvcc; "
                "this package has no CPU fallback") from None
    l = C.CDLL(path)
    for name, (res, args) in SIGNATURES.items():
        f = getattr(l, name)          # AttributeError if the .so lacks a declared symbol
        f.restype = res
        f.argtypes = args
    _lib = l
    return l


class DedispError(RuntimeError):
    def __init__(self, code: int, where: str):
        l = lib()
        self.code = code
        detail = l.dd_last_error().decode()
        super().__init__("%s: %s (%d)%s" % (where, l.dd_strerror(code).decode(), code,
                                            ": " + detail if detail else ""))


def _check(code: int, where: str) -> int:
    if code < 0:
        raise DedispError(int(code), where)
    return int(code)


def _ptr(obj) -> int:
    """Raw address of a torch tensor, numpy array, or int (None -> 0)."""
    if obj is None:
        return 0
    if isinstance(obj, int):
        return obj
    if hasattr(obj, "data_ptr"):
        return int(obj.data_ptr())
    if isinstance(obj, np.ndarray):
        return int(obj.ctypes.data)
    raise TypeError("expected a tensor, ndarray or integer address, got %r" % type(obj))


def _dms(dm_list):
    a = np.ascontiguousarray(np.asarray(dm_list, dtype=np.float64))
    return a, a.ctypes.data_as(_dp), int(a.size)


def _stream_ptr(stream) -> int:
    if stream is None:
        return 0
    if isinstance(stream, int):
        return stream
    return int(stream.cuda_stream)       # torch.cuda.Stream


# ------------------------------------------------------------------ plain calls

def dd_version() -> str:
    return lib().dd_version().decode()


def dd_max_shift(nchans, fch1, foff, tsamp, dm_list) -> int:
    a, p, n = _dms(dm_list)
    return _check(lib().dd_max_shift(nchans, fch1, foff, tsamp, p, n), "dd_max_shift")


def dd_shift_table(nchans, fch1, foff, tsamp, dm_list) -> np.ndarray:
    a, p, n = _dms(dm_list)
    out = np.empty((n, nchans), dtype=np.int32)
    _check(lib().dd_shift_table(nchans, fch1, foff, tsamp, p, n, out.ctypes.data), "dd_shift_table")
    return out


def dd_release_workspaces() -> None:
    _check(lib().dd_release_workspaces(), "dd_release_workspaces")


def dd_dedisperse_f32(X, nchans, nsamp, fch1, foff, tsamp, dm_list, D) -> None:
    a, p, n = _dms(dm_list)
    _check(lib().dd_dedisperse_f32(_ptr(X), nchans, nsamp, fch1, foff, tsamp, p, n, _ptr(D)), "dd_dedisperse_f32")


def dd_dedisperse_u8_i32(X, nchans, nsamp, fch1, foff, tsamp, dm_list, D) -> None:
    a, p, n = _dms(dm_list)
    _check(lib().dd_dedisperse_u8_i32(_ptr(X), nchans, nsamp, fch1, foff, tsamp, p, n, _ptr(D)), "dd_dedisperse_u8_i32")


def dd_dedisperse_f32_host(X, nchans, nsamp, fch1, foff, tsamp, dm_list, D) -> None:
    a, p, n = _dms(dm_list)
    _check(lib().dd_dedisperse_f32_host(_ptr(X), nchans, nsamp, fch1, foff, tsamp, p, n, _ptr(D)), "dd_dedisperse_f32_host")


def dd_dedisperse_u8_i32_host(X, nchans, nsamp, fch1, foff, tsamp, dm_list, D) -> None:
    a, p, n = _dms(dm_list)
    _check(lib().dd_dedisperse_u8_i32_host(_ptr(X), nchans, nsamp, fch1, foff, tsamp, p, n, _ptr(D)), "dd_dedisperse_u8_i32_host")


def post_params(median_window=0, detrend=True, normalise=True, nsigma=None) -> dd_post_params:
    """Fills a dd_post_params (thresholding on when nsigma is given)."""
    return dd_post_params(int(median_window), int(bool(detrend)), int(bool(normalise)), int(nsigma is not None),
                          float(nsigma if nsigma is not None else 0.0))


def dd_postprocess(dtype, D, stride, beam_stride, ndm, nsamp, nbeams, params, Z=None, z_stride=0, z_beam_stride=0,
                   stats=None, cand=None, capacity=0, count=None, stream=None) -> None:
    _check(lib().dd_postprocess(dtype, _ptr(D), stride, beam_stride, ndm, nsamp, nbeams, C.byref(params), _ptr(Z),
                                z_stride, z_beam_stride, _ptr(stats), _ptr(cand), capacity, _ptr(count),
                                _stream_ptr(stream)), "dd_postprocess")


POSTPROCESS_STATIC_MAX_SERIES = 16384      # DD_POSTPROCESS_STATIC_MAX_SERIES of include/dedisp_b200.h


def dd_postprocess_static(dtype, D, stride, beam_stride, ndm, nsamp, nbeams, params, Z=None, z_stride=0,
                          z_beam_stride=0, cand=None, capacity=0, count=None, stream=None) -> None:
    """dd_postprocess without device allocations (statistics in the library's static device array)."""
    _check(lib().dd_postprocess_static(dtype, _ptr(D), stride, beam_stride, ndm, nsamp, nbeams, C.byref(params),
                                       _ptr(Z), z_stride, z_beam_stride, _ptr(cand), capacity, _ptr(count),
                                       _stream_ptr(stream)), "dd_postprocess_static")


def dd_rfi_mitigate(X, nchans, nsamp, stride, beam_stride, nbeams, params, bandpass=None, fit=None, stats=None,
                    chan_flags=None, spec_flags=None, stream=None) -> None:
    _check(lib().dd_rfi_mitigate(_ptr(X), nchans, nsamp, stride, beam_stride, nbeams, C.byref(params), _ptr(bandpass),
                                 _ptr(fit), _ptr(stats), _ptr(chan_flags), _ptr(spec_flags), _stream_ptr(stream)),
           "dd_rfi_mitigate")


def dd_beamform_power_u4(V, nants, nchans, nsamp, W, nbeams, P, out_stride, out_beam_stride, stream=None) -> None:
    _check(lib().dd_beamform_power_u4(_ptr(V), nants, nchans, nsamp, _ptr(W), nbeams, _ptr(P), out_stride,
                                      out_beam_stride, _stream_ptr(stream)), "dd_beamform_power_u4")


def dd_postprocess_launches(params, want_series) -> int:
    return _check(lib().dd_postprocess_launches(C.byref(params), int(bool(want_series))), "dd_postprocess_launches")


# ------------------------------------------------------------------ plan / stream handles

class Plan:
    """Owns a ``dd_plan*``; methods are the dd_plan_* / dd_execute* calls."""

    def __init__(self, dtype, nchans, fch1, foff, tsamp, dm_list):
        a, p, n = _dms(dm_list)
        h = _vp()
        _check(lib().dd_plan_create(C.byref(h), dtype, nchans, fch1, foff, tsamp, p, n), "dd_plan_create")
        self._h = h
        self.dtype, self.nchans, self.ndm = dtype, nchans, n

    def destroy(self):
        if getattr(self, "_h", None):
            lib().dd_plan_destroy(self._h)
            self._h = None

    __del__ = destroy

    def max_shift(self) -> int:
        return _check(lib().dd_plan_max_shift(self._h), "dd_plan_max_shift")

    def shift_table(self) -> np.ndarray:
        out = np.empty((self.ndm, self.nchans), dtype=np.int32)
        _check(lib().dd_plan_shift_table(self._h, out.ctypes.data), "dd_plan_shift_table")
        return out

    def set_kernel(self, kernel: int) -> None:
        _check(lib().dd_plan_set_kernel(self._h, kernel), "dd_plan_set_kernel")

    def kernel_for(self, X, in_stride, in_beam_stride, D, out_stride, out_beam_stride, nsamp_out, nbeams=1) -> int:
        return _check(lib().dd_plan_kernel_for(self._h, _ptr(X), in_stride, in_beam_stride, _ptr(D), out_stride,
                                               out_beam_stride, nsamp_out, nbeams), "dd_plan_kernel_for")

    def launches_for(self, X, in_stride, in_beam_stride, D, out_stride, out_beam_stride, nsamp_out, nbeams=1) -> int:
        return _check(lib().dd_plan_launches_for(self._h, _ptr(X), in_stride, in_beam_stride, _ptr(D), out_stride,
                                                 out_beam_stride, nsamp_out, nbeams), "dd_plan_launches_for")

    def describe(self) -> str:
        buf = C.create_string_buffer(1024)
        _check(lib().dd_plan_describe(self._h, buf, len(buf)), "dd_plan_describe")
        return buf.value.decode()

    def execute(self, X, in_stride, in_beam_stride, D, out_stride, out_beam_stride, nsamp_out, nbeams=1,
                stream=None) -> None:
        _check(lib().dd_execute(self._h, _ptr(X), in_stride, in_beam_stride, _ptr(D), out_stride,
                                out_beam_stride, nsamp_out, nbeams, _stream_ptr(stream)), "dd_execute")

    def execute_host(self, X, in_stride, in_beam_stride, D, out_stride, out_beam_stride, nsamp_out,
                     nbeams=1) -> None:
        _check(lib().dd_execute_host(self._h, _ptr(X), in_stride, in_beam_stride, _ptr(D), out_stride,
                                     out_beam_stride, nsamp_out, nbeams), "dd_execute_host")


    def search_host(self, X, in_stride, in_beam_stride, nsamp_out, nbeams, params, cand, capacity) -> int:
        """dd_search_host: cand is a HOST buffer (numpy array of CANDIDATE_DTYPE or pinned tensor); returns count."""
        n = _i64(0)
        _check(lib().dd_search_host(self._h, _ptr(X), in_stride, in_beam_stride, nsamp_out, nbeams, C.byref(params),
                                    _ptr(cand), capacity, C.byref(n)), "dd_search_host")
        return int(n.value)


class Stream:
    """Owns a ``dd_stream*`` (chunked streaming with the maxshift carry)."""

    def __init__(self, plan: Plan, max_chunk: int, nbeams: int = 1):
        h = _vp()
        _check(lib().dd_stream_create(C.byref(h), plan._h, max_chunk, nbeams), "dd_stream_create")
        self._h = h
        self.plan = plan            # keep the plan alive

    def destroy(self):
        if getattr(self, "_h", None):
            lib().dd_stream_destroy(self._h)
            self._h = None

    __del__ = destroy

    def push(self, X_new, in_stride, in_beam_stride, n_new, D_out, out_stride, out_beam_stride,
             stream=None) -> int:
        n_out = _i64(0)
        _check(lib().dd_stream_push(self._h, _ptr(X_new), in_stride, in_beam_stride, n_new, _ptr(D_out),
                                    out_stride, out_beam_stride, C.byref(n_out), _stream_ptr(stream)),
               "dd_stream_push")
        return int(n_out.value)

    def reset(self) -> None:
        _check(lib().dd_stream_reset(self._h), "dd_stream_reset")


# ------------------------------------------------------------------ approximate variants (f2)

def dd_diagonal_dm(nchans, fch1, foff, tsamp) -> float:
    return float(lib().dd_diagonal_dm(nchans, fch1, foff, tsamp))


def dd_downsample2_f32(X, Y, nrows, n_in, stride_in, stride_out, stream=None) -> None:
    _check(lib().dd_downsample2_f32(_ptr(X), _ptr(Y), nrows, n_in, stride_in, stride_out, _stream_ptr(stream)),
           "dd_downsample2_f32")


class TimeBin:
    """Owns a ``dd_timebin*`` (time-binned dedispersion)."""

    def __init__(self, nchans, fch1, foff, tsamp, dm_list, dm_diag=0.0, max_level=8):
        a, p, n = _dms(dm_list)
        h = _vp()
        _check(lib().dd_timebin_create(C.byref(h), nchans, fch1, foff, tsamp, p, n, dm_diag, max_level),
               "dd_timebin_create")
        self._h, self.ndm = h, n

    def destroy(self):
        if getattr(self, "_h", None):
            lib().dd_timebin_destroy(self._h)
            self._h = None

    __del__ = destroy

    def levels(self) -> np.ndarray:
        out = np.zeros(self.ndm, dtype=np.int32)
        _check(lib().dd_timebin_levels(self._h, out.ctypes.data), "dd_timebin_levels")
        return out

    def input_samples(self, nsamp_out) -> int:
        return _check(lib().dd_timebin_input_samples(self._h, nsamp_out), "dd_timebin_input_samples")

    def execute(self, X, in_stride, n_in, D, out_stride, nsamp_out, stream=None) -> None:
        _check(lib().dd_timebin_execute(self._h, _ptr(X), in_stride, n_in, _ptr(D), out_stride, nsamp_out,
                                        _stream_ptr(stream)), "dd_timebin_execute")


class Subband:
    """Owns a ``dd_subband*`` (two-step subband dedispersion)."""

    def __init__(self, nchans, fch1, foff, tsamp, dm_list, chans_per_subband, dms_per_nominal):
        a, p, n = _dms(dm_list)
        h = _vp()
        _check(lib().dd_subband_create(C.byref(h), nchans, fch1, foff, tsamp, p, n, chans_per_subband,
                                       dms_per_nominal), "dd_subband_create")
        self._h, self.ndm = h, n

    def destroy(self):
        if getattr(self, "_h", None):
            lib().dd_subband_destroy(self._h)
            self._h = None

    __del__ = destroy

    def max_shift(self) -> int:
        return _check(lib().dd_subband_max_shift(self._h), "dd_subband_max_shift")

    def execute(self, X, in_stride, D, out_stride, nsamp_out, stream=None) -> None:
        _check(lib().dd_subband_execute(self._h, _ptr(X), in_stride, _ptr(D), out_stride, nsamp_out,
                                        _stream_ptr(stream)), "dd_subband_execute")
