"""CPU-only checks of the product's host side: the C-ABI library loads and exports every symbol
the header declares, the plan's delay table (plan.cpp) equals the oracle's independently written
one on all five workloads, and argument errors come back as codes.  No compute call is made."""
import ctypes as C
import os
import re

import numpy as np
import pytest

import oracle
import paper_1401_8258_b200 as dd
from paper_1401_8258_b200 import binding, synth

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _declared_symbols():
    text = open(os.path.join(ROOT, "include", "dedisp_b200.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(dd_[a-z0-9_]+)\s*\(", text)))


def test_library_loads_and_exports_every_declared_symbol():
    lib = dd.lib()
    names = _declared_symbols()
    assert len(names) >= 20
    for n in names:
        assert hasattr(lib, n), "libdedisp_b200.so lacks %s" % n
    # and the binding marshals every one of them
    assert sorted(binding.SIGNATURES) == names
    assert "sm_100a" in dd.dd_version()


def test_library_is_sm100a_only():
    import subprocess
    out = subprocess.run(["cuobjdump", "--list-elf", binding._build.LIB], capture_output=True, text=True).stdout
    archs = set(re.findall(r"sm_\d+a?", out))
    assert archs == {"sm_100a"}, archs


@pytest.mark.parametrize("idx", [1, 2, 3, 4, 5])
def test_plan_table_equals_oracle_table(idx):
    w = synth.WORKLOADS[idx]
    got = dd.dd_shift_table(w.nchans, w.fch1, w.foff, w.tsamp, w.dm_list)
    want = oracle.shift_table(w.nchans, w.fch1, w.foff, w.tsamp, w.dm_list)
    assert got.dtype == np.int32 and np.array_equal(got, want)
    assert dd.dd_max_shift(w.nchans, w.fch1, w.foff, w.tsamp, w.dm_list) == want.max()


def test_table_rows_follow_caller_order_for_unsorted_lists():
    g = np.random.default_rng(5)
    dms = g.uniform(0, 300, 37)
    dms[5] = dms[20]                      # duplicate
    dms[0] = 0.0
    got = dd.dd_shift_table(96, 1400.0, -0.5, 64e-6, dms)
    want = oracle.shift_table(96, 1400.0, -0.5, 64e-6, dms)
    assert np.array_equal(got, want)
    assert dd.dd_max_shift(96, 1400.0, -0.5, 64e-6, dms) == want.max()
    # foff == 0: all delays are zero
    assert not dd.dd_shift_table(8, 400.0, 0.0, 1e-3, [0.0, 50.0]).any()


def test_argument_errors_are_codes_not_crashes():
    ok = dict(nchans=4, fch1=400.0, foff=-1.0, tsamp=1e-3, dm_list=[0.0, 1.0])
    bad = [dict(nchans=0), dict(fch1=0.0), dict(fch1=-5.0), dict(foff=1.0), dict(tsamp=0.0),
           dict(tsamp=-1.0), dict(dm_list=[0.0, -1.0]), dict(dm_list=[float("nan")]),
           dict(dm_list=[float("inf")]), dict(foff=-200.0),          # bottom channel <= 0 MHz
           dict(tsamp=1e-30, dm_list=[1e6])]                         # shift overflows int32
    for b in bad:
        kw = dict(ok, **b)
        with pytest.raises(dd.DedispError) as e:
            dd.dd_max_shift(**kw)
        assert e.value.code == dd.DD_ERR_BAD_ARG, b
        with pytest.raises(dd.DedispError):
            dd.dd_shift_table(**kw)
    assert dd.dd_max_shift(4, 400.0, -1.0, 1e-3, []) == 0
    lib = dd.lib()
    assert lib.dd_strerror(dd.DD_ERR_BAD_ARG) == b"bad argument"
    # null handles are rejected, not dereferenced
    assert lib.dd_plan_max_shift(None) == dd.DD_ERR_BAD_ARG
    assert lib.dd_execute(None, None, 0, 0, None, 0, 0, 0, 1, None) == dd.DD_ERR_BAD_ARG
    assert lib.dd_stream_reset(None) == dd.DD_ERR_BAD_ARG
    n = C.c_int64(7)
    assert lib.dd_stream_push(None, None, 0, 0, 0, None, 0, 0, C.byref(n), None) == dd.DD_ERR_BAD_ARG


def test_no_gpu_means_unsupported_not_fallback():
    import torch
    if torch.cuda.is_available():
        pytest.skip("this check is for the CPU box")
    with pytest.raises(dd.DedispError) as e:
        dd.Plan(dd.DD_F32, 4, 400.0, -1.0, 1e-3, [0.0, 1.0])
    assert e.value.code in (dd.DD_ERR_UNSUPPORTED, dd.DD_ERR_CUDA)


def test_product_does_not_import_the_oracle():
    pkg = os.path.join(ROOT, "paper_1401_8258_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cpp", ".h", ".cuh")):
                src = open(os.path.join(dirpath, f)).read()
                assert not re.search(r"^\s*(import|from)\s+oracle|#include.*oracle|dedisp_oracle",
                                     src, flags=re.M), f
