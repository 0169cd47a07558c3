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


# ---------------------------------------------------------------- delay patterns behind the partial-sum kernels

def _patterns_from_oracle_table(tab, group, tile):
    """Mean / max number of distinct relative-delay vectors per (tile of sorted trials, channel group),
    recomputed with numpy from the ORACLE's table (rows sorted by DM by construction of the workloads)."""
    ndm, nch = tab.shape
    counts = []
    for t0 in range(0, ndm, tile):
        rows = np.minimum(np.arange(t0, t0 + tile), ndm - 1)
        for c0 in range(0, nch, group):
            rel = tab[rows][:, c0:c0 + group] - tab[rows][:, c0:c0 + 1]
            counts.append(len(np.unique(rel, axis=0)))
    return float(np.mean(counts)), int(np.max(counts))


@pytest.mark.parametrize("idx,nchans,ndm", [(2, 256, 200), (3, 512, 300), (4, 128, 130), (5, 301, 257)])
@pytest.mark.parametrize("group,tile", [(1, 64), (2, 16), (4, 64), (8, 128), (3, 7)])
def test_pattern_stats_match_a_numpy_recount_on_the_oracle_table(idx, nchans, ndm, group, tile):
    w0 = synth.WORKLOADS[idx]
    w = synth.scaled(w0, nchans=nchans, ndm=ndm, foff=w0.foff * w0.nchans / nchans)
    mean, mx = dd.dd_pattern_stats(w.nchans, w.fch1, w.foff, w.tsamp, w.dm_list, group, tile)
    tab = oracle.shift_table(w.nchans, w.fch1, w.foff, w.tsamp, w.dm_list)
    want_mean, want_max = _patterns_from_oracle_table(np.asarray(tab, dtype=np.int64), group, tile)
    assert mx == want_max and abs(mean - want_mean) < 1e-9
    if group == 1:
        assert mx == 1                                            # a single channel has one (empty) pattern
    assert 1 <= mean <= min(tile, ndm)


def test_pattern_counts_of_the_benchmark_workloads_stay_small():
    # the premise of DESIGN.md 5.3: a handful of patterns per 64-trial tile and 4-channel group
    for idx, lo, hi in [(2, 3, 8), (3, 2, 6), (5, 2, 7)]:
        w = synth.scaled(synth.WORKLOADS[idx], ndm=512)
        mean, mx = dd.dd_pattern_stats(w.nchans, w.fch1, w.foff, w.tsamp, w.dm_list, 4, 64)
        assert lo <= mean <= hi and mx <= 12, (idx, mean, mx)
