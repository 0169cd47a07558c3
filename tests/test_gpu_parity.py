"""GPU parity tests proper: the CUDA path (through the C ABI) against the oracle, element by
element, on the same seeded inputs.  Bit-exact for uint8->int32; |D_gpu - D_oracle| <=
1e-5 * sum_c|X| per element for float32 (north_star)."""
import os

import numpy as np
import pytest

import oracle
import paper_1401_8258_b200 as dd
from paper_1401_8258_b200 import synth

from _util import (assert_parity, assert_row_checksums, assert_sampled_parity, assert_whole_rows, dd_dtype,
                   gpu_dedisperse, make_case, p8_rows, small)

pytestmark = pytest.mark.gpu

KERNELS = [pytest.param(dd.DD_KERNEL_GENERIC, id="generic"), pytest.param(dd.DD_KERNEL_AUTO, id="auto"),
           pytest.param(dd.DD_KERNEL_DIRECT, id="direct")]
# AUTO takes the partial-sum kernels (uint8 and float32; float32 through a re-pitched copy when X is not
# 16-byte aligned) whenever the plan's delay steps are fine enough, else the generic kernel


@pytest.fixture(scope="module", autouse=True)
def _need_gpu():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    assert torch.cuda.get_device_capability(0)[0] == 10, "these kernels are sm_100a only"


# ------------------------------------------------------------------ configs, shrunk to oracle size

@pytest.mark.parametrize("kernel", KERNELS)
def test_config1_full(kernel):
    # BASELINE.json configs[0] exactly: 64 ch, 32 DMs, 8192 samples, pulse of amplitude 3 at DM 10
    w = synth.WORKLOADS[1]
    X, ms = make_case(w)
    tab = oracle.shift_table(w.nchans, w.fch1, w.foff, w.tsamp, w.dm_list)
    synth.inject_pulse(X, 4000, 1, 3.0, tab[10])
    D = gpu_dedisperse(w, X, kernel)
    assert_parity(w, X, D)
    d, t = np.unravel_index(D.argmax(), D.shape)
    assert (d, t) == (10, 4000) and abs(D[10, 4000] / 8.0 - 24.0) < 4.0      # S/N ~ A*sqrt(nchans)
    if kernel == dd.DD_KERNEL_AUTO:                                           # a tiny plan: the direct kernel
        plan = dd.Plan(dd.DD_F32, w.nchans, w.fch1, w.foff, w.tsamp, w.dm_list)
        assert plan.kernel_for(0x1000, 1 << 20, 0, 0x2000, w.nsamp, 0, w.nsamp, 1) == dd.DD_KERNEL_DIRECT
        assert "dd_direct_kernel" in plan.describe()
        plan.destroy()


CASES = [
    # (workload, nchans, ndm, nsamp): several tiles of every kernel plus a ragged tail
    (2, 256, 70, 9000 + 37),
    (2, 1024, 40, 4096 + 1),
    (3, 512, 50, 8192 + 333),
    (4, 128, 100, 5000),
    (5, 300, 61, 7001),
    (5, 2048, 16, 3000),
]


@pytest.mark.parametrize("kernel", KERNELS)
@pytest.mark.parametrize("idx,nchans,ndm,nsamp", CASES)
def test_shrunk_configs(idx, nchans, ndm, nsamp, kernel):
    w = small(idx, nchans, ndm, nsamp)
    X, ms = make_case(w, pulses=3)
    D = gpu_dedisperse(w, X, kernel)
    assert_parity(w, X, D)


@pytest.mark.parametrize("kernel", KERNELS)
@pytest.mark.parametrize("idx", [2, 3])
def test_top_of_the_dm_grid(idx, kernel):
    # the last trials of the full-size grids (largest shifts and spreads), few of them
    w0 = synth.WORKLOADS[idx]
    w = synth.scaled(w0, ndm=24, nsamp=3000)
    dms = w0.dm_list[-24:]
    ms = oracle.max_shift(w.nchans, w.fch1, w.foff, w.tsamp, dms)
    X = synth.make_input(w, w.nsamp + ms)
    D = gpu_dedisperse(w, X, kernel, dms=dms)
    assert_parity(w, X, D, dms=dms)


# ------------------------------------------------------------------ edge cases

@pytest.mark.parametrize("kernel", KERNELS)
@pytest.mark.parametrize("dtype", ["f32", "u8"])
def test_edges(dtype, kernel):
    base = synth.scaled(synth.WORKLOADS[2], dtype=dtype)
    # nchans = 1: identity for every DM; DM = 0 only; a single output sample; tiny everything
    for nchans, ndm, nsamp in [(1, 5, 100), (7, 1, 1), (3, 2, 5), (33, 17, 1025), (64, 33, 2049)]:
        w = synth.scaled(base, nchans=nchans, ndm=ndm, nsamp=nsamp, foff=-20.0 / nchans, dm_step=7.0)
        X, ms = make_case(w)
        D = gpu_dedisperse(w, X, kernel)
        assert_parity(w, X, D)
        if nchans == 1:
            assert np.array_equal(D, np.broadcast_to(X[0, :nsamp].astype(D.dtype), D.shape))
        if dtype == "u8":                                          # DM = 0 row = channel sum
            assert np.array_equal(D[0], X[:, :nsamp].sum(axis=0, dtype=np.int64))


def test_empty_inputs_write_nothing():
    import torch
    w = small(2, 16, 4, 64)
    plan = dd.Plan(dd.DD_U8, w.nchans, w.fch1, w.foff, w.tsamp, w.dm_list)
    D = torch.full((4, 64), -7, dtype=torch.int32, device="cuda")
    X = torch.zeros((16, 64 + plan.max_shift()), dtype=torch.uint8, device="cuda")
    plan.execute(X, X.shape[1], 0, D, 64, 0, 0, 1)                 # nsamp_out = 0
    torch.cuda.synchronize()
    assert int((D != -7).sum()) == 0
    empty = dd.Plan(dd.DD_U8, w.nchans, w.fch1, w.foff, w.tsamp, [])   # ndm = 0
    empty.execute(X, X.shape[1], 0, D, 64, 0, 64, 1)
    torch.cuda.synchronize()
    assert int((D != -7).sum()) == 0 and empty.max_shift() == 0
    with pytest.raises(dd.DedispError) as e:                       # stride shorter than the row
        plan.execute(X, 10, 0, D, 64, 0, 64, 1)
    assert e.value.code == dd.DD_ERR_BAD_ARG


@pytest.mark.parametrize("kernel", KERNELS)
def test_unsorted_duplicate_nonuniform_dm_list(kernel):
    w = small(3, 200, 45, 3000)
    g = np.random.default_rng(11)
    dms = g.uniform(0, 900, 45)
    dms[3] = dms[30]
    dms[7] = 0.0
    ms = oracle.max_shift(w.nchans, w.fch1, w.foff, w.tsamp, dms)
    X = synth.make_input(w, w.nsamp + ms)
    D = gpu_dedisperse(w, X, kernel, dms=dms)
    assert_parity(w, X, D, dms=dms)
    assert np.array_equal(D[3], D[30])


@pytest.mark.parametrize("kernel", KERNELS)
def test_large_dm_steps_fall_back_to_narrow_tiles(kernel):
    # per-trial shift steps of hundreds of samples (Fig 2.9 regime)
    w = small(1, 64, 9, 2500, dm_step=40.0)
    X, ms = make_case(w)
    assert ms > 8 * 512      # > 512 samples per trial step: only the KB=1 tiling fits
    D = gpu_dedisperse(w, X, kernel)
    assert_parity(w, X, D)


@pytest.mark.parametrize("kernel", KERNELS)
def test_all_255_input_does_not_overflow(kernel):
    # P13: 2048 channels of 255 -> every element = 522240 exactly (packed partial sums must flush)
    w = small(5, 2048, 12, 2100)
    ms = oracle.max_shift(w.nchans, w.fch1, w.foff, w.tsamp, w.dm_list)
    X = np.full((w.nchans, w.nsamp + ms), 255, dtype=np.uint8)
    D = gpu_dedisperse(w, X, kernel)
    assert np.all(D == 255 * 2048)


@pytest.mark.parametrize("kernel", KERNELS)
@pytest.mark.parametrize("dtype", ["f32", "u8"])
def test_impulse_response_against_the_table(dtype, kernel):
    # P6: X = delta at (c0, u0) => D[d][u0 - s(d,c0)] = 1, everything else 0
    w = small(2, 96, 40, 5000, dtype=dtype)
    tab = oracle.shift_table(w.nchans, w.fch1, w.foff, w.tsamp, w.dm_list)
    ms = int(tab.max())
    X = np.zeros((w.nchans, w.nsamp + ms), dtype=w.np_dtype)
    c0, u0 = 77, 4100
    X[c0, u0] = 1
    D = gpu_dedisperse(w, X, kernel)
    want = np.zeros_like(D)
    for d in range(w.ndm):
        want[d, u0 - tab[d, c0]] = 1
    assert np.array_equal(D, want)


# ------------------------------------------------------------------ strides, batch, streaming

@pytest.mark.parametrize("kernel", KERNELS)
@pytest.mark.parametrize("dtype", ["f32", "u8"])
def test_strides_offsets_and_batch_equal_loop_of_singles(dtype, kernel):
    import torch
    nb = 3
    w = small(4, 96, 37, 3001, dtype=dtype, nbeams=nb)
    tdt = torch.float32 if dtype == "f32" else torch.uint8
    odt = torch.float32 if dtype == "f32" else torch.int32
    plan = dd.Plan(dd_dtype(w), w.nchans, w.fch1, w.foff, w.tsamp, w.dm_list)
    plan.set_kernel(kernel)
    ms = plan.max_shift()
    assert ms == oracle.max_shift(w.nchans, w.fch1, w.foff, w.tsamp, w.dm_list)
    xs = [synth.make_input(w, w.nsamp + ms, beam=b) for b in range(nb)]
    # padded, offset (unaligned for u8) layout: rows of in_stride elements starting 3 elements in
    in_stride, out_stride = w.nsamp + ms + 13, w.nsamp + 5
    in_bs, out_bs = w.nchans * in_stride + 101, w.ndm * out_stride + 7
    Xd = torch.zeros(3 + nb * in_bs, dtype=tdt, device="cuda")
    for b in range(nb):
        v = Xd[3 + b * in_bs: 3 + b * in_bs + w.nchans * in_stride].view(w.nchans, in_stride)
        v[:, :w.nsamp + ms] = torch.from_numpy(xs[b]).cuda()
    Dd = torch.full((1 + nb * out_bs,), -7, dtype=odt, device="cuda")
    plan.execute(Xd[3:], in_stride, in_bs, Dd[1:], out_stride, out_bs, w.nsamp, nb)
    torch.cuda.synchronize()
    Dh = Dd.cpu().numpy()
    for b in range(nb):
        blk = Dh[1 + b * out_bs: 1 + b * out_bs + w.ndm * out_stride].reshape(w.ndm, out_stride)
        assert_parity(w, xs[b], np.ascontiguousarray(blk[:, :w.nsamp]))
        assert np.all(blk[:, w.nsamp:] == -7)                       # padding untouched
        single = gpu_dedisperse(w, xs[b], kernel)                   # batch == loop of singles, bit for bit
        assert np.array_equal(single, blk[:, :w.nsamp])
    plan.destroy()


@pytest.mark.parametrize("kernel", KERNELS)
@pytest.mark.parametrize("dtype", ["f32", "u8"])
def test_streaming_equals_one_shot_bit_for_bit(dtype, kernel):
    import torch
    nb = 2
    w = small(5, 160, 50, 6000, dtype=dtype, nbeams=nb)
    odt = torch.float32 if dtype == "f32" else torch.int32
    plan = dd.Plan(dd_dtype(w), w.nchans, w.fch1, w.foff, w.tsamp, w.dm_list)
    plan.set_kernel(kernel)
    ms = plan.max_shift()
    total = w.nsamp + ms
    xs = np.stack([synth.make_input(w, total, beam=b) for b in range(nb)])
    Xd = torch.from_numpy(xs).cuda()
    one = torch.empty((nb, w.ndm, w.nsamp), dtype=odt, device="cuda")
    plan.execute(Xd, total, w.nchans * total, one, w.nsamp, w.ndm * w.nsamp, w.nsamp, nb)
    # chunks: smaller than maxshift, larger, ragged, and a 1-sample push
    chunks, left = [], total
    for c in [ms // 3 + 1, 1, 1500, 777, 2048]:
        c = min(c, left); chunks.append(c); left -= c
    while left > 0:
        c = min(1900, left); chunks.append(c); left -= c
    st = dd.Stream(plan, max(chunks), nb)
    out = torch.full((nb, w.ndm, w.nsamp), -7, dtype=odt, device="cuda")
    pos = emitted = 0
    for c in chunks:
        if c == 0:
            continue
        chunk = Xd[:, :, pos:pos + c].contiguous()
        tmp = torch.empty((nb, w.ndm, c), dtype=odt, device="cuda")
        n = st.push(chunk, c, w.nchans * c, c, tmp, c, w.ndm * c)
        pos += c
        assert n == max(0, pos - ms) - emitted
        out[:, :, emitted:emitted + n] = tmp[:, :, :n]
        emitted += n
    torch.cuda.synchronize()
    assert emitted == w.nsamp
    assert torch.equal(out, one)
    for b in range(nb):
        assert_parity(w, xs[b], one[b].cpu().numpy())
    with pytest.raises(dd.DedispError) as e:
        st.push(Xd, total, 0, max(chunks) + 1, out, w.nsamp, 0)
    assert e.value.code == dd.DD_ERR_STATE
    st.destroy(); plan.destroy()


@pytest.mark.parametrize("dtype", ["f32", "u8"])
def test_one_shot_and_host_calls(dtype):
    import torch
    w = small(2, 128, 48, 20000 + 11, dtype=dtype)
    X, ms = make_case(w)
    odt = np.float32 if dtype == "f32" else np.int32
    Xd = torch.from_numpy(X).cuda()
    Dd = torch.empty((w.ndm, w.nsamp), dtype=torch.float32 if dtype == "f32" else torch.int32, device="cuda")
    f = dd.dd_dedisperse_f32 if dtype == "f32" else dd.dd_dedisperse_u8_i32
    f(Xd, w.nchans, w.nsamp, w.fch1, w.foff, w.tsamp, w.dm_list, Dd)
    D1 = Dd.cpu().numpy()
    assert_parity(w, X, D1)
    fh = dd.dd_dedisperse_f32_host if dtype == "f32" else dd.dd_dedisperse_u8_i32_host
    D2 = np.full((w.ndm, w.nsamp), -7, dtype=odt)
    fh(X, w.nchans, w.nsamp, w.fch1, w.foff, w.tsamp, w.dm_list, D2)      # pageable host memory
    assert np.array_equal(D1, D2)
    # pinned host memory through the plan form, twice (cached workspace)
    plan = dd.Plan(dd_dtype(w), w.nchans, w.fch1, w.foff, w.tsamp, w.dm_list)
    Xp = torch.from_numpy(X).pin_memory()
    Dp = torch.empty((w.ndm, w.nsamp), dtype=Dd.dtype).pin_memory()
    for _ in range(2):
        Dp.fill_(-7)
        plan.execute_host(Xp, X.shape[1], 0, Dp, w.nsamp, 0, w.nsamp, 1)
        assert np.array_equal(Dp.numpy(), D1)
    plan.destroy()


# ------------------------------------------------------------------ float32 partial-sum kernel, direct (aligned) path

@pytest.mark.parametrize("idx,nchans,ndm,nsamp", [(3, 517, 130, 2000), (4, 256, 200, 1500), (3, 64, 70, 5000), (3, 130, 70, 600)])
def test_ps_kernel_reads_aligned_input_directly(idx, nchans, ndm, nsamp):
    """16-byte aligned X with strides that are multiples of four elements is staged by TMA straight from
    the caller's buffer (no re-pitch copy): several DM tiles, several time tiles, ragged tails, a
    channel count that is not a multiple of the group size.

    The cases must be plans the partial-sum kernel takes (the test asserts kernel_for == DD_KERNEL_PS):
    `small()` keeps a workload's band, so 64 channels over config 4's 20 MHz at 418 MHz have delay steps of
    ~150 samples between adjacent channels at the top trial -- too many delay patterns per tile for shared
    memory once tiles hold 128 trials -- and such plans run the generic kernel (covered by
    test_shrunk_configs / test_large_dm_steps_fall_back_to_narrow_tiles through AUTO).  That is why the
    config-4 case here has 256 channels; the 64-channel case uses config 3's L-band (steps of a few samples)."""
    import torch
    w = small(idx, nchans, ndm, nsamp, dtype="f32")
    X, ms = make_case(w, pulses=2)
    stride = (w.nsamp + ms + 63) // 64 * 64
    plan = dd.Plan(dd.DD_F32, w.nchans, w.fch1, w.foff, w.tsamp, w.dm_list)
    Xd = torch.zeros((w.nchans, stride), dtype=torch.float32, device="cuda")
    Xd[:, :w.nsamp + ms] = torch.from_numpy(X).cuda()
    Dd = torch.full((w.ndm, w.nsamp), -7.0, dtype=torch.float32, device="cuda")
    assert plan.kernel_for(Xd, stride, 0, Dd, w.nsamp, 0, w.nsamp, 1) == dd.DD_KERNEL_PS
    plan.execute(Xd, stride, 0, Dd, w.nsamp, 0, w.nsamp, 1)
    torch.cuda.synchronize()
    D = Dd.cpu().numpy()
    assert_parity(w, X, D)
    # forced generic kernel on the same plan: both within tolerance of the oracle, and the
    # partial-sum result does not depend on the path the input took (re-pitched copy vs direct)
    D2 = gpu_dedisperse(w, X, dd.DD_KERNEL_PS)
    assert np.array_equal(D, D2)
    plan.destroy()


def test_config3_channels_and_trials_full_time_cut():
    # BASELINE.json configs[2] in the launch configuration bench.py times (4096 ch x 4096 DMs, float32,
    # partial-sum kernel, aligned direct path), cut to 8192 samples: sampled elements + whole rows
    import torch
    w = synth.scaled(synth.WORKLOADS[3], nsamp=8192)
    tab = oracle.shift_table(w.nchans, w.fch1, w.foff, w.tsamp, w.dm_list)
    ms = int(tab.max())
    X = synth.make_input(w, w.nsamp + ms)
    for d, t0, width in synth.pulse_plan(w, 5):
        synth.inject_pulse(X, t0, width, 0.25, tab[d])
    stride = (w.nsamp + ms + 63) // 64 * 64
    plan = dd.Plan(dd.DD_F32, w.nchans, w.fch1, w.foff, w.tsamp, w.dm_list)
    Xd = torch.zeros((w.nchans, stride), dtype=torch.float32, device="cuda")
    Xd[:, :w.nsamp + ms] = torch.from_numpy(X).cuda()
    Dd = torch.empty((w.ndm, w.nsamp), dtype=torch.float32, device="cuda")
    assert plan.kernel_for(Xd, stride, 0, Dd, w.nsamp, 0, w.nsamp, 1) == dd.DD_KERNEL_PS
    plan.execute(Xd, stride, 0, Dd, w.nsamp, 0, w.nsamp, 1)
    torch.cuda.synchronize()
    D = Dd.cpu().numpy()
    plan.destroy()
    assert_sampled_parity(w, X, D, n=100000, seed=3)
    rows = sorted({0, w.ndm - 1, w.ndm // 2, 63, 64} | {d for d, _, _ in synth.pulse_plan(w, 5)})
    assert_parity(w, X, D, rows=rows)


# ------------------------------------------------------------------ full sizes, bench configuration

def _full_size(idx):
    import torch
    w = synth.WORKLOADS[idx]
    tab = oracle.shift_table(w.nchans, w.fch1, w.foff, w.tsamp, w.dm_list)
    ms = int(tab.max())
    X = synth.make_input(w, w.nsamp + ms)
    for d, t0, width in synth.pulse_plan(w, 5):
        synth.inject_pulse(X, t0, width, 0.25 if w.dtype == "f32" else 8, tab[d])
    D = gpu_dedisperse(w, X, dd.DD_KERNEL_AUTO)        # the launch configuration bench.py times
    assert_sampled_parity(w, X, D, n=100000, seed=idx)
    assert_row_checksums(w, X, D, tab)
    rows = sorted({0, w.ndm - 1, w.ndm // 2} | {d for d, _, _ in synth.pulse_plan(w, 5)})
    assert_parity(w, X, D, rows=rows)
    return w, X, D, tab


def test_config2_full_size_sampled_rows_and_checksums():
    # BASELINE.json configs[1] as benchmarked: 1024 ch x 1024 DMs x 2^17 samples, uint8 -> int32
    w, X, D, tab = _full_size(2)
    assert np.array_equal(D[0], X[:, :w.nsamp].sum(axis=0, dtype=np.int64).astype(np.int32))   # DM = 0 row


def test_config2_full_size_every_element():
    # the metric's workload, complete: all 1024 x 131072 outputs of the launch bench.py times against a full
    # pass of the oracle (1.4e11 adds on the host cores), bit for bit
    w = synth.WORKLOADS[2]
    ms = oracle.max_shift(w.nchans, w.fch1, w.foff, w.tsamp, w.dm_list)
    X = synth.make_input(w, w.nsamp + ms)
    D = gpu_dedisperse(w, X, dd.DD_KERNEL_AUTO)
    want = oracle.dedisperse_u8(X, w.nsamp, w.fch1, w.foff, w.tsamp, w.dm_list)
    assert D.dtype == np.int32 and D.shape == want.shape
    assert np.array_equal(D, want)


# ------------------------------------------------------------------ configs 3-5 at full size, as bench.py launches them

def _sampled(w, X, d_idx, t_idx, got):
    if w.dtype == "u8":
        want = oracle.elements(X, w.fch1, w.foff, w.tsamp, w.dm_list, d_idx, t_idx)
        assert np.array_equal(got.astype(np.int64), want)
    else:
        want, A = oracle.elements(X, w.fch1, w.foff, w.tsamp, w.dm_list, d_idx, t_idx)
        err = np.abs(got.astype(np.float64) - want)
        assert np.all(err <= 1e-5 * A), (err / (1e-5 * A)).max()


def _sample_points(w, n, seed):
    g = np.random.default_rng(seed)
    di = g.integers(0, w.ndm, n)
    ti = g.integers(0, w.nsamp, n)
    # corners and the seams of the 64-trial x 512/1024-sample tiles
    di[:8] = [0, 0, w.ndm - 1, w.ndm - 1, 63, 64, min(w.ndm - 1, 127), min(w.ndm - 1, 128)]
    ti[:8] = [0, w.nsamp - 1, 0, w.nsamp - 1, 511, 512, 1023, 1024]
    return di, ti


FULL_PARITY = bool(int(os.environ.get("DD_FULL_PARITY", "0")))   # every-element passes of configs 3-5 (minutes of CPU)


def _every_element(w, X, Dd, label, block=64):
    """All ndm x nsamp outputs of one beam against the oracle's interchanged nest (pinned bit-identical to
    the literal nest), 64 trials at a time; returns the worst err / (1e-5 * A) (0 for uint8)."""
    worst = 0.0
    for r0 in range(0, w.ndm, block):
        rows = np.arange(r0, min(w.ndm, r0 + block), dtype=np.int32)
        worst = max(worst, assert_whole_rows(w, X, Dd[r0:r0 + len(rows)].cpu().numpy(), rows))
    print("FULL_PARITY %s: %d x %d = %d elements, worst err/(1e-5*A) = %.4f" % (
        label, w.ndm, w.nsamp, w.ndm * w.nsamp, worst))
    return worst


def test_config3_full_size_checksums_rows_and_samples():
    # BASELINE.json configs[2] exactly as bench.py times it: 4096 ch x 4096 DMs x 2^18 samples, float32,
    # one dd_execute on 16-byte aligned input (partial-sum kernel).  P7: prefix-sum checksum of EVERY trial
    # row; P8: whole rows for the first / last / every 64th trial, the tile seams and the pulse DMs;
    # P9: sampled elements; with DD_FULL_PARITY=1 every element.
    import torch
    w = synth.WORKLOADS[3]
    tab = oracle.shift_table(w.nchans, w.fch1, w.foff, w.tsamp, w.dm_list)
    ms = int(tab.max())
    X = synth.make_input(w, w.nsamp + ms)
    pulses = synth.pulse_plan(w, 5)
    for d, t0, width in pulses:
        synth.inject_pulse(X, t0, width, 0.25, tab[d])
    stride = (w.nsamp + ms + 63) // 64 * 64
    plan = dd.Plan(dd.DD_F32, w.nchans, w.fch1, w.foff, w.tsamp, w.dm_list)
    Xd = torch.zeros((w.nchans, stride), dtype=torch.float32, device="cuda")
    Xd[:, :w.nsamp + ms] = torch.from_numpy(X).cuda()
    Dd = torch.empty((w.ndm, w.nsamp), dtype=torch.float32, device="cuda")
    assert plan.kernel_for(Xd, stride, 0, Dd, w.nsamp, 0, w.nsamp, 1) == dd.DD_KERNEL_PS
    plan.execute(Xd, stride, 0, Dd, w.nsamp, 0, w.nsamp, 1)
    torch.cuda.synchronize()
    del Xd
    assert_row_checksums(w, X, Dd, tab)
    rows = p8_rows(w, pulses)
    assert_whole_rows(w, X, Dd[torch.from_numpy(rows).long().cuda()].cpu().numpy(), rows)
    di, ti = _sample_points(w, 40000, 33)
    got = Dd[torch.from_numpy(di).cuda(), torch.from_numpy(ti).cuda()].cpu().numpy()
    _sampled(w, X, di, ti, got)
    # the injected pulses peak at their trial and start sample (S/N ~ A sqrt(nchans) = 16 per sample)
    for d, t0, width in pulses:
        row = Dd[d].cpu().numpy()
        assert abs(int(np.argmax(np.convolve(row, np.ones(width), "valid"))) - t0) <= 1
    if FULL_PARITY:
        _every_element(w, X, Dd, w.name)
    plan.destroy()


def test_config4_full_size_batch_checksums_rows_and_samples():
    # BASELINE.json configs[3] as bench.py times it: 32 beams x 512 ch x 2048 DMs x 2^16 samples in ONE
    # dd_execute (grid.z = beam).  P7 on every trial row of ALL 32 beams, P8 whole rows and sampled
    # elements on three beams; with DD_FULL_PARITY=1 every element of those three beams.
    import torch
    w = synth.WORKLOADS[4]
    plan = dd.Plan(dd.DD_F32, w.nchans, w.fch1, w.foff, w.tsamp, w.dm_list)
    tab = oracle.shift_table(w.nchans, w.fch1, w.foff, w.tsamp, w.dm_list)
    ms = plan.max_shift()
    assert ms == int(tab.max()) == 9760
    stride = (w.nsamp + ms + 63) // 64 * 64
    Xd = torch.zeros((w.nbeams, w.nchans, stride), dtype=torch.float32, device="cuda")
    xs = []
    for b in range(w.nbeams):
        X = synth.make_input(w, w.nsamp + ms, beam=b)
        Xd[b, :, :w.nsamp + ms] = torch.from_numpy(X).cuda()
        xs.append(X)
    Dd = torch.empty((w.nbeams, w.ndm, w.nsamp), dtype=torch.float32, device="cuda")
    assert plan.kernel_for(Xd, stride, w.nchans * stride, Dd, w.nsamp, w.ndm * w.nsamp, w.nsamp, w.nbeams) == dd.DD_KERNEL_PS
    plan.execute(Xd, stride, w.nchans * stride, Dd, w.nsamp, w.ndm * w.nsamp, w.nsamp, w.nbeams)
    torch.cuda.synchronize()
    del Xd
    ws = synth.scaled(w, nbeams=1)
    for b in range(w.nbeams):
        assert_row_checksums(ws, xs[b], Dd[b], tab)
    rows = p8_rows(w)
    for b in (0, 13, 31):
        assert_whole_rows(ws, xs[b], Dd[b][torch.from_numpy(rows).long().cuda()].cpu().numpy(), rows)
        di, ti = _sample_points(w, 30000, 40 + b)
        got = Dd[b][torch.from_numpy(di).cuda(), torch.from_numpy(ti).cuda()].cpu().numpy()
        _sampled(w, xs[b], di, ti, got)
        if FULL_PARITY:
            _every_element(ws, xs[b], Dd[b], "%s beam %d" % (w.name, b))
    plan.destroy()


def test_config5_full_size_streamed_checksums_rows_and_samples():
    # BASELINE.json configs[4] as bench.py times it: 2048 ch uint8, 10000 DMs, 2^18 samples fed through
    # dd_stream_push in 4 chunks (the first carries maxshift extra samples).  Bit-exact: P7 on every trial
    # row of the concatenated output, P8 whole rows, sampled elements around the chunk seams; with
    # DD_FULL_PARITY=1 every element.
    import torch
    w = synth.WORKLOADS[5]
    plan = dd.Plan(dd.DD_U8, w.nchans, w.fch1, w.foff, w.tsamp, w.dm_list)
    tab = oracle.shift_table(w.nchans, w.fch1, w.foff, w.tsamp, w.dm_list)
    ms = plan.max_shift()
    assert ms == 37599                                               # golden maxshift of config 5
    X = synth.make_input(w, w.nsamp + ms)
    Xd = torch.from_numpy(X).cuda()
    Dd = torch.full((w.ndm, w.nsamp), -7, dtype=torch.int32, device="cuda")
    chunk = w.nsamp // w.nchunks
    st = dd.Stream(plan, chunk + ms, 1)
    pos = emitted = 0
    for k in range(w.nchunks):
        n_new = chunk + (ms if k == 0 else 0)
        n = st.push(Xd[:, pos:], X.shape[1], 0, n_new, Dd[:, emitted:], w.nsamp, 0)
        assert n == chunk
        pos += n_new
        emitted += n
    torch.cuda.synchronize()
    assert emitted == w.nsamp
    del Xd
    assert_row_checksums(w, X, Dd, tab)
    rows = p8_rows(w)
    assert_whole_rows(w, X, Dd[torch.from_numpy(rows).long().cuda()].cpu().numpy(), rows)
    di, ti = _sample_points(w, 40000, 55)
    ti[8:16] = [chunk - 1, chunk, 2 * chunk - 1, 2 * chunk, 3 * chunk - 1, 3 * chunk, chunk + 1, 3 * chunk + 1]
    got = Dd[torch.from_numpy(di).cuda(), torch.from_numpy(ti).cuda()].cpu().numpy()
    _sampled(w, X, di, ti, got)
    assert np.array_equal(Dd[0].cpu().numpy().astype(np.int64), X[:, :w.nsamp].sum(axis=0, dtype=np.int64))   # DM = 0 row
    if FULL_PARITY:
        _every_element(w, X, Dd, w.name)
    st.destroy(); plan.destroy()


# ------------------------------------------------------------------ plan-level hazards

def test_two_live_plans_do_not_undo_each_others_kernel_attributes():
    # a plan with a large shared-memory need, then a small plan and a one-shot call on the same kernel
    # instantiations, then the large plan again (the dynamic shared-memory attribute belongs to the
    # kernel function, not to a plan)
    import torch
    for dtype in ("f32", "u8"):
        big = small(3 if dtype == "f32" else 5, 512, 300, 3000, dtype=dtype)
        # same channel width and trial grid, fewer channels: a plan the same partial-sum kernels take with a
        # much smaller shared-memory need
        tiny = synth.scaled(big, nchans=32, ndm=130, nsamp=700)
        Xb, _ = make_case(big)
        Xt, _ = make_case(tiny)
        pb = dd.Plan(dd_dtype(big), big.nchans, big.fch1, big.foff, big.tsamp, big.dm_list)
        odt = torch.float32 if dtype == "f32" else torch.int32
        Xbd = torch.from_numpy(Xb).cuda()
        Db = torch.empty((big.ndm, big.nsamp), dtype=odt, device="cuda")
        pb.execute(Xbd, Xb.shape[1], 0, Db, big.nsamp, 0, big.nsamp, 1)
        torch.cuda.synchronize()
        first = Db.clone()
        pt = dd.Plan(dd_dtype(tiny), tiny.nchans, tiny.fch1, tiny.foff, tiny.tsamp, tiny.dm_list)
        Dt = gpu_dedisperse(tiny, Xt, dd.DD_KERNEL_AUTO)
        assert_parity(tiny, Xt, Dt)
        f = dd.dd_dedisperse_f32 if dtype == "f32" else dd.dd_dedisperse_u8_i32
        Dt2 = torch.empty((tiny.ndm, tiny.nsamp), dtype=odt, device="cuda")
        f(torch.from_numpy(Xt).cuda(), tiny.nchans, tiny.nsamp, tiny.fch1, tiny.foff, tiny.tsamp, tiny.dm_list, Dt2)
        assert np.array_equal(Dt2.cpu().numpy(), Dt)
        Db.fill_(-7)
        pb.execute(Xbd, Xb.shape[1], 0, Db, big.nsamp, 0, big.nsamp, 1)      # the older, larger plan still launches
        torch.cuda.synchronize()
        assert torch.equal(Db, first)
        assert_parity(big, Xb, Db.cpu().numpy())
        pt.destroy(); pb.destroy()


def test_many_beams_times_channels_stay_on_the_partial_sum_kernel():
    # 64 beams x 1024 channels = 65536 rows: more than a grid.y of the front end could hold (the rows are on
    # grid.x); AUTO must not drop to the generic kernel, and the result must stay exact
    import torch
    nb = 64
    w = synth.scaled(synth.WORKLOADS[2], ndm=64, nsamp=600, nbeams=nb)
    plan = dd.Plan(dd.DD_U8, w.nchans, w.fch1, w.foff, w.tsamp, w.dm_list)
    ms = plan.max_shift()
    total = w.nsamp + ms
    g = torch.Generator(device="cuda").manual_seed(5)
    Xd = torch.randint(0, 256, (nb, w.nchans, total), dtype=torch.uint8, device="cuda", generator=g)
    Dd = torch.empty((nb, w.ndm, w.nsamp), dtype=torch.int32, device="cuda")
    assert plan.kernel_for(Xd, total, w.nchans * total, Dd, w.nsamp, w.ndm * w.nsamp, w.nsamp, nb) == dd.DD_KERNEL_PS
    assert plan.launches_for(Xd, total, w.nchans * total, Dd, w.nsamp, w.ndm * w.nsamp, w.nsamp, nb) == 2
    plan.execute(Xd, total, w.nchans * total, Dd, w.nsamp, w.ndm * w.nsamp, w.nsamp, nb)
    torch.cuda.synchronize()
    ws = synth.scaled(w, nbeams=1)
    for b in (0, 31, 63):
        assert_parity(ws, Xd[b].cpu().numpy(), Dd[b].cpu().numpy())
    assert "dd_ps_u8_kernel" in plan.describe()
    plan.destroy()
    # a plan the partial-sum kernel cannot take says so
    coarse = small(1, 64, 70, 2500, dm_step=40.0)                    # 4480 cells: not a tiny plan either
    pc = dd.Plan(dd.DD_F32, coarse.nchans, coarse.fch1, coarse.foff, coarse.tsamp, coarse.dm_list)
    assert pc.kernel_for(0x1000, 1 << 20, 0, 0x2000, 2500, 0, 2500, 1) == dd.DD_KERNEL_GENERIC
    assert "unavailable" in pc.describe() and pc.launches_for(0x1000, 1 << 20, 0, 0x2000, 2500, 0, 2500, 1) == 1
    pc.destroy()


def test_execute_host_with_beams():
    import torch
    nb = 3
    for dtype in ("f32", "u8"):
        w = small(4, 128, 70, 9000 + 5, dtype=dtype, nbeams=nb)
        plan = dd.Plan(dd_dtype(w), w.nchans, w.fch1, w.foff, w.tsamp, w.dm_list)
        ms = plan.max_shift()
        total = w.nsamp + ms
        xs = np.stack([synth.make_input(w, total, beam=b) for b in range(nb)])
        Xp = torch.from_numpy(xs).pin_memory()
        Dp = torch.full((nb, w.ndm, w.nsamp), -7, dtype=torch.float32 if dtype == "f32" else torch.int32).pin_memory()
        plan.execute_host(Xp, total, w.nchans * total, Dp, w.nsamp, w.ndm * w.nsamp, w.nsamp, nb)
        ws = synth.scaled(w, nbeams=1)
        for b in range(nb):
            assert_parity(ws, xs[b], Dp[b].numpy())
        Dd = torch.empty((nb, w.ndm, w.nsamp), dtype=Dp.dtype, device="cuda")
        plan.execute(torch.from_numpy(xs).cuda(), total, w.nchans * total, Dd, w.nsamp, w.ndm * w.nsamp, w.nsamp, nb)
        torch.cuda.synchronize()
        assert torch.equal(Dd.cpu(), Dp)                                # host path == resident path, bit for bit
        plan.destroy()
    dd.dd_release_workspaces()


def test_uint8_partial_sum_kernel_takes_unaligned_output():
    # D rows that are not 16-byte aligned (odd row length, offset base): the partial-sum kernel flushes
    # element by element instead of falling back to the generic kernel; results stay bit-exact
    import torch
    w = small(2, 256, 70, 9000 + 37)
    X, ms = make_case(w, pulses=3)
    plan = dd.Plan(dd.DD_U8, w.nchans, w.fch1, w.foff, w.tsamp, w.dm_list)
    Xd = torch.from_numpy(X).cuda()
    buf = torch.full((1 + w.ndm * w.nsamp,), -7, dtype=torch.int32, device="cuda")
    Dd = buf[1:]
    assert plan.kernel_for(Xd, X.shape[1], 0, Dd, w.nsamp, 0, w.nsamp, 1) == dd.DD_KERNEL_PS
    plan.execute(Xd, X.shape[1], 0, Dd, w.nsamp, 0, w.nsamp, 1)
    torch.cuda.synchronize()
    assert int(buf[0]) == -7
    assert_parity(w, X, Dd.view(w.ndm, w.nsamp).cpu().numpy())
    plan.destroy()


# ------------------------------------------------------------------ seeded random shapes (all kernels through AUTO)

def _random_case(g, dtype):
    nchans = int(g.choice([1, 2, 3, 5, 8, 13, 31, 64, 100, 257, 300]))
    ndm = int(g.integers(1, 140))
    nsamp = int(g.integers(1, 2600))
    fch1 = float(g.uniform(150.0, 1600.0))
    band = float(g.uniform(0.01, 0.2)) * fch1                 # 1 % .. 20 % fractional bandwidth
    tsamp = float(g.choice([51.2e-6, 64e-6, 1e-4, 1e-3]))
    dm_step = float(g.choice([0.01, 0.05, 0.1, 0.25, 1.0]))
    return synth.scaled(synth.WORKLOADS[2], dtype=dtype, nchans=nchans, ndm=ndm, nsamp=nsamp, fch1=fch1,
                        foff=-band / nchans, tsamp=tsamp, dm_step=dm_step, nbeams=1)


@pytest.mark.parametrize("dtype", ["f32", "u8"])
def test_random_shapes_against_the_oracle(dtype):
    g = np.random.default_rng(20140128 + (dtype == "u8"))
    kinds = set()
    done = 0
    while done < 24:
        w = _random_case(g, dtype)
        ms = oracle.max_shift(w.nchans, w.fch1, w.foff, w.tsamp, w.dm_list)
        if ms > 60000 or (w.nsamp + ms) * w.nchans > 3e7:
            continue                                             # keep the oracle pass in seconds
        X = synth.make_input(synth.scaled(w, seed=int(g.integers(1, 1 << 30))), w.nsamp + ms)
        plan = dd.Plan(dd_dtype(w), w.nchans, w.fch1, w.foff, w.tsamp, w.dm_list)
        kinds.add(plan.kernel_for(0x1000, w.nsamp + ms, 0, 0x2000, w.nsamp, 0, w.nsamp, 1))
        plan.destroy()
        D = gpu_dedisperse(w, X, dd.DD_KERNEL_AUTO)
        assert_parity(w, X, D)
        done += 1
    assert dd.DD_KERNEL_PS in kinds and len(kinds) >= 2            # the draw exercises fast and fallback kernels


def test_many_random_plans_partial_sum_kernel_agrees_with_the_channel_vector_kernel():
    """Breadth beyond what the oracle can cover in seconds: 120 random plans (channel counts that are not multiples
    of the group size, sorted random and uniform DM lists, one or two beams, ragged sizes) through the float32
    partial-sum kernel and through the channel-vector kernel (itself compared with the oracle above); the two
    add in different orders, so they must agree within twice north_star's tolerance, |D1 - D2| <= 2e-5 * A."""
    import torch
    rng = np.random.default_rng(20261105)
    nps = 0
    for it in range(120):
        nch = int(rng.choice([16, 24, 37, 64, 100, 128, 200, 256, 333, 512]))
        ndm = int(rng.integers(1, 400))
        nsamp = int(rng.integers(1, 5000))
        fch1 = float(rng.choice([150.0, 418.0, 800.0, 1550.0]))
        band = float(rng.choice([5.0, 20.0, 100.0, 300.0])) * fch1 / 1550.0
        tsamp = float(rng.choice([51.2e-6, 64e-6, 1e-3]))
        step = float(rng.choice([0.01, 0.05, 0.1, 0.25, 1.0]))
        dms = np.sort(rng.uniform(0, step * ndm, ndm)) if it % 3 else np.arange(ndm) * step
        p = dd.Plan(dd.DD_F32, nch, fch1, -band / nch, tsamp, dms)
        ms = p.max_shift()
        if ms > 60000:
            p.destroy()
            continue
        nb = int(rng.integers(1, 3))
        stride = (nsamp + ms + 3) // 4 * 4
        X = torch.randn((nb, nch, stride), device="cuda")
        D1 = torch.empty((nb, ndm, nsamp), device="cuda")
        D2, A = torch.empty_like(D1), torch.empty_like(D1)
        a = lambda x, d: (x, stride, nch * stride, d, nsamp, ndm * nsamp, nsamp, nb)
        p.set_kernel(dd.DD_KERNEL_GENERIC)
        p.execute(*a(X, D2))
        p.execute(*a(X.abs(), A))
        try:
            p.set_kernel(dd.DD_KERNEL_PS)
        except dd.DedispError:                      # delay steps too coarse for shared partial sums
            p.destroy()
            continue
        assert p.kernel_for(*a(X, D1)) == dd.DD_KERNEL_PS
        p.execute(*a(X, D1))
        torch.cuda.synchronize()
        r = ((D1 - D2).abs() / (2e-5 * A + 1e-30)).max().item()
        assert r <= 1.0, (it, nch, ndm, nsamp, fch1, band, tsamp, step, r)
        nps += 1
        p.destroy()
    assert nps >= 60
