"""GPU parity of the approximate variants f2 (time binning, subband dedispersion)
against oracle/approx.py.  Tolerance: every stage is one of the exact float32 kernels, whose
error is bounded by 1e-5 x the sum of the magnitudes it adds; a second stage adds the same again on its own
inputs, so |D_gpu - D_oracle| <= 2e-5 * A with A the same two steps applied to |X| (one stage: 1e-5 * A)."""
import numpy as np
import pytest

import oracle
import paper_1401_8258_b200 as dd
from oracle import approx
from paper_1401_8258_b200 import synth

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module", autouse=True)
def _need_gpu():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"


def test_downsample2():
    import torch
    g = np.random.default_rng(1)
    for nrows, n, off in [(3, 1001, 0), (5, 4096, 1), (1, 1, 0), (2, 2, 3)]:
        X = g.standard_normal((nrows, n + 5)).astype(np.float32)
        buf = torch.from_numpy(np.r_[np.zeros(off, np.float32), X.ravel()]).cuda()
        Y = torch.full((nrows, n // 2 + 3), -7.0, dtype=torch.float32, device="cuda")
        dd.dd_downsample2_f32(buf[off:], Y, nrows, n, n + 5, n // 2 + 3)
        torch.cuda.synchronize()
        want = (X[:, 0:2 * (n // 2):2] + X[:, 1:2 * (n // 2):2])
        got = Y.cpu().numpy()
        assert np.array_equal(got[:, :n // 2], want) and np.all(got[:, n // 2:] == -7.0)
        assert np.allclose(want, approx.downsample2(X[:, :n]), rtol=1e-6, atol=1e-6)


@pytest.mark.parametrize("nchans,ndm,dm_step,nsamp,max_level", [(128, 60, 2.0, 4096, 8), (64, 40, 5.0, 2048 + 64, 2),
                                                                 (256, 33, 0.5, 3000, 8)])
def test_time_binning_against_the_oracle(nchans, ndm, dm_step, nsamp, max_level):
    import torch
    w = synth.scaled(synth.WORKLOADS[4], nbeams=1, nchans=nchans, foff=-20.0 / nchans, ndm=ndm, dm_step=dm_step, nsamp=nsamp)
    dms = w.dm_list
    tb = dd.TimeBin(w.nchans, w.fch1, w.foff, w.tsamp, dms, 0.0, max_level)
    dg = approx.diagonal_dm(w.nchans, w.fch1, w.foff, w.tsamp)
    assert dd.dd_diagonal_dm(w.nchans, w.fch1, w.foff, w.tsamp) == dg
    lv = tb.levels()
    assert np.array_equal(lv, approx.timebin_levels(dms, dg, max_level))
    n_in = tb.input_samples(w.nsamp)
    assert n_in == approx.timebin_input_samples(w.nchans, w.fch1, w.foff, w.tsamp, dms, w.nsamp, dg, max_level)
    X = synth.make_input(w, n_in)
    tab = oracle.shift_table(w.nchans, w.fch1, w.foff, w.tsamp, dms)
    synth.inject_pulse(X, w.nsamp // 3, 32, 0.5, tab[ndm - 2])
    Xd = torch.from_numpy(X).cuda()
    Dd = torch.full((ndm, w.nsamp + 7), -7.0, dtype=torch.float32, device="cuda")
    tb.execute(Xd, n_in, n_in, Dd, w.nsamp + 7, w.nsamp)
    torch.cuda.synchronize()
    D = Dd.cpu().numpy()
    out, scale, lvo = approx.timebin_dedisperse(X, w.nsamp, w.fch1, w.foff, w.tsamp, dms, max_level=max_level)
    assert lv.max() >= 1                                                        # the case does bin
    for d in range(ndm):
        n = w.nsamp >> int(lv[d])
        err = np.abs(D[d, :n].astype(np.float64) - out[d])
        assert np.all(err <= 1e-5 * scale[d]), (d, (err / (1e-5 * scale[d])).max())
        assert np.all(D[d, n:] == -7.0)                                         # the rest of the row is not written
    tb.destroy()


@pytest.mark.parametrize("nchans,ndm,nsamp,ncs,nds", [(128, 60, 3000, 16, 8), (96, 37, 2000 + 11, 32, 5), (200, 50, 2500, 7, 4),
                                                      (64, 20, 1500, 64, 1), (48, 24, 1200, 1, 6)])
def test_subband_against_the_oracle(nchans, ndm, nsamp, ncs, nds):
    import torch
    w = synth.scaled(synth.WORKLOADS[2], dtype="f32", nchans=nchans, foff=-20.0 / nchans, ndm=ndm, nsamp=nsamp, dm_step=0.5)
    dms = w.dm_list
    sb = dd.Subband(w.nchans, w.fch1, w.foff, w.tsamp, dms, ncs, nds)
    ms1, ms2 = approx.subband_max_shifts(w.nchans, w.fch1, w.foff, w.tsamp, dms, ncs, nds)
    assert sb.max_shift() == ms1 + ms2
    total = w.nsamp + ms1 + ms2
    X = synth.make_input(w, total)
    tab = oracle.shift_table(w.nchans, w.fch1, w.foff, w.tsamp, dms)
    synth.inject_pulse(X, w.nsamp // 2, 4, 1.0, tab[ndm // 2])
    Xd = torch.from_numpy(X).cuda()
    Dd = torch.full((ndm, w.nsamp), -7.0, dtype=torch.float32, device="cuda")
    sb.execute(Xd, total, Dd, w.nsamp, w.nsamp)
    torch.cuda.synchronize()
    D = Dd.cpu().numpy()
    want, A = approx.subband_dedisperse(X, w.nsamp, w.fch1, w.foff, w.tsamp, dms, ncs, nds)
    err = np.abs(D.astype(np.float64) - want)
    assert np.all(err <= 2e-5 * A), (err / (2e-5 * A)).max()
    if ncs == nchans and nds == 1 or ncs == 1:
        # the limits in which the method is exact: same result as the exact plan (oracle tolerance), and for
        # one subband / own nominal DMs the very same bits
        exact, Ae = oracle.dedisperse_f32(X, w.nsamp, w.fch1, w.foff, w.tsamp, dms)
        assert np.all(np.abs(D - exact) <= 1e-5 * Ae)
        if ncs == nchans:
            plan = dd.Plan(dd.DD_F32, w.nchans, w.fch1, w.foff, w.tsamp, dms)
            # the composite runs its (few-channel, few-trial) plans over whole observations and therefore takes the
            # partial-sum kernel where the plan allows it, else the channel-vector kernel -- never the direct
            # kernel AUTO gives tiny plans; the same choice here must give the same bits
            try:
                plan.set_kernel(dd.DD_KERNEL_PS)
            except dd.DedispError:
                plan.set_kernel(dd.DD_KERNEL_GENERIC)
            De = torch.empty((ndm, w.nsamp), dtype=torch.float32, device="cuda")
            plan.execute(Xd, total, 0, De, w.nsamp, 0, w.nsamp, 1)
            torch.cuda.synchronize()
            assert torch.equal(De, Dd)
            plan.destroy()
    sb.destroy()


def test_subband_config2_shape_full_size():
    # the shape of BASELINE.json configs[1] as float32 (1024 ch x 1024 trials x 2^17 samples), 32-channel
    # subbands, 16 trials per nominal DM: every element against the oracle's two steps
    import torch
    w = synth.scaled(synth.WORKLOADS[2], dtype="f32")
    dms = w.dm_list
    sb = dd.Subband(w.nchans, w.fch1, w.foff, w.tsamp, dms, 32, 16)
    total = w.nsamp + sb.max_shift()
    X = synth.make_input(w, total)
    Xd = torch.from_numpy(X).cuda()
    Dd = torch.empty((w.ndm, w.nsamp), dtype=torch.float32, device="cuda")
    sb.execute(Xd, total, Dd, w.nsamp, w.nsamp)
    torch.cuda.synchronize()
    want, A = approx.subband_dedisperse(X, w.nsamp, w.fch1, w.foff, w.tsamp, dms, 32, 16)
    worst = 0.0
    for r0 in range(0, w.ndm, 128):
        err = np.abs(Dd[r0:r0 + 128].cpu().numpy().astype(np.float64) - want[r0:r0 + 128])
        worst = max(worst, float((err / (2e-5 * A[r0:r0 + 128])).max()))
    assert worst <= 1.0, worst
    sb.destroy()


def test_argument_errors():
    dms = np.arange(10) * 1.0
    with pytest.raises(dd.DedispError) as e:
        dd.Subband(64, 400.0, -0.1, 1e-4, dms[::-1].copy(), 8, 2)               # decreasing DM list (R30)
    assert e.value.code == dd.DD_ERR_BAD_ARG
    with pytest.raises(dd.DedispError):
        dd.Subband(64, 400.0, -0.1, 1e-4, dms, 0, 2)
    with pytest.raises(dd.DedispError):
        dd.TimeBin(64, 400.0, -0.1, 1e-4, dms[::-1].copy())
    with pytest.raises(dd.DedispError):
        dd.TimeBin(64, 400.0, 0.1, 1e-4, dms)                                   # foff > 0
    tb = dd.TimeBin(64, 400.0, -0.1, 1e-4, dms)
    with pytest.raises(dd.DedispError):
        tb.execute(0x1000, 10, 10, 0x2000, 100, 100)                            # input shorter than required
    tb.destroy()
