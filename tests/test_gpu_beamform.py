"""GPU parity of the coherent beamformer of row f4 (dd_beamform_power_u4) against
oracle/beamform.py, and the beamformer feeding the dedisperser on the device.

Tolerance: the 4-bit voltages are exact in fp16; every weight is carried as hi + lo fp16
terms with |W - hi - lo| <= 2^-22 |W| (+ 6e-8 absolute from fp16 subnormals); the tensor cores accumulate in
float32.  The beam voltage therefore errs by at most ~1e-6 S, S = sum_a |W||v|, and the detected power by
2 |b| 1e-6 S + (1e-6 S)^2 <= 1e-5 S^2 -- the bound the header states and this file asserts."""
import numpy as np
import pytest

import oracle
import paper_1401_8258_b200 as dd
from oracle import beamform as bf
from paper_1401_8258_b200 import synth

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module", autouse=True)
def _need_gpu():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"


def gpu_beamform(V, W, pad=0, beam_pad=0):
    import torch
    nch, nt, na = V.shape
    nb = W.shape[1]
    stride = nt + pad
    bs = nch * stride + beam_pad
    Wd = torch.from_numpy(np.ascontiguousarray(W.astype(np.complex64)).view(np.float32)).cuda()
    Vd = torch.from_numpy(V).cuda()
    P = torch.full((nb * bs,), -7.0, dtype=torch.float32, device="cuda")
    dd.dd_beamform_power_u4(Vd, na, nch, nt, Wd, nb, P, stride, bs)
    torch.cuda.synchronize()
    h = P.cpu().numpy()
    out = np.empty((nb, nch, nt), dtype=np.float32)
    for b in range(nb):
        v = h[b * bs: b * bs + nch * stride].reshape(nch, stride)
        assert np.all(v[:, nt:] == -7.0) and np.all(h[b * bs + nch * stride:(b + 1) * bs] == -7.0)
        out[b] = v[:, :nt]
    return out


@pytest.mark.parametrize("nch,nt,na,nb", [(4, 300, 32, 16), (3, 1000 + 13, 32, 5), (2, 64, 8, 1), (5, 257, 4, 3),
                                          (2, 500, 64, 24), (1, 130, 36, 9), (2, 1, 32, 16),
                                          (2, 300, 128, 40),     # four K atoms, two beam groups (tcgen05 kernel)
                                          (1, 200, 132, 10)])    # more than 128 antennas: the warp-level MMA kernel
def test_against_the_oracle(nch, nt, na, nb):
    g = np.random.default_rng(nch * 1000 + nt + na + nb)
    V = g.integers(0, 256, (nch, nt, na), dtype=np.uint8)
    W = (g.standard_normal((nch, nb, na)) + 1j * g.standard_normal((nch, nb, na))) * g.uniform(0.01, 2.0, (nch, nb, 1))
    W = W.astype(np.complex64)                                           # the weights the device receives
    want, S = bf.beamform_power(V, W)
    got = gpu_beamform(V, W, pad=3, beam_pad=5)
    err = np.abs(got.astype(np.float64) - want)
    assert np.all(err <= 1e-5 * S ** 2), (err / (1e-5 * S ** 2)).max()
    print("beamformer worst err / (1e-5 S^2) = %.3g" % (err / (1e-5 * S ** 2)).max())


def test_extreme_voltages_and_unit_weights_are_exact():
    # every byte value, weights +-1 and +-i (exact in fp16): integer arithmetic, exact result
    V = np.arange(256, dtype=np.uint8).reshape(1, 8, 32)
    g = np.random.default_rng(3)
    W = g.choice(np.array([1, -1, 1j, -1j]), size=(1, 16, 32)).astype(np.complex64)
    want, _ = bf.beamform_power(V, W)
    assert np.array_equal(gpu_beamform(V, W).astype(np.float64), want)


def test_beams_feed_the_dedisperser_on_the_device():
    # BEST-II-like: 32 antennas, 20 MHz in 64 channels here, 8 beams; a dispersed broadband pulse arrives as a
    # plane wave from the direction of beam 5: beamform on the device, dedisperse the 8 beam filterbanks in ONE
    # multi-beam dd_execute on the beamformer's output buffer, and find the pulse in beam 5 at its DM -- the same
    # chain through the two oracles agrees element by element
    import torch
    nch, na, nb, ndm, nsamp = 64, 32, 8, 24, 1500
    w = synth.scaled(synth.WORKLOADS[2], dtype="f32", nchans=nch, foff=-20.0 / nch, ndm=ndm, dm_step=4.0, nsamp=nsamp)
    tab = oracle.shift_table(w.nchans, w.fch1, w.foff, w.tsamp, w.dm_list)
    ms = int(tab.max())
    nt = nsamp + ms
    g = np.random.default_rng(8)
    freqs = w.fch1 + np.arange(nch) * w.foff
    pos = np.zeros((na, 3))
    pos[:, 0] = np.arange(na) * 0.36                                     # ~half a wavelength at 418 MHz
    th = np.deg2rad(np.linspace(-20, 20, nb))
    dirs = np.stack([np.sin(th), np.zeros(nb), np.cos(th)], axis=1)
    W = bf.steering_weights(freqs, pos, dirs).astype(np.complex64)       # [nch][nb][na]
    z = g.standard_normal((nch, nt, na)) + 1j * g.standard_normal((nch, nt, na))
    src = bf.steering_weights(freqs, pos, dirs[[5]])[:, 0, :].conj()     # plane wave from beam 5's direction
    d_true, t_true, width = 17, 600, 6
    for c in range(nch):
        a = t_true + tab[d_true, c]
        ph = np.exp(2j * np.pi * g.random(width))
        z[c, a:a + width, :] += 2.0 * src[c][None, :] * ph[:, None]
    V = bf.encode_voltages(np.clip(np.rint(z.real), -8, 7) + 1j * np.clip(np.rint(z.imag), -8, 7))
    stride = (nt + 3) // 4 * 4
    Wd = torch.from_numpy(np.ascontiguousarray(W).view(np.float32)).cuda()
    Pd = torch.zeros((nb, nch, stride), dtype=torch.float32, device="cuda")
    dd.dd_beamform_power_u4(torch.from_numpy(V).cuda(), na, nch, nt, Wd, nb, Pd, stride, nch * stride)
    plan = dd.Plan(dd.DD_F32, w.nchans, w.fch1, w.foff, w.tsamp, w.dm_list)
    Dd = torch.empty((nb, ndm, nsamp), dtype=torch.float32, device="cuda")
    plan.execute(Pd, stride, nch * stride, Dd, nsamp, ndm * nsamp, nsamp, nb)
    torch.cuda.synchronize()
    D = Dd.cpu().numpy()
    b, d, t = np.unravel_index(D.argmax(), D.shape)
    assert b == 5 and abs(d - d_true) <= 1 and t_true <= t < t_true + width
    # the oracle chain: beam power (float64) -> float32 filterbank -> dedispersion oracle
    Pw, S = bf.beamform_power(V, W)
    assert np.all(np.abs(Pd.cpu().numpy()[:, :, :nt] - Pw) <= 1e-5 * S ** 2)
    for beam in (0, 5):
        want, A = oracle.dedisperse_f32(Pw[beam].astype(np.float32), nsamp, w.fch1, w.foff, w.tsamp, w.dm_list)
        # dedispersion tolerance on its own input plus the beamformer's tolerance summed along the same tracks
        extra, _ = oracle.dedisperse_f32((1e-5 * S[beam] ** 2).astype(np.float32), nsamp, w.fch1, w.foff, w.tsamp, w.dm_list)
        assert np.all(np.abs(D[beam] - want) <= 1e-5 * A + 1.001 * extra)
    plan.destroy()


def test_argument_errors():
    import torch
    V = torch.zeros((2, 10, 8), dtype=torch.uint8, device="cuda")
    W = torch.zeros((2, 3, 8, 2), dtype=torch.float32, device="cuda")
    P = torch.zeros((3, 2, 10), dtype=torch.float32, device="cuda")
    for args in [(V, 6, 2, 10, W, 3, P, 10, 20), (V, 8, 2, 10, W, 0, P, 10, 20), (V, 8, 2, 10, W, 3, P, 5, 20),
                 (V, 8, 2, 10, W, 3, P, 10, 5), (None, 8, 2, 10, W, 3, P, 10, 20)]:
        with pytest.raises(dd.DedispError) as e:
            dd.dd_beamform_power_u4(*args)
        assert e.value.code == dd.DD_ERR_BAD_ARG
    P.fill_(-7.0)
    dd.dd_beamform_power_u4(V, 8, 2, 0, W, 3, P, 10, 20)                  # nsamp = 0: nothing written
    torch.cuda.synchronize()
    assert bool((P == -7.0).all())
