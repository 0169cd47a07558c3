"""GPU parity of the RFI front end f3 (dd_rfi_mitigate) against oracle/rfi.py.

Tolerances: the device path evaluates row / window / spectrum means, the polynomial fit and
every threshold comparison in double, like the oracle, so averaged bandpass, fit, RMSE, mu and sigma agree to
~1e-12 relative (different summation order; normal equations in a Legendre basis against numpy's SVD least
squares), flags are IDENTICAL unless a mean lies within 1e-9 (relative) of its threshold -- the tests assert
their cases keep clear of that -- and the output, rounded once from double to float32, satisfies
|out - oracle| <= 2^-23 |oracle| + 1e-10 max|B|."""
import numpy as np
import pytest

import paper_1401_8258_b200 as dd
from oracle import rfi

from test_rfi_pins import rfi_test_buffer

pytestmark = pytest.mark.gpu

EPS32 = 2.0 ** -23


@pytest.fixture(scope="module", autouse=True)
def _need_gpu():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"


def run(Xs, order, window, t_chan, t_spec, pad=0, beam_pad=0):
    """Xs: list of per-beam arrays [nchans][n] -> per-beam dicts like oracle.rfi.mitigate's."""
    import torch
    nb, (nch, n) = len(Xs), Xs[0].shape
    stride = n + pad
    bs = nch * stride + beam_pad
    buf = torch.full((nb * bs,), -7.0, dtype=torch.float32, device="cuda")
    for b, X in enumerate(Xs):
        buf[b * bs: b * bs + nch * stride].view(nch, stride)[:, :n] = torch.from_numpy(X).cuda()
    nwin = (n + window - 1) // window
    bp = torch.zeros((nb, nch), dtype=torch.float64, device="cuda")
    fit = torch.zeros((nb, nch), dtype=torch.float64, device="cuda")
    st = torch.zeros((nb, 4), dtype=torch.float64, device="cuda")
    cf = torch.full((nb, nch, nwin), 9, dtype=torch.uint8, device="cuda")
    sf = torch.full((nb, n), 9, dtype=torch.uint8, device="cuda")
    prm = dd.dd_rfi_params(order, window, t_chan, t_spec)
    dd.dd_rfi_mitigate(buf, nch, n, stride, bs, nb, prm, bp, fit, st, cf, sf)
    torch.cuda.synchronize()
    h = buf.cpu().numpy()
    out = []
    for b in range(nb):
        v = h[b * bs: b * bs + nch * stride].reshape(nch, stride)
        assert np.all(v[:, n:] == -7.0) and np.all(h[b * bs + nch * stride:(b + 1) * bs] == -7.0)   # padding untouched
        s = st[b].cpu().numpy()
        out.append({"out": v[:, :n].copy(), "bandpass": bp[b].cpu().numpy(), "fit": fit[b].cpu().numpy(),
                    "rmse": s[0], "fit_mean": s[1], "spec_mu": s[2], "spec_sigma": s[3],
                    "chan_flags": cf[b].cpu().numpy().astype(bool), "spec_flags": sf[b].cpu().numpy().astype(bool)})
    return out


def compare(X, got, order, window, t_chan, t_spec):
    want = rfi.mitigate(X, order, window, t_chan, t_spec)
    scale = np.abs(want["fit"]).max() + 1e-30
    assert np.abs(got["bandpass"] - want["bandpass"]).max() <= 1e-12 * scale
    assert np.abs(got["fit"] - want["fit"]).max() <= 1e-9 * scale
    assert abs(got["rmse"] - want["rmse"]) <= 1e-9 * scale
    assert abs(got["fit_mean"] - want["fit"].mean()) <= 1e-9 * scale
    # the cases must keep clear of the thresholds, else flags could legitimately differ
    n = X.shape[1]
    starts = np.arange(0, n, window)
    M = np.add.reduceat(X.astype(np.float64), starts, axis=1) / np.minimum(window, n - starts)[None, :]
    margin = np.abs(np.abs(M - want["fit"][:, None]) - t_chan * want["rmse"])
    assert margin.min() > 1e-7 * scale, "test case too close to the channel threshold"
    assert np.array_equal(got["chan_flags"], want["chan_flags"])
    assert abs(got["spec_mu"] - want["spec_mu"]) <= 1e-9 * scale and abs(got["spec_sigma"] - want["spec_sigma"]) <= 1e-9 * scale
    assert np.array_equal(got["spec_flags"], want["spec_flags"])
    err = np.abs(got["out"].astype(np.float64) - want["out"])
    tol = EPS32 * np.abs(want["out"]) + 1e-10 * scale
    assert np.all(err <= tol), (err / tol).max()
    return want


def noisy(seed, nch, n, level=20.0):
    g = np.random.default_rng(seed)
    x = rfi.channel_abscissa(nch)
    shape = 1.0 + 0.2 * x - 0.25 * x ** 2 + 0.02 * np.sin(9 * x)
    X = (g.standard_normal((nch, n)) + level) * shape[:, None]
    X[nch // 3, : n // 2] += 4.0                                      # narrowband, half the buffer
    X[:, n // 5: n // 5 + 7] += 3.0                                   # broadband burst
    X[(2 * nch) // 3, n - 40:] -= 15.0                                # a drop-out at the very end (two-sided test)
    return X.astype(np.float32)


@pytest.mark.parametrize("nch,n,order,window", [(64, 4096, 3, 256), (200, 5000 + 37, 4, 512), (33, 777, 0, 100),
                                                 (512, 9000, 8, 64), (7, 300, 2, 1), (1, 500, 0, 50), (96, 40, 2, 64)])
def test_against_the_oracle(nch, n, order, window):
    X = noisy(nch * 7 + n, nch, n)
    got = run([X], order, window, 5.0, 4.0, pad=3)[0]
    want = compare(X, got, order, window, 5.0, 4.0)
    if nch >= 64 and n >= 4096 and order >= 3:
        assert want["chan_flags"].any() and want["spec_flags"].any()   # the case exercises both stages


@pytest.mark.parametrize("nch,n,order,window", [(64, 4099, 3, 256), (128, 6001, 4, 512), (256, 5000, 2, 100),
                                                 (512, 9002, 8, 64), (1024, 3003, 4, 12), (64, 300, 1, 512)])
def test_against_the_oracle_on_aligned_rows(nch, n, order, window):
    """16-byte aligned rows, window % 4 == 0: the first pass is the fused one (window sums + column sums of tiles of
    8 / 16 / 32 / 64 channels), the spectrum means come from the column sums except in windows with replaced
    channels; ragged lengths, a last window shorter than the rest, a window longer than the series."""
    X = noisy(nch * 5 + n, nch, n)
    got = run([X], order, window, 5.0, 4.0, pad=(-n) % 4)[0]
    want = compare(X, got, order, window, 5.0, 4.0)
    if n >= 4096 and order >= 3:
        assert want["chan_flags"].any() and want["spec_flags"].any()
    # several beams, padded aligned strides
    Xs = [noisy(nch + n + b, nch, n) for b in range(2)]
    for Xb, gb in zip(Xs, run(Xs, order, window, 5.0, 4.0, pad=(-n) % 4 + 8, beam_pad=12)):
        compare(Xb, gb, order, window, 5.0, 4.0)


def test_aligned_rows_with_every_channel_replaced_in_some_windows():
    """Fused first pass, worst case for the per-window lists of replaced channels: a broadband burst that lasts two
    whole windows replaces ALL channels there (and in the neighbouring windows); a narrowband interferer keeps every
    window of the buffer in the list path."""
    nch, n, window = 256, 8192 + 40, 256
    X = noisy(77, nch, n)
    X[:, 3 * window: 5 * window] += 6.0
    X[10, :] += 5.0
    got = run([X], 3, window, 5.0, 4.0, pad=(-n) % 4)[0]
    want = compare(X, got, 3, window, 5.0, 4.0)
    assert want["chan_flags"][:, 2:6].all() and want["chan_flags"][10].all()


def test_beams_and_strides():
    Xs = [noisy(100 + b, 48, 3000) for b in range(3)]
    res = run(Xs, 3, 128, 5.0, 4.0, pad=5, beam_pad=11)
    for X, got in zip(Xs, res):
        compare(X, got, 3, 128, 5.0, 4.0)


def test_section_3_3_4_recipe_on_the_device():
    # the thesis' own RFI test: same flags and corrected spectra as the oracle, the
    # narrowband channels end at exactly 0, the dispersed pulse is untouched
    X, info = rfi_test_buffer()
    got = run([X], 4, 512, 7.0, 5.0)[0]
    want = compare(X, got, 4, 512, 7.0, 5.0)
    assert got["chan_flags"][300:304].all() and not got["out"][300:304][:, ~got["spec_flags"]].any()
    p0, w10, tab = info["pulse"]
    for c in (0, 250, 511):
        seg = slice(p0 + tab[c], p0 + tab[c] + w10)
        assert np.array_equal(got["out"][c, seg], (X[c, seg].astype(np.float64) - got["fit"][c]).astype(np.float32))


def test_config2_shaped_buffer_full_size():
    # 1024 channels x (2^17 + 4883) samples float32: the input shape of BASELINE.json configs[1], every element
    X = noisy(2, 1024, (1 << 17) + 4883)
    got = run([X], 4, 512, 7.0, 5.0)[0]
    compare(X, got, 4, 512, 7.0, 5.0)


def test_argument_errors_and_empty_input():
    import torch
    X = torch.zeros((4, 100), dtype=torch.float32, device="cuda")
    ok = dict(poly_order=2, window=10, t_chan=5.0, t_spec=5.0)
    for bad in (dict(poly_order=-1), dict(poly_order=13), dict(window=0), dict(t_chan=-1.0), dict(t_spec=float("nan"))):
        kw = dict(ok, **bad)
        with pytest.raises(dd.DedispError) as e:
            dd.dd_rfi_mitigate(X, 4, 100, 100, 0, 1, dd.dd_rfi_params(kw["poly_order"], kw["window"], kw["t_chan"], kw["t_spec"]))
        assert e.value.code == dd.DD_ERR_BAD_ARG
    with pytest.raises(dd.DedispError):
        dd.dd_rfi_mitigate(X, 4, 100, 50, 0, 1, dd.dd_rfi_params(2, 10, 5.0, 5.0))       # stride < nsamp
    X.fill_(-7.0)
    dd.dd_rfi_mitigate(X, 4, 0, 100, 0, 1, dd.dd_rfi_params(2, 10, 5.0, 5.0))             # nsamp = 0: nothing written
    torch.cuda.synchronize()
    assert bool((X == -7.0).all())
    # a constant buffer: RMSE ~0, output ~0 (the fit reproduces the constant to rounding)
    X.fill_(3.5)
    dd.dd_rfi_mitigate(X, 4, 100, 100, 0, 1, dd.dd_rfi_params(2, 10, 5.0, 5.0))
    torch.cuda.synchronize()
    assert float(X.abs().max()) < 1e-12
