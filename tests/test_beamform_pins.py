"""Pins for the beamformer oracle (oracle/beamform.py; eq 5.1, Alg. 2), CPU only."""
import numpy as np

from oracle import beamform as bf


def test_nibble_decoding_by_hand():
    # low nibble real, high nibble imaginary, 4-bit two's complement (R34)
    assert bf.decode_voltages([0x00, 0x7F, 0x80, 0x18, 0xF1, 0x97]).tolist() == [0, -1 + 7j, -8j, -8 + 1j, 1 - 1j, 7 - 7j]
    z = np.array([[3 - 4j, -8 + 7j], [0, -1 - 1j]])
    assert np.array_equal(bf.decode_voltages(bf.encode_voltages(z)), z)
    assert np.array_equal(bf.encode_voltages(bf.decode_voltages(np.arange(256, dtype=np.uint8))), np.arange(256))


def test_explicit_loops_and_single_antenna():
    g = np.random.default_rng(0)
    nf, nt, na, nb = 3, 5, 6, 4
    V = g.integers(0, 256, (nf, nt, na), dtype=np.uint8)
    W = g.standard_normal((nf, nb, na)) + 1j * g.standard_normal((nf, nb, na))
    P, S = bf.beamform_power(V, W)
    v = bf.decode_voltages(V)
    for b in range(nb):
        for f in range(nf):
            for t in range(nt):
                acc = sum(W[f, b, a] * v[f, t, a] for a in range(na))            # Alg. 2: one accumulator per beam
                assert abs(P[b, f, t] - abs(acc) ** 2) < 1e-9
                assert abs(S[b, f, t] - sum(abs(W[f, b, a]) * abs(v[f, t, a]) for a in range(na))) < 1e-12
    # one antenna, unit weight: the detected power of the voltage itself
    P, _ = bf.beamform_power(V[:, :, :1], np.ones((nf, 1, 1)))
    assert np.array_equal(P[0], v[:, :, 0].real ** 2 + v[:, :, 0].imag ** 2)


def test_coherent_gain_and_array_factor_eq_5_1():
    c = 299792458.0
    na, f_mhz = 16, 408.0
    lam = c / (f_mhz * 1e6)
    pos = np.zeros((na, 3))
    pos[:, 0] = np.arange(na) * lam / 2                                          # uniform line array, half-wavelength spacing
    th0 = np.deg2rad(12.0)
    src = np.array([np.sin(th0), 0.0, np.cos(th0)])
    # a plane wave of amplitude 4 from direction th0, quantised on the 4-bit grid only through rounding of the phase term
    wave = 4.0 * bf.steering_weights([f_mhz], pos, src[None])[0, 0].conj()      # exp(+i k0.r_a)
    thetas = np.deg2rad(np.linspace(-60, 60, 241))
    dirs = np.stack([np.sin(thetas), np.zeros_like(thetas), np.cos(thetas)], axis=1)
    W = bf.steering_weights([f_mhz], pos, dirs)                                  # [1][nb][na]
    b = np.einsum("ba,a->b", W[0], wave)
    # closed form of eq 5.1 for identical elements: |sum_n exp(i n psi)|^2 = sin^2(N psi / 2) / sin^2(psi / 2)
    psi = np.pi * (np.sin(th0) - np.sin(thetas))
    with np.errstate(divide="ignore", invalid="ignore"):
        af = np.where(np.abs(psi) < 1e-12, float(na) ** 2, np.sin(na * psi / 2) ** 2 / np.sin(psi / 2) ** 2)
    assert np.abs(np.abs(b) ** 2 - 16.0 * af).max() < 1e-8
    # through the full oracle with 4-bit voltages: the beam pointed at the source has the coherent gain N^2
    # over one antenna, random pointing ~N
    g = np.random.default_rng(1)
    nt = 4000
    phase = np.exp(2j * np.pi * g.random(nt))                                    # the source's own random phase per sample
    z = np.rint(wave[None, :] * phase[:, None])                                  # integer grid, |.| <= 4 sqrt 2 < 8
    V = bf.encode_voltages(z)[None]                                              # [1][nt][na]
    on = bf.steering_weights([f_mhz], pos, src[None])
    off = bf.steering_weights([f_mhz], pos, dirs[[20]])                          # a direction far from the source
    P_on, _ = bf.beamform_power(V, on)
    P_off, _ = bf.beamform_power(V, off)
    one = np.mean(np.abs(z[:, 0]) ** 2)
    assert abs(P_on.mean() / (na ** 2 * one) - 1.0) < 0.05                       # coherent: N^2
    assert P_off.mean() < 0.1 * P_on.mean()
