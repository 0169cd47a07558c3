"""ORACLE — test infrastructure only.  Coherent multi-beam beamformer of the thesis (PAPER.md:1600-1665,
ch. 5, eq 5.1 and Alg. 2), plain numpy in complex128 / float64.  Shares no code with the CUDA library.

"The beamforming process is essentially a matrix-vector multiplication, which involves multiplying a vector
of N_a antennas by an N_b x N_a matrix of coefficients to form N_b beams, per frequency channel"
(PAPER.md:1639); the coefficients are held fixed over the buffer; the antenna voltages are
"4-bit, two's complement ... complex voltages", one byte per antenna sample, four antennas per 32-bit word
(PAPER.md:1645).  Each beam then "can be treated as if it is a signal from a single antenna ... fed directly
to backend detectors": the detected power of every beam is a filterbank [beam][chan][time]
for the dedisperser.

Readings (R34-R37):
  R34 voltage byte: low nibble = real part, high nibble = imaginary part, each a 4-bit two's complement
      integer (-8..7) ("floating point" in the text is taken as a slip: a 4-bit field has no exponent);
  R35 layouts: V uint8 [nchans][nsamp][nants] (antenna fastest: "groups of 4 antennas ... 32-bit words"),
      W complex [nchans][nbeams][nants], output float [nbeams][nchans][nsamp] (beams are
      [beam][chan][time] for the transient pipeline);
  R36 beam voltage b(f,t,beam) = sum_a W[f][beam][a] * v[f][t][a] (no conjugation: the caller supplies the
      weights that point the beam, e.g. exp(-i k0.r_a) of eq 5.1);
  R37 output = detected power |b|^2, no integration in time.
Pins (tests/test_beamform_pins.py): nibble decoding by hand; explicit Python loops; one-antenna identity;
coherent N^2 versus incoherent N gain; the closed-form array factor of a uniform line array (eq 5.1).
Nothing here is "parity unpinned".
"""
from __future__ import annotations

import numpy as np


def decode_voltages(V) -> np.ndarray:
    """uint8 -> complex128 (R34)."""
    V = np.asarray(V, dtype=np.uint8)
    re = (V & 0x0F).astype(np.int16)
    im = (V >> 4).astype(np.int16)
    re = np.where(re >= 8, re - 16, re)
    im = np.where(im >= 8, im - 16, im)
    return re.astype(np.float64) + 1j * im.astype(np.float64)


def encode_voltages(z) -> np.ndarray:
    """complex (integer parts in -8..7) -> uint8; inverse of decode_voltages (test-input helper)."""
    re = np.asarray(np.real(z)).astype(np.int16) & 0x0F
    im = np.asarray(np.imag(z)).astype(np.int16) & 0x0F
    return (re | (im << 4)).astype(np.uint8)


def beamform_power(V, W):
    """V uint8 [nchans][nsamp][nants], W complex [nchans][nbeams][nants] -> (P float64 [nbeams][nchans][nsamp],
    S same shape = sum_a |W||v|, the scale of the float tolerance)  (R35-R37)."""
    v = decode_voltages(V)
    W = np.asarray(W, dtype=np.complex128)
    b = np.einsum("fba,fta->bft", W, v)
    S = np.einsum("fba,fta->bft", np.abs(W), np.abs(v))
    return b.real ** 2 + b.imag ** 2, S


def steering_weights(freqs_mhz, positions_m, directions):
    """Phase weights pointing beams (eq 5.1): W[f][b][a] = exp(-i k0 . r_a), k0 = 2 pi f / c * unit vector of
    direction b.  positions [nants][3] metres, directions [nbeams][3] unit vectors."""
    c = 299792458.0
    f = np.asarray(freqs_mhz, dtype=np.float64) * 1e6
    phase = (2.0 * np.pi / c) * f[:, None, None] * (np.asarray(directions) @ np.asarray(positions_m).T)[None, :, :]
    return np.exp(-1j * phase)
