"""Seeded synthetic filterbanks and the five BASELINE.json workload shapes.

This module is shared by the oracle tests, the GPU parity tests and bench.py.
It holds NONE of the method's arithmetic: no delay formula, no shift table, no
dedispersion.  Anything that depends on s(d,c) (row length = nsamp + maxshift,
the per-channel delays of an injected pulse) is passed in by the caller, who
gets it from whichever side it is exercising (``oracle`` in the oracle tests,
the C-ABI library in the product / bench).

Shapes and distributions follow the thesis' simulated data: Gaussian noise
mu=0 sigma=1 with top-hat pulses, 408/418 MHz 20 MHz
1024-channel 51.2 us BEST-II data, 8-bit quantised
power as a storage format.  They stand in for the thesis'
simulated files and BEST-II recordings, which are not available.

Random numbers: numpy Philox (counter-based), keyed by (seed, channel row), so
rows can be generated independently, in any order, in parallel.
"""
from __future__ import annotations

import dataclasses
from concurrent.futures import ThreadPoolExecutor

import numpy as np

BASE_SEED = 14018258


@dataclasses.dataclass(frozen=True)
class Workload:
    """One BASELINE.json config (parameters only)."""
    name: str
    index: int
    dtype: str            # "f32" or "u8"
    nbeams: int
    nchans: int
    fch1: float           # MHz, channel 0 = top of band = reference
    foff: float           # MHz, negative
    tsamp: float          # s
    ndm: int
    dm_step: float
    nsamp: int            # OUTPUT samples per DM trial (per beam)
    nchunks: int = 1      # >1: fed through the streaming API in this many pushes
    seed: int = BASE_SEED

    @property
    def dm_list(self) -> np.ndarray:
        # DM_d = d * step as a double product (not a running sum)
        return np.arange(self.ndm, dtype=np.float64) * np.float64(self.dm_step)

    @property
    def np_dtype(self):
        return np.float32 if self.dtype == "f32" else np.uint8

    @property
    def adds(self) -> int:
        """DM * channel * samples — the unit of BASELINE.json's metric."""
        return self.nbeams * self.nchans * self.ndm * self.nsamp


# foff = -band/nchans exactly (reading R6); BASELINE.json prints rounded literals.
WORKLOADS = {
    1: Workload("cfg1_tiny_f32", 1, "f32", 1, 64, 420.0, -0.25, 100e-6, 32, 1.0, 8192,
                seed=BASE_SEED + 1),
    2: Workload("cfg2_u8_1024ch_1024dm", 2, "u8", 1, 1024, 418.0, -20.0 / 1024, 51.2e-6,
                1024, 0.1, 1 << 17, seed=BASE_SEED + 2),
    3: Workload("cfg3_f32_lband_4096ch_4096dm", 3, "f32", 1, 4096, 1550.0, -300.0 / 4096, 64e-6,
                4096, 0.25, 1 << 18, seed=BASE_SEED + 3),
    4: Workload("cfg4_f32_32beams_512ch_2048dm", 4, "f32", 32, 512, 418.0, -20.0 / 512, 51.2e-6,
                2048, 0.1, 1 << 16, seed=BASE_SEED + 4),
    5: Workload("cfg5_u8_lowfreq_2048ch_10000dm_stream4", 5, "u8", 1, 2048, 165.0, -30.0 / 2048,
                1e-3, 10000, 0.05, 1 << 18, nchunks=4, seed=BASE_SEED + 5),
}


def scaled(w: Workload, **kw) -> Workload:
    """A shrunk / altered copy of a workload (for CPU-sized parity cases)."""
    return dataclasses.replace(w, **kw)


def _rows(fn, nrows, out, threads=8):
    if nrows * out.shape[1] < (1 << 22) or threads <= 1:
        for r in range(nrows):
            fn(r)
        return
    with ThreadPoolExecutor(max_workers=threads) as ex:
        list(ex.map(fn, range(nrows)))


def noise_f32(seed: int, nchans: int, nsamp_in: int, out: np.ndarray | None = None) -> np.ndarray:
    """float32 N(0,1), [nchans][nsamp_in]; row r drawn from Philox(key=(seed, r))."""
    X = out if out is not None else np.empty((nchans, nsamp_in), dtype=np.float32)
    assert X.shape == (nchans, nsamp_in) and X.dtype == np.float32

    def one(r):
        g = np.random.Generator(np.random.Philox(key=[seed, r]))
        g.standard_normal(nsamp_in, dtype=np.float32, out=X[r])

    _rows(one, nchans, X)
    return X


def noise_u8(seed: int, nchans: int, nsamp_in: int, mean: float = 128.0, std: float = 16.0,
             out: np.ndarray | None = None) -> np.ndarray:
    """uint8 clamp(round_half_even(mean + std*z), 0, 255), z~N(0,1) (reading R13)."""
    X = out if out is not None else np.empty((nchans, nsamp_in), dtype=np.uint8)
    assert X.shape == (nchans, nsamp_in) and X.dtype == np.uint8

    def one(r):
        g = np.random.Generator(np.random.Philox(key=[seed, r]))
        z = g.standard_normal(nsamp_in, dtype=np.float32)
        np.multiply(z, np.float32(std), out=z)
        np.add(z, np.float32(mean), out=z)
        np.rint(z, out=z)
        np.clip(z, 0, 255, out=z)
        X[r] = z.astype(np.uint8)

    _rows(one, nchans, X)
    return X


def inject_pulse(X: np.ndarray, t0: int, width: int, amp, delays) -> None:
    """Add a top-hat of height `amp`, `width` samples wide, to every channel c at
    columns t0 + delays[c] + [0, width).  `delays` (one integer per channel) comes
    from the caller — this module does not know the dispersion law."""
    delays = np.asarray(delays)
    assert delays.shape == (X.shape[0],)
    for c in range(X.shape[0]):
        a = int(t0 + delays[c])
        assert 0 <= a and a + width <= X.shape[1], "pulse sweep out of range"
        if X.dtype == np.uint8:
            X[c, a:a + width] = np.clip(X[c, a:a + width].astype(np.int32) + int(amp), 0, 255)
        else:
            X[c, a:a + width] += X.dtype.type(amp)


def beam_seed(seed: int, beam: int) -> int:
    return seed * 1000 + beam


def make_input(w: Workload, nsamp_in: int, beam: int = 0, out: np.ndarray | None = None) -> np.ndarray:
    """Noise-only input of one beam of workload `w`, rows `nsamp_in` long."""
    s = beam_seed(w.seed, beam) if w.nbeams > 1 else w.seed
    if w.dtype == "f32":
        return noise_f32(s, w.nchans, nsamp_in, out=out)
    return noise_u8(s, w.nchans, nsamp_in, out=out)


def pulse_plan(w: Workload, npulses: int, nsamp_in_margin: int = 0):
    """Seeded (dm_index, t0, width) triples for config-3 style injections: DMs drawn
    from the trial grid, widths from {1,2,4,8,16}, t0 uniform in the output range."""
    g = np.random.Generator(np.random.Philox(key=[w.seed, 0xFACADE]))
    out = []
    for _ in range(npulses):
        d = int(g.integers(0, w.ndm))
        width = int(2 ** g.integers(0, 5))
        t0 = int(g.integers(0, max(1, w.nsamp - width - nsamp_in_margin)))
        out.append((d, t0, width))
    return out
