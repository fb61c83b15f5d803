"""
Seeded synthetic FDAS inputs, shared by the oracle tests, the GPU parity tests and bench.py.

This module holds NONE of the method's arithmetic (no templates, no correlation): a
spectrum is complex Gaussian noise plus the discrete Fourier transform of linearly
drifting complex sinusoids synthesised IN THE TIME DOMAIN,

    x_n = sum_c a_c exp( i phi_c + 2 pi i [ r_c u + z_c (u^2 - u)/2 ] ),  u = n/N,  n = 0..N-1
    A   = FFT(x) / N + noise                                   (DFT sign: eq. 5)

so a chirp "at (r_c, z_c)" has instantaneous frequency r_c + z_c (u - 1/2) bins: mean
frequency r_c, total drift z_c bins (eq. 2; reading R2).

They stand in for the paper's SIGPROC `fake` pulsar spectra, which are not
available here; shapes and sizes follow BASELINE.json's five configs.
"""
from __future__ import annotations

import numpy as np

# BASELINE.json configs 1..5 (index 0..4).  `chirps` = fixed list or a count drawn from the seed.
CONFIGS = [
    dict(name="config1_tiny", nbins=1 << 16, zmax=20.0, dz=2.0, seglen=1024, interbin=0, batch=1,
         seed=1001, chirps=[(20000.25, 8.0, 30.0)], zlim=None, whiten=False),
    dict(name="config2_smem", nbins=1 << 21, zmax=84.0, dz=2.0, seglen=2048, interbin=0, batch=1,
         seed=1002, chirps=8, zlim=80.0, whiten=False),
    dict(name="config3_interbin", nbins=1 << 23, zmax=84.0, dz=2.0, seglen=4096, interbin=1, batch=1,
         seed=1003, chirps=16, zlim=80.0, whiten=False),
    dict(name="config4_wide", nbins=1 << 23, zmax=200.0, dz=2.0, seglen=8192, interbin=0, batch=1,
         seed=1004, chirps=16, zlim=190.0, whiten=True),
    dict(name="config5_batched", nbins=1 << 21, zmax=84.0, dz=2.0, seglen=2048, interbin=1, batch=64,
         seed=5000, chirps="0-2", zlim=80.0, whiten=False),
]


def _rng(seed: int) -> np.random.Generator:
    return np.random.Generator(np.random.Philox(int(seed)))


def noise(nbins: int, rng: np.random.Generator) -> np.ndarray:
    """Unit-variance complex Gaussian bins: re, im ~ N(0, 1/2), so E|A|^2 = 1 (complex128)."""
    s = np.sqrt(0.5)
    return s * rng.standard_normal(nbins) + 1j * s * rng.standard_normal(nbins)


def chirp_spectrum(nbins: int, chirps, phases=None) -> np.ndarray:
    """
    FFT(x)/N of the sum of time-domain chirps (r_c, z_c, a_c) -- complex128, N bins.
    Synthesised in blocks to bound memory; phases default to 0.
    """
    x = np.zeros(nbins, dtype=np.complex128)
    if len(chirps) == 0:
        return x
    if phases is None:
        phases = [0.0] * len(chirps)
    blk = 1 << 20
    for lo in range(0, nbins, blk):
        hi = min(nbins, lo + blk)
        u = np.arange(lo, hi, dtype=np.float64) / nbins
        for (r, z, a), ph in zip(chirps, phases):
            x[lo:hi] += a * np.exp(1j * (ph + 2.0 * np.pi * (r * u + z * (u * u - u) / 2.0)))
    return np.fft.fft(x) / nbins


def draw_chirps(rng: np.random.Generator, count: int, nbins: int, zlim: float):
    """r ~ U(0.05N, 0.95N) real, z ~ U(-zlim, zlim) real, a ~ U(8, 40), phase ~ U(0, 2pi)."""
    chirps, phases = [], []
    for _ in range(count):
        r = rng.uniform(0.05 * nbins, 0.95 * nbins)
        z = rng.uniform(-zlim, zlim)
        a = rng.uniform(8.0, 40.0)
        chirps.append((float(r), float(z), float(a)))
        phases.append(float(rng.uniform(0.0, 2.0 * np.pi)))
    return chirps, phases


def make_spectrum(nbins: int, seed: int, chirps=(), phases=None, whiten: bool = False) -> np.ndarray:
    """Noise + chirps, rounded once to complex64 (what both the GPU and the oracle receive)."""
    rng = _rng(seed)
    a = noise(nbins, rng)
    if whiten:                       # "noise whitened to unit mean power" (BASELINE.json config 4)
        a /= np.sqrt(np.mean(a.real ** 2 + a.imag ** 2))
    a += chirp_spectrum(nbins, list(chirps), phases)
    return a.astype(np.complex64)


def config_spectrum(idx: int, b: int = 0, nbins: int | None = None):
    """
    Spectrum `b` of BASELINE.json config idx (0-based), optionally at a reduced `nbins`
    (same laws; for parity cases the oracle finishes quickly).  Returns (spectrum, chirps).
    """
    c = CONFIGS[idx]
    n = int(nbins or c["nbins"])
    seed = c["seed"] + b
    rng = _rng(seed + 77_000)        # chirp parameters come from their own stream
    spec = c["chirps"]
    if isinstance(spec, list):
        chirps = [(r * n / c["nbins"], z, a) for (r, z, a) in spec]
        phases = [0.0] * len(chirps)
    else:
        count = int(rng.integers(0, 3)) if spec == "0-2" else int(spec)
        chirps, phases = draw_chirps(rng, count, n, c["zlim"])
    return make_spectrum(n, seed, chirps, phases, c["whiten"]), chirps


def noise_only_c64(nbins: int, seed: int) -> np.ndarray:
    """Fast generator for throughput runs: unit-variance complex64 noise, no chirps."""
    rng = _rng(seed)
    out = np.empty(nbins, dtype=np.complex64)
    s = np.float32(np.sqrt(0.5))
    out.real = s * rng.standard_normal(nbins, dtype=np.float32)
    out.imag = s * rng.standard_normal(nbins, dtype=np.float32)
    return out
