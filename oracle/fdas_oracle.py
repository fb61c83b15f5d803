"""
FDAS oracle -- TEST INFRASTRUCTURE ONLY.  Never imported by the product path
(`paper_1804_05335_b200/`); only tests/, __graft_entry__.smoke() and bench.py's
cpu_baseline / `--impl reference` legs may use it.  It shares no code, tables or
constants with the CUDA path.

What it computes (fp64 throughout), each function citing the passage it follows:

  * template taps  h_z[d]  -- the "predicted normalised Fourier response" of
    PAPER.md:65 (section 2).  The paper cites the formula (Ransom et al. 2002) but does
    not print it; reading R1 defines it as the response, at bin offset d from
    the mid-observation frequency, of a unit-amplitude tone drifting linearly by z bins:
        h_z(d) = integral_0^1 exp( 2 pi i [ -d u + z (u^2 - u)/2 ] ) du
    evaluated HERE BY NUMERICAL QUADRATURE of that integral (the CUDA path uses the
    Fresnel closed form instead, so the two share no formula path).
  * the correlation of eq. 3 by direct summation (C, oracle/fdas_oracle.c),
  * Fourier power and interbinning, eq. 4 applied to the
    correlated complex amplitudes.

Pins (tests/test_oracle_pins.py): closed form via scipy's Fresnel integrals, the z=0
sinc/delta special case, brute-force time-domain chirp + DFT, injected-chirp peak,
reversal / shift / linearity invariants, noise statistics, the paper's printed
interbinning losses, fp64 FFT overlap-save at two segment lengths,
and a pure-Python triple loop on tiny inputs; the threshold search (`candidates`) by the
exponential tail law of noise powers, the 0 / +inf thresholds and an injected chirp's cell; the
2-bin Fourier interpolation (`interbin = 2`) by a brute-force DFT of a time series zero-padded to
twice its length, a half-bin tone's full recovery and the time-domain chirp at a half-integer centre.
  * the real-to-complex transform in front of the correlations: eq. 5
    summed directly for a real series, `dft_real_at` / `dft_real` (reading R17),
  * harmonic summing of the plane (reading R18), `harmonic_sum` /
    `harmonic_candidates`.

More pins: `dft_real*` by a literal O(n^2) Python loop, a pure tone's bin and amplitude, Parseval, conjugate
symmetry, linearity, the shift theorem and numpy's rfft as a third opinion; `harmonic_sum` by literal loops on a
tiny plane, the identity at one harmonic, a time-domain signal with power in harmonics 1, 2 and 4 peaking at the
fundamental's cell, and the Erlang tail law of summed noise powers; `harmonic_sums_cumulative` (one walk over the
harmonics for H = 2, 4, 8, 16) by equality with `harmonic_sum` level by level and a hand-computed cell.
  * the two steps between that transform and the correlations (Fig. 2): red-noise removal by a local
    median filter, `deredden`, and the normalisation of each block, `normalise_blocks` (readings R19, R20).

Pins of those two (tests/test_oracle_pins_whiten.py, P15): a hand-sorted tiny input, the exponential law's
median = mean x ln 2 (white noise keeps unit mean power), a power-law spectrum coming out flat, a strong narrow tone
surviving within 1/block of its amplitude, block mean exactly 1 after normalisation, scale invariance / idempotence,
the ragged last block and the all-zero block.
No function here is "parity unpinned".
"""
from __future__ import annotations

import ctypes
import functools
import math

import numpy as np

from . import build as _build

# --------------------------------------------------------------------------------------
# template bank (readings R4, R9; BASELINE.json configs: "half-width ceil(|z|/2)+16")
# --------------------------------------------------------------------------------------


def bank_z(zmax: float, dz: float) -> np.ndarray:
    """Trial z values, ascending: z_k = -zmax + k*dz, k = 0..K-1 (reading R9)."""
    nhalf = int(round(zmax / dz))
    if abs(nhalf * dz - zmax) > 1e-9 * max(1.0, abs(zmax)):
        raise ValueError("zmax/dz must be an integer")
    zs = np.array([-zmax + k * dz for k in range(2 * nhalf + 1)], dtype=np.float64)
    zs[nhalf] = 0.0                      # the centre template is z = 0 exactly, also for a fractional dz
    return zs


def halfwidth(z: float) -> int:
    """Per-template half-width m_z = ceil(|z|/2) + 16 bins (BASELINE.json config 1)."""
    return int(math.ceil(abs(z) / 2.0 - 1e-12)) + 16


@functools.lru_cache(maxsize=None)
def _gauss_legendre(n: int):
    x, w = np.polynomial.legendre.leggauss(n)
    return x, w


def response(z: float, d) -> np.ndarray:
    """
    h_z(d) for real bin offsets d (array-like), by composite Gauss-Legendre quadrature of
        integral_0^1 exp(2 pi i [ -d u + z (u^2 - u)/2 ]) du        (reading R1)
    The panel count is chosen so the phase advances by at most ~pi/4 per panel; with 12
    nodes per panel the quadrature error is far below 1e-15.
    """
    d = np.atleast_1d(np.asarray(d, dtype=np.float64))
    nodes, weights = _gauss_legendre(12)
    # |d phase/du| <= 2 pi (|d| + |z|/2)
    rate = float(np.max(np.abs(d))) + abs(z) / 2.0 + 1.0
    npanel = int(math.ceil(8.0 * rate))
    edges = np.linspace(0.0, 1.0, npanel + 1)
    half = 0.5 * (edges[1:] - edges[:-1])
    mid = 0.5 * (edges[1:] + edges[:-1])
    u = (mid[:, None] + half[:, None] * nodes[None, :]).ravel()          # all nodes
    w = (half[:, None] * weights[None, :]).ravel()                       # all weights
    out = np.empty(d.shape, dtype=np.complex128)
    chirp = z * (u * u - u) / 2.0
    for i, di in enumerate(d):
        phase = 2.0 * np.pi * (-di * u + chirp)
        out[i] = np.sum(w * np.cos(phase)) + 1j * np.sum(w * np.sin(phase))
    return out


@functools.lru_cache(maxsize=None)
def _taps_cached(z: float, m: int) -> np.ndarray:
    t = response(z, np.arange(-m, m + 1, dtype=np.float64))
    t.setflags(write=False)
    return t


def taps(z: float, m: int | None = None) -> np.ndarray:
    """Taps h_z[d], d = -m..+m (complex128, index d+m); m defaults to halfwidth(z)."""
    if m is None:
        m = halfwidth(z)
    return _taps_cached(float(z), int(m))


# --------------------------------------------------------------------------------------
# correlation, eq. 3 -- C direct sum
# --------------------------------------------------------------------------------------

_lib = None


def _load():
    global _lib
    if _lib is None:
        lib = ctypes.CDLL(_build.build())
        i64, i32, vp = ctypes.c_int64, ctypes.c_int32, ctypes.c_void_p
        lib.fdas_oracle_correlate.argtypes = [vp, i64, vp, i32, i64, i64, vp]
        lib.fdas_oracle_correlate.restype = None
        lib.fdas_oracle_correlate_at.argtypes = [vp, i64, vp, i32, vp, i64, vp]
        lib.fdas_oracle_correlate_at.restype = None
        lib.fdas_oracle_threads.restype = i32
        lib.fdas_oracle_dft_real_at.argtypes = [vp, i64, vp, i64, vp]
        lib.fdas_oracle_dft_real_at.restype = None
        _lib = lib
    return _lib


def threads() -> int:
    """OpenMP threads the C direct sum will use."""
    return int(_load().fdas_oracle_threads())


def _as_c64(spectrum) -> np.ndarray:
    a = np.ascontiguousarray(spectrum, dtype=np.complex64)
    if a.ndim != 1:
        raise ValueError("spectrum must be 1-D")
    return a


def correlate(spectrum, h: np.ndarray, r_begin: int = 0, r_count: int | None = None) -> np.ndarray:
    """y[r] = sum_d A[r+d] conj(h[d]) for r in [r_begin, r_begin+r_count); zero extension (R7)."""
    a = _as_c64(spectrum)
    h = np.ascontiguousarray(h, dtype=np.complex128)
    m = (h.size - 1) // 2
    assert h.size == 2 * m + 1
    if r_count is None:
        r_count = a.size - r_begin
    y = np.empty(r_count, dtype=np.complex128)
    _load().fdas_oracle_correlate(a.ctypes.data, a.size, h.ctypes.data, m,
                                  int(r_begin), int(r_count), y.ctypes.data)
    return y


def correlate_at(spectrum, h: np.ndarray, cols) -> np.ndarray:
    """y at the listed columns only (sampled checks at full size)."""
    a = _as_c64(spectrum)
    h = np.ascontiguousarray(h, dtype=np.complex128)
    m = (h.size - 1) // 2
    cols = np.ascontiguousarray(cols, dtype=np.int64)
    y = np.empty(cols.size, dtype=np.complex128)
    _load().fdas_oracle_correlate_at(a.ctypes.data, a.size, h.ctypes.data, m,
                                     cols.ctypes.data, cols.size, y.ctypes.data)
    return y


def correlate_numpy(spectrum, h: np.ndarray) -> np.ndarray:
    """Same sum as `correlate` over all N columns, written with numpy slices (cross-check of the C)."""
    a = _as_c64(spectrum).astype(np.complex128)
    n = a.size
    m = (h.size - 1) // 2
    y = np.zeros(n, dtype=np.complex128)
    for d in range(-m, m + 1):
        lo, hi = max(0, -d), min(n, n - d)          # r with 0 <= r+d < n
        if hi > lo:
            y[lo:hi] += a[lo + d:hi + d] * np.conj(h[d + m])
    return y


# --------------------------------------------------------------------------------------
# power and interbinning
# --------------------------------------------------------------------------------------

INTERBIN_SCALE = math.pi / 4.0            # eq. 4


def power_from_amplitudes(y: np.ndarray) -> np.ndarray:
    """P = |y|^2."""
    return y.real * y.real + y.imag * y.imag


def interbin_from_amplitudes(y_ext: np.ndarray) -> np.ndarray:
    """
    y_ext = y[0..N] (N+1 amplitudes, y[N] from the zero-extended sum, reading R7).
    Returns 2N powers: P[2r] = |y[r]|^2, P[2r+1] = |(pi/4)(y[r] - y[r+1])|^2
    -- eq. 4 applied to the correlated amplitudes,
    interleaved in natural frequency order (reading R8).
    """
    n = y_ext.size - 1
    out = np.empty(2 * n, dtype=np.float64)
    out[0::2] = power_from_amplitudes(y_ext[:n])
    half = INTERBIN_SCALE * (y_ext[:n] - y_ext[1:])
    out[1::2] = power_from_amplitudes(half)
    return out


@functools.lru_cache(maxsize=None)
def _taps2_cached(z: float, m: int) -> np.ndarray:
    t = response(z, 0.5 * np.arange(-2 * m, 2 * m + 1, dtype=np.float64))
    t.setflags(write=False)
    return t


def taps2(z: float, m: int | None = None) -> np.ndarray:
    """Double-resolution template h_z[j/2], j = -2m..+2m (index j + 2m): the template of the 2-bin
    Fourier interpolation, PAPER.md:89 ("doubling the template and signal resolution")."""
    if m is None:
        m = halfwidth(z)
    return _taps2_cached(float(z), int(m))


def interleave_zeros(spectrum) -> np.ndarray:
    """A2[2k] = A[k], A2[2k+1] = 0: "interleaving zeros prior to the correlations"."""
    a = _as_c64(spectrum)
    a2 = np.zeros(2 * a.size, dtype=np.complex64)
    a2[0::2] = a
    return a2


def plane_row(spectrum, z: float, interbin=False, m: int | None = None) -> np.ndarray:
    """One row of the f-fdot plane (float64): N columns; 2N interbinned (interbin = 1/True, eq. 4) or
    with 2-bin Fourier interpolation (interbin = 2, reading R16: the zero-interleaved spectrum
    correlated with the double-resolution template, column c <-> frequency c/2 bins)."""
    a = _as_c64(spectrum)
    if int(interbin) == 2:
        return power_from_amplitudes(correlate(interleave_zeros(a), taps2(z, m), 0, 2 * a.size))
    h = taps(z, m)
    if interbin:
        return interbin_from_amplitudes(correlate(a, h, 0, a.size + 1))
    return power_from_amplitudes(correlate(a, h, 0, a.size))


def plane(spectrum, zmax: float, dz: float, interbin=False) -> np.ndarray:
    """Whole plane, K rows ascending in z (reading R9).  For sizes that fit in memory."""
    zs = bank_z(zmax, dz)
    return np.stack([plane_row(spectrum, z, interbin) for z in zs])


def plane_cells(spectrum, z: float, cols, interbin=False) -> np.ndarray:
    """
    Sampled cells of one row.  `cols` are plane column indices (0..N-1, or 0..2N-1 when
    interbinned: even 2r -> bin r, odd 2r+1 -> bin r+1/2).
    """
    a = _as_c64(spectrum)
    cols = np.asarray(cols, dtype=np.int64)
    if int(interbin) == 2:
        return power_from_amplitudes(correlate_at(interleave_zeros(a), taps2(z), cols))
    h = taps(z)
    if not interbin:
        return power_from_amplitudes(correlate_at(a, h, cols))
    r = cols // 2
    y0 = correlate_at(a, h, r)
    y1 = correlate_at(a, h, r + 1)
    odd = (cols % 2) == 1
    return np.where(odd, power_from_amplitudes(INTERBIN_SCALE * (y0 - y1)),
                    power_from_amplitudes(y0))


def candidates(spectrum, zmax: float, dz: float, threshold: float, interbin=False):
    """
    Threshold search of the plane ("calculating the power spectrum, and comparing the
    resulting Fourier power to a pre-calculated threshold"; PAPER.md:331 names search / candidate
    selection next to the correlation as the step to fuse; reading R15): every cell with
    P[k][c] > threshold (strict), as three arrays (row k, column c, power) sorted by (row, column).
    Row by row, so the plane is never held.
    """
    rows, cols, pows = [], [], []
    for k, z in enumerate(bank_z(zmax, dz)):
        p = plane_row(spectrum, z, interbin)
        c = np.nonzero(p > threshold)[0]
        rows.append(np.full(c.size, k, dtype=np.int64))
        cols.append(c.astype(np.int64))
        pows.append(p[c])
    return np.concatenate(rows), np.concatenate(cols), np.concatenate(pows)


def cmacs(n: int, zmax: float, dz: float) -> int:
    """Complex multiply-accumulates of the direct sum for one spectrum: N * sum_z (2 m_z + 1)."""
    return int(n) * int(sum(2 * halfwidth(z) + 1 for z in bank_z(zmax, dz)))


# --------------------------------------------------------------------------------------
# the real-to-complex transform in front of the correlations
# --------------------------------------------------------------------------------------

def dft_real_at(x, bins) -> np.ndarray:
    """X[k] = sum_j x[j] exp(-2 pi i j k / n) (eq. 5; unnormalised) of the REAL series x (float32
    samples, up-converted) at the listed bins, by direct summation in C (O(n) per bin)."""
    x = np.ascontiguousarray(x, dtype=np.float32)
    if x.ndim != 1:
        raise ValueError("time series must be 1-D")
    bins = np.ascontiguousarray(bins, dtype=np.int64)
    out = np.empty(bins.size, dtype=np.complex128)
    _load().fdas_oracle_dft_real_at(x.ctypes.data, x.size, bins.ctypes.data, bins.size, out.ctypes.data)
    return out


def dft_real(x) -> np.ndarray:
    """The spectrum the correlations take (reading R17): bins k = 0 .. n/2 - 1 of the real series'
    DFT (DC kept, the Nyquist bin dropped), unnormalised.  O(n^2): small n only."""
    n = np.asarray(x).size
    if n % 2:
        raise ValueError("even number of samples")
    return dft_real_at(x, np.arange(n // 2))


# --------------------------------------------------------------------------------------
# harmonic summing (reading R18)
# --------------------------------------------------------------------------------------

def harmonic_rows(zmax: float, dz: float, nharm: int) -> np.ndarray:
    """Rows k of the bank whose harmonics h z_k, h = 1..nharm, all lie inside the bank (|z_k| <= zmax / nharm)."""
    zs = bank_z(zmax, dz)
    nhalf = (zs.size - 1) // 2
    lim = nhalf // int(nharm)
    return np.arange(nhalf - lim, nhalf + lim + 1)


def harmonic_sum(plane: np.ndarray, zmax: float, dz: float, nharm: int) -> np.ndarray:
    """
    S_H[k][c] = sum_{h=1}^{H} P[row(h z_k)][h c]: a signal whose fundamental sits at column c with drift z_k has its
    h-th harmonic at column h c with drift h z_k (frequency AND frequency derivative scale with h), so its power is
    collected at the fundamental's cell.  Defined for the rows of `harmonic_rows` and the columns c with
    H c <= ncols - 1; returned as a (rows, ceil(ncols / H)) float64 array, row i <-> bank row harmonic_rows()[i].
    """
    p = np.asarray(plane, dtype=np.float64)
    k_all, ncols = p.shape
    nharm = int(nharm)
    rows = harmonic_rows(zmax, dz, nharm)
    nhalf = (k_all - 1) // 2
    nc = (ncols - 1) // nharm + 1
    out = np.zeros((rows.size, nc), dtype=np.float64)
    for i, k in enumerate(rows):
        for h in range(1, nharm + 1):
            kh = nhalf + h * (int(k) - nhalf)          # row of h z_k
            out[i] += p[kh, 0:h * (nc - 1) + 1:h]
    return out


def harmonic_candidates(plane: np.ndarray, zmax: float, dz: float, nharm: int, threshold: float):
    """Cells of the H-harmonic sum above the threshold (strict): (bank row k, fundamental column c, S) sorted by
    (row, column)."""
    s = harmonic_sum(plane, zmax, dz, nharm)
    rows = harmonic_rows(zmax, dz, nharm)
    i, c = np.nonzero(s > threshold)
    return rows[i].astype(np.int64), c.astype(np.int64), s[i, c]


def harmonic_sums_cumulative(plane: np.ndarray, zmax: float, dz: float, levels=(2, 4, 8, 16)) -> dict:
    """
    The sums S_H of `harmonic_sum` for an increasing list of H, formed the way a search does it in ONE walk over the
    harmonics of a fundamental cell ("adding the power that is distributed in the harmonics to that of
    the fundamental"; reading R18):  S_{H_l}[k][c] = S_{H_{l-1}}[k][c] + sum_{h = H_{l-1}+1}^{H_l} P[row(h z_k)][h c],
    S_{H_0 = 0} = 0, on the rows and columns of level l (|z_k| <= zmax / H_l, H_l c <= ncols - 1), which shrink with l.
    Returns {H: (rows, S_H)} with S_H as `harmonic_sum` shapes it.  A literal loop over cells; small planes only.
    """
    p = np.asarray(plane, dtype=np.float64)
    k_all, ncols = p.shape
    nhalf = (k_all - 1) // 2
    levels = [int(h) for h in levels]
    if any(b <= a for a, b in zip([0] + levels, levels)):
        raise ValueError("levels must be increasing and positive")
    out = {h: (harmonic_rows(zmax, dz, h), np.zeros((harmonic_rows(zmax, dz, h).size, (ncols - 1) // h + 1)))
           for h in levels}
    rows0 = harmonic_rows(zmax, dz, levels[0])
    for k in rows0:
        for c in range((ncols - 1) // levels[0] + 1):
            s, h_done = 0.0, 0
            for hl in levels:
                lim = nhalf // hl
                if abs(int(k) - nhalf) > lim or hl * c > ncols - 1:
                    break                                     # this cell is outside level hl and every later one
                for h in range(h_done + 1, hl + 1):
                    s += p[nhalf + h * (int(k) - nhalf), h * c]
                h_done = hl
                out[hl][1][int(k) - (nhalf - lim), c] = s
    return out


# --------------------------------------------------------------------------------------
# red-noise removal and block normalisation (Fig. 2; readings R19, R20)
# --------------------------------------------------------------------------------------


def _scale_blocks(spectrum: np.ndarray, block: int, statistic) -> np.ndarray:
    """out[j] = A[j] / sqrt(statistic(powers of A's block)): consecutive blocks of `block` bins from bin 0, the last
    one shorter when `block` does not divide N; a block whose statistic is 0 is copied unchanged."""
    a = np.asarray(spectrum).astype(np.complex128).reshape(-1)
    block = int(block)
    if block < 1:
        raise ValueError("block must be >= 1")
    out = a.copy()
    for start in range(0, a.size, block):
        seg = a[start:start + block]
        stat = float(statistic(seg.real ** 2 + seg.imag ** 2))
        if stat > 0.0:
            out[start:start + block] = seg / math.sqrt(stat)
    return out


def deredden(spectrum: np.ndarray, block: int) -> np.ndarray:
    """
    "low frequency (red) noise is removed with the use of a local median filter".  Reading R19: the
    local noise level of a block of `block` consecutive bins is estimated by the MEDIAN of its Fourier powers
    |A[j]|^2 (the median ignores the few bins a signal occupies); noise powers are exponentially distributed, whose
    median is mean x ln 2, so the block is divided by sqrt(median / ln 2) and its noise comes out at unit mean power.
    Median of an even count = mean of the two middle values.  fp64, complex128 out.
    """
    return _scale_blocks(spectrum, block, lambda p: np.median(p) / math.log(2.0))


def normalise_blocks(spectrum: np.ndarray, block: int) -> np.ndarray:
    """
    "After a short step of normalization on the data of each block, the matched filtering is performed"
    (PAPER.md:79).  Reading R20: the blocks are the overlap-save blocks (`block` = the useful bins B of a segment)
    and each is scaled to unit MEAN power, A[j] / sqrt(mean_j |A[j]|^2).  fp64, complex128 out.
    """
    return _scale_blocks(spectrum, block, np.mean)
