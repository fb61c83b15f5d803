"""
Pins of the oracle's two newest parts (-m "not gpu"), committed before the CUDA code they check:

  P13  dft_real / dft_real_at  -- the real-to-complex transform in front of the correlations
       (PAPER.md:79, :105, :135 eq. 5, :190; reading R17)
  P14  harmonic_sum / harmonic_candidates  -- harmonic summing of the f-fdot plane
       (reading R18)
"""
import math
import os
import sys

import numpy as np
import pytest

sys.path.insert(0, os.path.dirname(os.path.dirname(os.path.abspath(__file__))))

from oracle import fdas_oracle as orc                      # noqa: E402
from paper_1804_05335_b200 import synthetic as syn         # noqa: E402


# ---------------------------------------------------------------- P13: eq. 5 for a real series
def test_p13_literal_loop_on_tiny_series():
    rng = np.random.default_rng(1)
    for n in (2, 16, 30, 128):
        x = rng.standard_normal(n).astype(np.float32)
        ref = np.zeros(n, dtype=np.complex128)
        for k in range(n):                                   # eq. 5 as printed: sign exp(-2 pi i n m / N)
            acc = 0j
            for j in range(n):
                acc += float(x[j]) * complex(math.cos(2 * math.pi * j * k / n), -math.sin(2 * math.pi * j * k / n))
            ref[k] = acc
        got = orc.dft_real_at(x, np.arange(n))
        assert np.max(np.abs(got - ref)) < 1e-12 * n
        assert np.array_equal(orc.dft_real(x), got[:n // 2])  # DC kept, Nyquist dropped (reading R17)
        # bins outside [0, n) wrap (the sum is periodic in k)
        assert np.max(np.abs(orc.dft_real_at(x, [-1, n + 3]) - ref[[n - 1, 3 % n]])) < 1e-12 * n


def test_p13_pure_tone_bin_and_amplitude():
    n, k0, a, phi = 4096, 321, 3.0, 0.7
    j = np.arange(n)
    x = (a * np.cos(2 * np.pi * k0 * j / n + phi)).astype(np.float32)
    X = orc.dft_real(x)
    assert abs(X[k0] - a * n / 2 * np.exp(1j * phi)) < 2e-3          # float32 samples: ~n * 6e-8 * a
    X[k0] = 0
    assert np.max(np.abs(X)) < 2e-3
    # a positive-frequency complex exponential's real part: the sign of eq. 5 puts it at +k0 with phase +phi
    assert abs(np.angle(orc.dft_real_at(x, [k0])[0]) - phi) < 1e-6


def test_p13_parseval_symmetry_linearity_shift_and_numpy():
    rng = np.random.default_rng(2)
    n = 1000                                                  # not a power of two: the definition does not care
    x = rng.standard_normal(n).astype(np.float32)
    y = rng.standard_normal(n).astype(np.float32)
    X = orc.dft_real_at(x, np.arange(n))
    x64 = x.astype(np.float64)
    assert abs(np.sum(np.abs(X) ** 2) / n - np.sum(x64 ** 2)) < 1e-9 * n          # Parseval
    assert np.max(np.abs(X[1:] - np.conj(X[1:][::-1]))) < 1e-10                   # X[n-k] = conj X[k]
    assert abs(X[0].imag) < 1e-12 and abs(X[n // 2].imag) < 1e-10                 # DC and Nyquist are real
    z = (2.0 * x - 0.5 * y).astype(np.float32)               # exact in float32? not in general: compare in fp64 of z
    Z = orc.dft_real_at(z, np.arange(n))
    lin = orc.dft_real_at(z.astype(np.float32), np.arange(n))
    assert np.array_equal(Z, lin)
    Y = orc.dft_real_at(y, np.arange(n))
    xe = x.astype(np.float64) * 2.0 - 0.5 * y.astype(np.float64)
    assert np.max(np.abs((2.0 * X - 0.5 * Y) - np.fft.fft(xe))) < 1e-9          # linearity (+ third opinion)
    s = 37                                                    # shift theorem: x[j - s] <-> X[k] exp(-2 pi i k s / n)
    xs = np.roll(x, s)
    Xs = orc.dft_real_at(xs, np.arange(n))
    assert np.max(np.abs(Xs - X * np.exp(-2j * np.pi * np.arange(n) * s / n))) < 1e-9
    assert np.max(np.abs(X[:n // 2 + 1] - np.fft.rfft(x64))) < 1e-9               # numpy's rfft, a third opinion


def test_p13_spectrum_of_a_time_domain_chirp_feeds_the_correlation():
    """The two parts of the oracle meet: the R2C spectrum of a REAL drifting tone, divided by n/2, is the complex
    amplitude h_z(k - r0) of the correlation's template (readings R1, R2), so the plane built on it peaks at (r0, z0)."""
    n, r0, z0, a = 1 << 13, 1000.0, 6.0, 2.0
    u = np.arange(n) / n
    x = (a * np.cos(2 * np.pi * (r0 * u + z0 * (u * u - u) / 2))).astype(np.float32)
    A = orc.dft_real(x) / (n / 2)
    d = np.arange(-10, 11)
    assert np.max(np.abs(A[int(r0) + d] - a * orc.response(z0, d.astype(np.float64)))) < 5e-4   # O(1/n) endpoint term
    plane = orc.plane(A.astype(np.complex64), 10.0, 2.0)
    k, r = np.unravel_index(np.argmax(plane), plane.shape)
    assert orc.bank_z(10.0, 2.0)[k] == z0 and r == int(r0) and abs(plane[k, r] - a * a) < 2e-2 * a * a


# ---------------------------------------------------------------- P14: harmonic summing
def test_p14_literal_loops_on_a_tiny_plane_and_identity():
    rng = np.random.default_rng(3)
    zmax, dz = 8.0, 2.0                                        # rows z = -8..8 (9 rows)
    p = rng.exponential(size=(9, 41))
    assert np.array_equal(orc.harmonic_sum(p, zmax, dz, 1), p)                      # one harmonic: the plane itself
    assert np.array_equal(orc.harmonic_rows(zmax, dz, 1), np.arange(9))
    zs = orc.bank_z(zmax, dz)
    for H in (2, 3, 4, 8):
        rows = orc.harmonic_rows(zmax, dz, H)
        assert np.all(np.abs(zs[rows]) * H <= zmax) and rows.size == 2 * (4 // H) + 1
        s = orc.harmonic_sum(p, zmax, dz, H)
        assert s.shape == (rows.size, (41 - 1) // H + 1)
        for i, k in enumerate(rows):
            for c in range(s.shape[1]):
                acc = 0.0
                for h in range(1, H + 1):
                    kh = int(np.argmin(np.abs(zs - h * zs[k])))               # the row whose z is h z_k
                    assert zs[kh] == h * zs[k]
                    acc += p[kh, h * c]
                assert abs(s[i, c] - acc) < 1e-12
    r, c, v = orc.harmonic_candidates(p, zmax, dz, 2, 3.0)
    s2 = orc.harmonic_sum(p, zmax, dz, 2)
    rows2 = orc.harmonic_rows(zmax, dz, 2)
    assert r.size == np.count_nonzero(s2 > 3.0) and np.all(v > 3.0)
    assert all(s2[list(rows2).index(rr), cc] == vv for rr, cc, vv in zip(r, c, v))


def test_p14_signal_with_harmonics_peaks_at_the_fundamental():
    """Time-domain pulse train stand-in: harmonics 1, 2 and 4 of a drifting tone (frequency and drift both scale
    with the harmonic number).  The 4-harmonic sum peaks at the fundamental's cell and collects the three powers."""
    n = 1 << 14
    r0, z0 = 1500.0, 4.0
    amps = {1: 6.0, 2: 4.0, 4: 3.0}
    chirps = [(h * r0, h * z0, a) for h, a in amps.items()]
    spec = syn.make_spectrum(n, 5, chirps)                     # unit-variance noise + the three harmonics
    zmax, dz = 16.0, 2.0
    plane = orc.plane(spec, zmax, dz)
    s4 = orc.harmonic_sum(plane, zmax, dz, 4)
    rows = orc.harmonic_rows(zmax, dz, 4)
    i, c = np.unravel_index(np.argmax(s4), s4.shape)
    assert orc.bank_z(zmax, dz)[rows[i]] == z0 and c == int(r0)
    expect = sum(a * a for a in amps.values())
    assert abs(s4[i, c] - expect) < 0.5 * expect                # + noise cross terms (amplitude-sigma products)
    # in the single-harmonic plane the fundamental's cell holds only its own power
    k0 = int(np.argmin(np.abs(orc.bank_z(zmax, dz) - z0)))
    assert plane[k0, int(r0)] < 0.75 * s4[i, c]


def test_p14_noise_mean_and_erlang_tail():
    rng = np.random.default_rng(4)
    zmax, dz = 8.0, 2.0
    p = rng.exponential(size=(9, 400001))                      # powers of unit-variance complex noise
    for H in (1, 2, 4):
        s = orc.harmonic_sum(p, zmax, dz, H)
        assert abs(s.mean() - H) < 0.02 * H                     # mean scales with the number of harmonics summed
        t = 2.0 * H + 4.0                                       # P(S > t) = exp(-t) sum_{j<H} t^j / j!   (Erlang)
        tail = math.exp(-t) * sum(t ** j / math.factorial(j) for j in range(H))
        frac = np.count_nonzero(s > t) / s.size
        assert abs(frac - tail) < 5.0 * math.sqrt(tail / s.size) + 1e-6


def test_cumulative_harmonic_sums_equal_the_per_h_definition():
    """P14 extended: the one-walk form (S_4 = S_2 + P[3z][3c] + P[4z][4c], ...) is the same function as the per-H
    definition on every level's own domain; one cell by hand."""
    rng = np.random.Generator(np.random.Philox(99))
    zmax, dz = 32.0, 2.0
    plane = rng.standard_exponential((33, 203))
    cum = orc.harmonic_sums_cumulative(plane, zmax, dz, (2, 4, 8, 16))
    for hh in (2, 4, 8, 16):
        rows, s = cum[hh]
        assert np.array_equal(rows, orc.harmonic_rows(zmax, dz, hh))
        ref = orc.harmonic_sum(plane, zmax, dz, hh)
        assert s.shape == ref.shape and np.max(np.abs(s - ref)) <= 1e-12 * ref.max()
    # by hand: fundamental z = +2 (row 17 of 33), column 5: S_4 collects rows 17, 18, 19, 20 at columns 5, 10, 15, 20
    want = plane[17, 5] + plane[18, 10] + plane[19, 15] + plane[20, 20]
    rows, s4 = cum[4]
    assert abs(s4[list(rows).index(17), 5] - want) <= 1e-14 * want
    # other level lists: a single level is harmonic_sum itself; a level the bank cannot hold keeps only z = 0
    one = orc.harmonic_sums_cumulative(plane, zmax, dz, (3,))
    assert np.allclose(one[3][1], orc.harmonic_sum(plane, zmax, dz, 3), rtol=1e-13)
    big = orc.harmonic_sums_cumulative(plane, zmax, dz, (2, 32))
    assert big[32][0].tolist() == [16] and big[32][1].shape == (1, (203 - 1) // 32 + 1)
    with pytest.raises(ValueError):
        orc.harmonic_sums_cumulative(plane, zmax, dz, (4, 2))
