"""
Pins for the oracle (CPU only).  Each test ties one part of oracle/ to something other
than itself: a closed form, a special case, a brute-force definition, an invariant, or a
number the paper prints.  See DESIGN.md "Oracle pins" (P1..P10).
"""
import math

import numpy as np
import pytest
import scipy.special

from oracle import fdas_oracle as orc
from paper_1804_05335_b200 import synthetic as syn


# ---------------------------------------------------------------- P1: closed form (Fresnel)
def _closed_form(z, d):
    """Reading R1's closed form written with scipy's Fresnel integrals (third opinion)."""
    d = np.asarray(d, dtype=np.float64)
    if z == 0:
        return np.exp(-1j * np.pi * d) * np.sinc(d)
    if z < 0:
        return np.conj(_closed_form(-z, -d))
    q = -d - z / 2.0
    s = math.sqrt(2.0 / z)
    SY, CY = scipy.special.fresnel(q * s)
    SZ, CZ = scipy.special.fresnel((q + z) * s)
    return np.exp(-1j * np.pi * q * q / z) / math.sqrt(2.0 * z) * ((CZ - CY) + 1j * (SZ - SY))


@pytest.mark.parametrize("z", [2.0, 8.0, -8.0, 84.0, -200.0, 0.5, 37.3, 0.0])
def test_p1_quadrature_equals_fresnel_closed_form(z):
    m = orc.halfwidth(z)
    d = np.arange(-m, m + 1, dtype=np.float64)
    assert np.max(np.abs(orc.taps(z) - _closed_form(z, d))) < 1e-12
    frac = np.array([-3.7, -0.25, 0.0, 0.5, 11.125])
    assert np.max(np.abs(orc.response(z, frac) - _closed_form(z, frac))) < 1e-12


# ---------------------------------------------------------------- P2: z = 0
def test_p2_z0_is_delta_and_sinc():
    h0 = orc.taps(0.0)
    m = orc.halfwidth(0.0)
    assert m == 16 and h0.size == 33
    expect = np.zeros(33, dtype=np.complex128)
    expect[m] = 1.0
    assert np.max(np.abs(h0 - expect)) < 1e-14
    # fractional offsets: the Fourier-interpolation sinc response of an un-accelerated tone
    d = np.linspace(-4.3, 4.3, 41)
    assert np.max(np.abs(orc.response(0.0, d) - np.exp(-1j * np.pi * d) * np.sinc(d))) < 1e-13
    # plane row z=0 is then exactly |A|^2
    a = syn.make_spectrum(4096, 7)
    p = orc.plane_row(a, 0.0)
    a64 = a.astype(np.complex128)
    assert np.max(np.abs(p - (a64.real ** 2 + a64.imag ** 2))) < 1e-12


# ---------------------------------------------------------------- P3: brute-force time-domain chirp + DFT
@pytest.mark.parametrize("nt,rc,z", [(4096, 300, 8.0), (8192, 1000, 40.0), (4096, 517, -13.0)])
def test_p3_time_domain_chirp_dft(nt, rc, z):
    u = np.arange(nt) / nt
    x = np.exp(2j * np.pi * (rc * u + z * (u * u - u) / 2.0))
    m = orc.halfwidth(z)
    ks = rc + np.arange(-m, m + 1)
    # O(nt * taps) DFT straight from eq. 5, normalised by nt
    n = np.arange(nt)
    dft = np.array([np.sum(x * np.exp(-2j * np.pi * n * k / nt)) for k in ks]) / nt
    assert np.max(np.abs(dft - orc.taps(z))) < 5.0 / nt ** 1.5 + 1e-6
    # sign of z (R3): positive z = frequency rising with time; the wrong sign is far off
    assert np.max(np.abs(dft - orc.taps(-z))) > 1e-2


# ---------------------------------------------------------------- symmetry of the bank (R2)
@pytest.mark.parametrize("z", [2.0, 20.0, 84.0, 200.0])
def test_conjugate_and_even_symmetry(z):
    hp, hm = orc.taps(z), orc.taps(-z)
    assert np.max(np.abs(hm - np.conj(hp))) < 1e-13          # h_{-z} = conj(h_z)
    assert np.max(np.abs(hp - hp[::-1])) < 1e-13             # even in the bin offset


def test_r5_tap_energy():
    # reading R5: unit-amplitude response, no renormalisation after truncation
    for z, e in [(0, 1.0), (2, 0.99999), (8, 0.99987), (20, 0.99956), (84, 0.99861), (200, 0.99803)]:
        assert abs(np.sum(np.abs(orc.taps(float(z))) ** 2) - e) < 6e-6
    # -> 1 as m grows (Parseval)
    assert abs(np.sum(np.abs(orc.taps(20.0, 400)) ** 2) - 1.0) < 2e-4


def test_bank_and_halfwidth():
    zs = orc.bank_z(20.0, 2.0)
    assert zs.size == 21 and zs[0] == -20.0 and zs[-1] == 20.0 and zs[10] == 0.0
    assert orc.halfwidth(20.0) == 26 and orc.halfwidth(84.0) == 58 and orc.halfwidth(200.0) == 116
    assert orc.halfwidth(-7.0) == 20
    with pytest.raises(ValueError):
        orc.bank_z(5.0, 2.0)


# ---------------------------------------------------------------- direct sum: C vs numpy vs pure Python
def test_c_direct_sum_matches_numpy_and_python_loops():
    a = syn.make_spectrum(600, 11)
    a128 = a.astype(np.complex128)
    for z in (0.0, 6.0, -20.0):
        h = orc.taps(z)
        m = (h.size - 1) // 2
        yc = orc.correlate(a, h, -5, 620)                    # includes columns outside [0,N)
        # eq. 3 as a literal double loop
        yp = np.zeros(620, dtype=np.complex128)
        for i in range(620):
            r = i - 5
            acc = 0j
            for d in range(-m, m + 1):
                if 0 <= r + d < 600:
                    acc += a128[r + d] * np.conj(h[d + m])
            yp[i] = acc
        assert np.max(np.abs(yc - yp)) < 1e-12
        assert np.max(np.abs(orc.correlate_numpy(a, h) - yp[5:605])) < 1e-12
        cols = np.array([0, 1, 57, 599, 600, 333])
        assert np.max(np.abs(orc.correlate_at(a, h, cols) - yp[cols + 5])) < 1e-12


# ---------------------------------------------------------------- P4: injected chirp peaks at its cell
def test_p4_injected_chirp_peak_config1_shape():
    a, chirps = syn.config_spectrum(0)
    (r0, z0, amp), = chirps
    plane = orc.plane(a, 20.0, 2.0)
    k, r = np.unravel_index(np.argmax(plane), plane.shape)
    assert orc.bank_z(20.0, 2.0)[k] == z0 and r == round(r0)
    # amplitude a at a quarter-bin offset: a^2 sinc^2(1/4) = 729.5, plus noise cross terms
    assert abs(plane[k, r] - amp ** 2 * np.sinc(0.25) ** 2) < 4 * 2 * amp
    # wrong-sign row is far weaker
    assert plane[20 - k, r] < 0.3 * plane[k, r]


def test_p4_off_grid_z_within_one_row():
    n = 1 << 14
    a = syn.make_spectrum(n, 5, [(5000.0, -11.0, 40.0)])
    plane = orc.plane(a, 20.0, 2.0)
    k, r = np.unravel_index(np.argmax(plane), plane.shape)
    assert abs(orc.bank_z(20.0, 2.0)[k] - (-11.0)) <= 1.0 + 1e-9 and abs(r - 5000) <= 1


# ---------------------------------------------------------------- P5: noiseless plane closed form
def test_p5_noiseless_plane_is_difference_template():
    n, rc, z0, amp = 4096, 2000, 12.0, 3.0
    k = np.arange(n)
    a = (amp * _closed_form(z0, (k - rc).astype(np.float64))).astype(np.complex64)
    for z, tol in [(12.0, 3e-3), (0.0, 1e-6), (4.0, 2e-2), (-20.0, 2e-2)]:
        y = orc.correlate(a, orc.taps(z))
        expect = amp * _closed_form(z0 - z, (k - rc).astype(np.float64))
        assert np.max(np.abs(y - expect)) < tol * amp
    # convergence with the half-width: the deviation shrinks as m grows
    e = [np.max(np.abs(orc.correlate(a, orc.taps(12.0, m)) - amp * _closed_form(0.0, (k - rc) * 1.0)))
         for m in (22, 60, 200)]
    assert e[0] > e[1] > e[2]


# ---------------------------------------------------------------- P6/P7: invariants
def test_p6_reversal_symmetry():
    a = syn.make_spectrum(3000, 21, [(1500.3, 9.0, 20.0)])
    ar = np.conj(a[::-1]).copy()
    for z in (4.0, 14.0):
        p = orc.plane_row(ar, z)
        q = orc.plane_row(a, -z)
        assert np.max(np.abs(p - q[::-1])) < 1e-9 * np.max(q)


def test_p7_shift_and_scale():
    a = syn.make_spectrum(3000, 22)
    z = 10.0
    p = orc.plane_row(a, z)
    b = np.zeros_like(a)
    b[37:] = a[:-37]
    pb = orc.plane_row(b, z)
    m = orc.halfwidth(z)
    assert np.max(np.abs(pb[37 + m:3000 - m] - p[m:3000 - 37 - m])) < 1e-10
    c = (a.astype(np.complex128) * (0.5 - 2.0j)).astype(np.complex64)
    a128, c128 = a.astype(np.complex128), c.astype(np.complex128)
    scale = np.abs(c128[100] / a128[100]) ** 2
    assert np.max(np.abs(orc.plane_row(c, z) - scale * p)) < 1e-5 * np.max(p)   # complex64 rounding of c


# ---------------------------------------------------------------- P8: noise statistics
def test_p8_noise_statistics():
    a = syn.make_spectrum(1 << 16, 33)
    for z in (0.0, 20.0, -84.0):
        p = orc.plane_row(a, z)
        e = np.sum(np.abs(orc.taps(z)) ** 2)
        assert abs(np.mean(p) - e) < 4.0 / math.sqrt(a.size) * 3
        # exponential distribution: variance = mean^2 (filtered samples are correlated -> loose)
        assert abs(np.var(p) / np.mean(p) ** 2 - 1.0) < 0.1


# ---------------------------------------------------------------- P9: interbinning, eq. 4 and PAPER.md:89
def _golden(golden_dir):
    vals = {}
    with open(golden_dir + "/interbin_loss.txt") as f:
        for line in f:
            if line.startswith("#") or not line.strip():
                continue
            name, v, tol = line.split()
            vals[name] = (float(v), float(tol))
    return vals


def test_p9_interbin_losses_printed_by_paper(golden_dir):
    g = _golden(golden_dir)
    n = 512
    worst_plain, worst_ib = 0.0, 0.0
    nn = np.arange(n) / n
    for off in np.linspace(0.0, 0.5, 201):
        x = np.exp(2j * np.pi * (100.0 + off) * nn)          # unit tone at bin 100 + off
        a = (np.fft.fft(x) / n).astype(np.complex64)
        row = orc.plane_row(a, 0.0, interbin=True)
        amp_plain = math.sqrt(np.max(row[0::2]))
        amp_ib = math.sqrt(np.max(row))
        worst_plain = max(worst_plain, 1.0 - amp_plain)
        worst_ib = max(worst_ib, 1.0 - amp_ib)
    v, tol = g["max_amplitude_loss_without_interbinning"]
    assert abs(100 * worst_plain - v) < tol          # 36.34 %
    v, tol = g["max_amplitude_loss_with_interbinning"]
    assert abs(100 * worst_ib - v) < tol             # 7.41 %


def test_p9_interbin_half_bin_tone_and_layout():
    n, amp = 1024, 5.0
    nn = np.arange(n) / n
    a = (np.fft.fft(amp * np.exp(2j * np.pi * 300.5 * nn)) / n).astype(np.complex64)
    row = orc.plane_row(a, 0.0, interbin=True)
    assert row.size == 2 * n
    assert np.argmax(row) == 2 * 300 + 1 and abs(row[601] - amp * amp) < 1e-3
    # on-bin tone: the neighbouring half-bins carry (pi/4)^2 a^2 (minus sign of eq. 4 kept, R8)
    b = np.zeros(n, dtype=np.complex64)
    b[300] = amp
    rb = orc.plane_row(b, 0.0, interbin=True)
    assert abs(rb[600] - 25.0) < 1e-12 and abs(rb[601] - (math.pi / 4) ** 2 * 25.0) < 1e-12
    assert abs(rb[599] - (math.pi / 4) ** 2 * 25.0) < 1e-12
    # last half-bin uses y[N] from the zero-extended sum (R7): spectrum with power in the last bin
    c = np.zeros(n, dtype=np.complex64)
    c[n - 1] = 2.0
    rc = orc.plane_row(c, 6.0, interbin=True)
    h = orc.taps(6.0)
    m = (h.size - 1) // 2
    y_last, y_n = 2.0 * np.conj(h[m]), 2.0 * np.conj(h[m - 1])
    assert abs(rc[2 * n - 1] - (math.pi / 4) ** 2 * abs(y_last - y_n) ** 2) < 1e-12
    # sampled-cell accessor agrees with the full row
    cols = np.array([0, 1, 2, 601, 2 * n - 1, 2 * n - 2])
    assert np.max(np.abs(orc.plane_cells(c, 6.0, cols, interbin=True) - rc[cols])) < 1e-14


# ---------------------------------------------------------------- P10: fp64 FFT overlap-save == direct sum
def _overlap_save_fp64(a, h, seglen):
    """PAPER.md:75-77 / Fig. 1 written with numpy's fp64 FFT (independent of the C direct sum)."""
    n = a.size
    m = (h.size - 1) // 2
    g = np.zeros(seglen, dtype=np.complex128)
    for d in range(-m, m + 1):
        g[(-d) % seglen] = np.conj(h[d + m])      # centred at bin 0, halves at both ends
    G = np.fft.fft(g)
    B = seglen - 2 * m
    nseg = -(-n // B)
    pad = np.zeros(m + nseg * B + m + seglen, dtype=np.complex128)
    pad[m:m + n] = a
    out = np.empty(nseg * B, dtype=np.complex128)
    for s in range(nseg):
        seg = pad[s * B:s * B + seglen]
        y = np.fft.ifft(np.fft.fft(seg) * G)
        out[s * B:(s + 1) * B] = y[m:m + B]
    return out[:n]


@pytest.mark.parametrize("seglen", [256, 1024])
def test_p10_overlap_save_equals_direct(seglen):
    a = syn.make_spectrum(5000, 44, [(2500.5, 15.0, 10.0)])
    for z in (-20.0, 0.0, 16.0):
        h = orc.taps(z)
        y_direct = orc.correlate(a, h)
        y_os = _overlap_save_fp64(a.astype(np.complex128), h, seglen)
        assert np.max(np.abs(y_direct - y_os)) < 1e-11


def test_cmacs_count():
    # 6.0e7 complex MACs for config 1
    assert orc.cmacs(1 << 16, 20.0, 2.0) == (1 << 16) * 913


# ---------------------------------------------------------------- P11: threshold search (reading R15)
def test_p11_threshold_limits_and_z0_row():
    a = syn.make_spectrum(1 << 14, 61)
    n = a.size
    for ib in (False, True):
        ncols = 2 * n if ib else n
        rows, cols, pows = orc.candidates(a, 4.0, 2.0, -1.0, ib)          # below every power: every cell
        assert rows.size == 5 * ncols and np.array_equal(cols[:ncols], np.arange(ncols))
        rows, cols, pows = orc.candidates(a, 4.0, 2.0, float("inf"), ib)  # above every power: nothing
        assert rows.size == 0
    # z = 0 row: h_0 is the Kronecker delta (P2), so its candidates are the raw bins with |A|^2 > thr
    rows, cols, pows = orc.candidates(a, 4.0, 2.0, 5.0)
    raw = np.abs(a.astype(np.complex128)) ** 2
    assert np.array_equal(cols[rows == 2], np.nonzero(raw > 5.0)[0])
    assert np.allclose(pows[rows == 2], raw[raw > 5.0], rtol=1e-14, atol=0)
    # sorted by (row, col), strict inequality
    key = rows * (1 << 40) + cols
    assert np.all(np.diff(key) > 0) and np.all(pows > 5.0)


def test_p11_noise_tail_law():
    # unit-power white noise -> filtered powers are exponential with mean E_z = sum|h_z|^2 (P8), so the
    # expected count above thr in row z is N exp(-thr / E_z)
    a = syn.make_spectrum(1 << 17, 62)
    thr = 6.0
    rows, cols, pows = orc.candidates(a, 20.0, 10.0, thr)
    for k, z in enumerate(orc.bank_z(20.0, 10.0)):
        e = np.sum(np.abs(orc.taps(z)) ** 2)
        expect = a.size * math.exp(-thr / e)
        got = int(np.sum(rows == k))
        assert abs(got - expect) < 5.0 * math.sqrt(expect) * 1.5, (z, got, expect)   # neighbours correlate: loose


def test_p11_injected_chirp_is_the_candidate():
    n, r0, z0, amp = 1 << 13, 3000, 8.0, 50.0
    a = syn.chirp_spectrum(n, [(float(r0), z0, amp)]).astype(np.complex64)
    zs = orc.bank_z(20.0, 2.0)
    k0 = int(np.nonzero(zs == z0)[0][0])
    rows, cols, pows = orc.candidates(a, 20.0, 2.0, 0.9 * amp ** 2)
    assert rows.size >= 1
    i = int(np.argmax(pows))
    assert (rows[i], cols[i]) == (k0, r0) and abs(pows[i] - amp ** 2) < 0.01 * amp ** 2
    assert np.all(np.abs(rows - k0) <= 1) and np.all(np.abs(cols - r0) <= 1)
    # half-bin tone, interbinned: the candidate sits in the odd column 2 r0 + 1 (P9 layout)
    b = syn.chirp_spectrum(n, [(r0 + 0.5, 0.0, amp)]).astype(np.complex64)
    rows, cols, pows = orc.candidates(b, 4.0, 2.0, 0.9 * amp ** 2, True)
    i = int(np.argmax(pows))
    assert (rows[i], cols[i]) == (2, 2 * r0 + 1)


# ---------------------------------------------------------------- P12: 2-bin Fourier interpolation (R16)
def test_p12_half_offset_response_is_the_dft_of_a_half_bin_chirp():
    # time-domain chirp centred on a half-integer frequency, DFT at integer bins k: h_z(k - r_c) with
    # k - r_c half-integer.  Endpoint (Riemann) term makes this O(1/Nt) for fractional r_c.
    nt, rc, z = 8192, 700.5, 12.0
    u = np.arange(nt) / nt
    x = np.exp(2j * np.pi * (rc * u + z * (u * u - u) / 2.0))
    spec = np.fft.fft(x) / nt
    m = orc.halfwidth(z)
    t2 = orc.taps2(z)                                   # h_z(j/2), j = -2m..2m
    odd = t2[1::2]                                      # j = -2m+1, -2m+3, ...: offsets d - 1/2, d = -m+1..m
    k = np.arange(-m + 1, m + 1) + int(rc - 0.5)        # k - rc = d - 1/2
    assert np.max(np.abs(spec[k] - odd)) < 3.0 / nt
    assert np.allclose(t2[0::2], orc.taps(z), rtol=0, atol=1e-15)         # even j: the integer-offset taps
    assert np.max(np.abs(odd + odd[::-1])) < 1e-14                        # h(x) = -h(-x) at half-integers


def test_p12_even_columns_are_the_plain_plane_and_z0_is_zero_padded_dft():
    nt = 4096
    rng = np.random.default_rng(5)
    x = rng.standard_normal(nt) + 1j * rng.standard_normal(nt)
    a = (np.fft.fft(x) / nt).astype(np.complex64)
    for z in (0.0, 6.0, -20.0):
        p2 = orc.plane_row(a, z, 2)
        assert p2.size == 2 * nt
        assert np.allclose(p2[0::2], orc.plane_row(a, z, 0), rtol=1e-12, atol=0)
    # z = 0: the half-bin amplitudes are the DFT of the time series zero-padded to 2 Nt (exact Fourier
    # interpolation) up to the truncation of the sinc taps, which shrinks as the half-width grows
    x64 = np.fft.ifft(a.astype(np.complex128)) * nt
    fine = np.abs(np.fft.fft(np.concatenate([x64, np.zeros(nt)])) / nt) ** 2
    errs = []
    for m in (16, 128, 1024):
        p2 = orc.plane_row(a, 0.0, 2, m=m)
        sl = slice(2 * m + 1, 2 * (nt - m) - 1, 2)      # odd columns away from the zero-extended edges
        errs.append(np.sqrt(np.mean((p2[sl] - fine[sl]) ** 2)) / np.mean(fine[sl]))
    assert errs[0] > errs[1] > errs[2] and errs[2] < 2e-2, errs


def test_p12_half_bin_chirp_peaks_in_its_odd_column():
    n, r0, z0, amp = 1 << 13, 3000, 8.0, 5.0
    a = syn.chirp_spectrum(n, [(r0 + 0.5, z0, amp)]).astype(np.complex64)
    zs = orc.bank_z(20.0, 2.0)
    pl = np.stack([orc.plane_row(a, z, 2) for z in zs])
    k, c = np.unravel_index(np.argmax(pl), pl.shape)
    assert zs[k] == z0 and c == 2 * r0 + 1
    e = np.sum(np.abs(orc.taps2(z0)[1::2]) ** 2)        # energy of the truncated half-offset taps
    assert abs(pl[k, c] - amp ** 2 * e ** 2) < 1e-3 * amp ** 2 and 0.95 < e < 1.0
    # unit white noise: odd columns average to that energy (as P8)
    b = syn.make_spectrum(1 << 16, 34)
    p = orc.plane_row(b, z0, 2)
    assert abs(np.mean(p[1::2]) - e) < 12.0 / math.sqrt(b.size)


def test_p12_sampled_cells_of_the_two_bin_plane_are_the_literal_interleaved_sum():
    """`plane_cells(..., interbin=2)` (sampled checks of the GPU's interbin = 2 planes): column c of the
    double-resolution plane written out as a literal loop over the ZERO-INTERLEAVED spectrum and
    the half-spaced template h_z(j/2) -- even and odd columns, both edges, z of both signs and z = 0 (whose odd
    columns are the zero-padded-DFT interpolation of P12's second pin)."""
    a = syn.make_spectrum(300, 13, [(140.5, 5.0, 8.0)])
    a128 = a.astype(np.complex128)
    cols = np.array([0, 1, 2, 3, 279, 280, 281, 598, 599])
    for z in (0.0, 6.0, -20.0):
        m = orc.halfwidth(z)
        t = orc.response(z, 0.5 * np.arange(-2 * m, 2 * m + 1))      # h_z(j/2), j = -2m..2m
        ref = np.zeros(cols.size)
        for i, c in enumerate(cols):
            acc = 0j
            for j in range(-2 * m, 2 * m + 1):
                q = c + j                                            # index in the interleaved spectrum
                if 0 <= q < 600 and q % 2 == 0:                      # odd entries are the interleaved zeros
                    acc += a128[q // 2] * np.conj(t[j + 2 * m])
            ref[i] = acc.real ** 2 + acc.imag ** 2
        got = orc.plane_cells(a, z, cols, 2)
        assert np.max(np.abs(got - ref)) < 1e-12 * max(1.0, ref.max())
        assert np.max(np.abs(got - orc.plane_row(a, z, 2)[cols])) < 1e-12 * max(1.0, ref.max())
    # even columns are the plain plane's cells
    assert np.allclose(orc.plane_cells(a, 6.0, cols[cols % 2 == 0], 2), orc.plane_cells(a, 6.0, cols[cols % 2 == 0] // 2, False),
                       rtol=1e-12, atol=1e-15)


def test_bank_centre_is_exactly_zero_for_fractional_dz():
    for zmax, dz in ((6.0, 0.5), (0.3, 0.1), (84.0, 2.0), (2.1, 0.7)):
        zs = orc.bank_z(zmax, dz)
        assert zs[zs.size // 2] == 0.0 and np.all(np.diff(zs) > 0)
