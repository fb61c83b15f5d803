"""
Pins of the oracle's red-noise removal and block normalisation (oracle.deredden / oracle.normalise_blocks;
PAPER.md:79, readings R19, R20) against what the mathematics fixes -- P15.  CPU only.
"""
import math

import numpy as np
import pytest

from oracle import fdas_oracle as orc

LN2 = 0.6931471805599453


def noise(n, seed):
    rng = np.random.Generator(np.random.Philox(seed))
    return (rng.standard_normal(n) + 1j * rng.standard_normal(n)) / math.sqrt(2.0)     # E|A|^2 = 1


def test_hand_sorted_tiny_blocks():
    # block of 5: powers 25, 1, 9, 4, 16 -> sorted 1 4 9 16 25 -> median 9; block of 4 (ragged tail):
    # powers 4, 1, 16, 9 -> sorted 1 4 9 16 -> median (4 + 9) / 2 = 6.5
    a = np.array([3 + 4j, 1j, -3, 2, -4j, 2j, 1, 4, -3j])
    out = orc.deredden(a, 5)
    assert np.allclose(out[:5], a[:5] / math.sqrt(9 / LN2), rtol=1e-15, atol=0)
    assert np.allclose(out[5:], a[5:] / math.sqrt(6.5 / LN2), rtol=1e-15, atol=0)
    out = orc.normalise_blocks(a, 5)
    assert np.allclose(out[:5], a[:5] / math.sqrt(55 / 5), rtol=1e-15, atol=0)
    assert np.allclose(out[5:], a[5:] / math.sqrt(30 / 4), rtol=1e-15, atol=0)
    # a literal selection-sort median, element by element, against the library median the oracle calls
    rng = np.random.default_rng(3)
    for w in (1, 2, 3, 6, 7, 32, 33):
        x = noise(w, 40 + w) * rng.uniform(0.5, 3.0)
        p = [abs(v) ** 2 for v in x]
        for i in range(w):                                      # selection sort
            m = min(range(i, w), key=p.__getitem__)
            p[i], p[m] = p[m], p[i]
        med = p[w // 2] if w % 2 else 0.5 * (p[w // 2 - 1] + p[w // 2])
        assert np.allclose(orc.deredden(x, w), x / math.sqrt(med / LN2), rtol=1e-14, atol=0)


def test_white_noise_keeps_unit_mean_power():
    n = 1 << 18
    a = noise(n, 7)
    for block in (64, 1000, 4096):
        out = orc.deredden(a, block)
        # median / ln 2 of w exponential powers estimates the mean with relative bias ~ 1/(2w) ... and scatter 1/sqrt(w)
        # per block; over the whole spectrum the mean power stays 1 within 3/sqrt(N) plus that bias
        assert abs(np.mean(np.abs(out) ** 2) - 1.0) < 3.0 / math.sqrt(n) + 2.0 / block
    out = orc.normalise_blocks(a, 1932)
    assert abs(np.mean(np.abs(out) ** 2) - 1.0) < 1e-12        # every block has mean power exactly 1


def test_power_law_spectrum_comes_out_flat():
    n, block = 1 << 18, 256
    f = np.arange(1, n + 1, dtype=np.float64)
    red = noise(n, 11) * np.sqrt(1.0 + (2000.0 / f) ** 2.5)     # red below bin ~2000, white above
    before = [np.mean(np.abs(red[lo:hi]) ** 2) for lo, hi in ((256, 512), (1024, 2048), (1 << 16, 1 << 17))]
    assert before[0] > 30 * before[2] and before[1] > 3 * before[2]
    out = orc.deredden(red, block)
    for lo, hi in ((256, 512), (1024, 2048), (8192, 16384), (1 << 16, 1 << 17)):
        m = np.mean(np.abs(out[lo:hi]) ** 2)
        # flat at 1: scatter of (hi-lo)/block block estimates, each good to ~1/sqrt(block); the slope inside one
        # block of the steepest part (bins 256..512: power changes by ~2.5 x 256/384) biases it by a few per cent
        assert abs(m - 1.0) < 0.12, (lo, hi, m)


def test_strong_narrow_tone_survives():
    n, block, a_tone, j0 = 1 << 14, 256, 50.0, 5000
    a = noise(n, 13)
    b = a.copy()
    b[j0] += a_tone
    clean, withtone = orc.deredden(a, block), orc.deredden(b, block)
    s = clean[j0 - 1] / a[j0 - 1]                              # the block's scale without the tone (real, > 0)
    assert abs(s.imag) < 1e-15 and abs(s.real - 1.0) < 0.2
    # one outlier moves the median of 256 values by at most one rank: the scale changes by O(1/block)
    assert abs(abs(withtone[j0]) - abs(b[j0]) * s.real) < 2.0 / block * abs(b[j0])
    assert abs(withtone[j0]) > 0.8 * a_tone
    other = np.ones(n, bool)
    other[j0 // block * block:(j0 // block + 1) * block] = False
    assert np.array_equal(clean[other], withtone[other])       # other blocks are untouched by it
    # the MEAN would have been dragged: 50^2 / 256 ~ 10 x the noise level -- the reason R19 reads "median"
    assert abs(orc.normalise_blocks(b, block)[j0]) < 0.35 * a_tone


def test_block_normalisation_invariants():
    n, block = 10007, 1932                                      # ragged last block of 347 bins
    a = noise(n, 17) * np.repeat(np.linspace(0.2, 5.0, 11), 1000)[:n]
    out = orc.normalise_blocks(a, block)
    for start in range(0, n, block):
        assert abs(np.mean(np.abs(out[start:start + block]) ** 2) - 1.0) < 1e-12
    assert np.allclose(orc.normalise_blocks(out, block), out, rtol=1e-12, atol=0)          # idempotent
    assert np.allclose(orc.normalise_blocks(3.7j * a, block), 1j * out, rtol=1e-12, atol=1e-300)   # scale-free
    assert np.allclose(orc.deredden(0.01 * a, 100), orc.deredden(a, 100), rtol=1e-12, atol=0)
    med = orc.deredden(a, block)
    for start in range(0, n, block):
        assert abs(np.median(np.abs(med[start:start + block]) ** 2) - LN2) < 1e-12
    # phases are untouched, the scale is one positive real number per block
    assert np.allclose(np.angle(out), np.angle(a), atol=1e-12)
    r = (out / a).reshape(-1)
    assert np.all(np.abs(r[:block] - r[0]) < 1e-12)


def test_degenerate_blocks():
    a = noise(300, 19)
    a[100:200] = 0.0                                            # an all-zero block is copied, not divided by zero
    for fn in (orc.deredden, orc.normalise_blocks):
        out = fn(a, 100)
        assert np.all(np.isfinite(out.real)) and np.all(out[100:200] == 0.0)
        assert fn(np.zeros(0, complex), 8).size == 0
        one = fn(np.array([3 + 4j]), 8)                         # a single bin: its own power is both statistics
    assert np.allclose(orc.normalise_blocks(np.array([3 + 4j]), 8), [(3 + 4j) / 5.0])
    assert np.allclose(orc.deredden(np.array([3 + 4j]), 8), [(3 + 4j) / math.sqrt(25 / LN2)])
    b = noise(64, 23)
    b[:40] = 0.0                                                # median 0 with a non-zero mean: deredden copies
    assert np.array_equal(orc.deredden(b, 64), b) and not np.array_equal(orc.normalise_blocks(b, 64), b)
    with pytest.raises(ValueError):
        orc.deredden(a, 0)
