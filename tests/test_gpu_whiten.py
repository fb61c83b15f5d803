"""
GPU parity (-m gpu) of red-noise removal and block normalisation (fdas_whiten, SURVEY.md section 8(f) F3,
DESIGN.md readings R19 / R20) against oracle.deredden / oracle.normalise_blocks, through the C ABI.

Tolerance: the kernel forms the powers in float32 (relative error 1.2e-7), selects the exact
median of those, forms the scale in double and rounds it to float32 (6e-8), and multiplies (6e-8): every output bin
is within 5e-7 of the oracle's, relative to its own magnitude; relative L2 <= 3e-7.
"""
import math

import numpy as np
import pytest

pytestmark = pytest.mark.gpu

ELEM_TOL, L2_TOL = 5e-7, 3e-7


@pytest.fixture(scope="module")
def torch():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    return torch


@pytest.fixture(scope="module")
def fd(torch):
    from paper_1804_05335_b200 import fdas
    return fdas


@pytest.fixture(scope="module")
def orc():
    from oracle import fdas_oracle
    return fdas_oracle


def red_spectrum(n, seed, tones=()):
    """Unit-power complex noise with a power-law excess below bin ~n/50 and a slow ripple, plus narrow tones."""
    rng = np.random.Generator(np.random.Philox(seed))
    a = (rng.standard_normal(n) + 1j * rng.standard_normal(n)) / math.sqrt(2.0)
    f = np.arange(1, n + 1, dtype=np.float64)
    a *= np.sqrt(1.0 + (n / 50.0 / f) ** 2.2) * (1.0 + 0.3 * np.sin(f / (n / 37.0)))
    for j, amp in tones:
        a[j] += amp
    return a.astype(np.complex64)


def run(torch, fd, spec, block, stat, inplace=False):
    n = spec.size
    d_in = torch.from_numpy(spec.view(np.float32).reshape(n, 2).copy()).cuda()
    d_out = d_in if inplace else torch.full((n, 2), float("nan"), dtype=torch.float32, device="cuda")
    fd.fdas_whiten(torch.cuda.current_stream(), d_in, d_out, n, block, stat)
    torch.cuda.synchronize()
    if not inplace:
        assert np.array_equal(d_in.cpu().numpy().view(np.complex64).reshape(-1), spec)     # input untouched
    return d_out.cpu().numpy().view(np.complex64).reshape(-1)


def check(got, ref):
    assert got.shape == ref.shape and np.all(np.isfinite(got.real)) and np.all(np.isfinite(got.imag))
    g = got.astype(np.complex128)
    err = np.abs(g - ref)
    nz = np.abs(ref) > 0
    assert np.all(err[~nz] == 0)
    worst = float(np.max(err[nz] / np.abs(ref[nz]))) if nz.any() else 0.0
    l2 = math.sqrt(np.sum(err ** 2) / max(np.sum(np.abs(ref) ** 2), 1e-300))
    print(f"whiten n={ref.size}: worst element {worst:.2e}, rel L2 {l2:.2e}")
    assert worst <= ELEM_TOL and l2 <= L2_TOL


CASES = [(1 << 21, 1024, 0), (1 << 21, 1920, 1), (1 << 21, 1920, 0), (1 << 23, 3968, 1), (1 << 23, 4096, 0),
         (1 << 22, 8192, 0), (1 << 22, 8191, 0), (1 << 22, 7936, 1), (100003, 97, 0), (100003, 97, 1), (100003, 32, 0),
         (5, 64, 0), (5, 64, 1), (1, 32, 0), (2, 32, 0), (1000, 8192, 0), (70001, 333, 0)]


@pytest.mark.parametrize("nbins,block,stat", CASES)
def test_whiten_matches_oracle(torch, fd, orc, nbins, block, stat):
    spec = red_spectrum(nbins, 900 + nbins % 1000 + block, [(nbins // 3, 40.0), (nbins // 2, 25.0)] if nbins > 100 else ())
    got = run(torch, fd, spec, block, stat)
    ref = (orc.normalise_blocks if stat else orc.deredden)(spec, block)
    check(got, ref)
    if stat and nbins > 100:                                   # R20: unit mean power per block, to float32 rounding
        p = np.abs(got.astype(np.complex128)) ** 2
        for start in (0, (nbins // block // 2) * block, (nbins - 1) // block * block):
            assert abs(np.mean(p[start:start + block]) - 1.0) < 1e-6


@pytest.mark.parametrize("stat", [0, 1])
def test_whiten_in_place_and_repeatable(torch, fd, stat):
    spec = red_spectrum(300007, 5, [(1000, 30.0)])
    a = run(torch, fd, spec, 1000, stat)
    assert np.array_equal(a, run(torch, fd, spec, 1000, stat))                  # bitwise repeatable
    assert np.array_equal(a, run(torch, fd, spec, 1000, stat, inplace=True))    # in place = out of place


def test_whiten_degenerate_blocks_and_exact_median(torch, fd, orc):
    spec = red_spectrum(640, 6)
    spec[64:128] = 0                                            # all-zero block: copied
    spec[128:168] = 0                                           # 40 of 64 zero: median 0 (copied), mean > 0 (scaled)
    for stat, fn in ((0, orc.deredden), (1, orc.normalise_blocks)):
        got = run(torch, fd, spec, 64, stat)
        check(got, fn(spec, 64))
        assert np.all(got[64:128] == 0)
    assert np.array_equal(run(torch, fd, spec, 64, 0)[128:192], spec[128:192])
    # many equal powers around the middle rank (ties in every radix pass), odd and even counts
    for n in (63, 64):
        amp = np.concatenate([np.full(n // 2 - 3, 0.5), np.full(8, 2.0), np.full(n - n // 2 - 5, 7.0)])
        rng = np.random.default_rng(n)
        s2 = (amp * np.exp(2j * np.pi * rng.random(n)))[rng.permutation(n)].astype(np.complex64)
        check(run(torch, fd, s2, 64, 0), orc.deredden(s2, 64))


def test_whiten_errors(torch, fd):
    x = torch.zeros((4096, 2), dtype=torch.float32, device="cuda")
    for block in (0, 16, 31, 8193):
        with pytest.raises(fd.FdasError) as e:
            fd.fdas_whiten(None, x, x, 4096, block, 0)
        assert e.value.status == 2 and str(block) in str(e.value)
    for args in ((None, x, 4096, 64, 0), (x, None, 4096, 64, 0), (x, x, 0, 64, 0), (x, x, 4096, 64, 2), (x, x, 4096, 64, -1)):
        with pytest.raises(fd.FdasError) as e:
            fd.fdas_whiten(None, *args)
        assert e.value.status == 1
    with pytest.raises(fd.FdasError) as e:
        fd.fdas_whiten(None, x.view(-1)[1:], x, 2000, 64, 0)
    assert e.value.status == 4


def test_red_series_to_plane_pipeline(torch, fd, orc):
    """Fig. 2 of the paper on one stream: series -> fdas_r2c_execute -> fdas_whiten (median, then per overlap-save
    block) -> fdas_execute, against the oracle's dft_real -> deredden -> normalise_blocks -> plane rows.  The series
    carries red noise (a random walk) and an accelerated tone, which must come out as the plane's peak."""
    n, zmax, dz, seglen = 1 << 15, 20.0, 2.0, 1024
    nb = n // 2
    rng = np.random.Generator(np.random.Philox(77))
    u = np.arange(n) / n
    r0, z0, amp = 3000.0, 8.0, 0.5
    x = rng.standard_normal(n) + 0.2 * np.cumsum(rng.standard_normal(n)) \
        + amp * np.cos(2 * np.pi * (r0 * u + z0 * (u * u - u) / 2))
    x = (x - x.mean()).astype(np.float32)
    scale = 1.0 / math.sqrt(n / 2)
    with fd.R2CPlan(n) as r2c, fd.Plan(nb, zmax, dz, seglen, 0) as plan:
        plan.make_templates()
        B = plan.info.useful
        st = torch.cuda.current_stream()
        d_x = torch.from_numpy(x).cuda()
        d_spec = torch.empty((nb, 2), dtype=torch.float32, device="cuda")
        d_plane = torch.full((plan.info.ntemplates, nb), float("nan"), dtype=torch.float32, device="cuda")
        r2c.execute(st, d_x, d_spec, scale)
        fd.fdas_whiten(st, d_spec, d_spec, nb, 256, fd.WHITEN_MEDIAN)
        fd.fdas_whiten(st, d_spec, d_spec, nb, B, fd.WHITEN_MEAN)
        plan.execute(st, d_spec, d_plane)
        torch.cuda.synchronize()
        plane = d_plane.cpu().numpy().astype(np.float64)
        spec_gpu = d_spec.cpu().numpy().view(np.complex64).reshape(-1)
    raw = orc.dft_real(x) * scale
    assert np.mean(np.abs(raw[8:64]) ** 2) > 20 * np.mean(np.abs(raw[nb // 2:]) ** 2)          # it IS red
    white = orc.normalise_blocks(orc.deredden(raw.astype(np.complex64), 256).astype(np.complex64), B)
    assert np.max(np.abs(spec_gpu - white)) <= 2e-5 * np.max(np.abs(white))
    # the median step alone flattens the spectrum: away from the first blocks (where a 1/f^2 slope crosses a block
    # and biases its median) and from the tone, the mean power is 1
    flat = np.abs(orc.deredden(raw.astype(np.complex64), 256)) ** 2
    assert abs(np.mean(flat[512:2048]) - 1.0) < 0.25 and abs(np.mean(flat[nb // 2:]) - 1.0) < 0.05
    zs = orc.bank_z(zmax, dz)
    w64 = white.astype(np.complex64)
    for k in (0, 10, 14, 20):
        ref = orc.plane_row(w64, zs[k], False)
        assert np.max(np.abs(plane[k] - ref)) <= 1e-4 * np.max(ref)
        assert math.sqrt(np.sum((plane[k] - ref) ** 2) / np.sum(ref ** 2)) <= 1e-4     # inputs differ at float32 rounding
    k, c = np.unravel_index(np.argmax(plane[:, 500:]), plane[:, 500:].shape)
    assert zs[k] == z0 and c + 500 == int(r0)
