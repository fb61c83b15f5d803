"""
GPU parity (-m gpu) of the two rows past the correlation: the real-to-complex transform in front of it
(fdas_r2c_*) and harmonic summing behind it (fdas_harmonic_sum_threshold, F2), each against
the oracle (oracle.dft_real* / oracle.harmonic_*), through the C ABI.

Tolerance of the transform: fp32 arithmetic over log2(n) <= 25 radix-2 levels with
fp64-evaluated twiddles: relative L2 error of the compared bins <= 3e-6 (measured: 1.1e-7 .. 1.9e-7) and
|dX| <= 1e-5 * max|X| per bin (a bin's rounding error scales with the largest amplitudes that pass through
its butterflies, i.e. with the injected tone's bin, not with the noise floor).
"""
import math

import numpy as np
import pytest

pytestmark = pytest.mark.gpu

R2C_L2, R2C_MAX = 3e-6, 1e-5


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


def series(n, seed, tones=()):
    rng = np.random.Generator(np.random.Philox(seed))
    x = rng.standard_normal(n)
    u = np.arange(n) / n
    for (r, z, a) in tones:
        x += a * np.cos(2 * np.pi * (r * u + z * (u * u - u) / 2))
    return x.astype(np.float32)


def run_r2c(torch, fd, x, scale=1.0):
    n = x.size
    with fd.R2CPlan(n) as plan:
        d_x = torch.from_numpy(x).cuda()
        d_out = torch.full((n // 2, 2), float("nan"), dtype=torch.float32, device="cuda")
        plan.execute(torch.cuda.current_stream(), d_x, d_out, scale)
        torch.cuda.synchronize()
        return d_out.cpu().numpy().view(np.complex64).reshape(-1).astype(np.complex128)


def check_bins(got, ref):
    rms = math.sqrt(np.mean(np.abs(ref) ** 2))
    assert np.all(np.isfinite(got.real)) and np.all(np.isfinite(got.imag))
    assert np.max(np.abs(got - ref)) <= R2C_MAX * np.max(np.abs(ref)), np.max(np.abs(got - ref)) / np.max(np.abs(ref))
    l2 = math.sqrt(np.sum(np.abs(got - ref) ** 2) / np.sum(np.abs(ref) ** 2))
    print(f"r2c n={2 * got.size}: max|dX|/rms = {np.max(np.abs(got - ref)) / rms:.2e}, rel L2 = {l2:.2e}")
    assert l2 <= R2C_L2


@pytest.mark.parametrize("n", [1 << 10, 1 << 11, 1 << 12, 1 << 13, 1 << 14])
def test_r2c_whole_spectrum_against_direct_sums(torch, fd, orc, n):
    x = series(n, 100 + n, [(n / 8 + 0.3, 3.0, 5.0)])
    got = run_r2c(torch, fd, x)
    assert got.size == n // 2
    check_bins(got, orc.dft_real(x))                          # every bin, O(n^2) direct sums (eq. 5)
    assert got[0].imag == 0.0                                  # DC is real; the Nyquist bin is dropped (R17)


@pytest.mark.parametrize("n", [1 << 17, 1 << 20, 1 << 21, 1 << 23, 1 << 24, 1 << 25])
def test_r2c_full_size_sampled_bins_and_properties(torch, fd, orc, n):
    """The paper's series lengths (2^20..2^24) and the largest supported one (2^25): sampled bins against direct sums, numpy's fp64 rfft
    over the whole output as a third opinion, Parseval."""
    x = series(n, 7 + n % 1000, [(0.1 * n + 0.5, 10.0, 4.0)])
    got = run_r2c(torch, fd, x)
    rng = np.random.default_rng(n % 97)
    m1 = 1 << ((int(math.log2(n)) - 1) // 2)                   # sample around the four-step seams as well
    bins = np.unique(np.concatenate([rng.integers(0, n // 2, 40), [0, 1, 2, m1 - 1, m1, m1 + 1, n // 4 - 1, n // 4,
                                                                    n // 4 + 1, n // 2 - 2, n // 2 - 1]]))
    ref = orc.dft_real_at(x, bins)
    full = np.fft.rfft(x.astype(np.float64))[: n // 2]
    assert np.max(np.abs(got[bins] - ref)) <= R2C_MAX * np.max(np.abs(full))
    assert np.max(np.abs(full[bins] - ref)) <= 1e-9 * np.max(np.abs(full))      # the third opinion agrees with the oracle
    check_bins(got, full)
    e_t = float(np.sum(x.astype(np.float64) ** 2))
    nyq = float(np.sum(x[0::2].astype(np.float64)) - np.sum(x[1::2].astype(np.float64)))
    e_f = (abs(got[0]) ** 2 + 2.0 * float(np.sum(np.abs(got[1:]) ** 2)) + nyq ** 2) / n
    assert abs(e_f - e_t) <= 1e-5 * e_t                        # Parseval, with the dropped Nyquist bin put back


def test_r2c_scale_linearity_repeatability_and_errors(torch, fd):
    n = 1 << 16
    x = series(n, 3)
    a = run_r2c(torch, fd, x, 1.0)
    assert np.array_equal(a, run_r2c(torch, fd, x, 1.0))       # bitwise repeatable
    assert np.array_equal(run_r2c(torch, fd, x, 0.5), 0.5 * a)  # power-of-two scale is exact
    assert np.array_equal(run_r2c(torch, fd, (2 * x).astype(np.float32), 1.0), 2.0 * a)
    for bad in (1000, 1 << 9, 1 << 26):
        with pytest.raises(fd.FdasError) as e:
            fd.R2CPlan(bad)
        assert e.value.status == 2                              # FDAS_ERR_UNSUPPORTED
    with fd.R2CPlan(n) as plan:
        d_x = torch.zeros(n + 2, dtype=torch.float32, device="cuda")
        d_out = torch.zeros(n // 2, 2, dtype=torch.float32, device="cuda")
        with pytest.raises(fd.FdasError) as e:
            fd.fdas_r2c_execute(plan.handle, None, d_x.data_ptr() + 4, d_out)
        assert e.value.status == 4                              # FDAS_ERR_ALIGNMENT
        with pytest.raises(fd.FdasError) as e:
            fd.fdas_r2c_execute(plan.handle, None, 0, d_out)
        assert e.value.status == 1


def test_time_series_to_plane_pipeline(torch, fd, orc):
    """Fig. 2 of the paper end to end on the device: real time series -> R2C -> correlations -> plane, one stream, no
    host copy in between.  A drifting tone (r0, z0) in the SERIES peaks at its cell of the plane, and the plane equals
    the oracle's built from the oracle's own direct-sum spectrum (two independent halves meeting)."""
    n, r0, z0, amp = 1 << 15, 3000.0, -8.0, 0.5
    x = series(n, 11, [(r0, z0, amp)])
    nb = n // 2
    with fd.R2CPlan(n) as r2c, fd.Plan(nb, 20.0, 2.0, 1024, 1) as plan:
        plan.make_templates()
        st = torch.cuda.current_stream()
        d_x = torch.from_numpy(x).cuda()
        d_spec = torch.empty((nb, 2), dtype=torch.float32, device="cuda")
        d_plane = torch.full((21, 2 * nb), float("nan"), dtype=torch.float32, device="cuda")
        r2c.execute(st, d_x, d_spec, 1.0 / math.sqrt(n / 2))   # unit-variance samples -> unit mean noise power per bin
        plan.execute(st, d_spec, d_plane)
        torch.cuda.synchronize()
        plane = d_plane.cpu().numpy().astype(np.float64)
    k, c = np.unravel_index(np.argmax(plane), plane.shape)
    assert orc.bank_z(20.0, 2.0)[k] == z0 and c == 2 * int(r0)
    # |X| = (a/2) n at the tone's bin, scaled by 1/sqrt(n/2): power a^2 n / 2 (+ noise)
    assert abs(plane[k, c] - amp ** 2 * n / 2) < 0.1 * amp ** 2 * n / 2
    spec_ref = (orc.dft_real(x) / math.sqrt(n / 2)).astype(np.complex64)
    zs = orc.bank_z(20.0, 2.0)
    for kk in (0, 6, 10, 20):
        ref = orc.plane_row(spec_ref, zs[kk], True)
        assert np.max(np.abs(plane[kk] - ref)) <= 1e-4 * np.max(ref)


# ---------------------------------------------------------------- harmonic summing
def read_cands(torch, d_cands, d_count, cap):
    cnt = int(d_count.item())
    assert cnt <= cap
    rec = d_cands[: cnt * 16].cpu().numpy().copy().view([("col", "<i8"), ("row", "<i4"), ("power", "<f4")])
    return rec[np.lexsort((rec["col"], rec["row"]))]


@pytest.mark.parametrize("nharm", [1, 2, 3, 4, 8, 16])
@pytest.mark.parametrize("interbin", [0, 1])
def test_harmonic_sum_candidates_match_oracle(torch, fd, orc, nharm, interbin):
    from paper_1804_05335_b200 import synthetic as syn
    n, zmax, dz = 60000, 32.0, 2.0
    r0, z0 = 2500.0, 2.0
    chirps = [(h * r0, h * z0, a) for h, a in ((1, 6.0), (2, 5.0), (4, 4.0), (8, 3.5), (16, 3.0))]
    spec = syn.make_spectrum(n, 77, chirps)
    with fd.Plan(n, zmax, dz, 1024, interbin) as plan:
        plan.make_templates()
        K, ncols = plan.info.ntemplates, plan.info.ncols
        st = torch.cuda.current_stream()
        d_spec = torch.from_numpy(spec.view(np.float32).reshape(n, 2)).cuda()
        d_plane = torch.empty((K, ncols), dtype=torch.float32, device="cuda")
        plan.execute(st, d_spec, d_plane)
        cap = 1 << 18
        d_cands = torch.zeros(cap * 16, dtype=torch.uint8, device="cuda")
        d_count = torch.zeros(1, dtype=torch.int64, device="cuda")
        thr = nharm + 4.0 * math.sqrt(nharm) + 4.0            # a few hundred noise cells and the signal
        plan.harmonic_sum_threshold(st, d_plane, nharm, thr, d_cands, cap, d_count)
        torch.cuda.synchronize()
        got = read_cands(torch, d_cands, d_count, cap)
        plane = d_plane.cpu().numpy()
    # exact: the sum of the stored float32 cells in harmonic order, as the kernel forms it
    rows = orc.harmonic_rows(zmax, dz, nharm)
    nhalf = (K - 1) // 2
    nc = (ncols - 1) // nharm + 1
    s32 = np.zeros((rows.size, nc), dtype=np.float32)
    for i, k in enumerate(rows):
        for h in range(1, nharm + 1):
            s32[i] += plane[nhalf + h * (k - nhalf), 0:h * (nc - 1) + 1:h]
    ii, cc = np.nonzero(s32 > np.float32(thr))
    assert got.size == ii.size > 0
    assert np.array_equal(got["row"], rows[ii]) and np.array_equal(got["col"], cc)
    assert np.array_equal(got["power"], s32[ii, cc])
    # against the oracle's fp64 sums of the oracle's own plane
    ref_plane = np.stack([orc.plane_row(spec, z, bool(interbin)) for z in orc.bank_z(zmax, dz)])
    r_o, c_o, v_o = orc.harmonic_candidates(ref_plane, zmax, dz, nharm, thr)
    s64 = orc.harmonic_sum(ref_plane, zmax, dz, nharm)
    assert np.max(np.abs(s32 - s64)) <= 1e-4 * s64.max()
    near = np.abs(s64 - thr) < 1e-3 * thr                      # cells within rounding of the threshold may differ
    want = set(zip(r_o.tolist(), c_o.tolist()))
    have = set(zip(got["row"].tolist(), got["col"].tolist()))
    for (rr, c_) in want ^ have:
        assert near[list(rows).index(rr), c_], (rr, c_)
    # the strongest summed cell is the fundamental's (harmonics up to nharm collected)
    best = got[np.argmax(got["power"])]
    cs = 2 if interbin else 1
    assert orc.bank_z(zmax, dz)[best["row"]] == z0 and best["col"] == cs * int(r0)


def test_harmonic_sum_errors(torch, fd):
    with fd.Plan(4096, 20.0, 2.0, 1024, 0) as plan:
        d_plane = torch.zeros(21, 4096, device="cuda")
        d_cands = torch.zeros(16 * 16, dtype=torch.uint8, device="cuda")
        d_count = torch.zeros(1, dtype=torch.int64, device="cuda")
        for bad in (0, -1):
            with pytest.raises(fd.FdasError) as e:
                plan.harmonic_sum_threshold(None, d_plane, bad, 1.0, d_cands, 16, d_count)
            assert e.value.status == 1
        with pytest.raises(fd.FdasError) as e:
            plan.harmonic_sum_threshold(None, d_plane, 2, float("nan"), d_cands, 16, d_count)
        assert e.value.status == 1
        plan.harmonic_sum_threshold(None, d_plane, 64, -1.0, d_cands, 16, d_count)     # H > nhalf: the z = 0 row only
        torch.cuda.synchronize()
        assert int(d_count.item()) == (4096 - 1) // 64 + 1
        # capacity 0 counts only: the candidate pointer is never written, so its alignment is not checked
        plan.harmonic_sum_threshold(None, d_plane, 1, -1.0, d_cands[8:], 0, d_count)
        torch.cuda.synchronize()
        assert int(d_count.item()) == 21 * 4096
        with pytest.raises(fd.FdasError) as e:
            plan.harmonic_sum_threshold(None, d_plane, 1, -1.0, d_cands[8:], 4, d_count)
        assert e.value.status == 4


@pytest.mark.parametrize("nharm", [1, 2, 5])
def test_harmonic_sum_bank_of_more_than_65535_rows(torch, fd, orc, nharm):
    """A bank finer than any BASELINE config (dz = 0.001: 70 001 rows) is legal for fdas_plan_create; the harmonic
    search must take it (rows used to sit in gridDim.y, which stops at 65 535: ADVICE r2).  Random exponential
    powers stand in for a plane; the sums are compared exactly with float32 sums in the kernel's order and with the
    oracle's fp64 sums."""
    zmax, dz, ncols = 35.0, 0.001, 300
    with fd.Plan(ncols, zmax, dz, 1024, 0) as plan:
        K = plan.info.ntemplates
        assert K == 70001 and plan.info.ncols == ncols
        rng = np.random.Generator(np.random.Philox(4242))
        plane = rng.standard_exponential((K, ncols)).astype(np.float32)
        d_plane = torch.from_numpy(plane).cuda()
        cap = 1 << 20
        d_cands = torch.zeros(cap * 16, dtype=torch.uint8, device="cuda")
        d_count = torch.zeros(1, dtype=torch.int64, device="cuda")
        thr = nharm + 3.0 * math.sqrt(nharm) + 2.0
        plan.harmonic_sum_threshold(torch.cuda.current_stream(), d_plane, nharm, thr, d_cands, cap, d_count)
        torch.cuda.synchronize()
        got = read_cands(torch, d_cands, d_count, cap)
    rows = orc.harmonic_rows(zmax, dz, nharm)
    assert rows.size == 2 * (35000 // nharm) + 1
    nhalf, nc = (K - 1) // 2, (ncols - 1) // nharm + 1
    s32 = np.zeros((rows.size, nc), dtype=np.float32)
    for h in range(1, nharm + 1):
        s32 += plane[nhalf + h * (rows - nhalf)][:, 0:h * (nc - 1) + 1:h]
    ii, cc = np.nonzero(s32 > np.float32(thr))
    assert got.size == ii.size > 1000
    assert np.array_equal(got["row"], rows[ii]) and np.array_equal(got["col"], cc)
    assert np.array_equal(got["power"], s32[ii, cc])
    if nharm == 1:
        assert rows.size > 65535 and got["row"].max() > 65535     # the case gridDim.y could not hold
    s64 = orc.harmonic_sum(plane, zmax, dz, nharm)
    assert np.max(np.abs(s32 - s64)) <= 1e-5 * s64.max()
    r_o, c_o, _ = orc.harmonic_candidates(plane, zmax, dz, nharm, thr)
    near = np.abs(s64 - thr) < 1e-5 * thr
    index_of = {int(r): i for i, r in enumerate(rows)}
    for (rr, c_) in set(zip(r_o.tolist(), c_o.tolist())) ^ set(zip(got["row"].tolist(), got["col"].tolist())):
        assert near[index_of[rr], c_], (rr, c_)


# ---------------------------------------------------------------- harmonic sums for several H in one pass
def read_level(torch, d_cands, d_counts, cap, level):
    cnt = int(d_counts[level].item())
    assert cnt <= cap
    rec = d_cands[level * cap * 16:(level * cap + cnt) * 16].cpu().numpy().copy().view(
        [("col", "<i8"), ("row", "<i4"), ("power", "<f4")])
    return rec[np.lexsort((rec["col"], rec["row"]))]


@pytest.mark.parametrize("levels", [(2, 4, 8, 16), (1, 2, 3), (4,), (2, 32)])
@pytest.mark.parametrize("interbin", [0, 1])
def test_one_pass_harmonic_sums_match_per_h_calls_and_oracle(torch, fd, orc, levels, interbin):
    """fdas_harmonic_sums_threshold: each level's list equals fdas_harmonic_sum_threshold's for that H bit for bit, and
    the sums agree with the oracle's cumulative walk (oracle.harmonic_sums_cumulative) over the same stored plane."""
    from paper_1804_05335_b200 import synthetic as syn
    n, zmax, dz = 9000, 32.0, 2.0
    r0, z0 = 400.0, 2.0
    chirps = [(h * r0, h * z0, a) for h, a in ((1, 6.0), (2, 5.0), (4, 4.0), (8, 3.5), (16, 3.0))]
    spec = syn.make_spectrum(n, 78, chirps)
    with fd.Plan(n, zmax, dz, 1024, interbin) as plan:
        plan.make_templates()
        K, ncols = plan.info.ntemplates, plan.info.ncols
        st = torch.cuda.current_stream()
        d_spec = torch.from_numpy(spec.view(np.float32).reshape(n, 2)).cuda()
        d_plane = torch.empty((K, ncols), dtype=torch.float32, device="cuda")
        plan.execute(st, d_spec, d_plane)
        cap = 1 << 16
        nl = len(levels)
        thr = [h + 3.0 * math.sqrt(h) + 3.0 for h in levels]
        d_cands = torch.zeros(nl * cap * 16, dtype=torch.uint8, device="cuda")
        d_counts = torch.full((nl,), 123, dtype=torch.int64, device="cuda")
        launches0 = fd.fdas_launch_count()
        plan.harmonic_sums_threshold(st, d_plane, levels, thr, d_cands, cap, d_counts)
        assert fd.fdas_launch_count() - launches0 == 1
        torch.cuda.synchronize()
        multi = [read_level(torch, d_cands, d_counts, cap, l) for l in range(nl)]
        d_c1 = torch.zeros(cap * 16, dtype=torch.uint8, device="cuda")
        d_n1 = torch.zeros(1, dtype=torch.int64, device="cuda")
        for l, h in enumerate(levels):
            plan.harmonic_sum_threshold(st, d_plane, h, thr[l], d_c1, cap, d_n1)
            torch.cuda.synchronize()
            single = read_cands(torch, d_c1, d_n1, cap)
            assert multi[l].size == single.size and multi[l].tobytes() == single.tobytes(), (l, h)
        plane = d_plane.cpu().numpy()
    assert multi[0].size > 0
    cum = orc.harmonic_sums_cumulative(plane, zmax, dz, levels)         # fp64 walk over the stored float32 cells
    for l, h in enumerate(levels):
        rows, s64 = cum[h]
        index_of = {int(r): i for i, r in enumerate(rows)}
        got = multi[l]
        ref = np.array([s64[index_of[int(r)], int(c)] for r, c in zip(got["row"], got["col"])])
        assert np.all(np.abs(got["power"] - ref) <= 2e-6 * np.maximum(ref, 1.0))
        ii, cc = np.nonzero(s64 > thr[l])
        near = np.abs(s64 - thr[l]) < 1e-5 * thr[l]
        for (rr, c_) in set(zip(rows[ii].tolist(), cc.tolist())) ^ set(zip(got["row"].tolist(), got["col"].tolist())):
            assert near[index_of[rr], c_], (h, rr, c_)


def test_one_pass_harmonic_sums_config2_full_size(torch, fd, orc):
    """BASELINE config 2 at its stated size (85 x 2^21 plane from fdas_execute): the one-pass search for H = 2, 4, 8, 16
    against (a) float32 sums of the stored plane in the kernel's order, every level, every cell -- exact; (b) the
    oracle's fp64 sums of the ORACLE'S OWN plane rows on sampled fundamentals (z = 6 at H = 2, z = 2 at H = 4, z = 0 at
    H = 8 and 16), as the config-5 parity test samples."""
    from paper_1804_05335_b200 import synthetic as syn
    c = syn.CONFIGS[1]
    n, zmax, dz = c["nbins"], c["zmax"], c["dz"]
    assert (n, c["seglen"]) == (1 << 21, 2048)
    spec, _ = syn.config_spectrum(1, 0)
    levels, thr = (2, 4, 8, 16), [13.0, 18.0, 24.0, 36.0]
    with fd.Plan(n, zmax, dz, c["seglen"], 0) as plan:
        plan.make_templates()
        K, ncols = plan.info.ntemplates, plan.info.ncols
        st = torch.cuda.current_stream()
        d_spec = torch.from_numpy(spec.view(np.float32).reshape(n, 2)).cuda()
        d_plane = torch.empty((K, ncols), dtype=torch.float32, device="cuda")
        plan.execute(st, d_spec, d_plane)
        cap = 1 << 20
        d_cands = torch.zeros(4 * cap * 16, dtype=torch.uint8, device="cuda")
        d_counts = torch.zeros(4, dtype=torch.int64, device="cuda")
        plan.harmonic_sums_threshold(st, d_plane, levels, thr, d_cands, cap, d_counts)
        torch.cuda.synchronize()
        multi = [read_level(torch, d_cands, d_counts, cap, l) for l in range(4)]
        plane = d_plane.cpu().numpy()
    nhalf = (K - 1) // 2
    zs = orc.bank_z(zmax, dz)
    for l, h in enumerate(levels):
        rows = orc.harmonic_rows(zmax, dz, h)
        nc = (ncols - 1) // h + 1
        s32 = np.zeros((rows.size, nc), dtype=np.float32)
        for hh in range(1, h + 1):
            s32 += plane[nhalf + hh * (rows - nhalf)][:, 0:hh * (nc - 1) + 1:hh]
        ii, cc = np.nonzero(s32 > np.float32(thr[l]))
        got = multi[l]
        assert got.size == ii.size > 0, (h, got.size, ii.size)
        assert np.array_equal(got["row"], rows[ii]) and np.array_equal(got["col"], cc)
        assert np.array_equal(got["power"], s32[ii, cc])
        # (b) the oracle's own plane rows for one fundamental per level
        zf = {2: 6.0, 4: 2.0, 8: 0.0, 16: 0.0}[h]
        kf = int(np.nonzero(zs == zf)[0][0])
        s_or = np.zeros(nc)
        for hh in range(1, h + 1):
            s_or += orc.plane_row(spec, hh * zf, False)[0:hh * (nc - 1) + 1:hh]
        i_f = int(np.nonzero(rows == kf)[0][0])
        assert np.max(np.abs(s32[i_f] - s_or)) <= 1e-4 * s_or.max()
        want = set(np.nonzero(s_or > thr[l])[0].tolist())
        have = set(got["col"][got["row"] == kf].tolist())
        for c_ in want ^ have:
            assert abs(s_or[c_] - thr[l]) < 1e-3 * thr[l], (h, c_)
        assert len(want) > 0


def test_one_pass_harmonic_sums_errors(torch, fd):
    with fd.Plan(4096, 20.0, 2.0, 1024, 0) as plan:
        d_plane = torch.zeros(21, 4096, device="cuda")
        d_cands = torch.zeros(4 * 16 * 16, dtype=torch.uint8, device="cuda")
        d_counts = torch.zeros(4, dtype=torch.int64, device="cuda")
        for levels in ((4, 2), (2, 2), (0, 2), (1, 2, 3, 4, 5)):
            with pytest.raises(fd.FdasError) as e:
                plan.harmonic_sums_threshold(None, d_plane, levels, [1.0] * len(levels), d_cands, 16, d_counts)
            assert e.value.status == 1
        with pytest.raises(fd.FdasError) as e:
            plan.harmonic_sums_threshold(None, d_plane, (2, 4), [1.0, float("nan")], d_cands, 16, d_counts)
        assert e.value.status == 1
        plan.harmonic_sums_threshold(None, d_plane, (2, 64), [-1.0, -1.0], d_cands, 0, d_counts)   # count only
        torch.cuda.synchronize()
        assert d_counts[:2].tolist() == [11 * 2048, 64]           # |z| <= 10: 11 rows x 2048 columns; z = 0 x 64 columns
