"""
GPU parity tests (-m gpu): the CUDA path, called through the C ABI, against the fp64 oracle on
the same seeded inputs.  Tolerances are BASELINE.json's (north_star): per row
max|dP| <= 1e-4 * max(row) and relative L2 <= 1e-5.
"""
import ctypes
import math

import numpy as np
import pytest

pytestmark = pytest.mark.gpu

TOL_MAX = 1e-4
TOL_L2 = 1e-5


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


@pytest.fixture(scope="module")
def syn():
    from paper_1804_05335_b200 import synthetic
    return synthetic


def run_gpu(torch, fd, spectrum, zmax, dz, seglen, interbin, prefill=float("nan")):
    """Whole plane through the C ABI; returns (numpy float32 plane, info dict)."""
    n = spectrum.size
    with fd.Plan(n, zmax, dz, seglen, interbin) as plan:
        plan.make_templates()
        info = plan.info.as_dict()
        d_spec = torch.from_numpy(spectrum.view(np.float32).reshape(n, 2)).cuda()
        d_plane = torch.full((info["ntemplates"], info["ncols"]), prefill, dtype=torch.float32, device="cuda")
        stream = torch.cuda.current_stream()
        plan.execute(stream, d_spec, d_plane)
        torch.cuda.synchronize()
        return d_plane.cpu().numpy(), info


def check_rows(orc, spectrum, plane, zmax, dz, interbin, rows=None):
    zs = orc.bank_z(zmax, dz)
    worst_max, worst_l2 = 0.0, 0.0
    for k in (range(zs.size) if rows is None else rows):
        ref = orc.plane_row(spectrum, zs[k], int(interbin))
        got = plane[k].astype(np.float64)
        assert got.shape == ref.shape
        assert np.all(np.isfinite(got)), f"row {k}: unwritten or non-finite cells"
        emax = np.max(np.abs(got - ref)) / np.max(ref)
        el2 = math.sqrt(np.sum((got - ref) ** 2) / np.sum(ref ** 2))
        worst_max, worst_l2 = max(worst_max, emax), max(worst_l2, el2)
        assert emax <= TOL_MAX, f"row {k} (z={zs[k]}): max|dP|/rowmax = {emax:.3e}"
        assert el2 <= TOL_L2, f"row {k} (z={zs[k]}): rel L2 = {el2:.3e}"
    return worst_max, worst_l2


# ------------------------------------------------------------------ templates (a0, a1)
@pytest.mark.parametrize("zmax,dz,seglen", [(20.0, 2.0, 1024), (84.0, 2.0, 2048), (84.0, 2.0, 4096),
                                            (6.0, 0.5, 1024), (200.0, 2.0, 8192)])
def test_taps_match_oracle_quadrature(torch, fd, orc, zmax, dz, seglen):
    with fd.Plan(1 << 14, zmax, dz, seglen, 0) as plan:
        plan.make_templates()
        torch.cuda.synchronize()
        zs = orc.bank_z(zmax, dz)
        assert plan.info.ntemplates == zs.size
        for k, z in enumerate(zs):
            got = fd.fdas_get_taps(plan.handle, k)
            ref = orc.taps(z)
            assert got.size == ref.size == 2 * orc.halfwidth(z) + 1
            assert np.max(np.abs(got - ref)) < 1e-12, (k, z)


@pytest.mark.parametrize("zmax,dz,seglen", [(20.0, 2.0, 1024), (84.0, 2.0, 2048), (84.0, 2.0, 4096),
                                            (200.0, 2.0, 8192), (20.0, 2.0, 8192)])
def test_template_spectra_match_fp64_fft_of_oracle_taps(torch, fd, orc, zmax, dz, seglen):
    with fd.Plan(1 << 14, zmax, dz, seglen, 0) as plan:
        plan.make_templates()
        zs = orc.bank_z(zmax, dz)
        for k in list(range(0, zs.size, 7)) + [zs.size // 2, zs.size - 1]:
            h = orc.taps(zs[k])
            m = (h.size - 1) // 2
            g = np.zeros(seglen, dtype=np.complex128)
            for d in range(-m, m + 1):
                g[(-d) % seglen] = np.conj(h[d + m])          # PAPER.md:77, :87 (Fig. 1)
            ref = np.fft.fft(g) / seglen
            got = fd.fdas_get_template_spectrum(plan.handle, k).astype(np.complex128)
            assert np.max(np.abs(got - ref)) < 1.5e-7 * np.max(np.abs(ref)), k


# ------------------------------------------------------------------ whole-plane parity
def test_config1_full_plane(torch, fd, orc, syn):
    spec, chirps = syn.config_spectrum(0)
    plane, info = run_gpu(torch, fd, spec, 20.0, 2.0, 1024, 0)
    assert plane.shape == (21, 1 << 16)
    check_rows(orc, spec, plane, 20.0, 2.0, 0)
    k, r = np.unravel_index(np.argmax(plane), plane.shape)
    assert k == 14 and r == 20000                       # z = +8, r = round(20000.25)
    # z = 0 row is |A|^2 up to fp32 rounding (P2)
    a = spec.astype(np.complex128)
    assert np.max(np.abs(plane[10] - (a.real ** 2 + a.imag ** 2))) < 2e-5 * np.max(plane[10])


@pytest.mark.parametrize("cfg,nbins", [(1, 1 << 18), (1, 100003), (2, 1 << 17), (4, 1 << 17), (2, 77777),
                                       (3, 1 << 17), (3, 55555)])
def test_reduced_configs_full_plane(torch, fd, orc, syn, cfg, nbins):
    c = syn.CONFIGS[cfg]
    spec, _ = syn.config_spectrum(cfg, 0, nbins)
    plane, info = run_gpu(torch, fd, spec, c["zmax"], c["dz"], c["seglen"], c["interbin"])
    assert plane.shape == (info["ntemplates"], nbins * (2 if c["interbin"] else 1))
    check_rows(orc, spec, plane, c["zmax"], c["dz"], c["interbin"])


def test_config2_full_size_full_plane(torch, fd, orc, syn):
    c = syn.CONFIGS[1]
    spec, chirps = syn.config_spectrum(1)
    plane, info = run_gpu(torch, fd, spec, c["zmax"], c["dz"], c["seglen"], 0)
    wm, wl = check_rows(orc, spec, plane, c["zmax"], c["dz"], 0)
    print(f"config2: worst max-err {wm:.3e}, worst rel-L2 {wl:.3e}")
    zs = orc.bank_z(c["zmax"], c["dz"])
    for (r0, z0, a0) in chirps:                          # P4: each chirp peaks at its cell
        k0 = int(np.argmin(np.abs(zs - z0)))
        lo, hi = int(r0) - 3, int(r0) + 4
        sub = plane[max(0, k0 - 2):k0 + 3, lo:hi]
        assert sub.max() > 0.3 * a0 * a0          # off-grid (r, z): scalloping in both axes
        kk, rr = np.unravel_index(np.argmax(sub), sub.shape)
        assert abs((max(0, k0 - 2) + kk) - k0) <= 1 and abs(lo + rr - r0) <= 1.0


def check_chirps_peak(orc, plane, chirps, zmax, dz, cols_per_bin):
    """P4 at full size: every injected chirp (r0, z0, a0) peaks at its own cell (within one row / one bin)."""
    zs = orc.bank_z(zmax, dz)
    for (r0, z0, a0) in chirps:
        k0 = int(np.argmin(np.abs(zs - z0)))
        klo = max(0, k0 - 2)
        lo, hi = cols_per_bin * (int(r0) - 3), cols_per_bin * (int(r0) + 4)
        sub = plane[klo:k0 + 3, lo:hi]
        assert sub.max() > 0.3 * a0 * a0          # off-grid (r, z): scalloping in both axes
        kk, rr = np.unravel_index(np.argmax(sub), sub.shape)
        assert abs(klo + kk - k0) <= 1 and abs((lo + rr) / cols_per_bin - r0) <= 1.0, (r0, z0, klo + kk, lo + rr)


def test_config3_full_size_full_plane(torch, fd, orc, syn):
    """BASELINE config 3 at its stated size on its own seeded input (2^23 bins, 16 chirps, seglen 4096,
    interbinned): every row of the 85 x 2^24 plane against the oracle, both criteria (eq. 3, eq. 4)."""
    c = syn.CONFIGS[2]
    spec, chirps = syn.config_spectrum(2)
    assert spec.size == 1 << 23 and len(chirps) == 16
    plane, info = run_gpu(torch, fd, spec, c["zmax"], c["dz"], c["seglen"], 1)
    assert plane.shape == (85, 1 << 24) and info["seglen"] == 4096
    wm, wl = check_rows(orc, spec, plane, c["zmax"], c["dz"], 1)
    print(f"config3: worst max-err {wm:.3e}, worst rel-L2 {wl:.3e}")
    check_chirps_peak(orc, plane, chirps, c["zmax"], c["dz"], 2)


def test_config4_full_size_full_plane(torch, fd, orc, syn):
    """BASELINE config 4 at its stated size on its own seeded input (2^23 bins whitened to unit mean power,
    16 chirps with |z| up to 190, 201 templates, seglen 8192 = 2 x 4096 kernel): every row against the oracle."""
    c = syn.CONFIGS[3]
    spec, chirps = syn.config_spectrum(3)
    assert spec.size == 1 << 23 and len(chirps) == 16 and max(abs(z) for _, z, _ in chirps) > 100.0
    plane, info = run_gpu(torch, fd, spec, c["zmax"], c["dz"], c["seglen"], 0)
    assert plane.shape == (201, 1 << 23)
    assert info["seglen"] == 8192 and info["useful"] + 2 * info["overlap"] == 8192
    wm, wl = check_rows(orc, spec, plane, c["zmax"], c["dz"], 0)
    print(f"config4: worst max-err {wm:.3e}, worst rel-L2 {wl:.3e}")
    check_chirps_peak(orc, plane, chirps, c["zmax"], c["dz"], 1)


@pytest.mark.parametrize("nbins", [1, 100, 7935, 7936, 7937, 20001])
def test_seglen_8192_tiny_and_ragged(torch, fd, orc, syn, nbins):
    spec = syn.make_spectrum(nbins, 800 + nbins, [(nbins / 2.0, -30.0, 10.0)] if nbins > 200 else [])
    plane, info = run_gpu(torch, fd, spec, 40.0, 4.0, 8192, 0)
    check_rows(orc, spec, plane, 40.0, 4.0, 0)


@pytest.mark.parametrize("nbins,zmax", [(1 << 17, 200.0), (30011, 40.0), (5, 40.0)])
def test_seglen_8192_interbin(torch, fd, orc, syn, nbins, zmax):
    """Interbinning at seglen 8192: the half-bin cells come from two more sub-units per slot whose input is
    scaled by (pi/4)(1 - exp(2 pi i k / L)) (fdas_kernel8k.cuh) -- same eq. 4, checked against the oracle."""
    chirps = [(0.37 * nbins + 0.5, 0.4 * zmax, 25.0), (nbins - 2.5, -0.8 * zmax, 18.0)] if nbins > 100 else []
    spec = syn.make_spectrum(nbins, 8192 + nbins, chirps)
    plane, info = run_gpu(torch, fd, spec, zmax, 4.0, 8192, 1)
    assert plane.shape == (info["ntemplates"], 2 * nbins) and info["overlap"] >= info["halfwidth"] + 1
    check_rows(orc, spec, plane, zmax, 4.0, 1)


@pytest.mark.parametrize("nbins,zmax,seglen", [(1 << 15, 20.0, 1024), (50021, 84.0, 2048), (1 << 16, 84.0, 4096),
                                               (3, 20.0, 1024), (1921, 84.0, 2048), (1 << 16, 84.0, 8192),
                                               (40003, 200.0, 8192), (7, 40.0, 8192)])
def test_two_bin_fourier_interpolation(torch, fd, orc, syn, nbins, zmax, seglen):
    """interbin = 2 (reading R16): even columns = the plain plane, odd columns = the correlation
    with the templates at half-integer offsets (second template bank); against the oracle's zero-interleaved
    double-resolution correlation.  Chirps sit on half bins, at z = 0 and at the right edge."""
    chirps = ([(int(0.3 * nbins) + 0.5, 0.5 * zmax, 30.0), (int(0.6 * nbins) + 0.5, 0.0, 15.0), (nbins - 1.5, -zmax, 25.0)]
              if nbins > 100 else [])
    spec = syn.make_spectrum(nbins, 222 + seglen, chirps)
    plane, info = run_gpu(torch, fd, spec, zmax, 2.0, seglen, 2)
    assert plane.shape == (info["ntemplates"], 2 * nbins) and info["interbin"] == 2
    check_rows(orc, spec, plane, zmax, 2.0, 2)
    if nbins > 100:
        k = int(np.argmax(plane.max(axis=1)))
        assert plane[k].argmax() % 2 == 1               # the strongest cell is a half-bin cell


def test_two_bin_fourier_interpolation_large_sampled(torch, fd, orc, syn):
    """interbin = 2 at 2^20 bins (several hundred segments, 2 x 43 slots each): sampled cells of every row
    against the oracle's literal zero-interleaved sum (`plane_cells(..., 2)`), plus whole rows at both ends and z = 0."""
    n, zmax = 1 << 20, 84.0
    spec = syn.make_spectrum(n, 2020, [(300000.5, 40.0, 30.0), (700000.0, -77.0, 20.0)])
    plane, info = run_gpu(torch, fd, spec, zmax, 2.0, 2048, 2)
    assert plane.shape == (85, 2 * n)
    check_rows(orc, spec, plane, zmax, 2.0, 2, rows=[0, 42, 84])
    rng = np.random.default_rng(7)
    zs = orc.bank_z(zmax, 2.0)
    for k, z in enumerate(zs):
        cols = np.concatenate([rng.integers(0, 2 * n, 1500), [0, 1, 2 * n - 2, 2 * n - 1]])
        ref = orc.plane_cells(spec, z, cols, 2)
        assert np.max(np.abs(plane[k, cols] - ref)) <= TOL_MAX * np.max(plane[k]), k


def test_half_bin_taps_match_oracle_quadrature(torch, fd, orc):
    """Bank 1 of interbin = 2: Fresnel closed form (and the z = 0 sinc) at half-integer offsets against the
    oracle's quadrature of the same integral."""
    for zmax, dz, seglen in [(20.0, 2.0, 1024), (84.0, 2.0, 2048), (6.0, 0.5, 1024)]:
        with fd.Plan(1 << 14, zmax, dz, seglen, 2) as plan:
            plan.make_templates()
            zs = orc.bank_z(zmax, dz)
            K = zs.size
            for k, z in enumerate(zs):
                got = fd.fdas_get_taps(plan.handle, K + k)              # index d + m_z <-> h_z(d - 1/2)
                ref = orc.taps2(z)[1::2]                                # offsets d - 1/2, d = -m_z+1..m_z
                assert got.size == 2 * orc.halfwidth(z) + 1 and got[0] == 0
                assert np.max(np.abs(got[1:] - ref)) < 1e-12, (k, z)
                assert np.max(np.abs(fd.fdas_get_taps(plan.handle, k) - orc.taps(z))) < 1e-12


def test_config5_batch_on_one_stream(torch, fd, orc, syn):
    c = syn.CONFIGS[4]
    nb = 3
    n = 1 << 17
    specs = [syn.config_spectrum(4, b, n)[0] for b in range(nb)]
    with fd.Plan(n, c["zmax"], c["dz"], c["seglen"], 1) as plan:
        plan.make_templates()
        K, ncols = plan.info.ntemplates, plan.info.ncols
        d_specs = [torch.from_numpy(s.view(np.float32).reshape(n, 2)).cuda() for s in specs]
        d_out = torch.full((nb, K, ncols), float("nan"), dtype=torch.float32, device="cuda")
        st = torch.cuda.Stream()
        with torch.cuda.stream(st):
            for b in range(nb):
                plan.execute(st, d_specs[b], d_out[b])      # no host sync between calls
        st.synchronize()
        out = d_out.cpu().numpy()
    for b in range(nb):
        check_rows(orc, specs[b], out[b], c["zmax"], c["dz"], 1, rows=range(0, 85, 6))


def test_config5_full_size_64_spectra_one_stream(torch, fd, orc, syn):
    """BASELINE config 5 as stated: 64 spectra of 2^21 bins (0-2 chirps each), one shared bank of 85 templates,
    seglen 2048, interbinned, 64 fdas_execute calls back to back on ONE stream with per-spectrum pointers and
    no host synchronisation in between (the launch configuration bench.py times).  91 GB of planes stay on
    the device; four whole planes and sampled cells of every other spectrum go to the oracle."""
    c = syn.CONFIGS[4]
    nb, n = c["batch"], c["nbins"]
    assert (nb, n, c["seglen"], c["interbin"]) == (64, 1 << 21, 2048, 1)
    free, _ = torch.cuda.mem_get_info()
    need = nb * 85 * 2 * n * 4 + nb * n * 8
    # config 5 as BASELINE.json states it is sized for one B200 (180 GB): too little free memory is a failure of the
    # box or of an earlier test that leaked, never a reason to pass without running
    assert free >= need + (2 << 30), f"needs {need / 1e9:.0f} GB of device memory, {free / 1e9:.0f} GB free"
    specs, chirps = [], []
    for b in range(nb):
        s_, ch = syn.config_spectrum(4, b)
        specs.append(s_)
        chirps.append(ch)
    assert {len(ch) for ch in chirps} == {0, 1, 2}
    with fd.Plan(n, c["zmax"], c["dz"], c["seglen"], 1) as plan:
        plan.make_templates()
        K, ncols, B = plan.info.ntemplates, plan.info.ncols, plan.info.useful
        d_specs = torch.stack([torch.from_numpy(s_.view(np.float32).reshape(n, 2)) for s_ in specs]).cuda()
        d_out = torch.full((nb, K, ncols), float("nan"), dtype=torch.float32, device="cuda")
        st = torch.cuda.Stream()
        st.wait_stream(torch.cuda.current_stream())
        launches0 = fd.fdas_launch_count()
        with torch.cuda.stream(st):
            for b in range(nb):
                plan.execute(st, d_specs[b], d_out[b])      # no host sync between calls
        assert fd.fdas_launch_count() - launches0 == nb     # one fused launch per spectrum
        st.synchronize()
    zs = orc.bank_z(c["zmax"], c["dz"])
    rng = np.random.default_rng(64)
    assert 0 < B < 2048 - 2 * 58                            # useful points per segment (plan.info): seams sit at multiples
    seams = 2 * np.array([B - 1, B, B + 1, 500 * B - 1, 500 * B, n - 1]) + np.array([1, 0, 0, 1, 0, 1])
    full = {0, 21, 42, 63}
    for b in range(nb):
        assert bool(torch.isfinite(d_out[b]).all()), f"spectrum {b}: unwritten or non-finite cells"
        if b in full:
            plane = d_out[b].cpu().numpy()
            wm, wl = check_rows(orc, specs[b], plane, c["zmax"], c["dz"], 1)
            print(f"config5 spectrum {b}: worst max-err {wm:.3e}, worst rel-L2 {wl:.3e}")
            check_chirps_peak(orc, plane, chirps[b], c["zmax"], c["dz"], 2)
            del plane
        else:
            rowmax = d_out[b].amax(dim=1).cpu().numpy().astype(np.float64)
            for k in rng.choice(K, 6, replace=False):
                cols = np.unique(np.concatenate([rng.integers(0, ncols, 3000), seams, [0, 1, ncols - 2, ncols - 1]]))
                got = d_out[b, int(k)][torch.from_numpy(cols).cuda()].cpu().numpy().astype(np.float64)
                ref = orc.plane_cells(specs[b], zs[k], cols, True)
                assert np.max(np.abs(got - ref)) <= TOL_MAX * rowmax[k], (b, k)
                # relative L2 over the sample: cells are exponentially distributed, so the sample's energy is a
                # fair estimate of the row's
                assert math.sqrt(np.sum((got - ref) ** 2) / np.sum(ref ** 2)) <= TOL_L2, (b, k)


# ------------------------------------------------------------------ edge cases
@pytest.mark.parametrize("nbins", [1, 31, 960, 961, 1921])
@pytest.mark.parametrize("interbin", [0, 1])
def test_tiny_and_ragged_spectra(torch, fd, orc, syn, nbins, interbin):
    spec = syn.make_spectrum(nbins, 900 + nbins, [(nbins / 2.0, 4.0, 10.0)] if nbins > 40 else [])
    plane, info = run_gpu(torch, fd, spec, 20.0, 2.0, 1024, interbin)
    check_rows(orc, spec, plane, 20.0, 2.0, interbin)


def test_single_template_bank(torch, fd, orc, syn):
    spec = syn.make_spectrum(5000, 71)
    plane, info = run_gpu(torch, fd, spec, 0.0, 2.0, 1024, 0)
    assert plane.shape == (1, 5000)
    check_rows(orc, spec, plane, 0.0, 2.0, 0)


def test_fractional_dz_bank(torch, fd, orc, syn):
    spec = syn.make_spectrum(20000, 72, [(9000.4, 2.5, 15.0)])
    plane, info = run_gpu(torch, fd, spec, 6.0, 0.5, 1024, 0)
    assert plane.shape[0] == 25
    check_rows(orc, spec, plane, 6.0, 0.5, 0)
    k, r = np.unravel_index(np.argmax(plane), plane.shape)
    assert orc.bank_z(6.0, 0.5)[k] == 2.5 and r == 9000


def test_deterministic_and_linear(torch, fd, syn):
    spec = syn.make_spectrum(1 << 16, 73)
    p1, _ = run_gpu(torch, fd, spec, 20.0, 2.0, 1024, 0)
    p2, _ = run_gpu(torch, fd, spec, 20.0, 2.0, 1024, 0)
    assert np.array_equal(p1, p2)
    p4, _ = run_gpu(torch, fd, (2.0 * spec).astype(np.complex64), 20.0, 2.0, 1024, 0)
    assert np.array_equal(p4, 4.0 * p1)                  # power-of-two scaling is exact in fp32


@pytest.mark.parametrize("seglen,interbin", [(1024, 0), (1024, 1), (1024, 2), (2048, 0), (2048, 1), (2048, 2),
                                             (4096, 0), (4096, 1), (4096, 2), (8192, 0), (8192, 1), (8192, 2)])
def test_bitwise_repeatable_all_kernels(torch, fd, syn, seglen, interbin):
    # compute-sanitizer is closed on this pool; a race in the shared-memory exchange pipeline
    # (split-phase mbarriers, per-warp regions, mailbox, tensor-memory parking) would show up as run-to-run
    # differences.  Both sinks: the plane store (MODE 0) and the threshold search (MODE 1).
    spec = syn.make_spectrum(300000, 75, [(150000.3, 6.0, 20.0)])
    ref, _ = run_gpu(torch, fd, spec, 20.0, 2.0, seglen, interbin)
    for _ in range(4):
        again, _ = run_gpu(torch, fd, spec, 20.0, 2.0, seglen, interbin)
        assert np.array_equal(ref, again)
    n = spec.size
    with fd.Plan(n, 20.0, 2.0, seglen, interbin) as plan:
        plan.make_templates()
        d_spec = torch.from_numpy(spec.view(np.float32).reshape(n, 2)).cuda()
        cap = 1 << 16
        d_cands = torch.zeros(cap * 16, dtype=torch.uint8, device="cuda")
        d_count = torch.zeros(1, dtype=torch.int64, device="cuda")
        found = []
        for _ in range(4):
            plan.execute_threshold(torch.cuda.current_stream(), d_spec, 9.0, d_cands, cap, d_count)
            torch.cuda.synchronize()
            cnt = int(d_count.item())
            assert 0 < cnt <= cap
            raw = d_cands[:cnt * 16].cpu().numpy().copy()
            cand = np.sort(raw.view([("col", "<i8"), ("row", "<i4"), ("power", "<f4")]), order=["row", "col"])
            found.append(cand)
        for other in found[1:]:
            assert np.array_equal(found[0], other)          # the same cells with the same powers (any order)
        # ... and they are exactly the cells of the stored plane above the threshold
        rows, cols = np.nonzero(ref > 9.0)
        assert found[0].size == rows.size
        assert np.array_equal(found[0]["row"], rows) and np.array_equal(found[0]["col"], cols)
        assert np.array_equal(found[0]["power"], ref[rows, cols])


def test_segmentation_independence_on_gpu(torch, fd, syn):
    # P10 on the device: the plane does not depend on the segment length
    spec = syn.make_spectrum(50000, 74, [(25000.0, -6.0, 12.0)])
    a, _ = run_gpu(torch, fd, spec, 20.0, 2.0, 1024, 0)
    b, _ = run_gpu(torch, fd, spec, 20.0, 2.0, 4096, 0)
    assert np.max(np.abs(a - b)) < 2e-5 * np.max(a)
    c, _ = run_gpu(torch, fd, spec, 20.0, 2.0, 8192, 0)
    assert np.max(np.abs(a - c)) < 2e-5 * np.max(a)


@pytest.mark.parametrize("interbin", [0, 1, 2])
def test_seglen_8192_matches_its_e1_sync_build(torch, fd, syn, interbin):
    """The 8192 kernel has no `empty` barrier on its two exchange buffers; it relies on program order (ADVICE r2,
    fdas_kernel8k.cuh).  FDAS_DEBUG_E1_SYNC=1 selects a build with a CTA barrier in front of every exchange store.
    Both must give the same bits, run after run: a later reordering that opens a write-after-read race shows here."""
    import os
    nbins = 300007                                             # 38 segments: every CTA walks many sub-units
    spec = syn.make_spectrum(nbins, 31 + interbin, [(nbins / 3 + 0.25, 150.0, 30.0)])
    d_spec = torch.from_numpy(spec.view(np.float32).reshape(nbins, 2)).cuda()
    st = torch.cuda.current_stream()
    planes = {}
    for dbg in ("0", "1"):
        os.environ["FDAS_DEBUG_E1_SYNC"] = dbg
        try:
            with fd.Plan(nbins, 200.0, 2.0, 8192, interbin) as plan:
                plan.make_templates()
                outs = []
                for _ in range(3):
                    d_plane = torch.full((plan.info.ntemplates, plan.info.ncols), float("nan"), dtype=torch.float32,
                                         device="cuda")
                    plan.execute(st, d_spec, d_plane)
                    torch.cuda.synchronize()
                    outs.append(d_plane)
                assert torch.equal(outs[0], outs[1]) and torch.equal(outs[0], outs[2])
                planes[dbg] = outs[0]
        finally:
            os.environ.pop("FDAS_DEBUG_E1_SYNC", None)
    assert bool(torch.isfinite(planes["0"]).all())
    assert torch.equal(planes["0"], planes["1"])


@pytest.mark.parametrize("interbin", [0, 1, 2])
def test_seglen_2048_grid_is_sized_from_computed_residency(torch, fd, interbin):
    """The 2048 kernel is built for three CTAs per SM; the occupancy API cannot confirm that for a tensor-memory
    kernel, so fdas_plan_create works it out from registers, shared memory and tensor-memory columns.
    On a B200 the answer must be 3 -- a later edit that costs registers or shared memory fails here instead of
    silently running a third of the grid as a serial tail."""
    with fd.Plan(1 << 16, 84.0, 2.0, 2048, interbin) as plan:
        I = plan.info
        prop = torch.cuda.get_device_properties(0)
        assert I.sm_count == prop.multi_processor_count
        assert I.ctas_per_sm == 3 and I.grid == 3 * I.sm_count
        assert ((I.regs + 7) // 8 * 8) * I.threads * 3 <= prop.regs_per_multiprocessor
        assert 3 * (I.smem_bytes + 1024) <= prop.shared_memory_per_multiprocessor


def test_error_codes_on_device(torch, fd):
    with fd.Plan(4096, 20.0, 2.0, 1024, 0) as plan:
        spec = torch.zeros(4096, 2, device="cuda")
        out = torch.zeros(21, 4096, device="cuda")
        with pytest.raises(fd.FdasError) as e:
            plan.execute(None, spec, out)
        assert e.value.status == 3                       # NOT_READY
        plan.make_templates()
        with pytest.raises(fd.FdasError) as e:
            fd.fdas_execute(plan.handle, None, spec.data_ptr() + 8, out)
        assert e.value.status == 4                       # ALIGNMENT
        with pytest.raises(fd.FdasError) as e:
            fd.fdas_execute(plan.handle, None, 0, out)
        assert e.value.status == 1
        plan.execute(None, spec, out)
        torch.cuda.synchronize()
        assert float(out.abs().max()) == 0.0


def test_execute_host_end_to_end(torch, fd, orc, syn):
    spec, _ = syn.config_spectrum(0)
    with fd.Plan(spec.size, 20.0, 2.0, 1024, 0) as plan:
        plan.make_templates()
        h_in = torch.from_numpy(spec.view(np.float32).reshape(-1, 2)).pin_memory()
        h_out = torch.empty(21, spec.size, dtype=torch.float32).pin_memory()
        plan.execute_host(torch.cuda.current_stream(), h_in, h_out)
        check_rows(orc, spec, h_out.numpy(), 20.0, 2.0, 0, rows=[0, 10, 14, 20])


def test_fp32_peak_probe(torch, fd):
    tf = fd.fdas_measure_fp32_peak(None, 2000)
    assert 20.0 < tf < 90.0, tf
    assert fd.fdas_launch_count() > 0


def test_two_plans_on_two_streams_share_the_gpu(torch, fd, orc, syn):
    """Two plans of the tensor-memory kernels (seglen 2048: three CTAs per SM, 128 columns each; seglen 8192: 128
    columns) enqueued on two streams at once: tensor-memory allocation and the persistent grids must coexist, and
    both planes must still match the oracle."""
    n = 1 << 18
    spec_a = syn.make_spectrum(n, 501, [(0.3 * n, 10.0, 20.0)])
    spec_b = syn.make_spectrum(n, 502, [(0.6 * n, -30.0, 25.0)])
    with fd.Plan(n, 84.0, 2.0, 2048, 1) as pa, fd.Plan(n, 84.0, 2.0, 8192, 0) as pb:
        pa.make_templates()
        pb.make_templates()
        torch.cuda.synchronize()
        sa, sb = torch.cuda.Stream(), torch.cuda.Stream()
        da = torch.from_numpy(spec_a.view(np.float32).reshape(n, 2)).cuda()
        db = torch.from_numpy(spec_b.view(np.float32).reshape(n, 2)).cuda()
        oa = torch.full((85, 2 * n), float("nan"), dtype=torch.float32, device="cuda")
        ob = torch.full((85, n), float("nan"), dtype=torch.float32, device="cuda")
        torch.cuda.synchronize()
        for _ in range(4):                                  # interleaved launches, no host sync in between
            pa.execute(sa, da, oa)
            pb.execute(sb, db, ob)
        sa.synchronize()
        sb.synchronize()
        check_rows(orc, spec_a, oa.cpu().numpy(), 84.0, 2.0, 1, rows=[0, 30, 47, 84])
        check_rows(orc, spec_b, ob.cpu().numpy(), 84.0, 2.0, 0, rows=[0, 27, 42, 84])


def test_execute_is_capturable_in_a_cuda_graph(torch, fd, orc, syn):
    """fdas_execute / fdas_r2c_execute allocate nothing and never synchronise, so a whole batch (time series -> R2C ->
    plane, several spectra) can be captured once into a CUDA graph and replayed: the replayed planes equal the
    eagerly computed ones bit for bit and match the oracle."""
    nb, n = 4, 1 << 16
    rng = np.random.Generator(np.random.Philox(2024))
    series = [rng.standard_normal(2 * n).astype(np.float32) for _ in range(nb)]
    with fd.R2CPlan(2 * n) as r2c, fd.Plan(n, 20.0, 2.0, 2048, 1) as plan:
        plan.make_templates()
        d_x = torch.stack([torch.from_numpy(s_) for s_ in series]).cuda()
        d_spec = torch.empty((nb, n, 2), dtype=torch.float32, device="cuda")
        d_eager = torch.full((nb, 21, 2 * n), float("nan"), dtype=torch.float32, device="cuda")
        d_graph = torch.full((nb, 21, 2 * n), float("nan"), dtype=torch.float32, device="cuda")
        scale = 1.0 / math.sqrt(n)
        st = torch.cuda.Stream()
        with torch.cuda.stream(st):
            for b in range(nb):
                r2c.execute(st, d_x[b], d_spec[b], scale)
                plan.execute(st, d_spec[b], d_eager[b])
        st.synchronize()
        spec0 = d_spec[0].cpu().numpy().view(np.complex64).reshape(-1).copy()
        d_spec.zero_()
        g = torch.cuda.CUDAGraph()
        with torch.cuda.graph(g, stream=st):
            for b in range(nb):
                r2c.execute(st, d_x[b], d_spec[b], scale)
                plan.execute(st, d_spec[b], d_graph[b])
        assert bool(torch.isnan(d_graph).all())              # capture enqueues nothing
        g.replay()
        torch.cuda.synchronize()
        assert torch.equal(d_eager, d_graph)
        d_graph.fill_(float("nan"))
        g.replay()                                           # a graph can be replayed
        torch.cuda.synchronize()
        assert torch.equal(d_eager, d_graph)
        check_rows(orc, spec0, d_graph[0].cpu().numpy(), 20.0, 2.0, 1, rows=[0, 10, 20])
