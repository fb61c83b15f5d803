"""
GPU parity of the fused threshold search (-m gpu): fdas_execute_threshold through the C ABI against the
oracle's `candidates` (reading R15) on the same seeded inputs.

Floating point decides a set here, so (task rules: "compare what is unique and check that the rest is
valid") with tol = 1e-4 * the row's max power (the plane tolerance of tests/test_gpu_parity.py):
  * every oracle cell with P > threshold + tol must be reported,
  * every reported cell must have oracle P > threshold - tol,
  * reported powers match the oracle's within tol,
  * no cell is reported twice (the z = 0 slot computes its row twice in the +-z pairing).
The list order is unspecified: both sides are sorted on (row, col).
"""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu


def run_threshold(torch, fd, spec, zmax, dz, seglen, interbin, thr, capacity):
    n = spec.size
    with fd.Plan(n, zmax, dz, seglen, interbin) as plan:
        plan.make_templates()
        d_spec = torch.from_numpy(spec.view(np.float32).reshape(n, 2)).cuda()
        d_cands = torch.zeros(max(capacity, 1) * 16, dtype=torch.uint8, device="cuda")
        d_count = torch.full((1,), 12345, dtype=torch.int64, device="cuda")     # the call must zero it
        plan.execute_threshold(torch.cuda.current_stream(), d_spec, thr, d_cands, capacity, d_count)
        torch.cuda.synchronize()
        count = int(d_count.item())
        rec = d_cands.cpu().numpy().view(fd.CANDIDATE_DTYPE)[: min(count, capacity)]
        info = plan.info.as_dict()
    order = np.lexsort((rec["col"], rec["row"]))
    return count, rec[order], info


def check_against_oracle(orc, spec, zmax, dz, interbin, thr, rec):
    zs = orc.bank_z(zmax, dz)
    key = rec["row"].astype(np.int64) * (1 << 40) + rec["col"]
    assert np.all(np.diff(key) > 0), "a cell was reported twice"
    for k, z in enumerate(zs):
        ref = orc.plane_row(spec, z, int(interbin))
        tol = 1e-4 * ref.max()
        got = rec[rec["row"] == k]
        assert np.all((got["col"] >= 0) & (got["col"] < ref.size))
        must = np.nonzero(ref > thr + tol)[0]
        assert np.all(np.isin(must, got["col"])), f"row {k}: a cell above threshold + tol is missing"
        assert np.all(ref[got["col"]] > thr - tol), f"row {k}: a reported cell is below threshold - tol"
        assert np.all(np.abs(got["power"].astype(np.float64) - ref[got["col"]]) <= tol), f"row {k}: power"
        assert np.all(got["power"] > np.float32(thr))


@pytest.mark.parametrize("nbins,zmax,seglen,interbin,thr", [
    (1 << 16, 20.0, 1024, 0, 9.0),
    (70001, 20.0, 1024, 1, 9.0),
    (1 << 17, 84.0, 2048, 0, 10.0),
    (99991, 84.0, 2048, 1, 10.0),
    (1 << 17, 84.0, 4096, 0, 10.0),
    (1 << 17, 84.0, 4096, 1, 10.0),
    (1 << 17, 200.0, 8192, 0, 11.0),
    (1 << 16, 84.0, 8192, 1, 10.0),
    (1 << 16, 84.0, 8192, 2, 10.0),
    (1 << 16, 84.0, 2048, 2, 10.0),
    (40009, 84.0, 4096, 2, 10.0),
])
def test_threshold_candidates_match_oracle(nbins, zmax, seglen, interbin, thr):
    import torch
    from oracle import fdas_oracle as orc
    from paper_1804_05335_b200 import fdas as fd, synthetic as syn
    spec = syn.make_spectrum(nbins, 900 + seglen + interbin,
                             [(0.31 * nbins + 0.25, 0.5 * zmax, 12.0), (0.77 * nbins, 0.0, 6.0),
                              (nbins - 3.0, -0.25 * zmax, 9.0)])         # one at z = 0, one at the right edge
    count, rec, info = run_threshold(torch, fd, spec, zmax, 2.0, seglen, interbin, thr, 1 << 20)
    assert count == rec.size and 10 < count < (1 << 20)
    check_against_oracle(orc, spec, zmax, 2.0, interbin, thr, rec)
    # the z = 0 chirp is found in the z = 0 row exactly once per cell
    k0 = info["ntemplates"] // 2
    assert np.any(rec["row"] == k0)


def test_threshold_limits_and_overflow():
    import torch
    from paper_1804_05335_b200 import fdas as fd, synthetic as syn
    n = 50000
    spec = syn.make_spectrum(n, 77)
    # +inf: nothing; count zeroed by the call
    count, rec, info = run_threshold(torch, fd, spec, 20.0, 2.0, 1024, 0, float("inf"), 16)
    assert count == 0 and rec.size == 0
    # below every power: every cell of the plane exactly once (ncols * K), capacity smaller than the count
    cap = 1000
    count, rec, info = run_threshold(torch, fd, spec, 20.0, 2.0, 1024, 1, -1.0, cap)
    assert count == info["ntemplates"] * info["ncols"] and rec.size == cap
    key = rec["row"].astype(np.int64) * (1 << 40) + rec["col"]
    assert np.all(np.diff(key) > 0)
    assert np.all((rec["row"] >= 0) & (rec["row"] < info["ntemplates"]) & (rec["col"] >= 0) & (rec["col"] < info["ncols"]))
    # capacity 0 with a NULL list: count only
    with fd.Plan(n, 20.0, 2.0, 1024, 0) as plan:
        plan.make_templates()
        d_spec = torch.from_numpy(spec.view(np.float32).reshape(n, 2)).cuda()
        d_count = torch.zeros(1, dtype=torch.int64, device="cuda")
        plan.execute_threshold(torch.cuda.current_stream(), d_spec, 8.0, None, 0, d_count)
        torch.cuda.synchronize()
        assert 0 < int(d_count.item()) < 21 * n
        with pytest.raises(fd.FdasError) as ei:
            plan.execute_threshold(None, d_spec, float("nan"), None, 0, d_count)
        assert ei.value.status == 1
        with pytest.raises(fd.FdasError) as ei:
            plan.execute_threshold(None, d_spec, 1.0, None, 4, d_count)
        assert ei.value.status == 1


@pytest.mark.parametrize("cfg", [2, 3, 4])
def test_threshold_full_size_equals_thresholded_plane(cfg):
    """BASELINE.json configs 2-4 at full size, launch configuration of bench.py: the candidate set equals
    the cells of fdas_execute's own plane above the threshold (same arithmetic, so exactly), and a sample
    of candidates is checked cell by cell against the oracle."""
    import torch
    from oracle import fdas_oracle as orc
    from paper_1804_05335_b200 import fdas as fd, synthetic as syn
    c = syn.CONFIGS[cfg - 1]
    spec, chirps = syn.config_spectrum(cfg - 1)
    n, thr = spec.size, 14.0
    with fd.Plan(n, c["zmax"], c["dz"], c["seglen"], c["interbin"]) as plan:
        plan.make_templates()
        K, ncols = plan.info.ntemplates, plan.info.ncols
        d_spec = torch.from_numpy(spec.view(np.float32).reshape(n, 2)).cuda()
        d_plane = torch.empty((K, ncols), dtype=torch.float32, device="cuda")
        st = torch.cuda.current_stream()
        plan.execute(st, d_spec, d_plane)
        cap = 1 << 22
        d_cands = torch.zeros(cap * 16, dtype=torch.uint8, device="cuda")
        d_count = torch.zeros(1, dtype=torch.int64, device="cuda")
        plan.execute_threshold(st, d_spec, thr, d_cands, cap, d_count)
        torch.cuda.synchronize()
        count = int(d_count.item())
        assert 0 < count <= cap
        rec = d_cands.cpu().numpy().view(fd.CANDIDATE_DTYPE)[:count]
        idx = torch.nonzero(d_plane > thr)
        assert idx.shape[0] == count
        flat_ref = np.sort((idx[:, 0] * ncols + idx[:, 1]).cpu().numpy())
        flat_got = np.sort(rec["row"].astype(np.int64) * ncols + rec["col"])
        assert np.array_equal(flat_ref, flat_got)
        pw = d_plane[torch.from_numpy(rec["row"].astype(np.int64)).cuda(), torch.from_numpy(rec["col"]).cuda()]
        assert np.array_equal(pw.cpu().numpy(), rec["power"])
    # sampled candidates against the oracle, one by one
    zs = orc.bank_z(c["zmax"], c["dz"])
    rng = np.random.default_rng(5)
    for i in rng.choice(count, size=min(count, 40), replace=False):
        ref = orc.plane_cells(spec, zs[rec["row"][i]], [rec["col"][i]], bool(c["interbin"]))[0]
        assert abs(rec["power"][i] - ref) <= 1e-4 * ref and ref > thr - 1e-2


def test_threshold_host_end_to_end():
    """fdas_execute_threshold_host (host buffers in, host candidates out) equals the device entry point."""
    import torch
    from paper_1804_05335_b200 import fdas as fd, synthetic as syn
    n, thr, cap = 1 << 17, 10.0, 1 << 16
    spec = syn.make_spectrum(n, 4321, [(0.4 * n, 30.0, 15.0)])
    count_d, rec_d, info = run_threshold(torch, fd, spec, 84.0, 2.0, 2048, 0, thr, cap)
    with fd.Plan(n, 84.0, 2.0, 2048, 0) as plan:
        plan.make_templates()
        h_spec = torch.from_numpy(spec.view(np.float32).reshape(n, 2)).pin_memory()
        h_cands = torch.zeros(cap * 16, dtype=torch.uint8).pin_memory()
        h_count = torch.zeros(1, dtype=torch.int64).pin_memory()
        for capacity in (16, cap):                       # growing capacity re-allocates the staging list
            plan.execute_threshold_host(torch.cuda.current_stream(), h_spec, thr, h_cands, capacity, h_count)
            assert int(h_count.item()) == count_d
        rec = h_cands.numpy().view(fd.CANDIDATE_DTYPE)[:count_d]
        rec = rec[np.lexsort((rec["col"], rec["row"]))]
        assert np.array_equal(rec, rec_d)


def test_execute_host_after_threshold_host_on_the_same_plan():
    """The host entry points share the input staging buffer but allocate their output staging independently:
    a plan whose first host call was the threshold search must still serve fdas_execute_host."""
    import torch
    from oracle import fdas_oracle as orc
    from paper_1804_05335_b200 import fdas as fd, synthetic as syn
    n, cap = 30000, 1 << 12
    spec = syn.make_spectrum(n, 99, [(0.5 * n, 6.0, 12.0)])
    with fd.Plan(n, 20.0, 2.0, 1024, 1) as plan:
        plan.make_templates()
        h_spec = torch.from_numpy(spec.view(np.float32).reshape(n, 2)).pin_memory()
        h_cands = torch.zeros(cap * 16, dtype=torch.uint8).pin_memory()
        h_count = torch.zeros(1, dtype=torch.int64).pin_memory()
        st = torch.cuda.current_stream()
        plan.execute_threshold_host(st, h_spec, 12.0, h_cands, cap, h_count)
        first = int(h_count.item())
        h_plane = torch.full((21, 2 * n), float("nan"), dtype=torch.float32).pin_memory()
        plan.execute_host(st, h_spec, h_plane)                     # used to return FDAS_ERR_INVALID_ARG
        plane = h_plane.numpy().astype(np.float64)
        assert np.all(np.isfinite(plane))
        for k in (0, 10, 13, 20):
            ref = orc.plane_row(spec, orc.bank_z(20.0, 2.0)[k], True)
            assert np.max(np.abs(plane[k] - ref)) <= 1e-4 * np.max(ref)
        plan.execute_threshold_host(st, h_spec, 12.0, h_cands, cap, h_count)
        assert int(h_count.item()) == first == int(np.count_nonzero(h_plane.numpy() > 12.0))
