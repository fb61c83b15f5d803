"""bench.py's algorithmic bytes / flops per spectrum (the roofline numerators) against the figures of
SURVEY.md section 8(d)'s table, which were derived independently from the same formulas."""
import os
import sys

import pytest

sys.path.insert(0, os.path.dirname(os.path.dirname(os.path.abspath(__file__))))


@pytest.mark.parametrize("cfg,gbytes,gflops,cells", [
    (2, 0.731, 12.19, 85 * 2 ** 21),
    (3, 5.774, 54.66, 85 * 2 ** 24),
    (4, 6.825, 128.84, 201 * 2 ** 23),
    (5, 92.34 / 64, 837.2 / 64, 85 * 2 ** 22),
])
def test_workload_matches_survey_table(cfg, gbytes, gflops, cells):
    import bench
    w = bench.workload(cfg)
    assert w["cells"] == cells
    assert abs(w["alg_bytes"] / 1e9 - gbytes) < 2e-3 * gbytes + 1e-3
    assert abs(w["alg_flops"] / 1e9 - gflops) < 2e-3 * gflops


def test_interbin_override_changes_only_the_half_bin_mode():
    import bench
    a, b, c = bench.workload(2), bench.workload(2, 1), bench.workload(2, 2)
    assert b["cells"] == 2 * a["cells"] == c["cells"] and b["nbins"] == a["nbins"]
    assert c["alg_flops"] > 1.9 * a["alg_flops"]          # two template banks: twice the inverse transforms
    assert bench.workload(3, 1) == bench.workload(3)


def test_default_workload_is_the_largest_single_gpu_config():
    import bench
    w = bench.workload(5)
    assert w["name"] == "config5_batched" and w["batch"] == 64 and w["interbin"] == 1 and w["seglen"] == 2048


def test_profiled_traffic_is_parsed_from_the_committed_summary(tmp_path, monkeypatch):
    import bench
    prof = tmp_path / "profiles"
    prof.mkdir()
    (prof / "rX_ncu_config7.md").write_text(
        "| metric | unit | launch 1 |\n|---|---|---|\n| dram__bytes_read.sum | Mbyte | 24.5 |\n"
        "| dram__bytes_write.sum | Gbyte | 1.25 |\n| gpu__time_duration.sum | us | 400 |\n")
    monkeypatch.setattr(bench, "ROOT", str(tmp_path))
    monkeypatch.setattr(bench, "PROFILE_ROUND", "rX")
    nbytes, name = bench.profiled_traffic(7)
    assert name == "rX_ncu_config7.md" and abs(nbytes - (24.5e6 + 1.25e9)) < 1.0
    assert bench.profiled_traffic(8) == (None, None)          # no capture: the bench line says null, not a constant


def test_committed_profiles_cover_the_bench_configs():
    import bench
    for c in (2, 3, 4, 5):
        nbytes, name = bench.profiled_traffic(c)
        assert name is not None, f"profiles/{bench.PROFILE_ROUND}_ncu_config{c}.md is missing"
        w = bench.workload(c)
        assert 0.8 * w["alg_bytes"] < nbytes < 1.3 * w["alg_bytes"], (c, nbytes, w["alg_bytes"])


def test_gpus_flag_spawns_one_rank_per_gpu():
    """`python bench.py --gpus 2` without a torchrun environment re-executes under torch.distributed.run with two
    ranks; --plumbing-only keeps the run on CPU (gloo): rendezvous, sharding of the job's spectra, barrier and the
    max / sum reductions, rank 0's JSON line."""
    import json
    import subprocess
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    env = {k: v for k, v in os.environ.items() if k not in ("RANK", "LOCAL_RANK", "WORLD_SIZE", "MASTER_ADDR", "MASTER_PORT")}
    res = subprocess.run([sys.executable, os.path.join(root, "bench.py"), "--gpus", "2", "--plumbing-only"],
                         capture_output=True, text=True, env=env, timeout=300)
    assert res.returncode == 0, res.stderr[-2000:]
    lines = [ln for ln in res.stdout.splitlines() if ln.startswith("{")]
    assert len(lines) == 1                                     # rank 0 alone prints
    out = json.loads(lines[0])
    assert out["n_gpus"] == 2 and out["requested_gpus"] == 2
    assert out["spectra_per_rank"] == 64 and out["spectra_total"] == 128 and out["max_over_ranks"] == 2.0
    assert out["scaling"] == "weak"
