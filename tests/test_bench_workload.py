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
