"""
Second, independent GPU cross-check (-m gpu): the fused kernel's plane against
the paper's variant A restated with library FFTs in bench.py (`CufftUnfused`: segment
copy, torch.fft forward, broadcast multiply, torch.fft inverse, discard + power / interbin).  This is NOT
the parity gate (that is the fp64 oracle, tests/test_gpu_parity.py): both sides are fp32 here, so the bound
is the sum of two fp32 roundings, and the comparator takes its taps from the plan.  It checks the fused
kernel's overlap-save plumbing (segment offsets, the +-z pairing, discard, interbin neighbours, tails)
against a structurally different implementation on whole planes at sizes the oracle would need minutes for.
"""
import math
import os
import sys

import numpy as np
import pytest

pytestmark = pytest.mark.gpu

sys.path.insert(0, os.path.dirname(os.path.dirname(os.path.abspath(__file__))))


@pytest.mark.parametrize("nbins,zmax,seglen,interbin", [
    (200_003, 20.0, 1024, 0),
    (300_001, 84.0, 2048, 0),
    (300_001, 84.0, 2048, 1),
    (1 << 19, 84.0, 4096, 1),
    (1 << 19, 200.0, 8192, 0),
    (1 << 19, 200.0, 8192, 1),
    (100003, 84.0, 8192, 1),
    (1 << 18, 84.0, 8192, 2),
    (200_003, 20.0, 1024, 2),
    (300_001, 84.0, 2048, 2),
    (1 << 19, 84.0, 4096, 2),
])
def test_fused_matches_unfused_cufft(nbins, zmax, seglen, interbin):
    import torch
    import bench
    from paper_1804_05335_b200 import fdas, synthetic

    assert torch.cuda.is_available()
    dev = torch.device("cuda", 0)
    spec = synthetic.make_spectrum(nbins, 31337 + seglen + interbin, [(0.4 * nbins + 0.3, -zmax * 0.6, 25.0)])
    with fdas.Plan(nbins, zmax, 2.0, seglen, interbin) as plan:
        plan.make_templates()
        K, ncols = plan.info.ntemplates, plan.info.ncols
        d_spec = torch.from_numpy(spec.view(np.float32).reshape(nbins, 2)).to(dev)
        ours = torch.full((K, ncols), float("nan"), dtype=torch.float32, device=dev)
        plan.execute(torch.cuda.current_stream(), d_spec, ours)
        ref = torch.full((K, ncols), float("nan"), dtype=torch.float32, device=dev)
        bench.CufftUnfused(torch, plan, dev).run(d_spec, ref)
        torch.cuda.synchronize()
    assert not torch.isnan(ours).any() and not torch.isnan(ref).any()
    o, r = ours.double(), ref.double()
    rowmax = r.max(dim=1).values
    emax = ((o - r).abs().max(dim=1).values / rowmax).max().item()
    el2 = torch.sqrt(((o - r) ** 2).sum(dim=1) / (r ** 2).sum(dim=1)).max().item()
    # two fp32 pipelines: twice the oracle tolerance of tests/test_gpu_parity.py
    assert emax <= 2e-4 and el2 <= 2e-5, (emax, el2)
