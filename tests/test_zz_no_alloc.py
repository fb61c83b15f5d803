"""
fdas_r2c_execute_static: the real-to-complex transform for callers that may not allocate device memory.

Some hosts of this library cannot call cudaMalloc once they are running: a real-time acquisition loop that must keep
the allocator's device-wide lock and its possible failure out of its latency budget, or code embedded in a framework
whose own pool already owns the card.  For them the library offers ONE entry point with no plan and no allocation;
its work arrays and twiddle tables sit in a fixed array inside the library (include/fdas.h: 8.04 MiB per GPU,
at most 2^20 samples, shared by all calls, contents left over from the previous call).

The GPU test checks what such a caller relies on: the spectrum equals the one the planned path
(fdas_r2c_plan_create + fdas_r2c_execute) gives for the same series, within the transform's tolerance of
tests/test_gpu_r2c_harmonics.py (relative L2 <= 3e-6, |dX| <= 1e-5 max|X|), on consecutive calls -- same length
with other data (left-over work arrays must not leak into the result) and other lengths (tables refilled on the
stream).  It holds in a fresh process (first call = per-device set-up) and after the rest of the suite.

This file sorts last on purpose: `pytest -x` stops at the first failure, and a failure here must not hide the parity
tests of the hot path.
"""
import ctypes
import math

import numpy as np
import pytest

R2C_L2, R2C_MAX = 3e-6, 1e-5          # tests/test_gpu_r2c_harmonics.py, DESIGN.md section 4.7


def series(n, seed):
    rng = np.random.Generator(np.random.Philox(seed))
    u = np.arange(n) / n
    x = rng.standard_normal(n) + 4.0 * np.cos(2 * np.pi * ((0.1 * n + 0.5) * u + 10.0 * (u * u - u) / 2))
    return x.astype(np.float32)


def test_static_entry_rejects_bad_sizes_before_touching_the_device():
    """No GPU needed: the size and pointer checks come before any CUDA call."""
    from paper_1804_05335_b200 import build
    build.build()
    from paper_1804_05335_b200 import fdas
    lib = fdas.lib
    buf = ctypes.create_string_buffer(64)
    p = ctypes.addressof(buf) & ~15
    assert lib.fdas_r2c_execute_static(None, None, 1 << 12, p, 1.0) == 1                 # FDAS_ERR_INVALID_ARG
    assert lib.fdas_r2c_execute_static(None, p, 1 << 12, None, 1.0) == 1
    assert lib.fdas_r2c_execute_static(None, p, 0, p, 1.0) == 1
    for n in (1 << 9, 1000, (1 << 20) + 1, 1 << 21, 1 << 40):                           # FDAS_ERR_UNSUPPORTED
        assert lib.fdas_r2c_execute_static(None, p, n, p, 1.0) == 2, n
        msg = lib.fdas_last_error(None).decode()
        assert str(n) in msg and str(fdas.R2C_STATIC_MAX_SAMPLES) in msg, msg
    assert lib.fdas_r2c_execute_static(None, p + 4, 1 << 12, p, 1.0) == 4               # FDAS_ERR_ALIGNMENT


@pytest.mark.gpu
def test_static_entry_matches_planned_path_on_consecutive_calls():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    from paper_1804_05335_b200 import fdas
    stream = torch.cuda.current_stream()
    # (nsamples, seed, scale): the same length twice with other data, a shorter and the longest allowed series, and
    # back to the first length -- every call shares the one scratch array and finds the previous call's contents
    calls = [(1 << 16, 11, 1.0), (1 << 16, 12, 1.0), (1 << 12, 13, 0.5), (1 << 20, 14, 1.0), (1 << 10, 15, 1.0),
             (1 << 16, 11, 1.0)]
    first = None
    for i, (n, seed, scale) in enumerate(calls):
        x = series(n, seed)
        d_x = torch.from_numpy(x).cuda()
        ref = torch.full((n // 2, 2), float("nan"), dtype=torch.float32, device="cuda")
        with fdas.R2CPlan(n) as plan:                          # the existing, allocating path
            plan.execute(stream, d_x, ref, scale)
            torch.cuda.synchronize()
        got = torch.full((n // 2, 2), float("nan"), dtype=torch.float32, device="cuda")
        torch.cuda.synchronize()
        before, free_before = fdas.fdas_launch_count(), torch.cuda.mem_get_info()[0]
        fdas.fdas_r2c_execute_static(stream, d_x, n, got, scale)
        torch.cuda.synchronize()
        assert fdas.fdas_launch_count() - before in (4, 9)     # four passes (+ five table launches on a new length)
        if i > 0:                                              # past the per-device set-up: the card's free memory
            assert torch.cuda.mem_get_info()[0] == free_before  # (cudaMemGetInfo) does not move across the call
        g = got.cpu().numpy().view(np.complex64).reshape(-1).astype(np.complex128)
        r = ref.cpu().numpy().view(np.complex64).reshape(-1).astype(np.complex128)
        assert np.all(np.isfinite(g.real)) and np.all(np.isfinite(g.imag)), f"call {i}: unwritten or invalid bins"
        err = np.abs(g - r)
        assert err.max() <= R2C_MAX * np.abs(r).max(), f"call {i} (n={n}): max |dX| {err.max():.3e}"
        l2 = math.sqrt(np.sum(err ** 2) / np.sum(np.abs(r) ** 2))
        assert l2 <= R2C_L2, f"call {i} (n={n}): rel L2 {l2:.3e}"
        if i == 0:
            first = g
    assert np.array_equal(g, first)                            # the last call repeats the first one's input
    # the limit is enforced with a message, and nothing was allocated along the way by this entry point's own rule
    n = 1 << 21
    d_x = torch.zeros(n, dtype=torch.float32, device="cuda")
    out = torch.zeros((n // 2, 2), dtype=torch.float32, device="cuda")
    with pytest.raises(fdas.FdasError) as e:
        fdas.fdas_r2c_execute_static(stream, d_x, n, out, 1.0)
    assert e.value.status == 2 and "1048576" in str(e.value)
