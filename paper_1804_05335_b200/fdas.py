"""
Thin ctypes binding over libfdas.so (include/fdas.h): same names, argument marshalling only.
Every step of the path runs in the library's CUDA kernels.  PyTorch is used by callers for
device memory and streams; this module accepts raw device pointers (ints) or torch tensors.

There is no CPU fallback: if the CUDA library has not been built, importing this module raises.
"""
from __future__ import annotations

import ctypes
import os

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libfdas.so")

FDAS_OK = 0
STATUS_NAMES = {0: "FDAS_OK", 1: "FDAS_ERR_INVALID_ARG", 2: "FDAS_ERR_UNSUPPORTED", 3: "FDAS_ERR_NOT_READY",
                4: "FDAS_ERR_ALIGNMENT", 5: "FDAS_ERR_CUDA", 6: "FDAS_ERR_NOMEM"}

# every symbol include/fdas.h declares
EXPORTS = ["fdas_plan_create", "fdas_make_templates", "fdas_execute", "fdas_execute_host", "fdas_execute_threshold",
           "fdas_execute_threshold_host",
           "fdas_destroy",
           "fdas_plan_info", "fdas_get_taps", "fdas_get_template_spectrum", "fdas_measure_fp32_peak",
           "fdas_launch_count", "fdas_status_string", "fdas_last_error",
           "fdas_harmonic_sum_threshold", "fdas_r2c_plan_create", "fdas_r2c_execute", "fdas_r2c_destroy",
           "fdas_r2c_execute_static", "fdas_whiten",
           "fdas_harmonic_sums_threshold"]

WHITEN_MEDIAN, WHITEN_MEAN = 0, 1     # fdas_whiten_statistic

R2C_STATIC_MAX_SAMPLES = 1 << 20      # FDAS_R2C_STATIC_MAX_SAMPLES of include/fdas.h


class FdasInfo(ctypes.Structure):
    _fields_ = [("nbins", ctypes.c_int64), ("ncols", ctypes.c_int64), ("row_stride", ctypes.c_int64),
                ("nseg", ctypes.c_int64), ("plane_bytes", ctypes.c_int64),
                ("zmax", ctypes.c_double), ("dz", ctypes.c_double),
                ("ntemplates", ctypes.c_int32), ("seglen", ctypes.c_int32), ("halfwidth", ctypes.c_int32),
                ("overlap", ctypes.c_int32), ("useful", ctypes.c_int32), ("interbin", ctypes.c_int32),
                ("npairs", ctypes.c_int32), ("threads", ctypes.c_int32), ("grid", ctypes.c_int32),
                ("ctas_per_sm", ctypes.c_int32), ("smem_bytes", ctypes.c_int32), ("regs", ctypes.c_int32),
                ("sm_count", ctypes.c_int32), ("reserved", ctypes.c_int32)]

    def as_dict(self):
        return {k: getattr(self, k) for k, _ in self._fields_ if k != "reserved"}


class FdasError(RuntimeError):
    def __init__(self, status: int, where: str, detail: str = ""):
        self.status = status
        super().__init__(f"{where}: {STATUS_NAMES.get(status, status)}" + (f" ({detail})" if detail else ""))


def _load() -> ctypes.CDLL:
    if not os.path.exists(LIB_PATH):
        raise ImportError(
            f"{LIB_PATH} is missing: build it with `python -m paper_1804_05335_b200.build` "
            "(there is no CPU fallback)")
    lib = ctypes.CDLL(LIB_PATH)
    vp, i32, i64, dbl = ctypes.c_void_p, ctypes.c_int32, ctypes.c_int64, ctypes.c_double
    lib.fdas_plan_create.argtypes = [ctypes.POINTER(vp), i64, dbl, dbl, i32, i32]
    lib.fdas_make_templates.argtypes = [vp, vp]
    lib.fdas_execute.argtypes = [vp, vp, vp, vp]
    lib.fdas_execute_host.argtypes = [vp, vp, vp, vp]
    lib.fdas_execute_threshold.argtypes = [vp, vp, vp, ctypes.c_float, vp, i64, vp]
    lib.fdas_execute_threshold_host.argtypes = [vp, vp, vp, ctypes.c_float, vp, i64, vp]
    lib.fdas_destroy.argtypes = [vp]
    lib.fdas_harmonic_sum_threshold.argtypes = [vp, vp, vp, i32, ctypes.c_float, vp, i64, vp]
    lib.fdas_r2c_plan_create.argtypes = [ctypes.POINTER(vp), i64]
    lib.fdas_r2c_execute.argtypes = [vp, vp, vp, vp, ctypes.c_float]
    lib.fdas_r2c_destroy.argtypes = [vp]
    lib.fdas_r2c_execute_static.argtypes = [vp, vp, i64, vp, ctypes.c_float]
    lib.fdas_whiten.argtypes = [vp, vp, vp, i64, i32, i32]
    lib.fdas_harmonic_sums_threshold.argtypes = [vp, vp, vp, i32, ctypes.POINTER(i32), ctypes.POINTER(ctypes.c_float), vp,
                                                 i64, vp]
    lib.fdas_plan_info.argtypes = [vp, ctypes.POINTER(FdasInfo)]
    lib.fdas_get_taps.argtypes = [vp, i32, vp, ctypes.POINTER(i32)]
    lib.fdas_get_template_spectrum.argtypes = [vp, i32, vp]
    lib.fdas_measure_fp32_peak.argtypes = [vp, i32, ctypes.POINTER(dbl)]
    for name in EXPORTS:
        getattr(lib, name).restype = ctypes.c_int
    lib.fdas_launch_count.restype = i64
    lib.fdas_launch_count.argtypes = []
    lib.fdas_status_string.restype = ctypes.c_char_p
    lib.fdas_status_string.argtypes = [ctypes.c_int]
    lib.fdas_last_error.restype = ctypes.c_char_p
    lib.fdas_last_error.argtypes = [vp]
    return lib


lib = _load()


def _ptr(x) -> int:
    """Device/host address of a torch tensor, numpy array, or a plain int."""
    if x is None:
        return 0
    if isinstance(x, int):
        return x
    if hasattr(x, "data_ptr"):
        return int(x.data_ptr())
    if hasattr(x, "ctypes"):
        return int(x.ctypes.data)
    raise TypeError(f"cannot take the address of {type(x)}")


def _stream(stream) -> int:
    if stream is None:
        return 0
    if isinstance(stream, int):
        return stream
    return int(stream.cuda_stream)  # torch.cuda.Stream


# ---- functions with the C names ------------------------------------------------------------
def fdas_plan_create(nbins: int, zmax: float, dz: float, seglen: int, interbin: int) -> int:
    h = ctypes.c_void_p()
    st = lib.fdas_plan_create(ctypes.byref(h), int(nbins), float(zmax), float(dz), int(seglen), int(interbin))
    if st != FDAS_OK:
        raise FdasError(st, "fdas_plan_create")
    return h.value


def _check(st: int, where: str, plan: int | None = None):
    if st != FDAS_OK:
        detail = lib.fdas_last_error(plan).decode() if plan else ""
        raise FdasError(st, where, detail)


def fdas_make_templates(plan: int, stream=None) -> None:
    _check(lib.fdas_make_templates(plan, _stream(stream)), "fdas_make_templates", plan)


def fdas_execute(plan: int, stream, d_spectrum, d_fdot_plane) -> None:
    _check(lib.fdas_execute(plan, _stream(stream), _ptr(d_spectrum), _ptr(d_fdot_plane)), "fdas_execute", plan)


def fdas_execute_host(plan: int, stream, h_spectrum, h_fdot_plane) -> None:
    _check(lib.fdas_execute_host(plan, _stream(stream), _ptr(h_spectrum), _ptr(h_fdot_plane)),
           "fdas_execute_host", plan)


def fdas_execute_threshold(plan: int, stream, d_spectrum, threshold: float, d_cands, capacity: int, d_count) -> None:
    """d_cands: device buffer of `capacity` 16-byte fdas_candidate records {int64 col, int32 row, float power};
    d_count: device uint64 (zeroed by the call)."""
    _check(lib.fdas_execute_threshold(plan, _stream(stream), _ptr(d_spectrum), float(threshold), _ptr(d_cands),
                                      int(capacity), _ptr(d_count)), "fdas_execute_threshold", plan)


def fdas_execute_threshold_host(plan: int, stream, h_spectrum, threshold: float, h_cands, capacity: int, h_count) -> None:
    _check(lib.fdas_execute_threshold_host(plan, _stream(stream), _ptr(h_spectrum), float(threshold), _ptr(h_cands),
                                           int(capacity), _ptr(h_count)), "fdas_execute_threshold_host", plan)


def fdas_harmonic_sum_threshold(plan: int, stream, d_plane, nharm: int, threshold: float, d_cands, capacity: int,
                                d_count) -> None:
    """Cells of the `nharm`-harmonic sum of a stored plane above `threshold` (candidate layout as above; row = bank
    row of the fundamental, col = its column)."""
    _check(lib.fdas_harmonic_sum_threshold(plan, _stream(stream), _ptr(d_plane), int(nharm), float(threshold),
                                           _ptr(d_cands), int(capacity), _ptr(d_count)),
           "fdas_harmonic_sum_threshold", plan)


def fdas_harmonic_sums_threshold(plan: int, stream, d_plane, nharm, thresholds, d_cands, capacity: int, d_counts) -> None:
    n = len(nharm)
    assert len(thresholds) == n
    _check(lib.fdas_harmonic_sums_threshold(plan, _stream(stream), _ptr(d_plane), n, (ctypes.c_int32 * n)(*map(int, nharm)),
                                            (ctypes.c_float * n)(*map(float, thresholds)), _ptr(d_cands), int(capacity),
                                            _ptr(d_counts)), "fdas_harmonic_sums_threshold", plan)


def fdas_r2c_plan_create(nsamples: int) -> int:
    h = ctypes.c_void_p()
    st = lib.fdas_r2c_plan_create(ctypes.byref(h), int(nsamples))
    if st != FDAS_OK:
        raise FdasError(st, "fdas_r2c_plan_create", lib.fdas_last_error(None).decode())
    return h.value


def fdas_r2c_execute(plan: int, stream, d_timeseries, d_spectrum, scale: float = 1.0) -> None:
    st = lib.fdas_r2c_execute(plan, _stream(stream), _ptr(d_timeseries), _ptr(d_spectrum), float(scale))
    if st != FDAS_OK:
        raise FdasError(st, "fdas_r2c_execute", lib.fdas_last_error(None).decode() if st == 5 else "")


def fdas_r2c_destroy(plan: int) -> None:
    _check(lib.fdas_r2c_destroy(plan), "fdas_r2c_destroy")


def fdas_r2c_execute_static(stream, d_timeseries, nsamples: int, d_spectrum, scale: float = 1.0) -> None:
    """The transform of fdas_r2c_execute without a plan and without any device allocation, for callers that may not
    call cudaMalloc (a real-time loop, a host whose memory pool owns the GPU): its scratch is a fixed array inside the
    library, so nsamples <= R2C_STATIC_MAX_SAMPLES, and calls that overlap on the GPU race (include/fdas.h)."""
    st = lib.fdas_r2c_execute_static(_stream(stream), _ptr(d_timeseries), int(nsamples), _ptr(d_spectrum), float(scale))
    if st != FDAS_OK:
        raise FdasError(st, "fdas_r2c_execute_static", lib.fdas_last_error(None).decode() if st in (2, 5) else "")


def fdas_whiten(stream, d_spectrum, d_out, nbins: int, block: int, statistic: int) -> None:
    st = lib.fdas_whiten(_stream(stream), _ptr(d_spectrum), _ptr(d_out), int(nbins), int(block), int(statistic))
    if st != FDAS_OK:
        raise FdasError(st, "fdas_whiten", lib.fdas_last_error(None).decode() if st in (2, 5) else "")


def fdas_destroy(plan: int) -> None:
    _check(lib.fdas_destroy(plan), "fdas_destroy")


def fdas_plan_info(plan: int) -> FdasInfo:
    info = FdasInfo()
    _check(lib.fdas_plan_info(plan, ctypes.byref(info)), "fdas_plan_info", plan)
    return info


def fdas_get_taps(plan: int, k: int):
    """Template k's taps as a complex128 numpy array (index d + m_k) -- for tests."""
    import numpy as np
    info = fdas_plan_info(plan)
    buf = np.zeros(2 * (2 * info.halfwidth + 1), dtype=np.float64)
    mk = ctypes.c_int32()
    _check(lib.fdas_get_taps(plan, int(k), buf.ctypes.data, ctypes.byref(mk)), "fdas_get_taps", plan)
    n = 2 * mk.value + 1
    return buf[:2 * n].view(np.complex128).copy()


def fdas_get_template_spectrum(plan: int, k: int):
    """Template k's spectrum H_k in natural frequency order, complex64 numpy array -- for tests."""
    import numpy as np
    info = fdas_plan_info(plan)
    buf = np.zeros(2 * info.seglen, dtype=np.float32)
    _check(lib.fdas_get_template_spectrum(plan, int(k), buf.ctypes.data), "fdas_get_template_spectrum", plan)
    return buf.view(np.complex64).copy()


def fdas_measure_fp32_peak(stream=None, iters: int = 4096) -> float:
    out = ctypes.c_double()
    _check(lib.fdas_measure_fp32_peak(_stream(stream), int(iters), ctypes.byref(out)), "fdas_measure_fp32_peak")
    return out.value


def fdas_launch_count() -> int:
    return int(lib.fdas_launch_count())


# numpy view of a candidate buffer copied to the host (marshalling only)
CANDIDATE_DTYPE = [("col", "<i8"), ("row", "<i4"), ("power", "<f4")]


# ---- small convenience wrapper (still marshalling only) --------------------------------------
class Plan:
    """RAII wrapper: Plan(nbins, zmax, dz, seglen, interbin).make_templates().execute(stream, spec, plane)."""

    def __init__(self, nbins, zmax, dz, seglen, interbin=0):
        self.handle = fdas_plan_create(nbins, zmax, dz, seglen, interbin)
        self.info = fdas_plan_info(self.handle)

    def make_templates(self, stream=None):
        fdas_make_templates(self.handle, stream)
        return self

    def execute(self, stream, d_spectrum, d_plane):
        fdas_execute(self.handle, stream, d_spectrum, d_plane)

    def execute_threshold(self, stream, d_spectrum, threshold, d_cands, capacity, d_count):
        fdas_execute_threshold(self.handle, stream, d_spectrum, threshold, d_cands, capacity, d_count)

    def execute_threshold_host(self, stream, h_spectrum, threshold, h_cands, capacity, h_count):
        fdas_execute_threshold_host(self.handle, stream, h_spectrum, threshold, h_cands, capacity, h_count)

    def harmonic_sum_threshold(self, stream, d_plane, nharm, threshold, d_cands, capacity, d_count):
        fdas_harmonic_sum_threshold(self.handle, stream, d_plane, nharm, threshold, d_cands, capacity, d_count)

    def harmonic_sums_threshold(self, stream, d_plane, nharm, thresholds, d_cands, capacity, d_counts):
        fdas_harmonic_sums_threshold(self.handle, stream, d_plane, nharm, thresholds, d_cands, capacity, d_counts)

    def execute_host(self, stream, h_spectrum, h_plane):
        fdas_execute_host(self.handle, stream, h_spectrum, h_plane)

    def close(self):
        if self.handle:
            fdas_destroy(self.handle)
            self.handle = None

    def __enter__(self):
        return self

    def __exit__(self, *exc):
        self.close()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


class R2CPlan:
    """RAII wrapper of the real-to-complex transform: R2CPlan(nsamples).execute(stream, d_series, d_spectrum, scale)."""

    def __init__(self, nsamples):
        self.handle = fdas_r2c_plan_create(nsamples)
        self.nsamples = int(nsamples)
        self.nbins = int(nsamples) // 2

    def execute(self, stream, d_timeseries, d_spectrum, scale=1.0):
        fdas_r2c_execute(self.handle, stream, d_timeseries, d_spectrum, scale)

    def close(self):
        if self.handle:
            fdas_r2c_destroy(self.handle)
            self.handle = None

    def __enter__(self):
        return self

    def __exit__(self, *exc):
        self.close()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass
