#!/usr/bin/env python
"""
bench.py -- throughput of the FDAS correlation hot path (BASELINE.json metric: f-fdot plane
cells/s, input bins/s, achieved HBM GB/s vs roofline) on synthetic spectra.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config 5] [--impl ours|reference]

A "step" is one pass of the whole hot path (segment fetch, forward FFT, multiply by every
template, inverse FFT, discard, power(/interbin), plane store) over one BATCH of the workload:
`batch` fdas_execute calls back to back on one CUDA stream (config 5, the default and the largest
single-GPU workload of BASELINE.json: 64 spectra per step; configs 2-4: one spectrum).  The same
JSON line carries a "configs" record with the kernel time and both roofline fractions of the
other full-size configs (2, 3, 4), so one run covers every workload BASELINE.json names.
N > 1: one process per GPU -- launched by torchrun, or by this script itself when WORLD_SIZE is
unset (`python bench.py --gpus N` re-executes under torch.distributed.run) -- the 64*N spectra of
the job are sharded across ranks with dist.shard, no data-path collective (weak scaling).
Prints ONE JSON line on rank 0.
"""
from __future__ import annotations

import argparse
import json
import math
import os
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

METRIC = "f-fdot plane cells/sec"
UNIT = "cells/s"


def load_peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        with open(path) as f:
            p = json.load(f)
        return {"hbm_gbs": float(p["hbm_gbs"]), "source": "measured (MEASURED_PEAKS.json)"}
    return {"hbm_gbs": 6650.0, "source": "fallback (B200_PROFILING.md)"}


# DRAM bytes (read + write) per launch of the fused kernel come from the committed `ncu --set full` summaries
# (dram__bytes_read.sum + dram__bytes_write.sum, first captured launch); None where no capture of the kernel
# that runs today exists.  The file is named in the JSON line next to the number.
PROFILE_ROUND = "r2"
_UNIT = {"byte": 1.0, "Kbyte": 1e3, "Mbyte": 1e6, "Gbyte": 1e9}


def profiled_traffic(cfg_idx: int):
    """(bytes per launch, file name) parsed from profiles/<round>_ncu_config<k>.md, or (None, None)."""
    name = f"{PROFILE_ROUND}_ncu_config{cfg_idx}.md"
    path = os.path.join(ROOT, "profiles", name)
    if not os.path.exists(path):
        return None, None
    total, seen = 0.0, 0
    with open(path) as f:
        for line in f:
            cells = [c.strip() for c in line.split("|")]
            if len(cells) >= 5 and cells[1] in ("dram__bytes_read.sum", "dram__bytes_write.sum") and cells[2] in _UNIT:
                total += float(cells[3]) * _UNIT[cells[2]]
                seen += 1
    return (total, name) if seen == 2 else (None, None)


def workload(cfg_idx: int, interbin=None):
    from paper_1804_05335_b200 import synthetic
    c = dict(synthetic.CONFIGS[cfg_idx - 1])
    if interbin is not None and interbin != c["interbin"]:      # --interbin: same spectra, other half-bin mode
        c["interbin"] = interbin
        c["name"] += f"+interbin{interbin}"
    K = 2 * int(round(c["zmax"] / c["dz"])) + 1
    m = int(math.ceil(c["zmax"] / 2.0)) + 16
    L = c["seglen"]
    N = c["nbins"]
    ncols = N * (2 if c["interbin"] else 1)
    # algorithmic costs per spectrum, SURVEY.md section 8(d) / DESIGN.md "Roofline":
    b_alg = L - 2 * m
    nseg_alg = -(-N // b_alg)
    nb = 2 if c["interbin"] == 2 else 1           # template banks (two-bin Fourier interpolation: 2)
    flops = nseg_alg * ((1 + nb * K) * 5 * L * math.log2(L) + 6 * nb * K * L + 3 * nb * K * b_alg
                        + (5 * K * b_alg if c["interbin"] == 1 else 0))
    nbytes = 8 * N + 8 * nb * K * L + 4 * K * ncols
    c.update(K=K, m=m, ncols=ncols, cells=K * ncols, alg_flops=flops, alg_bytes=nbytes)     # per spectrum
    return c


class ClockSampler:
    """nvidia-smi clocks/throttle reasons sampled DURING the timed region."""
    Q = ("index,clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.active,"
         "clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.index = index
        self.proc = None
        self.lines = []

    def start(self):
        try:
            self.proc = subprocess.Popen(
                ["nvidia-smi", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits", "-lms", "100",
                 "-i", str(self.index)], stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.th = threading.Thread(target=self._read, daemon=True)
            self.th.start()
        except OSError:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.lines.append((time.time(), line.strip()))

    def stop(self, t0=None, t1=None):
        if not self.proc:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except Exception:
            self.proc.kill()
        sm, smax, reasons, power = [], [], set(), []
        for ts, line in self.lines:
            if t0 is not None and not (t0 - 0.05 <= ts <= t1 + 0.15):
                continue
            f = [x.strip() for x in line.split(",")]
            if len(f) < 9:
                continue
            try:
                sm.append(float(f[1]))
                smax.append(float(f[2]))
                power.append(float(f[3]))
            except ValueError:
                continue
            for name, val in zip(("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"), f[5:9]):
                if val.lower().startswith("active"):
                    reasons.add(name)
        if not sm:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["no samples"]}
        sm.sort()
        return {"sm_mhz": sm[len(sm) // 2], "sm_max_mhz": max(smax), "reasons": sorted(reasons),
                "samples": len(sm), "power_w_max": max(power)}


def cpu_baseline(w, budget_s=15.0):
    """The oracle as it stands, timed on the host cores on a bounded sample of the same workload."""
    import numpy as np
    from oracle import fdas_oracle as orc
    from paper_1804_05335_b200 import synthetic
    spec = synthetic.noise_only_c64(w["nbins"], w["seed"])
    zs = orc.bank_z(w["zmax"], w["dz"])
    for z in zs:
        orc.taps(z)                           # templates are excluded from the timed region
    orc.plane_row(spec[:4096], zs[0], int(w["interbin"]))     # load the library
    t0 = time.perf_counter()
    cells, nrows = 0, 0
    while time.perf_counter() - t0 < budget_s:        # rows 0, 1, 2, ... (wrapping) until the budget is spent
        p = orc.plane_row(spec, zs[nrows % zs.size], int(w["interbin"]))
        cells += p.size
        nrows += 1
    dt = time.perf_counter() - t0
    return {"value": cells / dt, "unit": UNIT, "cores": orc.threads(), "kind": "oracle",
            "sample": f"{nrows} template rows (ascending z, wrapping over the {zs.size}-row bank) x all "
                      f"{w['nbins']} bins of {w['name']}, fp64 direct correlation, {dt:.1f} s"}


class CufftUnfused:
    """
    Same-box comparator: the paper's variant A restated with
    library FFTs -- overlapped segments copied out, cuFFT forward (torch.fft), a broadcast multiply by every
    template spectrum, cuFFT inverse, then discard + power (+ interbin), each step a global-memory round trip.
    Harness-side only: it is what the fused kernel is compared WITH (the paper's headline ratio is
    "custom vs cuFFT"), never part of the product path.  Segmentation (overlap, useful points)
    and the taps come from the plan so both sides compute the same function.
    """

    def __init__(self, torch, plan, dev):
        import numpy as np
        from paper_1804_05335_b200 import fdas
        self.torch = torch
        info = plan.info
        self.N, self.K, self.L = int(info.nbins), int(info.ntemplates), int(info.seglen)
        self.ov, self.B, self.nseg = int(info.overlap), int(info.useful), int(info.nseg)
        self.interbin = int(info.interbin)

        def bank(first):
            g = np.zeros((self.K, self.L), dtype=np.complex128)
            for k in range(self.K):
                h = fdas.fdas_get_taps(plan.handle, first + k)   # h[d + m_k], d = -m_k..m_k
                mk = (h.size - 1) // 2
                d = np.arange(-mk, mk + 1)
                g[k, (-d) % self.L] = np.conj(h)              # correlation as circular convolution
            return torch.from_numpy((np.fft.fft(g, axis=1) / self.L).astype(np.complex64)).to(dev)

        self.H = bank(0)
        self.H2 = bank(self.K) if self.interbin == 2 else None   # two-bin interpolation: taps h_z(d - 1/2)
        self.padded = torch.zeros(self.ov + self.nseg * self.B + self.L, dtype=torch.complex64, device=dev)

    def run(self, d_spec, d_plane):
        torch = self.torch
        N, K, L, ov, B, nseg = self.N, self.K, self.L, self.ov, self.B, self.nseg
        self.padded[ov:ov + N] = torch.view_as_complex(d_spec)                # zero extension both sides (R7)
        segs = self.padded.unfold(0, L, B)[:nseg].contiguous()               # step 1: overlapped segments
        X = torch.fft.fft(segs, dim=1)                                       # step 2: cuFFT forward
        Y = X.unsqueeze(0) * self.H.unsqueeze(1)                             # step 3: K x nseg x L products
        y = torch.fft.ifft(Y, dim=2, norm="forward")                         # step 4: cuFFT inverse (1/L in H)
        del Y
        if self.interbin == 2:                       # odd columns from the half-bin bank, even from the plain one
            y2 = torch.fft.ifft(X.unsqueeze(0) * self.H2.unsqueeze(1), dim=2, norm="forward")
            out = torch.empty((K, nseg * B, 2), dtype=torch.float32, device=d_plane.device)
            for j, yy in enumerate((y, y2)):
                v = torch.view_as_real(yy[:, :, ov:ov + B])
                out[:, :, j] = (v[..., 0] ** 2 + v[..., 1] ** 2).reshape(K, nseg * B)
            d_plane.copy_(out[:, :N].reshape(K, 2 * N))
        elif not self.interbin:                                              # step 5: discard + power
            yv = torch.view_as_real(y[:, :, ov:ov + B])
            P = (yv[..., 0] ** 2 + yv[..., 1] ** 2).reshape(K, nseg * B)
            d_plane.copy_(P[:, :N])
        else:
            yv = y[:, :, ov:ov + B + 1]
            a = torch.view_as_real(yv[:, :, :B])
            dd = torch.view_as_real(yv[:, :, :B] - yv[:, :, 1:])
            out = torch.empty((K, nseg * B, 2), dtype=torch.float32, device=d_plane.device)
            out[:, :, 0] = (a[..., 0] ** 2 + a[..., 1] ** 2).reshape(K, nseg * B)
            out[:, :, 1] = ((math.pi / 4) ** 2 * (dd[..., 0] ** 2 + dd[..., 1] ** 2)).reshape(K, nseg * B)
            d_plane.copy_(out[:, :N].reshape(K, 2 * N))


def time_cufft(torch, plan, dev, d_spec, d_plane, steps=5, warmup=2):
    cmp_ = CufftUnfused(torch, plan, dev)
    for _ in range(warmup):
        cmp_.run(d_spec, d_plane)
    torch.cuda.synchronize()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    for _ in range(steps):
        cmp_.run(d_spec, d_plane)
    e1.record()
    torch.cuda.synchronize()
    return e0.elapsed_time(e1) / steps


def run_reference(args, w):
    """--impl reference: the oracle timed on the host cores (rank 0 only)."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    import numpy as np
    from oracle import fdas_oracle as orc
    from paper_1804_05335_b200 import synthetic
    spec = synthetic.noise_only_c64(w["nbins"], w["seed"])
    zs = orc.bank_z(w["zmax"], w["dz"])
    for z in zs:
        orc.taps(z)
    rows_per_step = 2
    rng = np.random.default_rng(0)

    def step(i):
        cells = 0
        for k in rng.integers(0, zs.size, rows_per_step):
            cells += orc.plane_row(spec, zs[k], int(w["interbin"])).size
        return cells

    for i in range(args.warmup):
        step(i)
    t0 = time.perf_counter()
    cells = sum(step(i) for i in range(args.steps))
    dt = time.perf_counter() - t0
    val = cells / dt
    sample = f"each step = {rows_per_step} random template rows x all {w['nbins']} bins of {w['name']}"
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * dt / args.steps,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": w["name"], "nbins": w["nbins"], "templates": w["K"], "seglen": w["seglen"],
                   "interbin": w["interbin"]},
        "cpu_baseline": {"value": val, "unit": UNIT, "cores": orc.threads(), "kind": "oracle", "sample": sample},
        "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
    }))


# Paper's Table 4: independent time series processed in real time on a P100 with the
# custom-FFT code, sampling interval 64 us.  Rows: n samples -> {K templates: (count without, with interbinning)}.
# Time per series = n * 64e-6 / count; it INCLUDES the long R2C FFT, which is outside this library's path
# (BASELINE.md section 2): context, not a target.
PAPER_TABLE4 = {
    1 << 20: {64: (41427, 33893), 96: (24900, 19775), 128: (18847, 15277), 192: (12436, 9898), 256: (8039, 6620)},
    1 << 21: {64: (41645, 34086), 96: (26801, 21123), 128: (20147, 15568), 192: (12216, 9686), 256: (8338, 6757)},
    1 << 22: {64: (41850, 34322), 96: (27614, 21756), 128: (20455, 16079), 192: (12629, 10043), 256: (8477, 6867)},
    1 << 23: {64: (42099, 34196), 96: (27826, 21744), 128: (20627, 16199), 192: (12807, 10157), 256: (8600, 6954)},
}


def run_table4():
    """Table-4-shaped sweep (context): per-series time of fdas_execute for spectra of n/2 bins and K + 1 templates
    (z = -K..+K step 2; the paper's K is even, this bank is odd), both segment lengths 2048 and 4096, best of the two."""
    import numpy as np
    import torch
    from paper_1804_05335_b200 import fdas, synthetic
    torch.cuda.set_device(0)
    dev = torch.device("cuda", 0)
    stream = torch.cuda.Stream(device=dev)
    rows = []
    peaks = load_peaks()
    for n, per_k in PAPER_TABLE4.items():
        N = n // 2
        r2c_ms = time_r2c(torch, fdas, dev, stream, n, peaks, 10)["ms"]      # the long FFT the paper's times include
        spec = torch.from_numpy(synthetic.noise_only_c64(N, 4000 + n % 97).view(np.float32).reshape(N, 2)).to(dev)
        for K, counts in per_k.items():
            for ib in (0, 1):
                best = None
                for seglen in (2048, 4096):
                    with fdas.Plan(N, float(K), 2.0, seglen, ib) as plan:
                        plan.make_templates()
                        out = torch.empty((plan.info.ntemplates, plan.info.ncols), dtype=torch.float32, device=dev)
                        evs = [torch.cuda.Event(enable_timing=True) for _ in range(11)]
                        with torch.cuda.stream(stream):
                            for _ in range(3):
                                plan.execute(stream, spec, out)
                            evs[0].record(stream)
                            for i in range(10):
                                plan.execute(stream, spec, out)
                                evs[i + 1].record(stream)
                        stream.synchronize()
                        ms = sorted(evs[i].elapsed_time(evs[i + 1]) for i in range(10))[5]
                        if best is None or ms < best[0]:
                            best = (ms, seglen)
                        del out
                rows.append({"n_samples": n, "bins": N, "templates": K + 1, "interbin": ib, "seglen": best[1],
                             "ms": round(best[0], 4), "r2c_ms": round(r2c_ms, 4), "ms_incl_r2c": round(best[0] + r2c_ms, 4),
                             "paper_p100_ms_incl_r2c_fft": round(n * 64e-6 / counts[ib] * 1e3, 3)})
    print(json.dumps({"sweep": "paper Table 4 shape (PAPER.md:319, :335-366); ms = fdas_execute alone, ms_incl_r2c adds "
                               "fdas_r2c_execute of the n-sample series, as the paper's times do; other hardware: context, "
                               "not a target", "rows": rows}))


KERNEL_OF_SEGLEN = {1024: "fdas_fused_kernel", 2048: "fdas_fused_kernel3", 4096: "fdas_fused_kernel2 (interbinned: fdas_fused_kernel3)",
                    8192: "fdas_fused_kernel_8k"}


def roofline_record(w, info, kernel_ms, peaks, sm_max_mhz, cfg_idx, overridden, fp32_probe=None):
    """north_star's roofline for ONE launch (one spectrum): the slower of compulsory bytes at HBM bandwidth and
    FFT flops at FP32 peak; `achieved` = algorithmic bytes (flops) per launch / average launch duration."""
    fp32_peak = info.sm_count * 128 * 2 * sm_max_mhz * 1e6 / 1e12
    t_hbm = w["alg_bytes"] / (peaks["hbm_gbs"] * 1e9)
    t_alu = w["alg_flops"] / (fp32_peak * 1e12)
    s = kernel_ms * 1e-3
    ach_gbs, ach_tf = w["alg_bytes"] / s / 1e9, w["alg_flops"] / s / 1e12
    traffic, tfile = (None, None) if overridden else profiled_traffic(cfg_idx)
    hbm = {"bound": "hbm", "achieved": ach_gbs, "peak": peaks["hbm_gbs"], "unit": "GB/s",
           "frac": ach_gbs / peaks["hbm_gbs"], "traffic": traffic, "peak_source": peaks["source"]}
    alu = {"bound": "alu", "achieved": ach_tf, "peak": fp32_peak, "unit": "TFLOP/s", "frac": ach_tf / fp32_peak,
           "traffic": traffic,
           "peak_source": f"{info.sm_count} SMs x 128 FP32 lanes x 2 x {sm_max_mhz:.0f} MHz (DESIGN.md)"}
    if fp32_probe is not None:
        alu["fma_probe_tflops"] = fp32_probe
    roof = dict(alu if t_alu >= t_hbm else hbm)          # north_star: the slower bound is the roofline
    roof.update(kernel=KERNEL_OF_SEGLEN[w["seglen"]], kernel_ms=kernel_ms,
                traffic_source=f"ncu --set full, profiles/{tfile} (dram bytes per launch)" if tfile else None,
                alg_bytes=w["alg_bytes"], alg_flops=w["alg_flops"],
                t_bound_ms={"hbm": t_hbm * 1e3, "alu": t_alu * 1e3},
                hbm=hbm if roof["bound"] == "alu" else None, alu=alu if roof["bound"] == "hbm" else None)
    return roof


def time_config(torch, fdas, synthetic, dev, stream, w, steps, warmup, seed_off=0, nin=4):
    """Kernel time per spectrum (ms) of one config on this rank: `steps` launches between two CUDA events."""
    import numpy as np
    plan = fdas.Plan(w["nbins"], w["zmax"], w["dz"], w["seglen"], w["interbin"])
    plan.make_templates()
    info = plan.info
    N = info.nbins
    d_in = [torch.from_numpy(synthetic.noise_only_c64(N, w["seed"] + seed_off + i).view(np.float32).reshape(N, 2)).to(dev)
            for i in range(nin)]
    nout = 2 if info.plane_bytes * 2 < 20e9 else 1
    d_out = [torch.empty((info.ntemplates, info.ncols), dtype=torch.float32, device=dev) for _ in range(nout)]
    with torch.cuda.stream(stream):
        for i in range(warmup):
            plan.execute(stream, d_in[i % nin], d_out[i % nout])
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record(stream)
        for i in range(steps):
            plan.execute(stream, d_in[i % nin], d_out[i % nout])
        e1.record(stream)
    stream.synchronize()
    ms = e0.elapsed_time(e1) / steps
    rec = info.as_dict()
    plan.close()
    del d_in, d_out
    torch.cuda.empty_cache()
    return ms, rec


def time_r2c(torch, fdas, dev, stream, n, peaks, steps=20):
    """fdas_r2c_execute on n real samples (the long FFT in front of the correlations):
    four launches per call (three transform passes + untangle); HBM-bound, so its roofline is bytes: compulsory
    4n in + 4n out; the three-factor design itself moves 32n."""
    x = torch.randn(n, dtype=torch.float32, device=dev)
    out = torch.empty((n // 2, 2), dtype=torch.float32, device=dev)
    with fdas.R2CPlan(n) as plan:
        with torch.cuda.stream(stream):
            for _ in range(3):
                plan.execute(stream, x, out, 1.0)
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record(stream)
            for _ in range(steps):
                plan.execute(stream, x, out, 1.0)
            e1.record(stream)
        stream.synchronize()
    ms = e0.elapsed_time(e1) / steps
    gbs = 8.0 * n / (ms * 1e-3) / 1e9
    return {"nsamples": n, "ms": ms, "samples_per_s": n / (ms * 1e-3), "launches_per_call": 4,
            "alg_bytes": 8 * n, "design_bytes": 32 * n, "achieved_gbs": gbs, "frac_hbm": gbs / peaks["hbm_gbs"],
            "l2": "working set (series + 2 work arrays + spectrum) = %d MB: %s the 126 MB L2 between passes and calls"
                  % (16 * n >> 20, "stays in" if 16 * n < (120 << 20) else "larger than")}


def time_whiten(torch, fdas, dev, stream, n, block, statistic, peaks, steps=20):
    """fdas_whiten on n bins (red-noise removal by a local median filter / per-block normalisation):
    one launch, HBM-bound: 8n bytes read + 8n written.  Inputs rotate over > 126 MB so no call finds its input in L2."""
    nin = max(2, (160 << 20) // (8 * n) + 1)
    xs = torch.randn((nin, n, 2), dtype=torch.float32, device=dev)
    out = torch.empty((n, 2), dtype=torch.float32, device=dev)
    with torch.cuda.stream(stream):
        for i in range(3):
            fdas.fdas_whiten(stream, xs[i % nin], out, n, block, statistic)
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record(stream)
        for i in range(steps):
            fdas.fdas_whiten(stream, xs[i % nin], out, n, block, statistic)
        e1.record(stream)
    stream.synchronize()
    ms = e0.elapsed_time(e1) / steps
    gbs = 16.0 * n / (ms * 1e-3) / 1e9
    return {"nbins": n, "block": block, "statistic": "median" if statistic == 0 else "mean", "ms": ms,
            "bins_per_s": n / (ms * 1e-3), "alg_bytes": 16 * n, "achieved_gbs": gbs, "frac_hbm": gbs / peaks["hbm_gbs"],
            "launches_per_call": 1}


def time_harmonics(torch, fdas, synthetic, dev, stream, w, peaks):
    """fdas_harmonic_sum_threshold over a stored plane of config `w` for H = 2, 4, 8, 16."""
    import numpy as np
    N = w["nbins"]
    with fdas.Plan(N, w["zmax"], w["dz"], w["seglen"], w["interbin"]) as plan:
        plan.make_templates()
        K, ncols = plan.info.ntemplates, plan.info.ncols
        d_spec = torch.from_numpy(synthetic.noise_only_c64(N, 31).view(np.float32).reshape(N, 2)).to(dev)
        d_plane = torch.empty((K, ncols), dtype=torch.float32, device=dev)
        cap = 1 << 20
        d_cands = torch.empty(cap * 16, dtype=torch.uint8, device=dev)
        d_count = torch.zeros(1, dtype=torch.int64, device=dev)
        out = {}
        with torch.cuda.stream(stream):
            plan.execute(stream, d_spec, d_plane)
        for H in (2, 4, 8, 16):
            thr = H + 6.0 * math.sqrt(H) + 6.0
            with torch.cuda.stream(stream):
                for _ in range(2):
                    plan.harmonic_sum_threshold(stream, d_plane, H, thr, d_cands, cap, d_count)
                e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                e0.record(stream)
                for _ in range(10):
                    plan.harmonic_sum_threshold(stream, d_plane, H, thr, d_cands, cap, d_count)
                e1.record(stream)
            stream.synchronize()
            rows = 2 * (((K - 1) // 2) // H) + 1
            nc = (ncols - 1) // H + 1
            ms = e0.elapsed_time(e1) / 10
            out[str(H)] = {"ms": ms, "summed_cells": rows * nc, "cells_read": rows * nc * H,
                           "read_gbs": 4.0 * rows * nc * H / (ms * 1e-3) / 1e9, "threshold": thr,
                           "candidates": int(d_count.item())}
        # the same four searches in ONE pass (fdas_harmonic_sums_threshold): fundamentals read once
        levels = (2, 4, 8, 16)
        thrs = [H + 6.0 * math.sqrt(H) + 6.0 for H in levels]
        d_cands4 = torch.empty(4 * cap * 16, dtype=torch.uint8, device=dev)
        d_counts = torch.zeros(4, dtype=torch.int64, device=dev)
        with torch.cuda.stream(stream):
            for _ in range(2):
                plan.harmonic_sums_threshold(stream, d_plane, levels, thrs, d_cands4, cap, d_counts)
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record(stream)
            for _ in range(10):
                plan.harmonic_sums_threshold(stream, d_plane, levels, thrs, d_cands4, cap, d_counts)
            e1.record(stream)
        stream.synchronize()
        ms1 = e0.elapsed_time(e1) / 10
        cells_read, prev = 0, 0
        for H in levels:
            cells_read += (2 * (((K - 1) // 2) // H) + 1) * ((ncols - 1) // H + 1) * (H - prev)
            prev = H
        one_pass = {"ms": ms1, "levels": list(levels), "cells_read": cells_read,
                    "read_gbs": 4.0 * cells_read / (ms1 * 1e-3) / 1e9, "candidates": d_counts.tolist(),
                    "ms_of_the_four_separate_launches": sum(v["ms"] for v in out.values())}
    return {"workload": w["name"], "what": "S_H[z][r] = sum_h P[h z][h r] of the stored plane + threshold, one launch per H; "
                                             "one_pass: all four H in one launch (fdas_harmonic_sums_threshold)",
            "harmonics": out, "one_pass": one_pass}


def self_launch(args):
    """`python bench.py --gpus N` without a torchrun environment: re-execute under torch.distributed.run, one
    rank per GPU (the driver's own launch line), and pass its exit status on."""
    import socket
    with socket.socket() as sk:
        sk.bind(("127.0.0.1", 0))
        port = sk.getsockname()[1]
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={args.gpus}",
           "--master-addr", "127.0.0.1", "--master-port", str(port), os.path.abspath(__file__)] + sys.argv[1:]
    raise SystemExit(subprocess.call(cmd))


def plumbing_only(args, w):
    """--plumbing-only: everything of the N-rank path that is not GPU work (rendezvous, sharding of the job's spectra,
    barrier, max / sum over ranks, rank 0's JSON line) on the gloo backend: the CPU test of `--gpus N`."""
    from paper_1804_05335_b200 import dist
    rank, local_rank, world = dist.init("gloo")
    lo, hi = dist.shard(w["batch"] * world, rank, world)
    dist.barrier()
    t_max = dist.max_over_ranks(1.0 + rank)
    spectra = dist.sum_over_ranks(hi - lo)
    if rank == 0:
        print(json.dumps({"plumbing_only": True, "n_gpus": world, "requested_gpus": args.gpus,
                          "spectra_per_rank": hi - lo, "spectra_total": int(spectra), "max_over_ranks": t_max,
                          "config": {"workload": w["name"]}, "scaling": "weak"}))
    dist.finalize()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=None, help="timed steps (default 20; config 5: each step is 64 launches)")
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", type=int, default=5,
                    help="BASELINE.json config number 1..5 (default 5: the largest single-GPU workload)")
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--interbin", type=int, default=None, choices=[0, 1, 2],
                    help="override the config's half-bin mode (0 none, 1 interbinning, 2 two-bin Fourier interpolation)")
    ap.add_argument("--e2e-steps", type=int, default=None)
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-cufft", action="store_true",
                    help="skip the same-box unfused cuFFT comparator (variant A of the paper, N = 1 only)")
    ap.add_argument("--no-configs", action="store_true", help="skip the per-config record of configs 2, 3, 4")
    ap.add_argument("--table4", action="store_true",
                    help="sweep the shapes of the paper's Table 4 (n = 2^20..2^23 samples, 65..257 templates) and exit")
    ap.add_argument("--plumbing-only", action="store_true",
                    help="run only the multi-rank plumbing (gloo, no GPU work) and print its JSON line")
    args = ap.parse_args()
    if args.steps is None:
        args.steps = 20
    args.warmup = max(args.warmup, 3) if args.impl == "ours" else args.warmup

    w = workload(args.config, args.interbin)
    if args.gpus > 1 and "WORLD_SIZE" not in os.environ:
        if args.impl == "reference":
            run_reference(args, w)                      # rank 0 alone runs the reference arm
            return
        self_launch(args)
    if args.impl == "reference":
        run_reference(args, w)
        return
    if args.plumbing_only:
        plumbing_only(args, w)
        return

    import numpy as np
    import torch
    from paper_1804_05335_b200 import dist, fdas, synthetic

    if args.table4:
        if not torch.cuda.is_available():
            raise SystemExit("bench.py --table4 needs a CUDA device")
        run_table4()
        return
    rank, local_rank, world = dist.init()
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device (no CPU fallback)")
    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)
    peaks = load_peaks()

    plan = fdas.Plan(w["nbins"], w["zmax"], w["dz"], w["seglen"], w["interbin"])
    plan.make_templates()
    info = plan.info
    K, ncols, N = info.ntemplates, info.ncols, info.nbins
    batch = int(w["batch"])                        # spectra per step per GPU (config 5: 64)

    # inputs: this rank's shard of the job's batch * world spectra (distinct seeds), resident in HBM before
    # timing; at least 8 distinct spectra rotate.  The planes written per step (>= 713 MB, 91 GB for config 5)
    # are far larger than the 126 MB L2; NOUT output planes rotate.
    lo, hi = dist.shard(batch * world, rank, world)
    nin = max(8, hi - lo)
    d_in = []
    for i in range(nin):
        s = synthetic.noise_only_c64(N, w["seed"] + 1000 * (lo + i))
        d_in.append(torch.from_numpy(s.view(np.float32).reshape(N, 2)).to(dev))
    nout = 4 if info.plane_bytes * 4 < 40e9 else 1
    d_out = [torch.empty((K, ncols), dtype=torch.float32, device=dev) for _ in range(nout)]
    stream = torch.cuda.Stream(device=dev)

    def step(i):                                   # one step = `batch` launches on one stream, no host sync
        for b in range(batch):
            plan.execute(stream, d_in[(i * batch + b) % nin], d_out[(i * batch + b) % nout])

    with torch.cuda.stream(stream):
        for i in range(args.warmup):
            step(i)
    stream.synchronize()

    # ---- timed region: device-resident inputs ------------------------------------------------
    sampler = ClockSampler(local_rank)
    if rank == 0:
        sampler.start()
        time.sleep(0.3)
    dist.barrier()
    torch.cuda.synchronize()
    launches0 = fdas.fdas_launch_count()
    t_wall0 = time.time()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    with torch.cuda.stream(stream):
        e0.record(stream)
        for i in range(args.steps):
            step(i)
        e1.record(stream)
    stream.synchronize()
    torch.cuda.synchronize()
    t_wall1 = time.time()
    dist.barrier()
    launches = fdas.fdas_launch_count() - launches0
    clocks = sampler.stop(t_wall0, t_wall1) if rank == 0 else None
    total_ms = e0.elapsed_time(e1)
    total_ms_max = dist.max_over_ranks(total_ms, dev)
    value = world * args.steps * batch * w["cells"] / (total_ms_max * 1e-3)
    kernel_ms = total_ms / (args.steps * batch)    # average launch duration over the timed region (this rank)

    # ---- end to end through the C ABI with HOST buffers (pinned), copies inside the timed region:
    # one step = the whole batch through fdas_execute_host (H2D of each spectrum, kernel, D2H of each plane)
    e2e_steps = args.e2e_steps if args.e2e_steps is not None else (1 if batch > 1 else 3)
    nh = min(batch, 4)
    h_in = [torch.from_numpy(synthetic.noise_only_c64(N, w["seed"] + 77 + i).view(np.float32).reshape(N, 2)).pin_memory()
            for i in range(nh)]
    h_out = torch.empty((K, ncols), dtype=torch.float32).pin_memory()
    plan.execute_host(stream, h_in[0], h_out)          # warm-up (allocates the staging buffers)
    dist.barrier()
    torch.cuda.synchronize()
    e0.record(stream)
    for i in range(e2e_steps):
        for b in range(batch):
            plan.execute_host(stream, h_in[b % nh], h_out)
    e1.record(stream)
    stream.synchronize()
    e2e_ms = dist.max_over_ranks(e0.elapsed_time(e1), dev)
    e2e_value = world * e2e_steps * batch * w["cells"] / (e2e_ms * 1e-3)
    checksum = float(h_out[K // 2, : min(1024, ncols)].sum())

    # ---- threshold-search mode: the same fused kernel with a candidate
    # sink instead of the plane store; reported beside the headline, never instead of it (per spectrum)
    thr_val, thr_cap = 16.0, 1 << 20
    d_cands = torch.empty(thr_cap * 16, dtype=torch.uint8, device=dev)
    d_count = torch.zeros(1, dtype=torch.int64, device=dev)
    h_cands = torch.empty(thr_cap * 16, dtype=torch.uint8).pin_memory()
    h_count = torch.zeros(1, dtype=torch.int64).pin_memory()
    thr_steps = 20
    with torch.cuda.stream(stream):
        for i in range(3):
            plan.execute_threshold(stream, d_in[i % nin], thr_val, d_cands, thr_cap, d_count)
        t0e, t1e = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        t0e.record(stream)
        for i in range(thr_steps):
            plan.execute_threshold(stream, d_in[i % nin], thr_val, d_cands, thr_cap, d_count)
        t1e.record(stream)
    stream.synchronize()
    thr_ms = dist.max_over_ranks(t0e.elapsed_time(t1e), dev) / thr_steps
    plan.execute_threshold_host(stream, h_in[0], thr_val, h_cands, thr_cap, h_count)      # warm-up (staging)
    t0e.record(stream)
    for i in range(3):
        plan.execute_threshold_host(stream, h_in[i % nh], thr_val, h_cands, thr_cap, h_count)
    t1e.record(stream)
    stream.synchronize()
    thr_e2e_ms = dist.max_over_ranks(t0e.elapsed_time(t1e), dev) / 3
    thr_found = int(h_count.item())

    fp32_probe = fdas.fdas_measure_fp32_peak(stream, 4000) if rank == 0 else None

    # ---- same-box comparator: the paper's unfused cuFFT pipeline (harness-side, N = 1 only, one spectrum)
    cufft_ms, cufft_err = None, None
    if world == 1 and not args.no_cufft:
        del h_out
        try:
            cufft_ms = time_cufft(torch, plan, dev, d_in[0], d_out[0])
        except Exception as exc:                      # a comparator failure must not cost the bench line
            cufft_err = f"{type(exc).__name__}: {exc}"[:200]
    plan_rec = info.as_dict()
    plane_bytes = info.plane_bytes
    plan.close()
    del d_in, d_out, d_cands
    torch.cuda.empty_cache()

    # ---- the other full-size configs of BASELINE.json in the same line (rank 0's GPU, one spectrum per launch)
    sm_max_mhz = (clocks or {}).get("sm_max_mhz") or 1965.0
    others = {}
    ALG = {}
    if rank == 0 and not args.no_configs and args.interbin is None:
        for c in (2, 3, 4, 5):
            if c == args.config:
                continue
            wc = workload(c)
            try:
                ms, rec = time_config(torch, fdas, synthetic, dev, stream, wc, 20, 3)
            except Exception as exc:
                others[wc["name"]] = {"unavailable": f"{type(exc).__name__}: {exc}"[:200]}
                continue
            rc = roofline_record(wc, info, ms, peaks, sm_max_mhz, c, False)
            ALG[wc["name"]] = {"alg_bytes": wc["alg_bytes"], "alg_flops": wc["alg_flops"]}
            other = rc["hbm"] or rc["alu"]
            others[wc["name"]] = {
                "kernel_ms_per_spectrum": ms, "value": wc["cells"] / (ms * 1e-3), "unit": UNIT,
                "bins_per_s": wc["nbins"] / (ms * 1e-3), "bound": rc["bound"], "frac": rc["frac"],
                "frac_hbm": rc["frac"] if rc["bound"] == "hbm" else other["frac"],
                "frac_alu": rc["frac"] if rc["bound"] == "alu" else other["frac"],
                "achieved_gbs": wc["alg_bytes"] / (ms * 1e-3) / 1e9, "achieved_tflops": wc["alg_flops"] / (ms * 1e-3) / 1e12,
                "traffic": rc["traffic"], "traffic_source": rc["traffic_source"], "kernel": rc["kernel"],
                "templates": wc["K"], "nbins": wc["nbins"], "seglen": wc["seglen"], "interbin": wc["interbin"],
                "ctas_per_sm": rec["ctas_per_sm"], "regs": rec["regs"]}
    extra = {}
    if rank == 0 and world == 1 and not args.no_configs:
        try:
            extra["r2c"] = {str(n): time_r2c(torch, fdas, dev, stream, n, peaks) for n in (1 << 21, 1 << 23, 1 << 24)}
            extra["whiten"] = [time_whiten(torch, fdas, dev, stream, n, b, st_, peaks)
                               for (n, b, st_) in ((1 << 21, 1024, 0), (1 << 21, 1920, 1), (1 << 23, 1024, 0),
                                                   (1 << 23, 4096, 0), (1 << 23, 7936, 1))]
            extra["harmonic_sum"] = time_harmonics(torch, fdas, synthetic, dev, stream, workload(2), peaks)
        except Exception as exc:                      # the next-row extras must not cost the bench line
            extra["extras_unavailable"] = f"{type(exc).__name__}: {exc}"[:200]
    dist.barrier()

    if rank == 0:
        roof = roofline_record(w, info, kernel_ms, peaks, sm_max_mhz, args.config, args.interbin is not None, fp32_probe)
        out = {
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": total_ms_max / args.steps, "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "f32", "data": "synthetic",
            "config": {"workload": w["name"], "nbins": N, "templates": K, "zmax": w["zmax"], "dz": w["dz"],
                       "seglen": w["seglen"], "interbin": w["interbin"], "spectra_per_step_per_gpu": batch,
                       "launches_per_step": batch,
                       "l2": f"planes written per step = {batch * plane_bytes / 1e6:.0f} MB > 126 MB L2; "
                             f"{nin} distinct input spectra ({nin * 8 * N / 1e6:.0f} MB), {nout} rotating output planes",
                       "grid": plan_rec["grid"], "threads": plan_rec["threads"], "ctas_per_sm": plan_rec["ctas_per_sm"],
                       "regs": plan_rec["regs"], "smem_bytes": plan_rec["smem_bytes"], "overlap": plan_rec["overlap"],
                       "useful": plan_rec["useful"], "nseg": plan_rec["nseg"]},
            "bins_per_s": world * args.steps * batch * N / (total_ms_max * 1e-3),
            "e2e": {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": batch * 8 * N,
                    "d2h_bytes_per_step": batch * plane_bytes, "steps": e2e_steps,
                    "ms_per_step": e2e_ms / e2e_steps, "checksum": checksum},
            "gpu_launches": launches,
            "clocks": clocks,
            "roofline": roof,
        }
        if others:
            out["configs"] = others
            # the driver's record keeps `roofline` whole: every full-size config's bound and fraction go there too
            roof["configs"] = {name: {k: o.get(k) for k in ("bound", "frac", "frac_hbm", "frac_alu", "traffic", "kernel")}
                               | {"kernel_ms": o.get("kernel_ms_per_spectrum"),
                                  "alg_bytes": ALG.get(name, {}).get("alg_bytes"), "alg_flops": ALG.get(name, {}).get("alg_flops")}
                               for name, o in others.items() if "unavailable" not in o}
        out.update(extra)
        out["threshold_search"] = {
            "what": "fdas_execute_threshold: same fused kernel, cells with P > threshold appended to a candidate "
                    "list instead of the plane store (paper's stated next step, PAPER.md:73, :331); per spectrum",
            "threshold": thr_val, "candidates_found": thr_found, "ms_per_spectrum": thr_ms,
            "value": world * w["cells"] / (thr_ms * 1e-3), "unit": "cells searched/s",
            "e2e": {"value": world * w["cells"] / (thr_e2e_ms * 1e-3), "unit": "cells searched/s",
                    "ms_per_spectrum": thr_e2e_ms, "h2d_bytes_per_spectrum": 8 * N,
                    "d2h_bytes_per_spectrum": 8 + 16 * min(thr_found, thr_cap)}}
        if cufft_ms is not None:
            out["cufft_unfused"] = {"ms_per_spectrum": cufft_ms, "value": w["cells"] / (cufft_ms * 1e-3), "unit": UNIT,
                                    "fused_speedup": cufft_ms / kernel_ms,
                                    "what": "paper's variant A on this GPU (PAPER.md:101-119): segment copy, torch.fft "
                                            "(cuFFT) forward, broadcast multiply, cuFFT inverse, discard + power; "
                                            "context for the paper's custom-vs-cuFFT ratio (PAPER.md:237), not a target"}
        elif cufft_err:
            out["cufft_unfused"] = {"unavailable": cufft_err}
        if not args.no_cpu_baseline:
            out["cpu_baseline"] = cpu_baseline(w)
        # ONE compact line; the headline keys come last so that a tail cut off by a log viewer still holds them
        last = ("cpu_baseline", "config", "e2e", "roofline", "clocks", "metric", "value", "unit", "n_gpus", "steps", "warmup",
                "ms_per_step", "higher_is_better", "scaling", "vs_baseline", "dtype", "data", "bins_per_s", "gpu_launches")
        ordered = {k: v for k, v in out.items() if k not in last}
        ordered.update({k: out[k] for k in last if k in out})
        print(json.dumps(ordered, separators=(",", ":")))
    dist.finalize()


if __name__ == "__main__":
    main()
