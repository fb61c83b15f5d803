"""Build libfdas.so in-tree with nvcc for sm_100a.  `python -m paper_1804_05335_b200.build [--force] [-v]`."""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(HERE)
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libfdas.so")
SOURCES = [os.path.join(CSRC, "fdas_api.cu")]
DEPS = SOURCES + [os.path.join(CSRC, f) for f in ("fdas_fft.cuh", "fdas_kernel.cuh", "fdas_kernel8k.cuh", "fdas_kernel2.cuh", "fdas_kernel3.cuh", "fdas_r2c.cuh", "fdas_whiten.cuh", "fdas_templates.cuh")] + [
    os.path.join(ROOT, "include", "fdas.h")]


def nvcc_cmd(out=LIB, extra=()):
    return ["nvcc", "-O3", "-std=c++17", "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo",
            "--shared", "-Xcompiler", "-fPIC", "-Xcompiler", "-O2", *extra, "-o", out, *SOURCES]


def build(force: bool = False, verbose: bool = False) -> str:
    if not force and os.path.exists(LIB) and all(os.path.getmtime(LIB) >= os.path.getmtime(d) for d in DEPS):
        return LIB
    cmd = nvcc_cmd(extra=("-Xptxas", "-v") if verbose else ())
    res = subprocess.run(cmd, capture_output=True, text=True)
    if verbose or res.returncode != 0:
        sys.stderr.write(res.stdout + res.stderr)
    if res.returncode != 0:
        raise RuntimeError("nvcc failed: " + " ".join(cmd))
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
