"""Build the C part of the oracle (test infrastructure) with gcc.  `python -m oracle.build`.

Compiled with -O3 -march=native -fopenmp.  The library name carries a hash of this
machine's CPU flags: the repository travels between machines with different hosts, and a -march=native build
from one must not be loaded on another."""
import hashlib
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "fdas_oracle.c")


def _cpu_tag() -> str:
    flags = ""
    try:
        with open("/proc/cpuinfo") as f:
            for line in f:
                if line.startswith("flags") or line.startswith("model name"):
                    flags += line
                    if line.startswith("flags"):
                        break
    except OSError:
        pass
    return hashlib.sha1(flags.encode()).hexdigest()[:8]


LIB = os.path.join(HERE, f"libfdas_oracle_{_cpu_tag()}.so")


def build(force: bool = False) -> str:
    if (not force and os.path.exists(LIB)
            and os.path.getmtime(LIB) >= os.path.getmtime(SRC)):
        return LIB
    cmd = ["gcc", "-O3", "-march=native", "-fopenmp", "-fPIC", "-shared", "-o", LIB, SRC, "-lm"]
    subprocess.check_call(cmd)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv))
