"""Builds oracle/liboracle.so from aev_oracle.c with gcc (plain C99, fp64, OpenMP).

TEST INFRASTRUCTURE ONLY (see aev_oracle.c header).  Compiled -O3 -march=native (BASELINE.md
section 4) ON THE MACHINE THAT RUNS IT: the built library travels from the build container to the GPU
box, whose host CPU may differ, so a sidecar file records the CPU it was built for and a mismatch
triggers a rebuild.
"""
from __future__ import annotations

import os
import subprocess
import zlib

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "aev_oracle.c")
LIB = os.path.join(HERE, "liboracle.so")


def cpu_model() -> str:
    try:
        with open("/proc/cpuinfo") as fh:
            flags, name = "", ""
            for line in fh:
                if line.startswith("model name") and not name:
                    name = line.split(":", 1)[1].strip()
                if line.startswith("flags") and not flags:
                    flags = "%08x" % zlib.crc32(line.split(":", 1)[1].strip().encode())
            return "%s [%s]" % (name, flags)
    except OSError:
        return "unknown"


def build(force: bool = False) -> str:
    tag = LIB + ".host"
    here = cpu_model()
    built_for = open(tag).read() if os.path.exists(tag) else ""
    if (not force and os.path.exists(LIB) and built_for == here
            and os.path.getmtime(LIB) >= os.path.getmtime(SRC)):
        return LIB
    tmp = LIB + ".tmp%d" % os.getpid()
    # -ffp-contract=off: no fused multiply-adds, the arithmetic stays the one written in the source
    cmd = ["gcc", "-std=c99", "-O3", "-march=native", "-ffp-contract=off", "-fopenmp", "-fPIC", "-shared", "-Wall",
           "-Wextra", "-o", tmp, SRC, "-lm"]
    subprocess.run(cmd, check=True)
    os.replace(tmp, LIB)
    with open(tag, "w") as fh:
        fh.write(here)
    return LIB


if __name__ == "__main__":
    print(build(force=True))
