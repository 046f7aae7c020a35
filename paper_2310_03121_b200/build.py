"""Builds paper_2310_03121_b200/libaev_b200.so (the C-ABI library of include/aev.h) with
nvcc for sm_100a, in-tree.  nvcc cross-compiles without a GPU."""
from __future__ import annotations

import os
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libaev_b200.so")
SOURCES = ["aev_kernels.cu", "ani_mlp.cu", "ani_mlp_tc.cu", "aev_static.cu"]
HEADERS = ["aev_common.cuh", os.path.join("..", "..", "include", "aev.h")]
NVCC_FLAGS = [
    "-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17",
    "-Xcompiler", "-fPIC", "-shared", "-Xptxas", "-v",
]


def _stale() -> bool:
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    deps = [os.path.join(CSRC, f) for f in SOURCES + HEADERS] + [os.path.abspath(__file__)]
    return any(os.path.getmtime(d) > t for d in deps)


def _nvcc() -> str:
    return os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")


def compiler_present() -> bool:
    import shutil
    return shutil.which(_nvcc()) is not None


def build(force: bool = False, verbose: bool = False) -> str:
    if not force and not _stale():
        return LIB
    nvcc = _nvcc()
    tmp = LIB + ".tmp%d" % os.getpid()
    extra = os.environ.get("AEVB_NVCC_EXTRA", "").split()      # e.g. -DAEVB_TC_TIMING for debug builds
    cmd = [nvcc] + NVCC_FLAGS + extra + ["-o", tmp] + [os.path.join(CSRC, s) for s in SOURCES] + ["-lcudart"]
    res = subprocess.run(cmd, stdout=subprocess.PIPE, stderr=subprocess.STDOUT, text=True)
    if verbose or res.returncode != 0:
        print(res.stdout)
    if res.returncode != 0:
        raise RuntimeError("nvcc failed building libaev_b200.so")
    with open(os.path.join(HERE, "build_ptxas.log"), "w") as fh:
        fh.write(" ".join(cmd) + "\n" + res.stdout)
    os.replace(tmp, LIB)
    return LIB


if __name__ == "__main__":
    print(build(force=True, verbose=True))
