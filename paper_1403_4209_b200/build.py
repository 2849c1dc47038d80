"""Builds the C-ABI library libig.so in-tree with nvcc for sm_100a (cross-compiles without a GPU)."""
from __future__ import annotations

import os
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
SOURCES = ["ig_api.cu", "ig_sort.cu", "ig_ingest.cu", "ig_gridder.cu", "ig_gather.cu", "ig_bank.cu", "ig_finalize.cu", "ig_micro.cu", "ig_static.cu"]
LIB = os.path.join(HERE, "libig.so")
CUDA_HOME = os.environ.get("CUDA_HOME", "/usr/local/cuda")


def lib_path() -> str:
    return LIB


def needs_build() -> bool:
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    deps = [os.path.join(CSRC, f) for f in os.listdir(CSRC)] + [os.path.join(HERE, "..", "include", "ig.h")]
    return any(os.path.getmtime(d) > t for d in deps)


def build(force: bool = False, verbose: bool = False) -> str:
    if not force and not needs_build():
        return LIB
    nvcc = os.path.join(CUDA_HOME, "bin", "nvcc")
    cmd = [nvcc, "-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17",
           "-shared", "-Xcompiler", "-fPIC,-ffp-contract=off", "-fmad=true",
           "-o", LIB] + [os.path.join(CSRC, s) for s in SOURCES] + [
           "-L" + os.path.join(CUDA_HOME, "lib64"), "-lcufft",
           "-Xlinker", "-rpath," + os.path.join(CUDA_HOME, "lib64")]
    cmd[1:1] = os.environ.get("IG_NVCC_EXTRA", "").split()   # tuning experiments only (-DIG_RMAX=.. etc.)
    if verbose:
        cmd.insert(1, "-Xptxas=-v")
    subprocess.check_call(cmd)
    return LIB


if __name__ == "__main__":
    import sys
    print(build(force=True, verbose="-v" in sys.argv))
