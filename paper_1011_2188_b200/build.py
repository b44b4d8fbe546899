"""Build paper_1011_2188_b200/libfdc.so (the method) and libfdcpeaks.so (bench.py's roofline microbenchmarks) in-tree
with nvcc for sm_100a (cross-compiles without a GPU)."""
from __future__ import annotations

import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "csrc", "fdc.cu")
HDR = os.path.join(os.path.dirname(HERE), "include", "fdc.h")
LIB = os.path.join(HERE, "libfdc.so")
PEAKS_SRC = os.path.join(HERE, "csrc", "bench_peaks.cu")
PEAKS_LIB = os.path.join(HERE, "libfdcpeaks.so")

NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17",
              # arithmetic contract: no contraction, IEEE div/sqrt, denormals kept
              "-fmad=false", "-prec-div=true", "-prec-sqrt=true", "-ftz=false",
              "-Xcompiler", "-fPIC,-O2,-ffp-contract=off", "-shared"]


def build(force: bool = False, verbose: bool = False) -> str:
    stale = (not os.path.exists(LIB) or os.path.getmtime(LIB) < max(os.path.getmtime(SRC), os.path.getmtime(HDR)))
    if force or stale:
        nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
        tmp = LIB + ".tmp.%d" % os.getpid()
        cmd = [nvcc] + NVCC_FLAGS + (["-Xptxas", "-v"] if verbose else []) + ["-o", tmp, SRC]
        subprocess.check_call(cmd)
        os.replace(tmp, LIB)
    if force or not os.path.exists(PEAKS_LIB) or os.path.getmtime(PEAKS_LIB) < os.path.getmtime(PEAKS_SRC):
        nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
        tmp = PEAKS_LIB + ".tmp.%d" % os.getpid()
        subprocess.check_call([nvcc, "-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17",
                               "-Xcompiler", "-fPIC", "-shared", "-o", tmp, PEAKS_SRC])
        os.replace(tmp, PEAKS_LIB)
    return LIB


CHECKED_LIB = os.path.join(HERE, "libfdc_checked.so")


def build_checked() -> str:
    """libfdc_checked.so: the same source with -DFDC_CHECKED (device-side asserts on every material, step-record and tally
    address; csrc/fdc.cu).  Not built by default; run the GPU tests on it with FDC_LIB=<this path>."""
    nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
    tmp = CHECKED_LIB + ".tmp.%d" % os.getpid()
    subprocess.check_call([nvcc] + NVCC_FLAGS + ["-DFDC_CHECKED", "-o", tmp, SRC])
    os.replace(tmp, CHECKED_LIB)
    return CHECKED_LIB


if __name__ == "__main__":
    if "--checked" in sys.argv:
        print(build_checked())
    else:
        print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
