"""FP64 pipe microbenchmark: python -m paper_2607_08743_b200.fp64_peak

Builds csrc/fp64_peak.cu for sm_100a and prints the DFMA / DADD / DMUL instruction rates for a few (warps per SM,
independent chains per thread) points. Needs a GPU to run; the build needs none."""
from __future__ import annotations

import ctypes as C
import os
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
LIB = os.path.join(HERE, "libfp64peak.so")
SRC = os.path.join(HERE, "csrc", "fp64_peak.cu")
NVCC = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")


def build(force: bool = False) -> str:
    if force or not os.path.exists(LIB) or os.path.getmtime(LIB) < os.path.getmtime(SRC):
        subprocess.check_call([NVCC, "-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-shared",
                               "-Xcompiler", "-fPIC", "-cudart", "static", "-o", LIB, SRC])
    return LIB


def main():
    lib = C.CDLL(build())
    lib.fp64_chain_rate.restype = C.c_double
    lib.fp64_chain_rate.argtypes = [C.c_int] * 4
    for op, name in enumerate(("DFMA", "DADD", "DMUL")):
        for warps in (1, 8, 16, 32):
            for ilp in (1, 2, 4):
                r = lib.fp64_chain_rate(op, ilp, warps, 20000)
                print("%s warps/SM=%2d chains/thread=%d : %6.2f Tinst/s" % (name, warps, ilp, r / 1e12))


if __name__ == "__main__":
    main()
