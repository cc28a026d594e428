"""Build libsacra (the CUDA hot path + C ABI) in-tree for sm_100a.

    python -m paper_2607_08743_b200.build [--force] [--verbose]   ->  paper_2607_08743_b200/libsacra.so

nvcc cross-compiles without a GPU. -lineinfo keeps the ncu source page usable. No --use_fast_math
(-fno-fast-math on every platform) and -fmad=false: an FMA appears only where the
sources write fma() explicitly (csrc/z4c_stencil.cuh, z4c_fused.cuh).
"""
from __future__ import annotations

import hashlib
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(HERE)
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libsacra.so")
SRCS = ["sacra.cu"]
NVCC = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-std=c++17", "-lineinfo", "-fmad=false",
         "-shared", "-Xcompiler", "-fPIC", "-cudart", "static"]


def _deps():
    out = [os.path.join(ROOT, "include", "sacra.h"), os.path.abspath(__file__)]
    for f in os.listdir(CSRC):
        if f.endswith((".cu", ".cuh", ".h")):
            out.append(os.path.join(CSRC, f))
    return out


def _digest() -> str:
    h = hashlib.sha256(" ".join(FLAGS).encode())
    for d in sorted(_deps()):
        with open(d, "rb") as fh:
            h.update(fh.read())
    return h.hexdigest()


def build(force: bool = False, verbose: bool = False) -> str:
    """Compile if the sources' digest differs from the one stored beside the library (mtimes do not
    survive the copy to the GPU box; the digest does)."""
    stamp, dig = LIB + ".hash", _digest()
    if not force and os.path.exists(LIB) and os.path.exists(stamp) and open(stamp).read().strip() == dig:
        return LIB
    cmd = [NVCC, *FLAGS, *(["-Xptxas", "-v"] if verbose else []), "-o", LIB,
           *[os.path.join(CSRC, s) for s in SRCS]]
    subprocess.check_call(cmd)
    with open(stamp, "w") as fh:
        fh.write(dig + "\n")
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="--verbose" in sys.argv))
