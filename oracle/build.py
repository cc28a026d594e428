"""Build the oracle's shared library (TEST INFRASTRUCTURE; see z4c_oracle.hpp).

    python oracle/build.py        ->  oracle/liborc_z4c.so

Flags are the paper's reproducibility flags:
-fno-fast-math and -ffp-contract=off. -fopenmp only spreads z-planes over the
host cores for the timed CPU baseline.
"""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
LIB = os.path.join(HERE, "liborc_z4c.so")
SRCS = ["z4c_oracle_capi.cpp"]
DEPS = SRCS + ["z4c_oracle.hpp", "z4c_algebra.hpp", "z4c_grid.hpp", "z4c_amr.hpp", "z4c_boundary.hpp", "z4c_subcycle.hpp"]
FLAGS = ["-O2", "-std=c++17", "-fopenmp", "-ffp-contract=off", "-fno-fast-math",
         "-shared", "-fPIC", "-Wall"]


def build(force: bool = False) -> str:
    newest = max(os.path.getmtime(os.path.join(HERE, d)) for d in DEPS)
    if not force and os.path.exists(LIB) and os.path.getmtime(LIB) >= newest:
        return LIB
    cmd = ["g++", *FLAGS, "-o", LIB, *[os.path.join(HERE, s) for s in SRCS]]
    subprocess.check_call(cmd)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv))
