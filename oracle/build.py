"""Build the CPU oracle (TEST INFRASTRUCTURE ONLY) into oracle/libsnap_oracle.so.

    python oracle/build.py

Plain gcc, -O2, OpenMP over grid points.  No CUDA, no torch, nothing shared
with the product path under paper_2411_19617_b200/.
"""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "snap_oracle.c")
LIB = os.path.join(HERE, "libsnap_oracle.so")


def build(force: bool = False) -> str:
    if (not force) and os.path.exists(LIB) and os.path.getmtime(LIB) >= os.path.getmtime(SRC):
        return LIB
    cmd = ["gcc", "-O2", "-std=gnu99", "-fPIC", "-shared", "-fopenmp", "-fno-fast-math",
           "-Wall", "-Wextra", "-o", LIB, SRC, "-lm"]
    subprocess.check_call(cmd)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv))
