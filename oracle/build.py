"""Build the CPU oracle (test infrastructure) into oracle/libhsp_oracle.so with g++.

Usage: python -m oracle.build        (also called by __graft_entry__.build())
"""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "hsp_oracle.cpp")
LIB = os.path.join(HERE, "libhsp_oracle.so")


def build(force: bool = False) -> str:
    if (not force and os.path.exists(LIB)
            and os.path.getmtime(LIB) >= os.path.getmtime(SRC)):
        return LIB
    # -fopenmp only enables the `#pragma omp` of the timing-only FLAG_ROW_CHUNKS mode; the default (parity) path has none
    cmd = ["g++", "-O2", "-std=c++17", "-shared", "-fPIC", "-fno-fast-math", "-fopenmp", "-Wall", "-Wextra",
           "-o", LIB + ".tmp", SRC, "-lm"]
    subprocess.run(cmd, check=True)
    os.replace(LIB + ".tmp", LIB)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv))
