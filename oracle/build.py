"""Build the CPU oracle (test infrastructure) into oracle/libcrk_oracle.so with g++.

    python oracle/build.py

-ffp-contract=off pins the FP32 neighbour predicate (reading S3); -mavx2 -mfma only lets the
compiler vectorise the brute-force scan (IEEE results are identical lane by lane).
"""
from __future__ import annotations
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "crk_oracle.cpp")
HDR = os.path.join(HERE, "crk_oracle.h")
LIB = os.path.join(HERE, "libcrk_oracle.so")


def build(force: bool = False) -> str:
    if (not force and os.path.exists(LIB)
            and os.path.getmtime(LIB) >= max(os.path.getmtime(SRC), os.path.getmtime(HDR))):
        return LIB
    cmd = ["g++", "-O2", "-ftree-vectorize", "-std=c++17", "-fopenmp", "-ffp-contract=off", "-mavx2", "-mfma",
           "-fPIC", "-shared", "-Wall", "-Wextra", "-o", LIB, SRC]
    subprocess.run(cmd, check=True, cwd=HERE)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv))
