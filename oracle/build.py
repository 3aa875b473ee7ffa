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
    """CRK_ORACLE_SANITIZE=1 builds libcrk_oracle_san.so with AddressSanitizer + UndefinedBehaviorSanitizer instead (run the
    CPU tests with LD_PRELOAD=$(g++ -print-file-name=libasan.so); summary in profiles/r02_sanitizers.md)."""
    san = os.environ.get("CRK_ORACLE_SANITIZE", "0") == "1"
    lib = os.path.join(HERE, "libcrk_oracle_san.so") if san else LIB
    if (not force and os.path.exists(lib)
            and os.path.getmtime(lib) >= max(os.path.getmtime(SRC), os.path.getmtime(HDR))):
        return lib
    opt = ["-O1", "-g", "-fsanitize=address,undefined", "-fno-omit-frame-pointer"] if san else ["-O2", "-ftree-vectorize"]
    cmd = ["g++"] + opt + ["-std=c++17", "-fopenmp", "-ffp-contract=off", "-mavx2", "-mfma",
                           "-fPIC", "-shared", "-Wall", "-Wextra", "-o", lib, SRC]
    subprocess.run(cmd, check=True, cwd=HERE)
    return lib


if __name__ == "__main__":
    print(build(force="--force" in sys.argv))
