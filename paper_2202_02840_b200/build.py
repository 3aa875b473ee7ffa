"""Build libcrk.so (the C-ABI CUDA library) in-tree with nvcc for sm_100a.

    python -m paper_2202_02840_b200.build [--force] [--verbose]

nvcc cross-compiles without a GPU.  No --use_fast_math: the neighbour predicate and the pairwise-antisymmetric
force evaluation rely on IEEE round-to-nearest intrinsics (S3).
"""
from __future__ import annotations

import os
import subprocess
import sys
from concurrent.futures import ThreadPoolExecutor

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
INCLUDE = os.path.join(os.path.dirname(HERE), "include")
LIB = os.path.join(HERE, "libcrk.so")
SOURCES = ["sort.cu", "tree.cu", "lists.cu", "pairs.cu", "api.cu"]
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17",
              "-Xcompiler", "-fPIC", "-Xcompiler", "-O2"]


def _newest_dep() -> float:
    deps = [os.path.join(CSRC, f) for f in os.listdir(CSRC)] + [os.path.join(INCLUDE, "crk.h"), __file__]
    return max(os.path.getmtime(p) for p in deps)


def build(force: bool = False, verbose: bool = False, checked: bool = False) -> str:
    """checked=True: libcrk_checked.so with -DCRK_CHECKED (device-side range checks of every list / tile / arena index; the
    binding loads it when CRK_LIB points at it)."""
    lib = os.path.join(HERE, "libcrk_checked.so") if checked else LIB
    if not force and os.path.exists(lib) and os.path.getmtime(lib) >= _newest_dep():
        return lib
    nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
    flags = list(NVCC_FLAGS) + (["-Xptxas", "-v"] if verbose else []) + (["-DCRK_CHECKED"] if checked else [])
    objs = []

    def compile_one(src):
        obj = os.path.join(CSRC, src.replace(".cu", ".chk.o" if checked else ".o"))
        cmd = [nvcc] + flags + ["-c", os.path.join(CSRC, src), "-o", obj]
        r = subprocess.run(cmd, capture_output=True, text=True)
        return src, obj, r

    with ThreadPoolExecutor(max_workers=len(SOURCES)) as ex:
        results = list(ex.map(compile_one, SOURCES))
    for src, obj, r in results:
        if verbose or r.returncode != 0:
            sys.stderr.write(f"--- {src}\n{r.stdout}{r.stderr}\n")
        if r.returncode != 0:
            raise RuntimeError(f"nvcc failed on {src}")
        objs.append(obj)
    cmd = [nvcc, "-shared", "-o", lib] + objs + ["-lcudart"]
    subprocess.run(cmd, check=True)
    return lib


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="--verbose" in sys.argv, checked="--checked" in sys.argv))
