"""Build libagate.so (the C-ABI CUDA library) in-tree with nvcc for sm_100a.

    python -m paper_2503_20899_b200.build [--force] [--verbose]

The .so is git-ignored but travels to the GPU box with the gpurun snapshot.  nvcc cross-compiles without a GPU.
"""
from __future__ import annotations

import os
import subprocess
import sys

_HERE = os.path.dirname(os.path.abspath(__file__))
_ROOT = os.path.dirname(_HERE)
CSRC = os.path.join(_HERE, "csrc")
INCLUDE = os.path.join(_ROOT, "include")
LIB = os.path.join(_HERE, "libagate.so")
SOURCES = [os.path.join(CSRC, "agate.cu"), os.path.join(CSRC, "agate_noalloc.cu")]
DEPS = SOURCES + [os.path.join(CSRC, "agate_kernels.cuh"), os.path.join(CSRC, "agate_physics.cuh"),
                  os.path.join(CSRC, "agate_stage3d.cuh"), os.path.join(CSRC, "agate_stage2d.cuh"),
                  os.path.join(INCLUDE, "agate.h")]

NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17",
              "-Xcompiler", "-fPIC", "-shared", "-I", INCLUDE, "-I", CSRC]


def nvcc_path() -> str:
    for p in (os.environ.get("NVCC"), "/usr/local/cuda/bin/nvcc", "nvcc"):
        if p and (os.path.sep not in p or os.path.exists(p)):
            return p
    return "nvcc"


def is_stale() -> bool:
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    return any(os.path.getmtime(p) > t for p in DEPS)


def build(force: bool = False, verbose: bool = False) -> str:
    """Compile if the library is missing or older than its sources.  Returns the .so path."""
    if force or is_stale():
        tmp = LIB + f".tmp{os.getpid()}"
        cmd = [nvcc_path()] + NVCC_FLAGS + (["-Xptxas", "-v"] if verbose else []) + ["-o", tmp] + SOURCES
        res = subprocess.run(cmd, cwd=_HERE, capture_output=True, text=True)
        if verbose or res.returncode != 0:
            sys.stderr.write(res.stdout + res.stderr)
        if res.returncode != 0:
            raise RuntimeError("nvcc failed building libagate.so")
        os.replace(tmp, LIB)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="--verbose" in sys.argv))
