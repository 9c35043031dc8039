"""Build paper_2006_10142_b200/libwave2d.so from csrc/ with nvcc for sm_100a (in-tree, no JIT cache).

    python -m paper_2006_10142_b200.build [--force] [--verbose]

nvcc cross-compiles without a GPU.  The library links only the CUDA runtime (static); the one driver
entry point it needs (cuTensorMapEncodeTiled) is resolved at run time through cudaGetDriverEntryPoint.
"""
from __future__ import annotations

import os
import subprocess
import sys

_HERE = os.path.dirname(os.path.abspath(__file__))
_CSRC = os.path.join(_HERE, "csrc")
_LIB = os.path.join(_HERE, "libwave2d.so")
_SOURCES = ["wave2d.cu"]
_DEPS = ["wave2d.cu", "kernels.cuh", "exact.cuh", "line.cuh", "ptx.cuh", os.path.join("..", "..", "include", "wave2d.h")]


def nvcc_path() -> str:
    for cand in (os.environ.get("NVCC"), "/usr/local/cuda/bin/nvcc", "nvcc"):
        if cand and (os.path.isabs(cand) and os.path.exists(cand) or not os.path.isabs(cand)):
            return cand
    return "nvcc"


def needs_build() -> bool:
    if not os.path.exists(_LIB):
        return True
    t = os.path.getmtime(_LIB)
    return any(os.path.getmtime(os.path.join(_CSRC, d)) > t for d in _DEPS)


def build(force: bool = False, verbose: bool = False) -> str:
    if not force and not needs_build():
        return _LIB
    tmp = _LIB + f".tmp{os.getpid()}"
    cmd = [nvcc_path(), "-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-std=c++17", "-lineinfo",
           "-shared", "-Xcompiler", "-fPIC", "--cudart", "static",
           "-o", tmp] + [os.path.join(_CSRC, s) for s in _SOURCES]
    if verbose:
        cmd.insert(1, "-Xptxas=-v")
        print(" ".join(cmd), flush=True)
    subprocess.check_call(cmd)
    os.replace(tmp, _LIB)
    return _LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="--verbose" in sys.argv))
