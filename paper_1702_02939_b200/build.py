"""Build the CUDA library of the AVM hot path for sm_100a (in-tree, nvcc, no JIT cache).

    python -m paper_1702_02939_b200.build [--force]

nvcc cross-compiles without a GPU.  The resulting ``libavm_b200.so`` sits next to this file so that
it travels to the GPU box with the repository snapshot.
"""
from __future__ import annotations

import glob
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libavm_b200.so")
# same sources, reduced-precision storage (positions on a 2^-32 L grid, float records), fp64 arithmetic: NEXT-3
LIB_MIXED = os.path.join(HERE, "libavm_b200_mixed.so")
NVCC = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17",
              "-Xcompiler", "-fPIC", "-shared", "-cudart", "static"]


def sources():
    return sorted(glob.glob(os.path.join(CSRC, "*.cu")))


def _stale(lib: str = LIB) -> bool:
    if not os.path.exists(lib):
        return True
    t = os.path.getmtime(lib)
    deps = sources() + glob.glob(os.path.join(CSRC, "*.cuh")) + [os.path.join(HERE, "..", "include", "avm.h")]
    return any(os.path.getmtime(d) > t for d in deps)


def build(force: bool = False, verbose: bool = False) -> str:
    """builds both libraries; returns the path of the default (fp64) one"""
    for lib, defs in ((LIB, []), (LIB_MIXED, ["-DAVM_MIXED=1"])):
        if force or _stale(lib):
            tmp = lib + f".tmp{os.getpid()}"
            cmd = [NVCC] + NVCC_FLAGS + defs + (["-Xptxas", "-v"] if verbose else []) + ["-o", tmp] + sources()
            subprocess.check_call(cmd)
            os.replace(tmp, lib)
    return LIB


def build_variant(path: str, defines) -> str:
    """the fp64 library with extra -D flags at `path` (test builds: tests/test_gpu_skew.py)"""
    subprocess.check_call([NVCC] + NVCC_FLAGS + [f"-D{d}" for d in defines] + ["-o", path] + sources())
    return path


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
