"""Build step of the package: nvcc-compile csrc/ into libcpra.so, in-tree, for sm_100a only.

    python -m paper_2402_05283_b200.build [--force]

nvcc cross-compiles without a GPU.  The library is linked against the static CUDA runtime, so it
loads (and `cpra_plan` validates arguments) on a box without a driver; compute calls then fail with
CPRA_ERR_CUDA -- there is no CPU fallback."""
from __future__ import annotations

import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
LIB = os.path.join(HERE, "libcpra.so")
SOURCES = [os.path.join(HERE, "csrc", "cpra_api.cu")]
DEPENDS = SOURCES + [os.path.join(HERE, "csrc", f) for f in ("cpra_fft.cuh", "cpra_kernels.cuh", "cpra_layout.cuh", "cpra_image.cuh", "cpra_walk.cuh")] + [
    os.path.join(os.path.dirname(HERE), "include", "cpra.h")]
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17",
              "-shared", "-Xcompiler", "-fPIC", "-cudart", "static"]


def needs_build() -> bool:
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    return any(os.path.getmtime(d) > t for d in DEPENDS)


def build(force: bool = False, verbose: bool = False) -> str:
    if force or needs_build():
        nvcc = os.environ.get("NVCC", "nvcc")
        cmd = [nvcc] + NVCC_FLAGS + (["-Xptxas", "-v"] if verbose else []) + ["-o", LIB] + SOURCES
        subprocess.check_call(cmd)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
