"""Build step of the package: nvcc-compile csrc/ into libcpra.so, in-tree, for sm_100a only.

    python -m paper_2402_05283_b200.build [--force] [-v]

nvcc cross-compiles without a GPU.  The kernels of each image size N are one translation unit
(csrc/cpra_inst.cu with -DCPRA_INST_N=<N>), compiled in parallel with csrc/cpra_api.cu and linked into
one shared library.  The library is linked against the static CUDA runtime, so it loads (and
`cpra_plan` validates arguments) on a box without a driver; compute calls then fail with
CPRA_ERR_CUDA -- there is no CPU fallback."""
from __future__ import annotations

import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
OBJ = os.path.join(HERE, "build")
LIB = os.path.join(HERE, "libcpra.so")
SIZES = (16, 32, 64, 128, 256, 512, 1024)
HEADERS = ["cpra_generic.cuh", "cpra_generic_kernels.cuh", "cpra_fft.cuh", "cpra_kernels.cuh", "cpra_layout.cuh", "cpra_image.cuh", "cpra_walk.cuh", "cpra_plan.cuh", "cpra_next.cuh", "cpra_cluster.cuh"]
DEPENDS = [os.path.join(CSRC, f) for f in ["cpra_api.cu", "cpra_inst.cu", "cpra_generic.cu", "cpra_static.cu"] + HEADERS] + [
    os.path.join(os.path.dirname(HERE), "include", "cpra.h")]
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17",
              "-Xcompiler", "-fPIC", "-cudart", "static"]


def needs_build() -> bool:
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    return any(os.path.getmtime(d) > t for d in DEPENDS)


def build(force: bool = False, verbose: bool = False) -> str:
    if not (force or needs_build()):
        return LIB
    nvcc = os.environ.get("NVCC", "nvcc")
    os.makedirs(OBJ, exist_ok=True)
    extra = ["-Xptxas", "-v"] if verbose else []
    units = [("cpra_api.o", "cpra_api.cu", []), ("cpra_generic.o", "cpra_generic.cu", []), ("cpra_static.o", "cpra_static.cu", [])] + [(f"cpra_inst_{n}.o", "cpra_inst.cu", [f"-DCPRA_INST_N={n}"]) for n in SIZES]
    procs = []
    for obj, src, defs in units:
        cmd = [nvcc] + NVCC_FLAGS + extra + defs + ["-c", "-o", os.path.join(OBJ, obj), os.path.join(CSRC, src)]
        procs.append((cmd, subprocess.Popen(cmd, stdout=subprocess.PIPE, stderr=subprocess.STDOUT, text=True)))
    failed = None
    for cmd, pr in procs:
        out, _ = pr.communicate()
        if verbose or pr.returncode != 0:
            sys.stderr.write(out)
        if pr.returncode != 0 and failed is None:
            failed = cmd
    if failed is not None:
        raise subprocess.CalledProcessError(1, failed)
    subprocess.check_call([nvcc] + NVCC_FLAGS + ["-shared", "-o", LIB] + [os.path.join(OBJ, u[0]) for u in units])
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
