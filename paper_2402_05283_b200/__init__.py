"""paper_2402_05283_b200 -- the CPRA iteration loop (arXiv 2402.05283) as hand-written sm_100a CUDA
kernels behind a C ABI (include/cpra.h, libcpra.so), with a thin ctypes binding.

No CPU fallback exists: importing works anywhere (so that the build and symbol checks run on a box
without a GPU), but every compute call needs the CUDA library and a B200."""
from .binding import (CPRA_OK, ERR_CUDA, ERR_INVALID_ARG, ERR_NOT_READY, ERR_UNSUPPORTED_SIZE, ERR_WORKSPACE,
                      FLAG_DEFAULT, FLAG_FORCE_MULTIPASS, FLAG_NO_CHUNKING, FLAG_NO_WALK, ITERATE, MAX_K, SIGNATURES, SUPPORTED,
                      CpraError, Plan, fsc_static, lib, lib_path)
from .build import build
from . import pipeline

__all__ = ["CPRA_OK", "ERR_CUDA", "ERR_INVALID_ARG", "ERR_NOT_READY", "ERR_UNSUPPORTED_SIZE", "ERR_WORKSPACE",
           "FLAG_DEFAULT", "FLAG_FORCE_MULTIPASS", "FLAG_NO_CHUNKING", "FLAG_NO_WALK", "ITERATE", "MAX_K", "SIGNATURES",
           "SUPPORTED", "CpraError", "Plan", "build", "fsc_static", "lib", "lib_path", "pipeline"]
