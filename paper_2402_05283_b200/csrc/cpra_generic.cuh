// cpra_generic.cuh -- the CPRA loop for image sizes that are NOT powers of two (the paper's own detectors:
// N = 160 = 2^5 5; N = 700 = 2^2 5^2 7): any even N in [16, 1024] whose prime factors
// are 2, 3, 5, 7.  Same three-kernel structure as cpra_kernels.cuh (mix + row FFT | column FFT + error + modulus
// + inverse column FFT | inverse row FFT + support / HIO) on NATURAL [n][y][x] arrays, with a mixed-radix
// Stockham autosort FFT in shared memory: W lines of length N side by side (element x of line w at x * (W + 1) + w),
// one stage per radix r in {8, 4, 2, 3, 5, 7}, each butterfly = twiddle multiply + a direct r-point DFT, the roots of
// unity from one table e^{-2 pi i m / N} (computed in double, rounded once).  A functional path: the paper's sizes
// run and are parity-tested; it is not tuned (no packed arithmetic, no TMA, no fused row kernel).
#pragma once
#include "cpra_kernels.cuh"

namespace cpra {

constexpr int GEN_MAXF = 12;
struct GenGeo {
    int N, Np, W, nf;          // image size, projections, lines per tile, number of stages
    int radix[GEN_MAXF];
};
constexpr int GEN_NT = 256;
// line stride of a position in shared memory, in complex numbers: even, so that the pair of lines (w, w + 1), w
// even, is one aligned 16-byte access
__host__ __device__ __forceinline__ int gen_wp(int W) { return W + 2; }
__host__ __device__ __forceinline__ size_t gen_smem_bytes(int N, int W) { return (size_t)2 * N * gen_wp(W) * 8 + (size_t)N * 8 + 32 * 8 + 16; }

}  // namespace cpra
