// cpra_generic.cuh -- the CPRA loop for image sizes that are NOT powers of two (the paper's own detectors:
// N = 160 = 2^5 5; N = 700 = 2^2 5^2 7): any even N in [16, 1024] whose prime factors
// are 2, 3, 5, 7.  Same three-kernel structure as cpra_kernels.cuh (mix + row FFT | column FFT + error + modulus
// + inverse column FFT | inverse row FFT + support / HIO) with the state on NATURAL [n][y][x] arrays and a
// mixed-radix FFT done IN PLACE in shared memory on W lines side by side:
//   forward  decimation in frequency, stages r_0 .. r_{nf-1} (even radices first, odd ones last), natural order in,
//            digit-reversed order out: X[k], k = k_0 + r_0 (k_1 + r_1 (k_2 + ...)), ends at position
//            pos(k) = sum_s k_s M_s,  M_s = N / (r_0 ... r_s);
//   inverse  the mirror image (decimation in time), digit-reversed in, natural out.
// As in the power-of-two path the pointwise steps never need natural frequency order: K1 stores the spectrum with its
// columns in position order, K2 leaves the rows of a forward-only pass in position order, and sqrt(I) is stored once
// in that order (A_perm[pos(ky)][pos(kx)]); only cpra_fft2 and the assembly un-permute (one-off gathers).
// A position of the tile is W complex numbers (W / 2 packed pairs of lines, 16 bytes each); the pairs of position x
// are stored XOR-ed with a key of x, so that the butterflies (16-byte accesses, consecutive positions across the lanes)
// are bank-conflict free without padding and the transposing loads / stores of the row kernels (8-byte accesses, one
// line across the lanes) are 2-way at worst.  Each butterfly = a direct r-point DFT (the networks of cpra_fft.cuh for
// r = 2, 4, 8; real-coefficient sums for r = 3, 5, 7) + twiddles from one table e^{-2 pi i m / N} (computed in double,
// rounded once).  No TMA and no fused row kernel: this path serves the paper's sizes at about a quarter of the
// power-of-two path's bytes per second.
#pragma once
#include "cpra_kernels.cuh"

namespace cpra {

constexpr int GEN_MAXF = 12;
struct GenGeo {
    int N, Np, W, nf;          // image size, projections, lines per tile, number of stages
    int radix[GEN_MAXF];
    // per stage s (sub-transform length L_s = N / (r_0 ... r_{s-1})), filled by gen_make_geo so that no thread divides:
    int L[GEN_MAXF], M[GEN_MAXF], ts[GEN_MAXF];   // L_s, M_s = L_s / r_s, twiddle step N / L_s
    int nb[GEN_MAXF];                              // butterflies per line N / r_s (= the table step of the r_s-th roots of unity)
    float invM[GEN_MAXF];                          // 1 / M_s
};
constexpr int GEN_NT = 256;
// lines per tile: as many as leave four CTAs per SM their shared memory (N W 8 bytes each + the table)
__host__ __device__ __forceinline__ int gen_lines_per_tile(int N) { return N <= 360 ? 16 : 8; }
// the tile, the table of roots, 32 doubles of reduction scratch, the position table of the natural-order column modes
__host__ __device__ __forceinline__ size_t gen_smem_bytes(int N, int W) { return (size_t)N * W * 8 + (size_t)N * 8 + 32 * 8 + (size_t)N * 4 + 16; }
// position of frequency k after the forward transform
__host__ __device__ __forceinline__ int gen_pos(int k, const GenGeo& g)
{
    int M = g.N, p = 0;
    for (int s = 0; s < g.nf; ++s) {
        const int r = g.radix[s];
        M /= r;
        p += (k % r) * M;
        k /= r;
    }
    return p;
}

}  // namespace cpra
