// cpra_fft.cuh -- register/shared-memory FFT building blocks of the CPRA loop (sm_100a, complex fp32).
//
// The 2D FTs of the "conventional 2D CXDI" iteration (the N^2 log N term of
// PAPER.md:74) are done as 1D FFTs of length N along the SLOW index of a [N][16] tile whose fast
// index is a batch of 16 independent transforms (16 rows for the row pass, 16 columns for the
// column pass).  A warp's lanes run along the batch index, so every shared-memory access of every
// stage is 16 consecutive float2 = 128 B per half-warp: bank-conflict free for any stride pattern.
//
// Forward: in-place decimation-in-frequency, radices R0, R1[, R2] (first stage has stride N/R0),
//          natural order in, digit-reversed order out:  X[k] ends at position pos(k),
//          k = k0 + R0 (k1 + R1 k2)  ->  pos = k2 + R2 (k1 + R1 k0).
// Inverse: the mirror image (decimation-in-time), digit-reversed in, natural out.
// Each butterfly reads and writes the SAME R positions, so a stage needs one barrier, any number of
// butterflies per thread, and the last forward stage / pointwise step / first inverse stage fuse in
// registers.  The pointwise steps of the loop never need natural frequency order: sqrt(I) is stored
// once in the permuted order (cpra_set_data).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace cpra {

constexpr int TB = 16;  // tile width = batch of transforms = lanes of a half-warp

// ---- stage plan ------------------------------------------------------------------------------
template <int N> struct Radix;
template <> struct Radix<16>   { static constexpr int S = 2, R0 = 4,  R1 = 4,  R2 = 1; };
template <> struct Radix<32>   { static constexpr int S = 2, R0 = 8,  R1 = 4,  R2 = 1; };
template <> struct Radix<64>   { static constexpr int S = 2, R0 = 8,  R1 = 8,  R2 = 1; };
template <> struct Radix<128>  { static constexpr int S = 2, R0 = 16, R1 = 8,  R2 = 1; };
template <> struct Radix<256>  { static constexpr int S = 2, R0 = 16, R1 = 16, R2 = 1; };
template <> struct Radix<512>  { static constexpr int S = 3, R0 = 8,  R1 = 8,  R2 = 8; };
template <> struct Radix<1024> { static constexpr int S = 3, R0 = 16, R1 = 8,  R2 = 8; };

template <int N> __host__ __device__ constexpr int last_radix() { return Radix<N>::S == 3 ? Radix<N>::R2 : Radix<N>::R1; }

// position of frequency k after the forward transform (runtime radices: used by layout kernels)
__host__ __device__ __forceinline__ int fft_pos(int k, int R0, int R1, int R2)
{
    const int k0 = k % R0, k1 = (k / R0) % R1, k2 = k / (R0 * R1);
    return k2 + R2 * (k1 + R1 * k0);
}

// ---- complex helpers -------------------------------------------------------------------------
__device__ __forceinline__ float2 cadd(float2 a, float2 b) { return make_float2(a.x + b.x, a.y + b.y); }
__device__ __forceinline__ float2 csub(float2 a, float2 b) { return make_float2(a.x - b.x, a.y - b.y); }
// a * w
__device__ __forceinline__ float2 cmul(float2 a, float2 w)
{
    return make_float2(fmaf(a.x, w.x, -a.y * w.y), fmaf(a.x, w.y, a.y * w.x));
}
// a * conj(w)
__device__ __forceinline__ float2 cmulc(float2 a, float2 w)
{
    return make_float2(fmaf(a.x, w.x, a.y * w.y), fmaf(a.y, w.x, -a.x * w.y));
}

// a * exp(-+ 2 pi i q / 16)  (- forward, + inverse); q is a compile-time constant after unrolling
template <bool INV>
__device__ __forceinline__ float2 mul_w16(float2 a, int q)
{
    constexpr float H = 0.70710678118654752440f;
    constexpr float C1 = 0.92387953251128675613f, S1 = 0.38268343236508977173f;
    switch (q) {
        case 0: return a;
        case 4: return INV ? make_float2(-a.y, a.x) : make_float2(a.y, -a.x);
        case 2: return INV ? make_float2((a.x - a.y) * H, (a.x + a.y) * H) : make_float2((a.x + a.y) * H, (a.y - a.x) * H);
        case 6: return INV ? make_float2((-a.x - a.y) * H, (a.x - a.y) * H) : make_float2((a.y - a.x) * H, (-a.x - a.y) * H);
        default: {
            // q = 1, 3, 5, 7: c = cos(2 pi q/16), s = sin(2 pi q/16)
            const float c = (q == 1) ? C1 : (q == 3) ? S1 : (q == 5) ? -S1 : -C1;
            const float s = (q == 1 || q == 7) ? S1 : C1;
            return INV ? make_float2(fmaf(a.x, c, -a.y * s), fmaf(a.y, c, a.x * s))
                       : make_float2(fmaf(a.x, c, a.y * s), fmaf(a.y, c, -a.x * s));
        }
    }
}

// ---- radix-R DFT in registers, natural order in and out ----------------------------------------
template <int R, bool INV>
__device__ __forceinline__ void dft(float2 (&v)[R])
{
    if constexpr (R == 2) {
        const float2 a = v[0];
        v[0] = cadd(a, v[1]);
        v[1] = csub(a, v[1]);
    } else if constexpr (R == 4) {
        const float2 t0 = cadd(v[0], v[2]), t1 = csub(v[0], v[2]);
        const float2 t2 = cadd(v[1], v[3]), t3 = csub(v[1], v[3]);
        const float2 t3r = INV ? make_float2(-t3.y, t3.x) : make_float2(t3.y, -t3.x);
        v[0] = cadd(t0, t2); v[2] = csub(t0, t2);
        v[1] = cadd(t1, t3r); v[3] = csub(t1, t3r);
    } else {
        float2 e[R / 2], o[R / 2];
#pragma unroll
        for (int k = 0; k < R / 2; ++k) { e[k] = v[2 * k]; o[k] = v[2 * k + 1]; }
        dft<R / 2, INV>(e);
        dft<R / 2, INV>(o);
#pragma unroll
        for (int k = 0; k < R / 2; ++k) {
            const float2 t = mul_w16<INV>(o[k], k * (16 / R));
            v[k] = cadd(e[k], t);
            v[k + R / 2] = csub(e[k], t);
        }
    }
}

// ---- one in-place stage over a [N][TB] tile ------------------------------------------------------
// Sub-transform length L, radix R, M = L/R: butterfly (blk, n2) touches positions blk L + n2 + M r.
// tw[m] = exp(-2 pi i m / N) (shared memory).  ld(pos, b) / st(pos, b, value) move one element.
// Forward: butterfly, then outputs r >= 1 times w_L^{n2 r}.  Inverse: inputs times conj first.
template <int N, int R, int L, bool INV, int NT, int UNROLL, class LD, class ST>
__device__ __forceinline__ void fft_stage(const float2* __restrict__ tw, LD ld, ST st)
{
    constexpr int M = L / R;
    constexpr int NBF = TB * (N / R);
    constexpr int ITERS = (NBF + NT - 1) / NT;
#pragma unroll UNROLL
    for (int it = 0; it < ITERS; ++it) {
        const int bf = (int)threadIdx.x + it * NT;
        if ((NBF % NT) != 0 && bf >= NBF) break;
        const int b = bf % TB, q = bf / TB;
        const int blk = q / M, n2 = q % M;
        const int base = blk * L + n2;
        float2 v[R];
#pragma unroll
        for (int r = 0; r < R; ++r) v[r] = ld(base + M * r, b);
        if (INV && M > 1) {
#pragma unroll
            for (int r = 1; r < R; ++r) v[r] = cmulc(v[r], tw[n2 * r * (N / L)]);
        }
        dft<R, INV>(v);
        if (!INV && M > 1) {
#pragma unroll
            for (int r = 1; r < R; ++r) v[r] = cmul(v[r], tw[n2 * r * (N / L)]);
        }
#pragma unroll
        for (int r = 0; r < R; ++r) st(base + M * r, b, v[r]);
    }
}

// Last forward stage (L = R, contiguous positions R q + r) + pointwise step + first inverse stage,
// fused in registers.  pw(v, q, b) edits the R values in place.
template <int N, int R, int NT, int UNROLL, class LD, class PW, class ST>
__device__ __forceinline__ void fft_stage_mid(LD ld, PW pw, ST st)
{
    constexpr int NBF = TB * (N / R);
    constexpr int ITERS = (NBF + NT - 1) / NT;
#pragma unroll UNROLL
    for (int it = 0; it < ITERS; ++it) {
        const int bf = (int)threadIdx.x + it * NT;
        if ((NBF % NT) != 0 && bf >= NBF) break;
        const int b = bf % TB, q = bf / TB;
        float2 v[R];
#pragma unroll
        for (int r = 0; r < R; ++r) v[r] = ld(q * R + r, b);
        dft<R, false>(v);
        pw(v, q, b);
        dft<R, true>(v);
#pragma unroll
        for (int r = 0; r < R; ++r) st(q * R + r, b, v[r]);
    }
}

}  // namespace cpra
