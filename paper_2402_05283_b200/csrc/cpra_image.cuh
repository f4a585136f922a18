// cpra_image.cuh -- the whole iteration of one projection in ONE kernel, for N <= 128 (sm_100a).
//
// An N x N complex fp32 image is at most 128 KiB: it stays in one SM's shared memory for the full
// round trip  mix -> row FFT -> column FFT -> error + modulus -> inverse column FFT -> inverse row
// FFT -> support / HIO, so an iteration reads the state once, sqrt(I) once,
// writes the state once, and never touches the scratch.  One CTA per projection n; the CTA has as
// many threads as the image has last-stage butterflies, so both block transpositions (row layout
// <-> column layout of cpra_kernels.cuh, now over the whole image) happen in registers between two
// barriers and the image is transformed in place.
// Shared-memory layouts: "row"  quad index (rt N + x)  NPAIR + j          (= the HBM state layout)
//                        "col"  quad index (ct N + py) NPAIR + sw(j, py)  (= the HBM scratch layout)
#pragma once
#include "cpra_kernels.cuh"

namespace cpra {

template <int N> __host__ __device__ constexpr int image_quads() { return N * N / 2; }
template <int N> __host__ __device__ constexpr int image_bytes() { return N * N * 8; }
template <int N> __host__ __device__ constexpr int image_threads() { return (N / TB) * NPAIR * (N / last_radix<N>()); }
template <int N> __host__ __device__ constexpr int image_smem_bytes() { return image_bytes<N>() + tw_bytes<N>() + 16 + 32 * 4; }

// one in-place stage over all N/16 tiles of the image; ld(t, pos, j) / st(t, pos, j, v)
template <int N, int R, int L, bool INV, int NT, class LD, class ST>
__device__ __forceinline__ void image_stage(const float2* __restrict__ tws, LD ld, ST st)
{
    constexpr int M = L / R;
    constexpr int NBFT = NPAIR * (N / R), NBF = NBFT * (N / TB);
    constexpr int ITERS = (NBF + NT - 1) / NT;
#pragma unroll 1
    for (int it = 0; it < ITERS; ++it) {
        const int bfi = (int)threadIdx.x + it * NT;
        if ((NBF % NT) != 0 && bfi >= NBF) break;
        const int t = bfi / NBFT, bf = bfi % NBFT;
        const int j = bf % NPAIR, q = bf / NPAIR;
        const int blk = q / M, n2 = q % M;
        const int base = blk * L + n2;
        c2 v[R];
#pragma unroll
        for (int r = 0; r < R; ++r) v[r] = ld(t, base + M * r, j);
        if constexpr (INV && M > 1) twiddle<R, true>(v, tws, n2);
        dft<R, INV>(v);
        if constexpr (!INV && M > 1) twiddle<R, false>(v, tws, n2);
#pragma unroll
        for (int r = 0; r < R; ++r) st(t, base + M * r, j, v[r]);
    }
}

// block transposition over the whole image: the thread with last-stage butterfly (rt, q, j) owns
// rows (2j, 2j+1) of row tile rt at px slots RL q .. RL q + RL - 1, i.e. a 2 x RL piece of block
// (rt, ct = RL q / 16), which lives at rows 16 rt + 2j (+1) of column tile ct
template <int N, int RL>
__device__ __forceinline__ void store_transposed_img(float4* __restrict__ img, const c2 (&v)[RL], int rt, int q, int j)
{
    const int p0 = q * RL, ct = p0 / TB, jc0 = (p0 % TB) / 2;
    float4* __restrict__ d = img + (ct * N + rt * TB + 2 * j) * NPAIR;
#pragma unroll
    for (int i = 0; i < RL / 2; ++i) {
        const int slot = (jc0 + i) ^ j;
        d[slot] = make_float4(v[2 * i].re.x, v[2 * i + 1].re.x, v[2 * i].im.x, v[2 * i + 1].im.x);
        d[NPAIR + slot] = make_float4(v[2 * i].re.y, v[2 * i + 1].re.y, v[2 * i].im.y, v[2 * i + 1].im.y);
    }
}
template <int N, int RL>
__device__ __forceinline__ void load_transposed_img(const float4* __restrict__ img, c2 (&v)[RL], int rt, int q, int j)
{
    const int p0 = q * RL, ct = p0 / TB, jc0 = (p0 % TB) / 2;
    const float4* __restrict__ d = img + (ct * N + rt * TB + 2 * j) * NPAIR;
#pragma unroll
    for (int i = 0; i < RL / 2; ++i) {
        const int slot = (jc0 + i) ^ j;
        const float4 a = d[slot], b = d[NPAIR + slot];
        v[2 * i] = c2{make_float2(a.x, b.x), make_float2(a.z, b.z)};
        v[2 * i + 1] = c2{make_float2(a.y, b.y), make_float2(a.w, b.w)};
    }
}

// ------------------------------------------------------------------------------------------------
// K0: one CPRA iteration of projection n = n0 + blockIdx.x, image resident in shared memory.
// ------------------------------------------------------------------------------------------------
template <int N, int MIXMODE>
__global__ void __launch_bounds__(image_threads<N>())
k_image(const float4* __restrict__ cur, float4* __restrict__ nxt, const float* __restrict__ Aperm,
        const float2* __restrict__ twg, const uint16_t* __restrict__ S16, double* __restrict__ partial,
        MixParams mp, float beta, float scale, int Np, int n0)
{
    using RX = Radix<N>;
    static_assert(RX::S == 2 && tile_batch<N>() == TB, "whole-image kernel: 16-wide two-stage plans only");
    constexpr int NT = image_threads<N>(), NRT = N / TB, NCT = N / TB, R0 = RX::R0, RL = RX::R1;
    constexpr int NBFL = NPAIR * (N / RL);   // last-stage butterflies per tile; NT = NRT * NBFL
    extern __shared__ __align__(128) float4 sm[];
    float4* __restrict__ img = sm;
    const float2* __restrict__ tw0 = reinterpret_cast<const float2*>(sm + image_quads<N>());
    uint64_t* bar = reinterpret_cast<uint64_t*>(const_cast<float2*>(tw0) + tw_count<N>());
    float* red = reinterpret_cast<float*>(bar + 2);
    const int n = n0 + (int)blockIdx.x;
    const size_t istride = image_quads<N>();

    if (threadIdx.x == 0) mbar_init(bar, 1);
    __syncthreads();
    if (threadIdx.x == 0) {
        mbar_expect_tx(bar, image_bytes<N>() + tw_bytes<N>());
        bulk_load(img, cur + (size_t)n * istride, image_bytes<N>(), bar);
        bulk_load(const_cast<float2*>(tw0), twg, tw_bytes<N>(), bar);
    }
    const MixLoader<MIXMODE> mix(cur, istride, n, Np, mp, N, TB);
    mbar_wait(bar, 0);

    auto ld_row = [&](int t, int p, int j) -> c2 { return from_quad(img[(t * N + p) * NPAIR + j]); };
    auto st_row = [&](int t, int p, int j, c2 v) { st_quad(img + (t * N + p) * NPAIR + j, v); };
    auto ld_col = [&](int t, int p, int j) -> c2 { return from_quad(img[(t * N + p) * NPAIR + sw(j, p)]); };
    auto st_col = [&](int t, int p, int j, c2 v) { st_quad(img + (t * N + p) * NPAIR + sw(j, p), v); };
    auto ld_mix = [&](int t, int p, int j) -> c2 {
        const int i = (t * N + p) * NPAIR + j;
        return mix(from_quad(img[i]), (size_t)i);
    };
    // this thread's butterfly in the stages with contiguous positions
    const int lt = (int)threadIdx.x / NBFL, lbf = (int)threadIdx.x % NBFL, lj = lbf % NPAIR, lq = lbf / NPAIR;

    // ---- A1 + A2: mix, forward FFT along x, transposition into the column layout ----
    image_stage<N, R0, N, false, NT>(tw0, ld_mix, st_row);
    __syncthreads();
    {
        c2 v[RL];
#pragma unroll
        for (int r = 0; r < RL; ++r) v[r] = ld_row(lt, lq * RL + r, lj);
        dft<RL, false>(v);
        __syncthreads();
        store_transposed_img<N, RL>(img, v, lt, lq, lj);
    }
    __syncthreads();
    // ---- A2 along y, A3 + A4 in registers, A5 along y ----
    image_stage<N, R0, N, false, NT>(tw0, ld_col, st_col);
    __syncthreads();
    {
        const float* __restrict__ At = Aperm + ((size_t)n * NCT + lt) * N * TB + (size_t)(lq * NPAIR + lj) * (2 * RL);
        c2 v[RL];
#pragma unroll
        for (int r = 0; r < RL; ++r) v[r] = ld_col(lt, lq * RL + r, lj);
        dft<RL, false>(v);
        float2 acc2 = make_float2(0.f, 0.f);
#pragma unroll
        for (int r = 0; r < RL / 2; ++r) {
            const float4 a = __ldg(reinterpret_cast<const float4*>(At) + r);
            modulus_pair(v[2 * r], make_float2(a.x, a.y), scale, acc2);
            modulus_pair(v[2 * r + 1], make_float2(a.z, a.w), scale, acc2);
        }
        dft<RL, true>(v);
#pragma unroll
        for (int r = 0; r < RL; ++r) st_col(lt, lq * RL + r, lj, v[r]);
        float acc = acc2.x + acc2.y;
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, o);
        if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = acc;
    }
    __syncthreads();
    if (threadIdx.x == 0) {   // fixed order: deterministic.  Slot 0 of the image carries its whole sum.
        double e = 0.0;
        for (int w = 0; w < NT / 32; ++w) e += (double)red[w];
        partial[(size_t)n * NCT] = e;
        for (int c = 1; c < NCT; ++c) partial[(size_t)n * NCT + c] = 0.0;
    }
    image_stage<N, R0, N, true, NT>(tw0, ld_col, st_col);
    __syncthreads();
    // ---- A5 along x: transposition back, inverse stages ----
    {
        c2 v[RL];
        load_transposed_img<N, RL>(img, v, lt, lq, lj);
        dft<RL, true>(v);
        __syncthreads();
#pragma unroll
        for (int r = 0; r < RL; ++r) st_row(lt, lq * RL + r, lj, v[r]);
    }
    __syncthreads();
    image_stage<N, R0, N, true, NT>(tw0, ld_row, st_row);
    __syncthreads();
    // ---- A6: support / HIO over the quads of the image (ghat recomputed from the previous state) ----
    {
        const float4* __restrict__ own = cur + (size_t)n * istride;
        const uint16_t* __restrict__ Simg = S16 + (size_t)n * NRT * N;
#pragma unroll 4
        for (int i = threadIdx.x; i < image_quads<N>(); i += NT) {
            const int j = i % NPAIR, tx = i / NPAIR;   // tx = rt N + x
            unsigned bits = (unsigned)Simg[tx] >> (2 * j);
            const c2 gh = mix(from_quad(__ldg(own + i)), (size_t)i);
            const c2 gp = from_quad(img[i]);
            bits = inside_bits(mp, bits, gp.re);
            const float2 ore = update_outside(mp, gp.re, gh.re), oim = update_outside(mp, gp.im, gh.im);
            float4 o;
            o.x = (bits & 1) ? gp.re.x : ore.x;
            o.y = (bits & 2) ? gp.re.y : ore.y;
            o.z = (bits & 1) ? gp.im.x : oim.x;
            o.w = (bits & 2) ? gp.im.y : oim.y;
            img[i] = o;
        }
    }
    fence_async_smem();
    __syncthreads();
    if (threadIdx.x == 0) {
        bulk_store(nxt + (size_t)n * istride, img, image_bytes<N>());
        bulk_commit();
        bulk_wait_read0();
    }
}

}  // namespace cpra
