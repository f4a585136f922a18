// cpra_cluster.cuh -- the whole iteration of one projection in ONE kernel with the image spread over the
// shared memories of a thread-block CLUSTER (sm_100a, N <= 256).
//
// cpra_image.cuh keeps an image in one CTA: at N = 128 that is one 128 KiB CTA per SM, so 180 projections
// run as two waves with the second 22 % full, and nothing overlaps a CTA's load, barriers and store.  Here a
// cluster of C CTAs owns projection n; CTA c holds T = (N/16)/C row tiles during the row passes and the T
// column tiles with the same numbers during the column passes, so a CTA is 8 ... 64 KiB and several clusters
// are resident on every SM.  The two block transpositions go through distributed shared memory: the forward
// one is PUSHED (each thread stores its transposed 2 x RL piece into the owner's tile, st.shared::cluster),
// the backward one is PULLED (ld.shared::cluster), each between two cluster barriers whose arrive / wait
// halves enclose the register DFT of the stage.  ghat (the mixed input, needed again by the HIO update) is
// written to a global scratch and read back from L2 instead of being re-mixed from three images.
// Launched with programmatic dependent launch: the prologue of iteration t + 1 (barrier init, twiddles,
// L2 request for sqrt(I)) overlaps the tail of iteration t; griddepcontrol.wait precedes the first read of
// the state.
// HBM traffic per pixel: state in 8 + sqrt(I) 4 + support 1/8 + ghat out 8 (+ ghat in 8, an L2 hit) + state
// out 8 = 28.125 (36.125 if ghat misses L2); neighbours come from L2.
#pragma once
#include "cpra_image.cuh"

namespace cpra {

__device__ __forceinline__ uint32_t cluster_ctarank()
{
    uint32_t r;
    asm volatile("mov.u32 %0, %%cluster_ctarank;" : "=r"(r));
    return r;
}
__device__ __forceinline__ void cluster_arrive() { asm volatile("barrier.cluster.arrive.release.aligned;" ::: "memory"); }
__device__ __forceinline__ void cluster_wait() { asm volatile("barrier.cluster.wait.acquire.aligned;" ::: "memory"); }
// arrive without release semantics: for a barrier that only protects shared memory against being OVERWRITTEN
// after it was read (the reads have returned their values before the arrive is issued), so that the arrive
// does not wait for this thread's outstanding global stores (ghat)
__device__ __forceinline__ void cluster_arrive_relaxed() { asm volatile("barrier.cluster.arrive.relaxed.aligned;" ::: "memory"); }
// shared::cta address -> shared::cluster address of the same offset in CTA `rank`
__device__ __forceinline__ uint32_t mapa(uint32_t a, uint32_t rank)
{
    uint32_t r;
    asm volatile("mapa.shared::cluster.u32 %0, %1, %2;" : "=r"(r) : "r"(a), "r"(rank));
    return r;
}
__device__ __forceinline__ void st_dsmem(uint32_t a, float4 v)
{
    asm volatile("st.shared::cluster.v4.f32 [%0], {%1, %2, %3, %4};" ::"r"(a), "f"(v.x), "f"(v.y), "f"(v.z), "f"(v.w) : "memory");
}
__device__ __forceinline__ float4 ld_dsmem(uint32_t a)
{
    float4 v;
    asm volatile("ld.shared::cluster.v4.f32 {%0, %1, %2, %3}, [%4];" : "=f"(v.x), "=f"(v.y), "=f"(v.z), "=f"(v.w) : "r"(a) : "memory");
    return v;
}
__device__ __forceinline__ void pdl_wait() { asm volatile("griddepcontrol.wait;" ::: "memory"); }
__device__ __forceinline__ void pdl_launch_dependents() { asm volatile("griddepcontrol.launch_dependents;" ::: "memory"); }

template <int N, int C> __host__ __device__ constexpr int cl_tiles() { return (N / TB) / C; }
template <int N, int C> __host__ __device__ constexpr int cl_threads() { return cl_tiles<N, C>() * NPAIR * (N / last_radix<N>()); }
template <int N, int C> __host__ __device__ constexpr int cl_quads() { return cl_tiles<N, C>() * N * NPAIR; }
template <int N, int C> __host__ __device__ constexpr int cl_smem_bytes() { return cl_quads<N, C>() * 16 + tw_bytes<N>() + 16 + 32 * 4; }
// CTAs per SM the register allocation is held to: what shared memory allows, at no fewer than 80 registers per thread
template <int N, int C> __host__ __device__ constexpr int cl_min_blocks()
{
    const int by_smem = (220 * 1024) / cl_smem_bytes<N, C>(), by_regs = 65536 / (cl_threads<N, C>() * 80);
    const int m = by_smem < by_regs ? by_smem : by_regs;
    return m < 1 ? 1 : (m > 16 ? 16 : m);
}
template <int N, int C> __host__ __device__ constexpr bool cl_ok()
{
    return Radix<N>::S == 2 && tile_batch<N>() == TB && N >= 64 && N <= 256 && C >= 1 && C <= 16 && (N / TB) % C == 0 &&
           cl_threads<N, C>() >= 32 && cl_threads<N, C>() <= 1024 && cl_smem_bytes<N, C>() <= 227 * 1024;
}

// one in-place stage over the TILES tiles of this CTA; ld(t, pos, j) / st(t, pos, j, v)
template <int N, int R, int L, bool INV, int NT, int TILES, class LD, class ST>
__device__ __forceinline__ void cl_stage(const float2* __restrict__ tws, LD ld, ST st)
{
    constexpr int M = L / R;
    constexpr int NBFT = NPAIR * (N / R), NBF = NBFT * TILES;
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

template <int N, int C, int MIXMODE>
__global__ void __launch_bounds__(cl_threads<N, C>(), cl_min_blocks<N, C>())
k_image_cl(const float4* __restrict__ cur, float4* __restrict__ nxt, float4* __restrict__ gh, const float* __restrict__ Aperm,
           const float2* __restrict__ twg, const uint16_t* __restrict__ S16, double* __restrict__ partial,
           MixParams mp, float beta, float scale, int Np)
{
    using RX = Radix<N>;
    static_assert(cl_ok<N, C>(), "unsupported (N, cluster size)");
    constexpr int T = cl_tiles<N, C>(), NT = cl_threads<N, C>(), NRT = N / TB, NCT = N / TB, R0 = RX::R0, RL = RX::R1;
    constexpr int NBFL = NPAIR * (N / RL);   // last-stage butterflies per tile; NT = T * NBFL
    constexpr int QUADS = cl_quads<N, C>();
    extern __shared__ __align__(128) float4 sm[];
    float4* __restrict__ img = sm;
    const float2* __restrict__ tw0 = reinterpret_cast<const float2*>(sm + QUADS);
    uint64_t* bar = reinterpret_cast<uint64_t*>(const_cast<float2*>(tw0) + tw_count<N>());
    float* red = reinterpret_cast<float*>(bar + 2);
    const int n = (int)(blockIdx.x / C);
    const int c = C == 1 ? 0 : (int)cluster_ctarank();
    const size_t istride = (size_t)N * N / 2;
    const size_t coff = (size_t)c * QUADS;          // quad offset of this CTA's share inside an image
    const int t0 = c * T;                            // first (row / column) tile of this CTA

    if (threadIdx.x == 0) mbar_init(bar, 1);
    __syncthreads();
    if (threadIdx.x == 0) {
        mbar_expect_tx(bar, QUADS * 16 + tw_bytes<N>());
        bulk_load(const_cast<float2*>(tw0), twg, tw_bytes<N>(), bar);
    }
    {   // sqrt(I) of this CTA's column tiles: requested into L2 now (constant data: may precede the dependency wait)
        const char* pf = reinterpret_cast<const char*>(Aperm + ((size_t)n * NCT + t0) * N * TB);
        for (int l = threadIdx.x; l < T * N * TB * 4 / 128; l += NT) asm volatile("prefetch.global.L2 [%0];" ::"l"(pf + (size_t)l * 128));
    }
    pdl_wait();                                      // the previous kernel of the stream (iteration t - 1) is complete
    if (threadIdx.x == 0) bulk_load(img, cur + (size_t)n * istride + coff, QUADS * 16, bar);
    const MixLoader<MIXMODE> mix(cur, istride, n, Np, mp, N, TB);
    float4* __restrict__ ghn = gh + (size_t)n * istride + coff;
    mbar_wait(bar, 0);
    pdl_launch_dependents();                         // the next iteration's CTAs may start their prologue

    auto ld_row = [&](int t, int p, int j) -> c2 { return from_quad(img[(t * N + p) * NPAIR + j]); };
    auto st_row = [&](int t, int p, int j, c2 v) { st_quad(img + (t * N + p) * NPAIR + j, v); };
    auto ld_col = [&](int t, int p, int j) -> c2 { return from_quad(img[(t * N + p) * NPAIR + sw(j, p)]); };
    auto st_col = [&](int t, int p, int j, c2 v) { st_quad(img + (t * N + p) * NPAIR + sw(j, p), v); };
    auto ld_mix = [&](int t, int p, int j) -> c2 {
        const int i = (t * N + p) * NPAIR + j;
        const c2 v = mix(from_quad(img[i]), coff + (size_t)i);
        if constexpr (MIXMODE != MIX_NONE) ghn[i] = to_quad(v);   // ghat, for the update at the end
        return v;
    };
    const int lt = (int)threadIdx.x / NBFL, lbf = (int)threadIdx.x % NBFL, lj = lbf % NPAIR, lq = lbf / NPAIR;
    const int p0 = lq * RL, bct = p0 / TB, jc0 = (p0 % TB) / 2;      // this thread's 2 x RL piece lies in block (t0 + lt, bct)
    // address (in CTA bct / T) of rows (2 lj, 2 lj + 1) of block (t0 + lt, bct) in the column layout
    const uint32_t piece = mapa(smem_u32(img + ((bct % T) * N + (t0 + lt) * TB + 2 * lj) * NPAIR), (uint32_t)(bct / T));

    // ---- A1 + A2 along x ----
    cl_stage<N, R0, N, false, NT, T>(tw0, ld_mix, st_row);
    __syncthreads();
    {
        c2 v[RL];
#pragma unroll
        for (int r = 0; r < RL; ++r) v[r] = ld_row(lt, lq * RL + r, lj);
        dft<RL, false>(v);                           // (consumes the loads: they have returned)
        cluster_arrive_relaxed();                    // this CTA has read its rows ...
        cluster_wait();                              // ... and so has every CTA of the cluster: the tiles may be overwritten
#pragma unroll
        for (int i = 0; i < RL / 2; ++i) {
            const uint32_t a = piece + (uint32_t)(((jc0 + i) ^ lj) * 16);
            st_dsmem(a, make_float4(v[2 * i].re.x, v[2 * i + 1].re.x, v[2 * i].im.x, v[2 * i + 1].im.x));
            st_dsmem(a + NPAIR * 16, make_float4(v[2 * i].re.y, v[2 * i + 1].re.y, v[2 * i].im.y, v[2 * i + 1].im.y));
        }
    }
    cluster_arrive();
    cluster_wait();                                  // the column tiles of this CTA are complete
    // ---- A2 along y, A3 + A4 in registers, A5 along y ----
    cl_stage<N, R0, N, false, NT, T>(tw0, ld_col, st_col);
    __syncthreads();
    {
        const float* __restrict__ At = Aperm + ((size_t)n * NCT + t0 + lt) * N * TB + (size_t)(lq * NPAIR + lj) * (2 * RL);
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
    if (threadIdx.x == 0) {   // fixed order: deterministic.  The first slot of this CTA's tiles carries their sum.
        double e = 0.0;
        for (int w = 0; w < NT / 32; ++w) e += (double)red[w];
        partial[(size_t)n * NCT + t0] = e;
        for (int k = 1; k < T; ++k) partial[(size_t)n * NCT + t0 + k] = 0.0;
    }
    cl_stage<N, R0, N, true, NT, T>(tw0, ld_col, st_col);
    // ---- A5 along x: transposition back (pulled), inverse stages ----
    cluster_arrive();
    cluster_wait();                                  // every column tile of the cluster is final
    {
        c2 v[RL];
#pragma unroll
        for (int i = 0; i < RL / 2; ++i) {
            const uint32_t a = piece + (uint32_t)(((jc0 + i) ^ lj) * 16);
            const float4 x = ld_dsmem(a), y = ld_dsmem(a + NPAIR * 16);
            v[2 * i] = c2{make_float2(x.x, y.x), make_float2(x.z, y.z)};
            v[2 * i + 1] = c2{make_float2(x.y, y.y), make_float2(x.w, y.w)};
        }
        dft<RL, true>(v);                            // (consumes the loads: they have returned)
        cluster_arrive_relaxed();                    // this CTA has pulled its pieces ...
        cluster_wait();                              // ... and so has every CTA: the tiles may be overwritten
#pragma unroll
        for (int r = 0; r < RL; ++r) st_row(lt, lq * RL + r, lj, v[r]);
    }
    __syncthreads();
    cl_stage<N, R0, N, true, NT, T>(tw0, ld_row, st_row);
    __syncthreads();
    // ---- A6: support / HIO over the quads of this CTA's tiles ----
    {
        const float4* __restrict__ ghr = (MIXMODE != MIX_NONE) ? ghn : cur + (size_t)n * istride + coff;
        const uint16_t* __restrict__ Simg = S16 + ((size_t)n * NRT + t0) * N;
#pragma unroll 4
        for (int i = threadIdx.x; i < QUADS; i += NT) {
            const int j = i % NPAIR, tx = i / NPAIR;   // tx = (local row tile) N + x
            unsigned bits = (unsigned)Simg[tx] >> (2 * j);
            // ghat was written by this CTA earlier in this launch: a plain (coherent) load, not the read-only path
            const c2 g0 = from_quad((MIXMODE != MIX_NONE) ? ghr[i] : __ldg(ghr + i));
            const c2 gp = from_quad(img[i]);
            bits = inside_bits(mp, bits, gp.re);
            const float2 ore = update_outside(mp, gp.re, g0.re), oim = update_outside(mp, gp.im, g0.im);
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
        bulk_store(nxt + (size_t)n * istride + coff, img, QUADS * 16);
        bulk_commit();
        bulk_wait_read0();
    }
}

}  // namespace cpra
