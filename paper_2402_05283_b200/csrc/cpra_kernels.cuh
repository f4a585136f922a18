// cpra_kernels.cuh -- the three tile kernels of the CPRA loop (sm_100a).  See DESIGN.md "Kernels".
//
// HBM layouts.  The unit everywhere is the quad [re_a, re_b, im_a, im_b] (16 B) of a batch pair
// (cpra_fft.cuh).  A tile is N positions x TB/2 quads (TB = Radix<N>::TB transforms per tile: 16, or 8
// at N >= 512), contiguous in HBM, and has the SAME byte layout in shared memory, so it moves with
// asynchronous bulk / tensor copies (TMA) each way and never passes through registers on its way in
// or out.  Written for TB = 16:
//   state g   [n][rt][x][j]       rt = y/16; quad j = rows (16 rt + 2j, + 2j + 1) at column x
//   scratch   [n][ct][py][j^s]    ct = px/16; quad j = columns (16 ct + 2j, + 2j + 1) at row py,
//                                 stored at slot j ^ s, s = (py >> 1) & (TB/2 - 1).  py, px are
//                                 digit-reversed frequency positions after the respective forward
//                                 transform.  The XOR makes the TB x TB block transposition that the
//                                 row kernels do between their own layout and this one conflict-free.
//   A=sqrt(I) [n][ct][q][j][r][e] fp32; py = RL q + r, px = 16 ct + 2j + e: the 2 RL values one
//                                 thread needs in the fused middle stage are contiguous
//   support   [n][y/16][x] u16    bit b = S(y = 16 (y/16) + b, x)   (1 bit per pixel)
// With TB = 8 the positions of a tile are additionally permuted inside aligned pairs (ppos below).
#pragma once
#include <cuda.h>   // CUtensorMap (type only; the encoder is fetched through the runtime, see cpra_api.cu)

#include "cpra_fft.cuh"

namespace cpra {

constexpr int MAXK = 8;  // = CPRA_MAX_K
// sizes and radices of a plan, for the layout kernels of cpra_layout.cuh (runtime, not templated)
struct Geo {
    int N, Np, R0, R1, R2, RL, TB;   // TB = transforms per tile (Radix<N>::TB)
};
struct MixParams {
    int K;
    float a[MAXK + 1];
    // real-space update outside the support: g <- c_ghat ghat + c_gp g'   (HIO: 1, -beta;  RAAR: beta,
    // 1 - 2 beta;  ER: 0, 0;  cpra_set_update).  Inside the support g <- g' for all of them.
    float c_ghat, c_gp;
    // cpra_set_seam: a neighbour reached by wrapping round the end of the stack is read mirrored in u
    // (x -> (N - x) mod N about the centre pixel): the seam of a [0, 180) scan, reading A5b
    int flip_seam;
    // cpra_set_positivity: a pixel inside the support whose modulus-constrained estimate has a negative real part
    // is treated as lying outside it (the conventional positivity constraint of the real-space step)
    int positivity;
};
// the update outside the support on a pair; with c_ghat = 1 (HIO) the product is exact, so the result
// is the single fma ghat - beta g'
__device__ __forceinline__ float2 update_outside(const MixParams& mp, float2 gp, float2 gh)
{
    return pfma(bc(mp.c_gp), gp, pmul(bc(mp.c_ghat), gh));
}

// support bits of a pair after the optional positivity test on Re g'
__device__ __forceinline__ unsigned inside_bits(const MixParams& mp, unsigned bits, float2 re)
{
    if (mp.positivity) {
        if (re.x < 0.f) bits &= ~1u;
        if (re.y < 0.f) bits &= ~2u;
    }
    return bits;
}

enum { MIX_NONE = 0, MIX_K1 = 1, MIX_GEN = 2, MIX_MASK = 3, MIX_ABS = 4 };   // MIX_MASK: S g (assembly); MIX_ABS: (|S g|, 0) (shrink-wrap)
// (|a|, 0), (|b|, 0) of a pair: sqrt(re^2 + im^2) with one rounding of the sum of squares' product term (fma), as the
// scalar expression sqrtf(x * x + y * y) compiles
__device__ __forceinline__ c2 abs_pair(c2 v)
{
    const float2 m2 = pfma(v.re, v.re, pmul(v.im, v.im));
    return c2{make_float2(sqrtf(m2.x), sqrtf(m2.y)), make_float2(0.f, 0.f)};
}
enum { COL_FULL = 0, COL_FWD = 1, COL_INV = 2, COL_GAUSS = 3 };   // COL_GAUSS: forward, times a separable table, inverse (shrink-wrap's blur)
enum { ROWINV_HIO = 0, ROWINV_PLAIN = 1 };

template <int N> __host__ __device__ constexpr int tile_quads() { return N * tile_pairs<N>(); }
template <int N> __host__ __device__ constexpr int tile_bytes() { return N * tile_pairs<N>() * 16; }
template <int N> __host__ __device__ constexpr int tw_bytes() { return tw_count<N>() * 8; }
// tile + twiddle tables + mbarrier + the tile's support words (k_row_inv)
template <int N> __host__ __device__ constexpr int smem_bytes() { return tile_bytes<N>() + tw_bytes<N>() + 16 + 2 * N; }

// slot of column pair j at row py of a scratch tile with np pairs per position
__host__ __device__ __forceinline__ int sw(int j, int py, int np = NPAIR) { return j ^ ((py >> 1) & (np - 1)); }
// Physical place of logical position p of a tile.  With 16 transforms per tile a position is 128 B
// and any two positions are conflict-free.  With 8 (N = 1024) a position is 64 B = half of the bank
// window and a quarter-warp touches two positions (two butterflies): they must differ in parity.
// They do in every stage with stride > 1 (consecutive n2); in the stage with contiguous positions
// (radix 8) they are 8 apart, so odd 8-blocks swap their even and odd positions.  HBM tiles have the
// same order (they are bulk-copied verbatim).
// `par` (scratch tiles: the parity of the column tile ct) inverts the choice of the swapped blocks, so
// that the two 8 x 8 blocks (rt, ct), (rt, ct + 1) that a quarter-warp of a row kernel transposes at
// once have their rows in opposite halves of the bank window too.
__host__ __device__ __forceinline__ int ppos(int p, int tb, int par = 0) { return tb == 16 ? p : p ^ (((p >> 3) + par) & 1); }
template <int N> __host__ __device__ __forceinline__ int ppos(int p)
{
    static_assert(tile_batch<N>() == 16 || last_radix<N>() == 8, "8-wide tiles: the contiguous stage must be radix 8");
    return ppos(p, tile_batch<N>());
}

// The carousel mix of Eq. (4) evaluated at one quad: `q` = quad offset inside an
// image (same for every n), `istride` = quads per image.  `own` = the quad of image n itself.
template <int MODE>
struct MixLoader {
    const float4* __restrict__ cm;   // image n-1 (mod Np)
    const float4* __restrict__ cp;   // image n+1 (mod Np)
    const float4* __restrict__ base; // image 0
    size_t istride;
    int n, Np;
    MixParams mp;
    int N, tb;          // image size and transforms per tile (for the mirrored read across the seam)
    bool flm, flp;      // K = 1: the lower / upper neighbour lies across the seam and is read mirrored

    __device__ __forceinline__ MixLoader(const float4* cur, size_t istride_, int n_, int Np_, const MixParams& mp_, int N_, int tb_)
        : base(cur), istride(istride_), n(n_), Np(Np_), mp(mp_), N(N_), tb(tb_)
    {
        cm = cur + (size_t)(n_ == 0 ? Np_ - 1 : n_ - 1) * istride_;
        cp = cur + (size_t)(n_ == Np_ - 1 ? 0 : n_ + 1) * istride_;
        flm = mp_.flip_seam && n_ == 0;
        flp = mp_.flip_seam && n_ == Np_ - 1;
    }
    // quad offset (inside an image, state layout) of the pixel mirrored in x: same row tile and row pair,
    // position x -> (N - x) mod N
    __device__ __forceinline__ size_t mirrored(size_t q) const
    {
        const int np = tb / 2, tq = N * np;
        const int loc = (int)(q % (size_t)tq), j = loc % np, x = ppos(loc / np, tb);
        return q - (size_t)loc + (size_t)(ppos((N - x) & (N - 1), tb) * np + j);
    }
    __device__ __forceinline__ c2 ldm(size_t q) const { return from_quad(__ldg(cm + (flm ? mirrored(q) : q))); }
    __device__ __forceinline__ c2 ldp(size_t q) const { return from_quad(__ldg(cp + (flp ? mirrored(q) : q))); }
    // general K: image (n + d) mod Np, mirrored if the step d wrapped round the end of the stack
    __device__ __forceinline__ c2 ldk(int d, size_t q) const
    {
        int m = n + d;
        const bool wrapped = m < 0 || m >= Np;
        if (m < 0) m += Np;
        if (m >= Np) m -= Np;
        return from_quad(__ldg(base + (size_t)m * istride + ((wrapped && mp.flip_seam) ? mirrored(q) : q)));
    }
    // the neighbours' share of the mix at quad q: sum_k a_k (g_{n-k} + g_{n+k}), and its combination
    // with the own quad: a_0 own + nb
    __device__ __forceinline__ c2 nbsum(size_t q) const
    {
        if constexpr (MODE == MIX_K1) {
            const c2 m = ldm(q), p = ldp(q);
            const float2 a1 = bc(mp.a[1]);
            return c2{pmul(a1, padd(m.re, p.re)), pmul(a1, padd(m.im, p.im))};
        } else if constexpr (MODE == MIX_GEN) {
            c2 acc{make_float2(0.f, 0.f), make_float2(0.f, 0.f)};
            for (int k = 1; k <= mp.K; ++k) {
                const c2 m = ldk(-k, q);
                const c2 p = ldk(k, q);
                acc.re = pfma(bc(mp.a[k]), padd(m.re, p.re), acc.re);
                acc.im = pfma(bc(mp.a[k]), padd(m.im, p.im), acc.im);
            }
            return acc;
        } else {
            return c2{make_float2(0.f, 0.f), make_float2(0.f, 0.f)};
        }
    }
    __device__ __forceinline__ c2 combine(c2 own, c2 nb) const
    {
        if constexpr (MODE == MIX_K1 || MODE == MIX_GEN) {
            const float2 a0 = bc(mp.a[0]);
            return c2{pfma(a0, own.re, nb.re), pfma(a0, own.im, nb.im)};
        } else {
            return own;
        }
    }
    __device__ __forceinline__ c2 operator()(c2 own, size_t q) const
    {
        if constexpr (MODE == MIX_NONE || MODE == MIX_MASK || MODE == MIX_ABS) {
            return own;
        } else if constexpr (MODE == MIX_K1) {
            const c2 m = ldm(q), p = ldp(q);
            const float2 a0 = bc(mp.a[0]), a1 = bc(mp.a[1]);
            return c2{pfma(a0, own.re, pmul(a1, padd(m.re, p.re))), pfma(a0, own.im, pmul(a1, padd(m.im, p.im)))};
        } else {
            c2 acc{pmul(bc(mp.a[0]), own.re), pmul(bc(mp.a[0]), own.im)};
            for (int k = 1; k <= mp.K; ++k) {
                const c2 m = ldk(-k, q);
                const c2 p = ldk(k, q);
                acc.re = pfma(bc(mp.a[k]), padd(m.re, p.re), acc.re);
                acc.im = pfma(bc(mp.a[k]), padd(m.im, p.im), acc.im);
            }
            return acc;
        }
    }
};

// One TMA tensor instruction moves the N/TB blocks (TB x TB complex each, one per column tile) of a
// row tile between shared memory and a spectrum buffer, described as the contiguous 5D tensor
// [n][ct][rt][split][inner floats] (a block = split x inner floats, inner <= 256) with the box
// {inner, split, 1, N/TB, 1}.  (One bulk copy per block would have to be issued lane by lane: the
// copy instructions take their addresses from uniform registers.)
__device__ __forceinline__ void tma_load_tile(void* smem_dst, const CUtensorMap* tm, int rt, int n, uint64_t* bar)
{
    asm volatile("cp.async.bulk.tensor.5d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3, %4, %5, %6}], [%7];"
                 ::"r"(smem_u32(smem_dst)), "l"(tm), "r"(0), "r"(0), "r"(rt), "r"(0), "r"(n), "r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void tma_store_tile(const CUtensorMap* tm, int rt, int n, const void* smem_src)
{
    asm volatile("cp.async.bulk.tensor.5d.global.shared::cta.bulk_group [%0, {%1, %2, %3, %4, %5}], [%6];"
                 ::"l"(tm), "r"(0), "r"(0), "r"(rt), "r"(0), "r"(n), "r"(smem_u32(smem_src)) : "memory");
}

// Barrier between the two inner stages of a 3-stage plan.  With 4 pairs per position and radices
// R1 = RL = 8, butterfly bf of either stage works inside the 64-position block bf / 32, i.e. every
// warp owns whole blocks: the exchange stays inside the warp and a warp barrier is enough.
template <int N> __host__ __device__ constexpr bool inner_stages_warp_local()
{
    return Radix<N>::S == 3 && tile_pairs<N>() == 4 && Radix<N>::R1 == 8 && Radix<N>::R2 == 8;
}
template <int N> __device__ __forceinline__ void inner_sync()
{
    if constexpr (inner_stages_warp_local<N>()) __syncwarp(); else __syncthreads();
}

// ------------------------------------------------------------------------------------------------
// Stages of the 8-wide plans with inner radices 8 x 8 (N = 512, 1024) with the quad offsets of a
// butterfly written as ONE base (two where the positions cross 8-blocks of alternating parity, see
// ppos) plus compile-time multiples of r, instead of position arithmetic per access:
//   stage 0 (stride M0 = 64): p = n2 + M0 r            ppos(p) = ppos(n2) + M0 r,  slot key (p >> 1) & 3 = (n2 >> 1) & 3
//   stage 1 (stride 8):       p = 64 b + n2 + 8 r      ppos(p) = p ^ (r & 1),      slot key (n2 >> 1) & 3
//   last    (contiguous):     p = 8 q + r              ppos(p) = 8 q + (r ^ (q & 1)), slot key (r >> 1) & 3
// SWZ = the scratch layout (slot = pair ^ key); otherwise the state layout (slot = pair).
// ------------------------------------------------------------------------------------------------
template <int N, bool INV, bool SWZ, int NT>
__device__ __forceinline__ void stage0_8(float4* __restrict__ tile, const float2* __restrict__ tw0, int par = 0)
{
    constexpr int R = Radix<N>::R0, M0 = N / R, NP = 4, NBF = NP * M0, ITERS = (NBF + NT - 1) / NT;
    static_assert(M0 == 64, "stage 0 of the 8-wide plans has stride 64");
#pragma unroll 1
    for (int it = 0; it < ITERS; ++it) {
        const int bf = (int)threadIdx.x + it * NT;
        if ((NBF % NT) != 0 && bf >= NBF) break;
        const int j = bf % NP, n2 = bf / NP;
        float4* __restrict__ b = tile + ppos(n2, 8, par) * NP + (SWZ ? (j ^ ((n2 >> 1) & 3)) : j);
        c2 v[R];
#pragma unroll
        for (int r = 0; r < R; ++r) v[r] = from_quad(b[r * (M0 * NP)]);
        if constexpr (INV) twiddle<R, true>(v, tw0, n2);
        dft<R, INV>(v);
        if constexpr (!INV) twiddle<R, false>(v, tw0, n2);
#pragma unroll
        for (int r = 0; r < R; ++r) st_quad(b + r * (M0 * NP), v[r]);
    }
}
template <int N, bool INV, bool SWZ, int NT>
__device__ __forceinline__ void stage1_8(float4* __restrict__ tile, const float2* __restrict__ tw1, int par = 0)
{
    constexpr int R = 8, NP = 4, NBF = NP * (N / R), ITERS = (NBF + NT - 1) / NT;
#pragma unroll 1
    for (int it = 0; it < ITERS; ++it) {
        const int bf = (int)threadIdx.x + it * NT;
        if ((NBF % NT) != 0 && bf >= NBF) break;
        const int j = bf % NP, q = bf / NP, blk = q / 8, n2 = q % 8;
        const int slot = SWZ ? (j ^ ((n2 >> 1) & 3)) : j;
        float4* __restrict__ be = tile + (blk * 64 + (n2 ^ par)) * NP + slot;         // even r (8-block 8 blk + r)
        float4* __restrict__ bo = tile + (blk * 64 + (n2 ^ 1 ^ par)) * NP + slot;     // odd r
        c2 v[R];
#pragma unroll
        for (int r = 0; r < R; ++r) v[r] = from_quad(((r & 1) ? bo : be)[r * (8 * NP)]);
        if constexpr (INV) twiddle<R, true>(v, tw1, n2);
        dft<R, INV>(v);
        if constexpr (!INV) twiddle<R, false>(v, tw1, n2);
#pragma unroll
        for (int r = 0; r < R; ++r) st_quad(((r & 1) ? bo : be) + r * (8 * NP), v[r]);
    }
}
// quad of element r of the contiguous butterfly q, pair j
template <bool SWZ>
struct Last8 {
    float4* pe;
    float4* po;
    int j;
    __device__ __forceinline__ Last8(float4* tile, int q, int j_, int par = 0) : j(j_)
    {
        const int s = (q + par) & 1;
        pe = tile + (8 * q + s) * 4;
        po = tile + (8 * q + 1 - s) * 4;
    }
    __device__ __forceinline__ float4* operator()(int r) const
    {
        return ((r & 1) ? po : pe) + (r & ~1) * 4 + (SWZ ? (j ^ (r >> 1)) : j);
    }
};

// shared-memory carve-up of the three kernels
template <int N>
struct Smem {
    float4* tile;
    const float2* tw0;
    const float2* tw1;
    uint64_t* bar;
    uint16_t* sup;   // [N] support words of the tile
    __device__ __forceinline__ explicit Smem(float4* sm)
        : tile(sm), tw0(reinterpret_cast<const float2*>(sm + tile_quads<N>())), tw1(tw0 + tw_count_stage0<N>()),
          bar(reinterpret_cast<uint64_t*>(const_cast<float2*>(tw0) + tw_count<N>())),
          sup(reinterpret_cast<uint16_t*>(bar + 2)) {}
};

// ------------------------------------------------------------------------------------------------
// The block transposition of the row kernels.  A thread of the stage with contiguous positions
// (radix RL, butterfly q, row pair j) owns rows (2j, 2j+1) x px slots RL q .. RL q + RL - 1 of the
// tile.  In the row layout these are RL quads (one per slot); in the scratch layout they are
// 2 x RL/2 quads (one per row and column pair) inside the 16 x 16 block ct = RL q / 16, which
// occupies the same 2 KiB of shared memory: position (16 ct + row) , slot jc ^ j.
// ------------------------------------------------------------------------------------------------
// `rt` = the row tile: inside its 8-row block the rows sit in the physical order of the column tile,
// ppos(TB rt + r, ct) = TB rt + (r ^ flip), flip = (rt + ct) & 1: the two blocks ct, ct + 1 that a
// quarter-warp handles together lie in opposite halves of the bank window (conflict-free).
template <int N>
__device__ __forceinline__ void store_transposed(float4* __restrict__ tile, const c2 (&v)[last_radix<N>()], int q, int j, int rt)
{
    constexpr int RL = last_radix<N>(), TBN = tile_batch<N>(), NP = tile_pairs<N>();
    const int p0 = q * RL, ct = p0 / TBN, jc0 = (p0 % TBN) / 2;
    const int r0 = ppos(TBN * rt + 2 * j, TBN, ct & 1) % TBN, r1 = ppos(TBN * rt + 2 * j + 1, TBN, ct & 1) % TBN;
#pragma unroll
    for (int i = 0; i < RL / 2; ++i) {
        const int slot = (jc0 + i) ^ j;
        tile[(ct * TBN + r0) * NP + slot] = make_float4(v[2 * i].re.x, v[2 * i + 1].re.x, v[2 * i].im.x, v[2 * i + 1].im.x);
        tile[(ct * TBN + r1) * NP + slot] = make_float4(v[2 * i].re.y, v[2 * i + 1].re.y, v[2 * i].im.y, v[2 * i + 1].im.y);
    }
}
template <int N>
__device__ __forceinline__ void load_transposed(const float4* __restrict__ tile, c2 (&v)[last_radix<N>()], int q, int j, int rt)
{
    constexpr int RL = last_radix<N>(), TBN = tile_batch<N>(), NP = tile_pairs<N>();
    const int p0 = q * RL, ct = p0 / TBN, jc0 = (p0 % TBN) / 2;
    const int r0 = ppos(TBN * rt + 2 * j, TBN, ct & 1) % TBN, r1 = ppos(TBN * rt + 2 * j + 1, TBN, ct & 1) % TBN;
#pragma unroll
    for (int i = 0; i < RL / 2; ++i) {
        const int slot = (jc0 + i) ^ j;
        const float4 a = tile[(ct * TBN + r0) * NP + slot];
        const float4 b = tile[(ct * TBN + r1) * NP + slot];
        v[2 * i] = c2{make_float2(a.x, b.x), make_float2(a.z, b.z)};
        v[2 * i + 1] = c2{make_float2(a.y, b.y), make_float2(a.w, b.w)};
    }
}

// ------------------------------------------------------------------------------------------------
// K1: mix (Eq. (4)) + forward FFT along x of 16 rows; writes the column-tiled scratch.
// grid = nimg * N/16 CTAs, n fastest (so that the three CTAs sharing a neighbour tile run together
// and the second and third read hit L2).  The tile of image n arrives by bulk copy; the neighbours
// n-1, n+1 are read with 128-bit loads inside the first stage.
// ------------------------------------------------------------------------------------------------
template <int N, int MODE>
__global__ void __launch_bounds__(Radix<N>::NT, (Radix<N>::PF && (MODE == MIX_K1 || MODE == MIX_GEN)) ? Radix<N>::MINBF : Radix<N>::MINB)
k_row_fwd(const float4* __restrict__ cur, const __grid_constant__ CUtensorMap tm_scr, const float2* __restrict__ twg,
          const uint16_t* __restrict__ S16, MixParams mp, int Np, int n0, int nimg, float4* __restrict__ ghat_out)
{
    // ghat_out != nullptr: the mixed input ghat_n is also stored (state layout) for the HIO update of
    // this iteration (read by k_row_inv / k_row_walk instead of being recomputed from three tiles)
    using RX = Radix<N>;
    constexpr int TBN = tile_batch<N>(), NP = tile_pairs<N>();
    constexpr int NT = RX::NT, NRT = N / TBN, NCT = N / TBN, RL = last_radix<N>();
    constexpr int B = NP * (N / RL) / NT;   // butterflies per thread in the last stage
    static_assert(B * NT == NP * (N / RL) && B >= 1, "last stage must fill the CTA exactly");
    constexpr int R0 = RX::R0, M0 = N / R0, NBF0 = NP * M0, IT0 = (NBF0 + NT - 1) / NT;
    constexpr bool PFMIX = RX::PF && (MODE == MIX_K1 || MODE == MIX_GEN);
    constexpr bool FAST = inner_stages_warp_local<N>();   // 8-wide, inner radices 8 x 8: affine offsets
    extern __shared__ __align__(128) float4 sm[];
    const Smem<N> s(sm);
    float4* __restrict__ tile = s.tile;
    const int n = n0 + (int)(blockIdx.x % (unsigned)nimg);
    const int rt = (int)(blockIdx.x / (unsigned)nimg);
    const size_t istride = (size_t)N * N / 2;             // quads per image
    const size_t toff = (size_t)rt * tile_quads<N>();      // tile offset inside an image

    if (threadIdx.x == 0) mbar_init(s.bar, 1);
    __syncthreads();
    if (threadIdx.x == 0) {
        mbar_expect_tx(s.bar, tile_bytes<N>() + tw_bytes<N>());
        bulk_load(tile, cur + (size_t)n * istride + toff, tile_bytes<N>(), s.bar);
        bulk_load(const_cast<float2*>(s.tw0), twg, tw_bytes<N>(), s.bar);
    }
    const MixLoader<MODE> mix(cur, istride, n, Np, mp, N, TBN);
    const uint16_t* __restrict__ Srow = S16 + ((size_t)n * (N / 16) + (rt * TBN) / 16) * N;   // 16-row words
    const int sshift = (rt * TBN) % 16;
    auto tq = [&](int p, int j) -> int { return ppos<N>(p) * NP + j; };   // quad of (position, pair) in a state tile
    if constexpr (!PFMIX && MODE == MIX_K1 && N <= 256) {
        // the two neighbour tiles (read with 128-bit loads inside the first stage) are requested into L2
        // before the own tile is waited for (N = 256: 148.5 -> 146.5 us per iteration at N_p = 180; at
        // N = 1024 the same requests make the kernel 8 % slower)
        const char* pm = reinterpret_cast<const char*>(mix.cm + toff);
        const char* pp = reinterpret_cast<const char*>(mix.cp + toff);
        for (int l = threadIdx.x; l < tile_bytes<N>() / 128; l += NT) {
            asm volatile("prefetch.global.L2 [%0];" ::"l"(pm + (size_t)l * 128));
            asm volatile("prefetch.global.L2 [%0];" ::"l"(pp + (size_t)l * 128));
        }
    }
    if constexpr (!PFMIX) mbar_wait(s.bar, 0);

    auto ld_first = [&](int x, int j) -> c2 {
        c2 v = mix(from_quad(tile[tq(x, j)]), toff + (size_t)tq(x, j));
        if constexpr (MODE == MIX_MASK || MODE == MIX_ABS) {
            const unsigned bits = (unsigned)Srow[x] >> (sshift + 2 * j);
            if (!(bits & 1)) { v.re.x = 0.f; v.im.x = 0.f; }
            if (!(bits & 2)) { v.re.y = 0.f; v.im.y = 0.f; }
        }
        if constexpr (MODE == MIX_ABS) v = abs_pair(v);
        if (ghat_out) ghat_out[(size_t)n * istride + toff + (size_t)tq(x, j)] = to_quad(v);
        return v;
    };
    auto ld_s = [&](int p, int j) -> c2 { return from_quad(tile[tq(p, j)]); };
    auto st_s = [&](int p, int j, c2 v) { st_quad(tile + tq(p, j), v); };

    if constexpr (PFMIX) {
        // the neighbours' share of every first-stage butterfly of this thread is requested before
        // the own tile is waited for
        c2 nbv[IT0][R0];
#pragma unroll
        for (int it = 0; it < IT0; ++it) {
            const int bf = (int)threadIdx.x + it * NT, j = bf % NP, q = bf / NP;
            if (bf < NBF0) {
#pragma unroll
                for (int r = 0; r < R0; ++r) nbv[it][r] = mix.nbsum(toff + (size_t)tq(q + M0 * r, j));
            }
        }
        mbar_wait(s.bar, 0);
#pragma unroll
        for (int it = 0; it < IT0; ++it) {
            const int bf = (int)threadIdx.x + it * NT, j = bf % NP, q = bf / NP;
            if (bf < NBF0) {
                c2 v[R0];
#pragma unroll
                for (int r = 0; r < R0; ++r) v[r] = mix.combine(ld_s(q + M0 * r, j), nbv[it][r]);
                if (ghat_out) {
#pragma unroll
                    for (int r = 0; r < R0; ++r) ghat_out[(size_t)n * istride + toff + (size_t)tq(q + M0 * r, j)] = to_quad(v[r]);
                }
                dft<R0, false>(v);
                twiddle<R0, false>(v, s.tw0, q);
#pragma unroll
                for (int r = 0; r < R0; ++r) st_s(q + M0 * r, j, v[r]);
            }
        }
    } else if constexpr (FAST) {
        // 8-wide plans: the butterfly's quads are one base + compile-time multiples of r, in shared
        // memory and (same layout) in the neighbours' tiles
#pragma unroll 1
        for (int it = 0; it < IT0; ++it) {
            const int bf = (int)threadIdx.x + it * NT;
            if ((NBF0 % NT) != 0 && bf >= NBF0) break;
            const int j = bf % NP, n2 = bf / NP, o = ppos(n2, 8) * NP + j;
            c2 v[R0];
#pragma unroll
            for (int r = 0; r < R0; ++r) {
                const int idx = o + r * (M0 * NP);
                v[r] = mix(from_quad(tile[idx]), toff + (size_t)idx);
                if constexpr (MODE == MIX_MASK || MODE == MIX_ABS) {
                    const unsigned bits = (unsigned)Srow[n2 + M0 * r] >> (sshift + 2 * j);
                    if (!(bits & 1)) { v[r].re.x = 0.f; v[r].im.x = 0.f; }
                    if (!(bits & 2)) { v[r].re.y = 0.f; v[r].im.y = 0.f; }
                }
                if constexpr (MODE == MIX_ABS) v[r] = abs_pair(v[r]);
                if (ghat_out) ghat_out[(size_t)n * istride + toff + (size_t)idx] = to_quad(v[r]);
            }
            dft<R0, false>(v);
            twiddle<R0, false>(v, s.tw0, n2);
#pragma unroll
            for (int r = 0; r < R0; ++r) st_quad(tile + o + r * (M0 * NP), v[r]);
        }
    } else {
        fft_stage<N, RX::R0, N, false, NT, 1>(s.tw0, ld_first, st_s);
    }
    __syncthreads();
    if constexpr (RX::S == 3) {
        if constexpr (FAST) stage1_8<N, false, false, NT>(tile, s.tw1);
        else fft_stage<N, RX::R1, N / RX::R0, false, NT, 1>(s.tw1, ld_s, st_s);
        inner_sync<N>();
    }
    // last stage (contiguous positions, no twiddles) + transposition into the scratch layout
    c2 v[B][RL];
#pragma unroll
    for (int b = 0; b < B; ++b) {
        const int bf = (int)threadIdx.x + b * NT, j = bf % NP, q = bf / NP;
#pragma unroll
        if constexpr (FAST) {
            const Last8<false> at(tile, q, j);
#pragma unroll
            for (int r = 0; r < RL; ++r) v[b][r] = from_quad(*at(r));
        } else {
#pragma unroll
            for (int r = 0; r < RL; ++r) v[b][r] = ld_s(q * RL + r, j);
        }
        dft<RL, false>(v[b]);
    }
    inner_sync<N>();   // (the block a butterfly is transposed into lies in its own 64-position block)
#pragma unroll
    for (int b = 0; b < B; ++b) {
        const int bf = (int)threadIdx.x + b * NT;
        store_transposed<N>(tile, v[b], bf / NP, bf % NP, rt);
    }
    fence_async_smem();
    __syncthreads();
    // block ct of the tile -> rows [TBN rt, TBN rt + TBN) of scratch tile (n, ct), all ct in one instruction
    if (threadIdx.x == 0) {
        tma_store_tile(&tm_scr, rt, n, tile);
        bulk_commit();
        bulk_wait_read0();
    }
}

// ------------------------------------------------------------------------------------------------
// K2: column pass on one scratch tile (16 columns x N rows): forward FFT along y, error metric +
// Fourier-modulus constraint in registers, inverse FFT along y, in place.
// A < 0 marks an unmeasured pixel (beamstop): left free.  `scale` (= 1/N^2, a power
// of two) is folded into the constraint.  partial[n][ct] = sum over the tile of (|G| - A)^2.
// ------------------------------------------------------------------------------------------------
// The error metric and the constraint on a pair of pixels, branch-free.  v = G (two pixels), a = A
// of the two pixels (A < 0: unmeasured).  Returns with v = G' / N^2 and acc += (|G| - A)^2 over the
// measured ones.  |G|^2 below the smallest normal number counts as |G| = 0: phase 0, G' = A
// (reading A13; rsqrt.approx.ftz would return +inf there).
__device__ __forceinline__ float rsqrt_ftz(float x)
{
    float r;
    asm("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x));
    return r;
}
__device__ __forceinline__ void modulus_pair(c2& v, float2 a, float scale, float2& acc)
{
    const float2 m2 = pfma(v.re, v.re, pmul(v.im, v.im));
    const bool p0 = m2.x >= 1.17549435e-38f, p1 = m2.y >= 1.17549435e-38f;   // |G| > 0
    const bool k0 = a.x >= 0.f, k1 = a.y >= 0.f;                              // measured
    float2 rs = make_float2(rsqrt_ftz(m2.x), rsqrt_ftz(m2.y));
    const float2 h = pmul(pmul(m2, bc(0.5f)), rs);                            // one Newton step: ~1 ulp
    rs = pfma(rs, pfma(neg2(h), rs, bc(0.5f)), rs);
    rs.x = p0 ? rs.x : 1.f;
    rs.y = p1 ? rs.y : 1.f;
    v.re.x = p0 ? v.re.x : 1.f;                                               // |G| = 0: G / |G| := (1, 0)
    v.re.y = p1 ? v.re.y : 1.f;
    const float2 mag = pmul(make_float2(p0 ? m2.x : 0.f, p1 ? m2.y : 0.f), rs);
    float2 d = psub(mag, a);
    d.x = k0 ? d.x : 0.f;
    d.y = k1 ? d.y : 0.f;
    acc = pfma(d, d, acc);
    float2 f = pmul(pmul(a, rs), bc(scale));                                   // G' = A G / |G|
    f.x = k0 ? f.x : scale;                                                    // unmeasured: G' = G
    f.y = k1 ? f.y : scale;
    // an unmeasured pixel with |G| = 0 stays 0 (v.re was set to 1 above)
    v.re.x = (k0 || p0) ? v.re.x : 0.f;
    v.re.y = (k1 || p1) ? v.re.y : 0.f;
    v.re = pmul(v.re, f);
    v.im = pmul(v.im, f);
}

template <int N, int MODE>
__global__ void __launch_bounds__(Radix<N>::NT, Radix<N>::MINB)
k_col(float4* __restrict__ scr, const float* __restrict__ Aperm, const float2* __restrict__ twg,
      double* __restrict__ partial, int n0, float scale)
{
    using RX = Radix<N>;
    constexpr int TBN = tile_batch<N>(), NP = tile_pairs<N>();
    constexpr int NT = RX::NT, NCT = N / TBN, RL = last_radix<N>();
    extern __shared__ __align__(128) float4 sm[];
    __shared__ float red[32];   // per-warp error sums of the tile
    const Smem<N> s(sm);
    float4* __restrict__ tile = s.tile;
    const int n = n0 + (int)(blockIdx.x / (unsigned)NCT);
    const int ct = (int)(blockIdx.x % (unsigned)NCT);
    float4* __restrict__ g = scr + ((size_t)n * NCT + ct) * tile_quads<N>();

    if (threadIdx.x == 0) mbar_init(s.bar, 1);
    __syncthreads();
    if (threadIdx.x == 0) {
        mbar_expect_tx(s.bar, tile_bytes<N>() + tw_bytes<N>());
        bulk_load(tile, g, tile_bytes<N>(), s.bar);
        bulk_load(const_cast<float2*>(s.tw0), twg, tw_bytes<N>(), s.bar);
    }
    if constexpr (MODE == COL_FULL) {
        // sqrt(I) of this tile (one contiguous chunk, read by the fused middle stage) is requested
        // into L2 now: it arrives while the forward stages run
        const char* pf = reinterpret_cast<const char*>(Aperm + ((size_t)n * NCT + ct) * N * TBN);
        for (int l = threadIdx.x; l < N * TBN * 4 / 128; l += NT) asm volatile("prefetch.global.L2 [%0];" ::"l"(pf + (size_t)l * 128));
    }
    mbar_wait(s.bar, 0);

    const int par = ct & 1;   // see ppos
    auto ld_s = [&](int p, int j) -> c2 { return from_quad(tile[ppos(p, TBN, par) * NP + sw(j, p, NP)]); };
    auto st_s = [&](int p, int j, c2 v) { st_quad(tile + ppos(p, TBN, par) * NP + sw(j, p, NP), v); };

    constexpr bool FAST = inner_stages_warp_local<N>();   // 8-wide, inner radices 8 x 8: affine offsets
    if constexpr (MODE == COL_FULL || MODE == COL_FWD || MODE == COL_GAUSS) {
        if constexpr (FAST) stage0_8<N, false, true, NT>(tile, s.tw0, par);
        else fft_stage<N, RX::R0, N, false, NT, 1>(s.tw0, ld_s, st_s);
        __syncthreads();
        if constexpr (RX::S == 3) {
            if constexpr (FAST) stage1_8<N, false, true, NT>(tile, s.tw1, par);
            else fft_stage<N, RX::R1, N / RX::R0, false, NT, 1>(s.tw1, ld_s, st_s);
            inner_sync<N>();
        }
    }
    if constexpr (MODE == COL_FWD) {
        fft_stage<N, RL, RL, false, NT, 1>(s.tw0, ld_s, st_s);
    }
    if constexpr (MODE == COL_FULL) {
        const float* __restrict__ At = Aperm + ((size_t)n * NCT + ct) * N * TBN;
        float2 acc2 = make_float2(0.f, 0.f);
        auto pw = [&](c2 (&v)[RL], int q, int j) {
            const float4* __restrict__ a4 = reinterpret_cast<const float4*>(At + (size_t)(q * NP + j) * (2 * RL));
            float2 a[RL];
#pragma unroll
            for (int r = 0; r < RL / 2; ++r) {
                const float4 t = __ldg(a4 + r);
                a[2 * r] = make_float2(t.x, t.y);
                a[2 * r + 1] = make_float2(t.z, t.w);
            }
#pragma unroll
            for (int r = 0; r < RL; ++r) modulus_pair(v[r], a[r], scale, acc2);
        };
        if constexpr (FAST) {
            constexpr int NBF = NP * (N / RL), ITERS = (NBF + NT - 1) / NT;
#pragma unroll 1
            for (int it = 0; it < ITERS; ++it) {
                const int bf = (int)threadIdx.x + it * NT, j = bf % NP, q = bf / NP;
                const Last8<true> at(tile, q, j, par);
                c2 v[RL];
#pragma unroll
                for (int r = 0; r < RL; ++r) v[r] = from_quad(*at(r));
                dft<RL, false>(v);
                pw(v, q, j);
                dft<RL, true>(v);
#pragma unroll
                for (int r = 0; r < RL; ++r) st_quad(at(r), v[r]);
            }
        } else {
            fft_stage_mid<N, RL, NT, 1>(ld_s, pw, st_s);
        }
        float acc = acc2.x + acc2.y;
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, o);
        if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = acc;
    }
    if constexpr (MODE == COL_GAUSS) {
        // the pointwise step of the blur: Aperm is a table of N floats over the scratch POSITIONS here, the factor of
        // element (row position py, column position px) is tab[py] tab[px] (cpra_shrinkwrap; reading A23)
        const float* __restrict__ tab = Aperm;
        auto pw = [&](c2 (&v)[RL], int q, int j) {
            const float2 fx = __ldg(reinterpret_cast<const float2*>(tab + ct * TBN + 2 * j));
#pragma unroll
            for (int r = 0; r < RL; ++r) {
                const float fy = __ldg(tab + q * RL + r);
                const float2 f = make_float2(fy * fx.x, fy * fx.y);
                v[r].re = pmul(v[r].re, f);
                v[r].im = pmul(v[r].im, f);
            }
        };
        if constexpr (FAST) {
            constexpr int NBF = NP * (N / RL), ITERS = (NBF + NT - 1) / NT;
#pragma unroll 1
            for (int it = 0; it < ITERS; ++it) {
                const int bf = (int)threadIdx.x + it * NT, j = bf % NP, q = bf / NP;
                const Last8<true> at(tile, q, j, par);
                c2 v[RL];
#pragma unroll
                for (int r = 0; r < RL; ++r) v[r] = from_quad(*at(r));
                dft<RL, false>(v);
                pw(v, q, j);
                dft<RL, true>(v);
#pragma unroll
                for (int r = 0; r < RL; ++r) st_quad(at(r), v[r]);
            }
        } else {
            fft_stage_mid<N, RL, NT, 1>(ld_s, pw, st_s);
        }
    }
    if constexpr (MODE == COL_INV) fft_stage<N, RL, RL, true, NT, 1>(s.tw0, ld_s, st_s);
    if constexpr (MODE != COL_FWD) {
        if constexpr (RX::S == 3) {
            inner_sync<N>();
            if constexpr (FAST) stage1_8<N, true, true, NT>(tile, s.tw1, par);
            else fft_stage<N, RX::R1, N / RX::R0, true, NT, 1>(s.tw1, ld_s, st_s);
        }
        __syncthreads();
        if constexpr (MODE == COL_FULL) {
            if (threadIdx.x == 0) {   // error numerator of the tile, fixed order: deterministic
                double t = 0.0;
                for (int w = 0; w < NT / 32; ++w) t += (double)red[w];
                partial[(size_t)n * NCT + ct] = t;
            }
        }
        if constexpr (FAST) stage0_8<N, true, true, NT>(tile, s.tw0, par);
        else fft_stage<N, RX::R0, N, true, NT, 1>(s.tw0, ld_s, st_s);
    }
    fence_async_smem();
    __syncthreads();
    if (threadIdx.x == 0) {
        bulk_store(g, tile, tile_bytes<N>());
        bulk_commit();
        bulk_wait_read0();
    }
}

// ------------------------------------------------------------------------------------------------
// K3: inverse FFT along x of 16 rows + support / HIO update (PAPER.md:98 ref [22], :104):
//   S = 1: g <- g';  S = 0: g <- ghat - beta g'   (ghat = the mixed input of this iteration,
// recomputed from the previous state).  Writes the new state (ping-pong buffer).
// The 16 x 16 blocks of the scratch arrive by N/16 bulk copies of 2 KiB; the first inverse stage
// transposes them into the row layout; the new state tile leaves by one bulk copy.
// ------------------------------------------------------------------------------------------------
template <int N, int MODE, int MIXMODE>
__global__ void __launch_bounds__(Radix<N>::NT, N == 1024 ? 3 : Radix<N>::MINB)   // (N = 1024: 84 registers without a cap; 80 lets a third CTA in)
k_row_inv(const __grid_constant__ CUtensorMap tm_scr, const float4* __restrict__ cur, float4* __restrict__ nxt,
          const float2* __restrict__ twg, const uint16_t* __restrict__ S16, MixParams mp, float beta,
          float scale, int Np, int n0, int nimg, const float4* __restrict__ ghat_in)
{
    using RX = Radix<N>;
    constexpr int TBN = tile_batch<N>(), NP = tile_pairs<N>();
    constexpr int NT = RX::NT, NRT = N / TBN, NCT = N / TBN, RL = last_radix<N>();
    constexpr int B = NP * (N / RL) / NT;
    constexpr bool FAST = inner_stages_warp_local<N>();   // 8-wide, inner radices 8 x 8: affine offsets
    extern __shared__ __align__(128) float4 sm[];
    const Smem<N> s(sm);
    float4* __restrict__ tile = s.tile;
    const int n = n0 + (int)(blockIdx.x % (unsigned)nimg);
    const int rt = (int)(blockIdx.x / (unsigned)nimg);
    const size_t istride = (size_t)N * N / 2;
    const size_t toff = (size_t)rt * tile_quads<N>();

    if (threadIdx.x == 0) mbar_init(s.bar, 1);
    __syncthreads();
    if (threadIdx.x == 0) {
        mbar_expect_tx(s.bar, tile_bytes<N>() + tw_bytes<N>() + (MODE == ROWINV_HIO ? 2 * N : 0));
        bulk_load(const_cast<float2*>(s.tw0), twg, tw_bytes<N>(), s.bar);
        if constexpr (MODE == ROWINV_HIO) bulk_load(s.sup, S16 + ((size_t)n * (N / 16) + (rt * TBN) / 16) * N, 2 * N, s.bar);
        tma_load_tile(tile, &tm_scr, rt, n, s.bar);
    }
    if constexpr (MODE != ROWINV_PLAIN && N >= 1024) {
        // the epilogue's own-tile loads (ghat, or the previous state it is recomputed from; the
        // neighbours' tiles are pulled in by the CTAs of n - 1 and n + 1) are requested into L2 now:
        // they arrive while the stages run.  Three CTAs per SM at N = 1024 do not hide that latency
        // (0.995 -> 0.883 ms); six at N = 512 do, and the early requests cost 15 % there.
        const char* pf = reinterpret_cast<const char*>((ghat_in ? ghat_in : cur) + (size_t)n * istride + toff);
        for (int l = threadIdx.x; l < tile_bytes<N>() / 128; l += NT) asm volatile("prefetch.global.L2 [%0];" ::"l"(pf + (size_t)l * 128));
    }
    mbar_wait(s.bar, 0);

    auto ld_s = [&](int p, int j) -> c2 { return from_quad(tile[ppos<N>(p) * NP + j]); };
    auto st_s = [&](int p, int j, c2 v) { st_quad(tile + ppos<N>(p) * NP + j, v); };

    // first inverse stage (contiguous positions, no twiddles), reading the scratch layout
    {
        c2 v[B][RL];
#pragma unroll
        for (int b = 0; b < B; ++b) {
            const int bf = (int)threadIdx.x + b * NT;
            load_transposed<N>(tile, v[b], bf / NP, bf % NP, rt);
            dft<RL, true>(v[b]);
        }
        inner_sync<N>();
#pragma unroll
        for (int b = 0; b < B; ++b) {
            const int bf = (int)threadIdx.x + b * NT, j = bf % NP, q = bf / NP;
            if constexpr (FAST) {
                const Last8<false> at(tile, q, j);
#pragma unroll
                for (int r = 0; r < RL; ++r) st_quad(at(r), v[b][r]);
            } else {
#pragma unroll
                for (int r = 0; r < RL; ++r) st_s(q * RL + r, j, v[b][r]);
            }
        }
    }
    inner_sync<N>();
    if constexpr (RX::S == 3) {
        if constexpr (FAST) stage1_8<N, true, false, NT>(tile, s.tw1);
        else fft_stage<N, RX::R1, N / RX::R0, true, NT, 1>(s.tw1, ld_s, st_s);
        __syncthreads();
    }
    if constexpr (FAST) stage0_8<N, true, false, NT>(tile, s.tw0);
    else fft_stage<N, RX::R0, N, true, NT, 1>(s.tw0, ld_s, st_s);
    __syncthreads();

    // epilogue over the quads of the tile: each thread rewrites its own quads in place
    if constexpr (MODE == ROWINV_PLAIN) {
        for (int i = threadIdx.x; i < tile_quads<N>(); i += NT) {
            float4 v = tile[i];
            v.x *= scale; v.y *= scale; v.z *= scale; v.w *= scale;
            tile[i] = v;
        }
    } else {
        const MixLoader<MIXMODE> mix(cur, istride, n, Np, mp, N, TBN);
        const float4* __restrict__ own = cur + (size_t)n * istride + toff;
#pragma unroll 4
        for (int i = threadIdx.x; i < tile_quads<N>(); i += NT) {
            const int x = ppos<N>(i / NP), j = i % NP;   // i runs over the physical quads of the tile
            unsigned bits = (unsigned)s.sup[x] >> ((rt * TBN) % 16 + 2 * j);
            // ghat: stored by k_row_fwd / k_row_walk (ghat_in), else recomputed from the previous state
            const c2 gh = ghat_in ? from_quad(__ldg(ghat_in + (size_t)n * istride + toff + i))
                                  : mix(from_quad(__ldg(own + i)), toff + (size_t)i);
            const c2 gp = from_quad(tile[i]);
            bits = inside_bits(mp, bits, gp.re);
            const float2 ore = update_outside(mp, gp.re, gh.re), oim = update_outside(mp, gp.im, gh.im);
            float4 o;
            o.x = (bits & 1) ? gp.re.x : ore.x;
            o.y = (bits & 2) ? gp.re.y : ore.y;
            o.z = (bits & 1) ? gp.im.x : oim.x;
            o.w = (bits & 2) ? gp.im.y : oim.y;
            tile[i] = o;
        }
    }
    fence_async_smem();
    __syncthreads();
    if (threadIdx.x == 0) {
        bulk_store(nxt + (size_t)n * istride + toff, tile, tile_bytes<N>());
        bulk_commit();
        bulk_wait_read0();
    }
}

// ------------------------------------------------------------------------------------------------
// f3: the z pass of the 3D transform of Step D ("3D FTs as a set of 2D
// FTs"): the 2D transforms of the N slices run through the loop's own row / column kernels; this kernel
// transforms the z lines of a natural-order cube vol[z][y][x] in place.  One CTA = TB columns x at one y:
// an [N][TB/2] tile of quads, the same stages as k_col; the forward transform leaves X[k] at position
// pos(k), so the store (forward) / load (inverse) goes through fft_pos.  One-shot, not on the timed path.
// ------------------------------------------------------------------------------------------------
template <int N, bool INV>
__global__ void __launch_bounds__(Radix<N>::NT)
k_fft_z(float2* __restrict__ vol, const float2* __restrict__ twg, float scale)
{
    using RX = Radix<N>;
    constexpr int TBN = tile_batch<N>(), NP = tile_pairs<N>(), NT = RX::NT, RL = last_radix<N>();
    extern __shared__ __align__(128) float4 sm[];
    float4* __restrict__ tile = sm;
    float2* tw0 = reinterpret_cast<float2*>(sm + tile_quads<N>());
    const float2* tw1 = tw0 + tw_count_stage0<N>();
    const int y = blockIdx.y, x0 = blockIdx.x * TBN;
    float4* __restrict__ v4 = reinterpret_cast<float4*>(vol);   // two complex numbers (re_a, im_a, re_b, im_b)
    for (int i = threadIdx.x; i < tw_count<N>(); i += NT) tw0[i] = twg[i];
    // all of a thread's loads are issued before the first is used (N NP / NT = 16 at N = 512: two batches of 8)
    constexpr int PER = N * NP / NT, UB = PER % 8 == 0 ? 8 : (PER % 4 == 0 ? 4 : 1);
    static_assert(PER * NT == N * NP, "whole loads per thread");
    for (int b = 0; b < PER; b += UB) {
        float4 a[UB];
#pragma unroll
        for (int u = 0; u < UB; ++u) {
            const int i = (int)threadIdx.x + (b + u) * NT, z = i / NP, j = i % NP;
            a[u] = v4[(((size_t)z * N + y) * N + x0) / 2 + j];
        }
#pragma unroll
        for (int u = 0; u < UB; ++u) {
            const int i = (int)threadIdx.x + (b + u) * NT, z = i / NP, j = i % NP;
            tile[(INV ? fft_pos(z, RX::R0, RX::R1, RX::R2) : z) * NP + j] = make_float4(a[u].x, a[u].z, a[u].y, a[u].w);
        }
    }
    __syncthreads();
    auto ld_s = [&](int p, int j) -> c2 { return from_quad(tile[p * NP + j]); };
    auto st_s = [&](int p, int j, c2 v) { st_quad(tile + p * NP + j, v); };
    if constexpr (!INV) {
        fft_stage<N, RX::R0, N, false, NT, 1>(tw0, ld_s, st_s);
        __syncthreads();
        if constexpr (RX::S == 3) { fft_stage<N, RX::R1, N / RX::R0, false, NT, 1>(tw1, ld_s, st_s); __syncthreads(); }
        fft_stage<N, RL, RL, false, NT, 1>(tw0, ld_s, st_s);
    } else {
        fft_stage<N, RL, RL, true, NT, 1>(tw0, ld_s, st_s);
        __syncthreads();
        if constexpr (RX::S == 3) { fft_stage<N, RX::R1, N / RX::R0, true, NT, 1>(tw1, ld_s, st_s); __syncthreads(); }
        fft_stage<N, RX::R0, N, true, NT, 1>(tw0, ld_s, st_s);
    }
    __syncthreads();
    for (int i = threadIdx.x; i < N * NP; i += NT) {
        const int z = i / NP, j = i % NP;
        const float4 q = tile[(INV ? z : fft_pos(z, RX::R0, RX::R1, RX::R2)) * NP + j];
        v4[(((size_t)z * N + y) * N + x0) / 2 + j] = make_float4(q.x * scale, q.z * scale, q.y * scale, q.w * scale);
    }
}

// The same z pass on a cube kept in the loop's own layouts (Step D's iterations, cpra_refine_3d): plane z of the cube is
// image z of the column-tiled scratch, so the z line of (column tile ct, scratch row `row`, pair j) is the quad
// scr[((z NCT + ct) N + row) NP + j], z = 0 .. N-1: the tile [z][NP] arrives as quads already.  The forward pass leaves
// frequency kz in plane pos(kz) and the inverse pass expects it there: the cube's planes stay in position order between
// the two, so nothing is permuted.  grid = (N rows, N / TB column tiles).
template <int N, bool INV>
__global__ void __launch_bounds__(Radix<N>::NT)
k_fft_z_scr(float4* __restrict__ scr, const float2* __restrict__ twg, float scale)
{
    using RX = Radix<N>;
    constexpr int TBN = tile_batch<N>(), NP = tile_pairs<N>(), NT = RX::NT, RL = last_radix<N>(), NCT = N / TBN;
    extern __shared__ __align__(128) float4 sm[];
    float4* __restrict__ tile = sm;
    float2* tw0 = reinterpret_cast<float2*>(sm + tile_quads<N>());
    const float2* tw1 = tw0 + tw_count_stage0<N>();
    const size_t plane = (size_t)NCT * N * NP;                                  // quads per plane
    float4* __restrict__ line = scr + ((size_t)blockIdx.y * N + blockIdx.x) * NP;   // (ct = blockIdx.y, row = blockIdx.x), plane 0
    for (int i = threadIdx.x; i < tw_count<N>(); i += NT) tw0[i] = twg[i];
    constexpr int PER = N * NP / NT, UB = PER % 8 == 0 ? 8 : (PER % 4 == 0 ? 4 : 1);
    static_assert(PER * NT == N * NP, "whole loads per thread");
    for (int b = 0; b < PER; b += UB) {
        float4 a[UB];
#pragma unroll
        for (int u = 0; u < UB; ++u) {
            const int i = (int)threadIdx.x + (b + u) * NT;
            a[u] = line[(size_t)(i / NP) * plane + i % NP];
        }
#pragma unroll
        for (int u = 0; u < UB; ++u) tile[(int)threadIdx.x + (b + u) * NT] = a[u];
    }
    __syncthreads();
    auto ld_s = [&](int p, int j) -> c2 { return from_quad(tile[p * NP + j]); };
    auto st_s = [&](int p, int j, c2 v) { st_quad(tile + p * NP + j, v); };
    if constexpr (!INV) {
        fft_stage<N, RX::R0, N, false, NT, 1>(tw0, ld_s, st_s);
        __syncthreads();
        if constexpr (RX::S == 3) { fft_stage<N, RX::R1, N / RX::R0, false, NT, 1>(tw1, ld_s, st_s); __syncthreads(); }
        fft_stage<N, RL, RL, false, NT, 1>(tw0, ld_s, st_s);
    } else {
        fft_stage<N, RL, RL, true, NT, 1>(tw0, ld_s, st_s);
        __syncthreads();
        if constexpr (RX::S == 3) { fft_stage<N, RX::R1, N / RX::R0, true, NT, 1>(tw1, ld_s, st_s); __syncthreads(); }
        fft_stage<N, RX::R0, N, true, NT, 1>(tw0, ld_s, st_s);
    }
    __syncthreads();
    for (int i = threadIdx.x; i < N * NP; i += NT) {
        const float4 q = tile[i];
        line[(size_t)(i / NP) * plane + i % NP] = make_float4(q.x * scale, q.y * scale, q.z * scale, q.w * scale);
    }
}

}  // namespace cpra
