// cpra_fft.cuh -- register / shared-memory FFT building blocks of the CPRA loop (sm_100a, complex fp32).
//
// The 2D FTs of the "conventional 2D CXDI" iteration (the N^2 log N term of
// PAPER.md:74) are done as 1D FFTs of length N along the SLOW index of a [N][16] tile whose fast
// index is a batch of 16 independent transforms (16 rows for the row pass, 16 columns for the
// column pass).
//
// Packed arithmetic: a thread owns a PAIR of batch members (a, b) and keeps them as
//     c2 = { re = (re_a, re_b), im = (im_a, im_b) }
// so that every add / multiply / fma of the butterflies is one sm_100 packed instruction
// (FADD2 / FMUL2 / FFMA2: two fp32 results per issue slot, negation and broadcast immediates free).
// The same 16 bytes [re_a, re_b, im_a, im_b] ("quad") are the unit of every shared-memory and
// global-memory layout of the loop: a position of the tile is 8 quads = 128 B, a quarter-warp of
// LDS.128 / STS.128 reads one whole position, so every stage is bank-conflict free for any stride.
//
// Forward: in-place decimation-in-frequency, radices R0, R1[, R2] (first stage has stride N/R0),
//          natural order in, digit-reversed order out:  X[k] ends at position pos(k),
//          k = k0 + R0 (k1 + R1 k2)  ->  pos = k2 + R2 (k1 + R1 k0).
// Inverse: the mirror image (decimation-in-time), digit-reversed in, natural out.
// Each butterfly reads and writes the SAME R positions, so a stage needs one barrier and the last
// forward stage / pointwise step / first inverse stage fuse in registers.  The pointwise steps of
// the loop never need natural frequency order: sqrt(I) is stored once in the permuted order.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace cpra {

constexpr int TB = 16;     // tile width = batch of transforms (Radix<N>::TB: 8 at N = 1024, so that a tile is 64 KiB)
constexpr int NPAIR = 8;   // batch pairs = quads per position (Radix<N>::TB / 2)

// ---- stage plan ------------------------------------------------------------------------------
// NT = threads per CTA, chosen so that the last stage has NPAIR * N / RL = B * NT butterflies with
// B in {1, 2}: the transposing stage of the row kernels keeps all of them in registers.  MINB = CTAs
// per SM the register allocation is held to (shared memory allows that many).  PF: k_row_fwd
// requests the neighbours' share of the mix for all its first-stage butterflies before it waits for its
// own tile (MINBF = its CTAs per SM: the prefetch needs 2 x 32 more registers).  N = 1024: three CTAs
// N = 256 runs the 8-wide 4 x 8 x 8 plan (16 KiB tiles, k_row_walk: 146 -> 120 us per iteration at N_p = 180).  The
// same 2 x 8 x 8 plan at N = 128 measured 36.9 us against 45.1 us for the whole-image kernel at N_p = 180 and
// 24.6 against 24.6 at N_p = 90 (config 2); N = 128 stays on the image-resident kernel (cpra_image.cuh).
// N = 1024: three CTAs of 256 threads (85 registers, 64 KiB tiles) beat two without a cap (k_col 112 -> 40 B of spills,
// k_row_fwd 128 -> 4 B): 2.498 -> 2.291 ms per iteration at N_p = 180; five instead of four at N = 256: no gain.
template <int N> struct Radix;
template <> struct Radix<16>   { static constexpr int TB = 16, S = 2, R0 = 4,  R1 = 4,  R2 = 1, NT = 32,  MINB = 8; static constexpr bool PF = false; static constexpr int MINBF = MINB; };
template <> struct Radix<32>   { static constexpr int TB = 16, S = 2, R0 = 8,  R1 = 4,  R2 = 1, NT = 64,  MINB = 8; static constexpr bool PF = false; static constexpr int MINBF = MINB; };
template <> struct Radix<64>   { static constexpr int TB = 16, S = 2, R0 = 8,  R1 = 8,  R2 = 1, NT = 64,  MINB = 8; static constexpr bool PF = false; static constexpr int MINBF = MINB; };
template <> struct Radix<128>  { static constexpr int TB = 16, S = 2, R0 = 8,  R1 = 16, R2 = 1, NT = 64,  MINB = 6; static constexpr bool PF = false; static constexpr int MINBF = MINB; };
template <> struct Radix<256>  { static constexpr int TB = 8, S = 3, R0 = 4,  R1 = 8,  R2 = 8, NT = 128, MINB = 8; static constexpr bool PF = false; static constexpr int MINBF = MINB; };
template <> struct Radix<512>  { static constexpr int TB = 8, S = 3, R0 = 8,  R1 = 8,  R2 = 8, NT = 128, MINB = 6; static constexpr bool PF = true; static constexpr int MINBF = 4; };
template <> struct Radix<1024> { static constexpr int TB = 8, S = 3, R0 = 16, R1 = 8,  R2 = 8, NT = 256, MINB = 3; static constexpr bool PF = false; static constexpr int MINBF = MINB; };

template <int N> __host__ __device__ constexpr int tile_batch() { return Radix<N>::TB; }
template <int N> __host__ __device__ constexpr int tile_pairs() { return Radix<N>::TB / 2; }
template <int N> __host__ __device__ constexpr int last_radix() { return Radix<N>::S == 3 ? Radix<N>::R2 : Radix<N>::R1; }

// position of frequency k after the forward transform (runtime radices: used by layout kernels)
__host__ __device__ __forceinline__ int fft_pos(int k, int R0, int R1, int R2)
{
    const int k0 = k % R0, k1 = (k / R0) % R1, k2 = k / (R0 * R1);
    return k2 + R2 * (k1 + R1 * k0);
}

// ---- twiddle tables ----------------------------------------------------------------------------
// One table per stage with M = L / R > 1, entry (n2, r) for r = 1 .. R-1 at index
// n2 (R - 1) + (r - 1):  (wr, wi),  w = exp(-2 pi i n2 r / L)  (computed in double, rounded once, on
// the host).  Stage 0 (L = N) first, then stage 1 (L = N / R0) if the plan has 3 stages.  A twiddle
// is one 64-bit shared-memory load; the packed instructions take wr and wi as scalar operands that
// the hardware broadcasts to both halves (SASS "R12.F32"), so no duplicated copy is stored or built.
template <int N> __host__ __device__ constexpr int tw_count_stage0() { return (N / Radix<N>::R0) * (Radix<N>::R0 - 1); }
template <int N> __host__ __device__ constexpr int tw_count_stage1()
{
    return Radix<N>::S == 3 ? (N / (Radix<N>::R0 * Radix<N>::R1)) * (Radix<N>::R1 - 1) : 0;
}
template <int N> __host__ __device__ constexpr int tw_count() { return tw_count_stage0<N>() + tw_count_stage1<N>(); }

// ---- packed helpers ----------------------------------------------------------------------------
struct c2 {
    float2 re, im;
};

__device__ __forceinline__ float2 bc(float a) { return make_float2(a, a); }
__device__ __forceinline__ float2 neg2(float2 a) { return make_float2(-a.x, -a.y); }
__device__ __forceinline__ float2 padd(float2 a, float2 b) { return __fadd2_rn(a, b); }
__device__ __forceinline__ float2 psub(float2 a, float2 b) { return __fadd2_rn(a, neg2(b)); }
__device__ __forceinline__ float2 pmul(float2 a, float2 b) { return __fmul2_rn(a, b); }
__device__ __forceinline__ float2 pfma(float2 a, float2 b, float2 c) { return __ffma2_rn(a, b, c); }

__device__ __forceinline__ c2 from_quad(float4 q) { return c2{make_float2(q.x, q.y), make_float2(q.z, q.w)}; }
__device__ __forceinline__ float4 to_quad(c2 v) { return make_float4(v.re.x, v.re.y, v.im.x, v.im.y); }
// store one quad to shared memory as two 64-bit halves: the packed results live in separate
// register pairs, and a 128-bit store would first have to gather them into four consecutive registers
__device__ __forceinline__ void st_quad(float4* q, c2 v)
{
    const uint32_t a = (uint32_t)__cvta_generic_to_shared(q);
    asm volatile("st.shared.v2.f32 [%0], {%1, %2};" ::"r"(a), "f"(v.re.x), "f"(v.re.y) : "memory");
    asm volatile("st.shared.v2.f32 [%0+8], {%1, %2};" ::"r"(a), "f"(v.im.x), "f"(v.im.y) : "memory");
}

__device__ __forceinline__ c2 cadd(c2 a, c2 b) { return c2{padd(a.re, b.re), padd(a.im, b.im)}; }
__device__ __forceinline__ c2 csub(c2 a, c2 b) { return c2{psub(a.re, b.re), psub(a.im, b.im)}; }
// a * w, w = (wr, wi) broadcast pairs
__device__ __forceinline__ c2 cmul(c2 a, float2 wr, float2 wi)
{
    return c2{pfma(a.re, wr, neg2(pmul(a.im, wi))), pfma(a.re, wi, pmul(a.im, wr))};
}
// a * conj(w)
__device__ __forceinline__ c2 cmulc(c2 a, float2 wr, float2 wi)
{
    return c2{pfma(a.re, wr, pmul(a.im, wi)), pfma(a.im, wr, neg2(pmul(a.re, wi)))};
}

// lo = e + W o, hi = e - W o with W = exp(-+ 2 pi i q / 16)  (- forward, + inverse); q is a
// compile-time constant after unrolling
template <bool INV>
__device__ __forceinline__ void tw_addsub(c2 e, c2 o, int q, c2& lo, c2& hi)
{
    constexpr float H = 0.70710678118654752440f;
    constexpr float C1 = 0.92387953251128675613f, S1 = 0.38268343236508977173f;
    if (q == 0) {
        lo = cadd(e, o);
        hi = csub(e, o);
    } else if (q == 4) {
        // forward W = -i: W o = (o.im, -o.re);  inverse W = +i: W o = (-o.im, o.re)
        const c2 p{padd(e.re, o.im), psub(e.im, o.re)};
        const c2 m{psub(e.re, o.im), padd(e.im, o.re)};
        lo = INV ? m : p;
        hi = INV ? p : m;
    } else if (q == 2 || q == 6) {
        // q = 2: W = (1 -+ i) H;  q = 6: W = (-1 -+ i) H
        const float2 s = padd(o.re, o.im), d = psub(o.im, o.re);   // o.re + o.im, o.im - o.re
        float2 tr, ti;   // W o = H (tr, ti)
        if (q == 2) { tr = INV ? neg2(d) : s;  ti = INV ? s : d; }
        else        { tr = INV ? neg2(s) : d;  ti = INV ? neg2(d) : neg2(s); }
        lo = c2{pfma(tr, bc(H), e.re), pfma(ti, bc(H), e.im)};
        hi = c2{pfma(tr, bc(-H), e.re), pfma(ti, bc(-H), e.im)};
    } else {
        // q = 1, 3, 5, 7: W = c -+ i s with c = cos(2 pi q / 16), s = sin(2 pi q / 16)
        const float c = (q == 1) ? C1 : (q == 3) ? S1 : (q == 5) ? -S1 : -C1;
        const float s0 = (q == 1 || q == 7) ? S1 : C1;
        const float s = INV ? -s0 : s0;
        // W o = (o.re c + o.im s, o.im c - o.re s)
        const float2 tr = pfma(o.re, bc(c), pmul(o.im, bc(s)));
        const float2 ti = pfma(o.im, bc(c), neg2(pmul(o.re, bc(s))));
        lo = c2{padd(e.re, tr), padd(e.im, ti)};
        hi = c2{psub(e.re, tr), psub(e.im, ti)};
    }
}

// ---- radix-R DFT in registers, natural order in and out ----------------------------------------
template <int R, bool INV>
__device__ __forceinline__ void dft(c2 (&v)[R])
{
    if constexpr (R == 2) {
        const c2 a = v[0];
        v[0] = cadd(a, v[1]);
        v[1] = csub(a, v[1]);
    } else {
        c2 e[R / 2], o[R / 2];
#pragma unroll
        for (int k = 0; k < R / 2; ++k) { e[k] = v[2 * k]; o[k] = v[2 * k + 1]; }
        dft<R / 2, INV>(e);
        dft<R / 2, INV>(o);
#pragma unroll
        for (int k = 0; k < R / 2; ++k) tw_addsub<INV>(e[k], o[k], k * (16 / R), v[k], v[k + R / 2]);
    }
}

// twiddle the R values of a butterfly: forward after the DFT (times w), inverse before it (times
// conj w); tws = this stage's table in shared memory, n2 = the butterfly's index inside its block
template <int R, bool INV>
__device__ __forceinline__ void twiddle(c2 (&v)[R], const float2* __restrict__ tws, int n2)
{
    const float2* __restrict__ t = tws + n2 * (R - 1);
#pragma unroll
    for (int r = 1; r < R; ++r) {
        const float2 w = t[r - 1];
        v[r] = INV ? cmulc(v[r], bc(w.x), bc(w.y)) : cmul(v[r], bc(w.x), bc(w.y));
    }
}

// ---- one in-place stage over a [N][NPAIR] tile of quads -------------------------------------------
// Sub-transform length L, radix R, M = L/R: butterfly (blk, n2) touches positions blk L + n2 + M r.
// ld(pos, j) / st(pos, j, value) move one quad of batch pair j.
template <int N, int R, int L, bool INV, int NT, int UNROLL, class LD, class ST>
__device__ __forceinline__ void fft_stage(const float2* __restrict__ tws, LD ld, ST st)
{
    constexpr int M = L / R, NP = tile_pairs<N>();
    constexpr int NBF = NP * (N / R);
    constexpr int ITERS = (NBF + NT - 1) / NT;
#pragma unroll UNROLL
    for (int it = 0; it < ITERS; ++it) {
        const int bf = (int)threadIdx.x + it * NT;
        if ((NBF % NT) != 0 && bf >= NBF) break;
        const int j = bf % NP, q = bf / NP;
        const int blk = q / M, n2 = q % M;
        const int base = blk * L + n2;
        c2 v[R];
#pragma unroll
        for (int r = 0; r < R; ++r) v[r] = ld(base + M * r, j);
        if constexpr (INV && M > 1) twiddle<R, true>(v, tws, n2);
        dft<R, INV>(v);
        if constexpr (!INV && M > 1) twiddle<R, false>(v, tws, n2);
#pragma unroll
        for (int r = 0; r < R; ++r) st(base + M * r, j, v[r]);
    }
}

// Last forward stage (L = R, contiguous positions R q + r) + pointwise step + first inverse stage,
// fused in registers.  pw(v, q, j) edits the R values in place.
template <int N, int R, int NT, int UNROLL, class LD, class PW, class ST>
__device__ __forceinline__ void fft_stage_mid(LD ld, PW pw, ST st)
{
    constexpr int NP = tile_pairs<N>();
    constexpr int NBF = NP * (N / R);
    constexpr int ITERS = (NBF + NT - 1) / NT;
#pragma unroll UNROLL
    for (int it = 0; it < ITERS; ++it) {
        const int bf = (int)threadIdx.x + it * NT;
        if ((NBF % NT) != 0 && bf >= NBF) break;
        const int j = bf % NP, q = bf / NP;
        c2 v[R];
#pragma unroll
        for (int r = 0; r < R; ++r) v[r] = ld(q * R + r, j);
        dft<R, false>(v);
        pw(v, q, j);
        dft<R, true>(v);
#pragma unroll
        for (int r = 0; r < R; ++r) st(q * R + r, j, v[r]);
    }
}

// ---- asynchronous bulk copies (TMA 1D; SASS: UBLKCP) and their mbarrier -----------------------------
__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void mbar_init(uint64_t* bar, uint32_t count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint64_t* bar, uint32_t bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t* bar, uint32_t parity)
{
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "WAIT_%=:\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
        "@p bra DONE_%=;\n"
        "bra WAIT_%=;\n"
        "DONE_%=:\n"
        "}\n" ::"r"(smem_u32(bar)), "r"(parity) : "memory");
}
// global -> shared, completion counted in bytes on the mbarrier; 16 B aligned, bytes % 16 == 0
__device__ __forceinline__ void bulk_load(void* smem_dst, const void* gsrc, uint32_t bytes, uint64_t* bar)
{
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                 ::"r"(smem_u32(smem_dst)), "l"(gsrc), "r"(bytes), "r"(smem_u32(bar)) : "memory");
}
// shared -> global (bulk async group)
__device__ __forceinline__ void bulk_store(void* gdst, const void* smem_src, uint32_t bytes)
{
    asm volatile("cp.async.bulk.global.shared::cta.bulk_group [%0], [%1], %2;"
                 ::"l"(gdst), "r"(smem_u32(smem_src)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void bulk_commit() { asm volatile("cp.async.bulk.commit_group;" ::: "memory"); }
__device__ __forceinline__ void bulk_wait_read0() { asm volatile("cp.async.bulk.wait_group.read 0;" ::: "memory"); }
// make generic-proxy shared-memory writes visible to the async proxy (before a bulk store)
__device__ __forceinline__ void fence_async_smem() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }

}  // namespace cpra
