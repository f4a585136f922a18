// cpra_walk.cuh -- K3 of iteration t fused with K1 of iteration t + 1 in a CTA that WALKS along n
// (sm_100a; plans with 8-row tiles: a tile is N x 64 B = 16 / 32 / 64 KiB at N = 256 / 512 / 1024).
//
// The carousel mix (Eq. (4)) needs the NEW states of projections n-1, n, n+1.  A CTA
// that owns a run of consecutive n for one row tile rt keeps the last three new tiles in shared
// memory (3 slots), so the mix reads no neighbour from L2 or HBM at all, and the forward row FFT of
// iteration t + 1 follows the support / HIO update of iteration t without the state ever being
// written as g:
//     A(i):  spectrum tile of projection m_i (after the column pass)  --bulk copies-->  slot i % 3
//            inverse FFT along x, in place; the last stage stays in registers:
//            g_new = S ? g' : ghat_old - beta g'   (ghat_old = the mixed input of iteration t, stored
//            by the previous walk: ONE 128-bit load per quad, requested before the tile is waited for)
//            g_new goes back to the slot and stays in the registers v
//     B(i):  ghat_new(m_i) = a0 g_new(m_i) + a1 (g_new(m_{i-1}) + g_new(m_{i+1})):  m_{i-1} from the
//            registers gm, m_i from slot i % 3, m_{i+1} from v (A(i+1) ran just before); stored for the
//            next HIO; forward FFT along x in place in slot i % 3, transposed, bulk-stored into the
//            OTHER scratch buffer; then the tile of m_{i+3} is loaded into that slot: it is needed
//            a whole step later, so its latency is covered.
// HBM traffic of a walk: spectrum in 8 + ghat_old 8 + support 1/8 + ghat_new 8 + spectrum out 8 =
// 32.125 B/px, against 16 + 24.125 for K1 + K3, and no neighbour loads.  The two tiles next to a run
// (halo) are inverse-transformed twice (by this CTA and by their owner): the spectra are therefore
// read from one scratch buffer and written to the other.
#pragma once
#include "cpra_kernels.cuh"

namespace cpra {

template <int N> __host__ __device__ constexpr bool walk_ok() { return tile_batch<N>() == 8 && Radix<N>::S == 3 && N <= 1024; }
// CTAs per SM that the three slots allow (N = 1024: 3 x 64 KiB, one CTA of 512 threads)
template <int N> __host__ __device__ constexpr int walk_ctas_per_sm() { return N >= 1024 ? 1 : (N >= 512 ? 2 : 4); }
constexpr int WALK_SLOTS = 3;
// slots + twiddles + 3 mbarriers + support words of the 3 slots
template <int N> __host__ __device__ constexpr int walk_smem_bytes()
{
    return WALK_SLOTS * tile_bytes<N>() + tw_bytes<N>() + 32 + WALK_SLOTS * 2 * N;
}
template <int N> __host__ __device__ constexpr int walk_threads() { return tile_pairs<N>() * (N / last_radix<N>()); }

// N = 1024: the two threads (lanes l, l ^ 8) that share a radix-16 first-stage butterfly
__device__ __forceinline__ c2 walk_xchg(c2 a)   // the partner's value
{
    return c2{make_float2(__shfl_xor_sync(0xffffffffu, a.re.x, 8), __shfl_xor_sync(0xffffffffu, a.re.y, 8)),
              make_float2(__shfl_xor_sync(0xffffffffu, a.im.x, 8), __shfl_xor_sync(0xffffffffu, a.im.y, 8))};
}
__device__ __forceinline__ c2 walk_sel(int c, c2 a, c2 b)
{
    return c2{make_float2(c ? a.re.x : b.re.x, c ? a.re.y : b.re.y), make_float2(c ? a.im.x : b.im.x, c ? a.im.y : b.im.y)};
}
// tw_addsub<INV>(e, o, k, lo, hi) of cpra_fft.cuh for k = m + 4 h0 with h0 known only at run time: the same operations
// on the same operands as the compile-time version (k and k + 4 share a code shape; constants and operand roles are selected)
template <bool INV>
__device__ __forceinline__ void walk_tw_addsub(c2 e, c2 o, int m, int h0, c2& lo, c2& hi)
{
    constexpr float H = 0.70710678118654752440f;
    constexpr float C1 = 0.92387953251128675613f, S1 = 0.38268343236508977173f;
    if (m == 0) {
        // k = 0: W o = o;  k = 4: W o = (o.im, -o.re) forward, (-o.im, o.re) inverse
        const float2 x = h0 ? (INV ? neg2(o.im) : o.im) : o.re, y = h0 ? (INV ? o.re : neg2(o.re)) : o.im;
        lo = c2{padd(e.re, x), padd(e.im, y)};
        hi = c2{psub(e.re, x), psub(e.im, y)};
    } else if (m == 2) {
        const float2 s = padd(o.re, o.im), d = psub(o.im, o.re);
        const float2 tr = h0 ? (INV ? neg2(s) : d) : (INV ? neg2(d) : s);
        const float2 ti = h0 ? (INV ? neg2(d) : neg2(s)) : (INV ? s : d);
        lo = c2{pfma(tr, bc(H), e.re), pfma(ti, bc(H), e.im)};
        hi = c2{pfma(tr, bc(-H), e.re), pfma(ti, bc(-H), e.im)};
    } else {
        // m = 1: k = 1 | 5;  m = 3: k = 3 | 7
        const float c = (m == 1) ? (h0 ? -S1 : C1) : (h0 ? -C1 : S1);
        const float s0 = (m == 1) ? (h0 ? C1 : S1) : (h0 ? S1 : C1);
        const float s = INV ? -s0 : s0;
        const float2 tr = pfma(o.re, bc(c), pmul(o.im, bc(s)));
        const float2 ti = pfma(o.im, bc(c), neg2(pmul(o.re, bc(s))));
        lo = c2{padd(e.re, tr), padd(e.im, ti)};
        hi = c2{psub(e.re, tr), psub(e.im, ti)};
    }
}
// The second half of dft<16>: a = the radix-8 DFT this thread computed over the inputs of parity h0 (E if h0 = 0, O if
// h0 = 1).  Thread h0 takes k = 4 h0 + m, m = 0 .. 3: it gets the four values of the other parity it needs, and ends with
// output k in a[m] and output k + 8 in a[4 + m].
template <bool INV>
__device__ __forceinline__ void walk_combine(c2 (&a)[8], int h0)
{
#pragma unroll
    for (int m = 0; m < 4; ++m) {
        const c2 recv = walk_xchg(walk_sel(h0, a[m], a[4 + m]));   // h0 = 0 sends E[4 + m] and gets O[m]; h0 = 1 the reverse
        c2 lo, hi;
        walk_tw_addsub<INV>(walk_sel(h0, recv, a[m]), walk_sel(h0, a[4 + m], recv), m, h0, lo, hi);
        a[m] = lo;
        a[4 + m] = hi;
    }
}

template <int N>
__global__ void __launch_bounds__(walk_threads<N>(), walk_ctas_per_sm<N>())
k_row_walk(const __grid_constant__ CUtensorMap tm_in, const __grid_constant__ CUtensorMap tm_out, const float4* __restrict__ gh_old,
           float4* __restrict__ gh_new, const float2* __restrict__ twg, const uint16_t* __restrict__ S16,
           MixParams mp, float beta, int Np, int per_cta)
{
    using RX = Radix<N>;
    constexpr int TBN = tile_batch<N>(), NP = tile_pairs<N>(), NT = walk_threads<N>();
    constexpr int NRT = N / TBN, NCT = N / TBN, R0 = RX::R0, R1 = RX::R1, RL = RX::R2, M0 = N / R0;
    // every thread owns E0 = 8 elements of the tile in the first-stage arrangement: B0 butterflies of radix R0
    // (N = 512: one of radix 8; N = 256: two of radix 4), and one radix-8 butterfly in each inner stage.
    // N = 1024 (R0 = 16, SPLIT = 2): a first-stage butterfly belongs to TWO threads of a warp (lanes l, l ^ 8).  The
    // radix-16 DFT of cpra_fft.cuh is two radix-8 DFTs over the inputs of even / odd index followed by 8 twiddled
    // add/subs that give outputs k and k + 8: thread h0 does the radix-8 DFT of the inputs of parity h0, the two
    // exchange 4 results each by shuffles, and thread h0 does the add/subs k = 4 h0 + m, m = 0 .. 3 (outputs k, k + 8).
    // Every operation is the one dft<16> does on the same operands: the results are bit-identical to the tile kernels'.
    // On the object side (g_new, ghat, the mix, the support) a thread therefore owns the elements
    // r(e) = 4 h0 + (e & 3) + 8 (e >> 2), on the spectrum side of the inverse the elements r = 2 e + h0; the forward
    // transform regroups by parity first (4 more exchanges).
    constexpr int SPLIT = R0 == 16 ? 2 : 1;
    constexpr int QN = NT / NP, B0 = SPLIT == 2 ? 1 : NP * M0 / NT, E0 = SPLIT == 2 ? R0 / 2 : B0 * R0;
    static_assert((SPLIT == 2 ? 2 * NP * M0 == NT : B0 * NT == NP * M0) && E0 == 8 && NP * (N / R1) == NT && RL == 8,
                  "8 first-stage elements and one inner butterfly per thread");
    static_assert(NP == 4 && R1 == 8, "the two inner stages of a 64-position block must belong to one warp");
    extern __shared__ __align__(128) float4 sm[];
    float4* const slots = sm;
    const float2* const tw0 = reinterpret_cast<const float2*>(sm + WALK_SLOTS * tile_quads<N>());
    const float2* const tw1 = tw0 + tw_count_stage0<N>();
    uint64_t* const full = reinterpret_cast<uint64_t*>(const_cast<float2*>(tw0) + tw_count<N>());   // [3] + 1 for the twiddles
    uint16_t* const sup = reinterpret_cast<uint16_t*>(full + 4);                                     // [3][N]
    const size_t istride = (size_t)N * N / 2;
    const int total = NRT * Np;
    const int u0 = (int)blockIdx.x * per_cta, u1 = min(total, u0 + per_cta);
    if (u0 >= u1) return;
    const int j = threadIdx.x % NP, q = threadIdx.x / NP;   // this thread's butterfly in every stage
    const bool io = threadIdx.x == 0;   // the thread that issues the copies

    if (threadIdx.x == 0) {
        for (int b = 0; b < 4; ++b) mbar_init(full + b, 1);
    }
    __syncthreads();
    if (threadIdx.x == 0) {
        mbar_expect_tx(full + 3, tw_bytes<N>());
        bulk_load(const_cast<float2*>(tw0), twg, tw_bytes<N>(), full + 3);
    }
    unsigned phase = 0;   // bit s = parity of the next completion of full[s]
    // Quad offsets of this thread's butterfly in the three stages, as one base (two for the stages
    // whose positions cross 8-blocks of alternating parity, see ppos) plus a compile-time multiple of r:
    //   stage 0 (stride M0):    p = q + QN b + M0 r     ppos(p) = ppos(q) + QN b + M0 r   (element e = R0 b + r)
    //   stage 1 (stride 8):     p = 64 b + n2 + 8 r     ppos(p) = p ^ (r & 1)
    //   last    (contiguous):   p = 8 q + r             ppos(p) = 8 q + (r ^ (q & 1))
    // first stage: SPLIT == 1: the thread's inner indices (q, j).  SPLIT == 2: lane bits [1:0] = pair, [2] = low bit
    // of the butterfly index q0 (a quarter-warp reads two neighbouring positions: conflict-free), [3] = half h0
    const int j0 = SPLIT == 2 ? (int)(threadIdx.x & 3) : j;
    const int q0 = SPLIT == 2 ? (int)(((threadIdx.x >> 4) << 1) | ((threadIdx.x >> 2) & 1)) : q;
    const int h0 = SPLIT == 2 ? (int)((threadIdx.x >> 3) & 1) : 0;
    const int o0 = ppos<N>(q0) * NP + j0;
    const int o1e = ((q / 8) * 64 + (q % 8)) * NP + j, o1o = ((q / 8) * 64 + ((q % 8) ^ 1)) * NP + j;
    const int oLe = (8 * q + (q & 1)) * NP + j, oLo = (8 * q + 1 - (q & 1)) * NP + j;
    // object side: position and quad of first-stage element e (SPLIT == 2: r = 4 h0 + (e & 3) + 8 (e >> 2))
    auto r0s = [&](int e) -> int { return 4 * h0 + (e & 3) + 8 * (e >> 2); };
    auto p0 = [&](int e) -> int { return SPLIT == 2 ? q0 + M0 * r0s(e) : q + QN * (e / R0) + M0 * (e % R0); };
    auto i0 = [&](int e) -> int { return SPLIT == 2 ? o0 + r0s(e) * (M0 * NP) : o0 + (e / R0) * (QN * NP) + (e % R0) * (M0 * NP); };
    // spectrum side of the inverse first stage: where its inputs are read (SPLIT == 2: r = 2 e + h0)
    auto iS = [&](int e) -> int { return SPLIT == 2 ? o0 + (2 * e + h0) * (M0 * NP) : i0(e); };
    auto i1 = [&](int r) -> int { return ((r & 1) ? o1o : o1e) + r * (8 * NP); };
    auto iL = [&](int r) -> int { return ((r & 1) ? oLo : oLe) + (r & ~1) * NP; };
    // the quad of the stage-0 element r of this thread MIRRORED in x (position p -> (N - p) mod N): read for a
    // halo tile that lies across the seam of a [0, 180) scan (cpra_set_seam, reading A5b)
    auto i0m = [&](int e) -> int { return ppos<N>((N - p0(e)) & (N - 1)) * NP + j0; };
    static_assert(N / R0 == 64 && QN % 16 == 0, "offsets above assume inner radices 8 x 8 (64-position blocks)");
    // the B0 first-stage butterflies of this thread (twiddle index n2 = q + QN b); SPLIT == 2: its half of one
    auto stage0_inv = [&](c2 (&a)[E0]) {
        if constexpr (SPLIT == 2) {
            const float2* __restrict__ t = tw0 + q0 * (R0 - 1);   // a[e] = input r = 2 e + h0, times conj w_r (r >= 1)
#pragma unroll
            for (int e = 0; e < E0; ++e) {
                const float2 w = t[e == 0 ? 0 : 2 * e + h0 - 1];
                const c2 x = cmulc(a[e], bc(w.x), bc(w.y));
                a[e] = e == 0 ? walk_sel(h0, x, a[e]) : x;
            }
            dft<E0, true>(a);
            walk_combine<true>(a, h0);
        } else {
#pragma unroll
            for (int b = 0; b < B0; ++b) {
                c2(&u)[R0] = *reinterpret_cast<c2(*)[R0]>(&a[b * R0]);
                twiddle<R0, true>(u, tw0, q + QN * b);
                dft<R0, true>(u);
            }
        }
    };
    auto stage0_fwd = [&](c2 (&a)[E0]) {
        if constexpr (SPLIT == 2) {
            // a[e] = element r(e); the radix-8 DFT of parity h0 needs r = 2 e' + h0: half of them are the partner's.
            // h0 = 0 owns r = 0 1 2 3 8 9 10 11 and sends the odd ones, h0 = 1 owns 4 5 6 7 12 13 14 15 and sends the even ones
            c2 n[E0];
#pragma unroll
            for (int i = 0; i < E0 / 2; ++i) {
                const c2 recv = walk_xchg(walk_sel(h0, a[2 * i], a[2 * i + 1]));
                const int lo_i = 4 * (i / 2) + (i % 2);   // r = 2 e' + h0 < 4 + 8 (i / 2): h0 = 0 has it, h0 = 1 receives it
                n[lo_i] = walk_sel(h0, recv, a[2 * i]);
                n[lo_i + 2] = walk_sel(h0, a[2 * i + 1], recv);
            }
            dft<E0, false>(n);
            walk_combine<false>(n, h0);
            const float2* __restrict__ t = tw0 + q0 * (R0 - 1);   // output r(m), times w_r (r >= 1)
#pragma unroll
            for (int m = 0; m < E0; ++m) {
                const float2 w = t[m == 0 ? 3 * h0 : r0s(m) - 1];
                const c2 x = cmul(n[m], bc(w.x), bc(w.y));
                a[m] = m == 0 ? walk_sel(h0, x, n[m]) : x;
            }
        } else {
#pragma unroll
            for (int b = 0; b < B0; ++b) {
                c2(&u)[R0] = *reinterpret_cast<c2(*)[R0]>(&a[b * R0]);
                dft<R0, false>(u);
                twiddle<R0, false>(u, tw0, q + QN * b);
            }
        }
    };
    const float2 a0 = bc(mp.a[0]), a1 = bc(mp.a[1]);

    // issue the loads of projection m's spectrum tile (row tile rt) and support words into slot s
    auto load_tile = [&](int m, int rt, int s) {
        mbar_expect_tx(full + s, tile_bytes<N>() + 2 * N);
        tma_load_tile(slots + s * tile_quads<N>(), &tm_in, rt, m, full + s);
        bulk_load(sup + s * N, S16 + ((size_t)m * (N / 16) + (rt * TBN) / 16) * N, 2 * N, full + s);
    };

    mbar_wait(full + 3, 0);
    for (int u = u0; u < u1;) {
        // a run: consecutive n in [na, nb] of one row tile rt
        const int rt = u / Np, na = u % Np, nb = min(Np - 1, na + (u1 - u) - 1), len = nb - na + 1;
        const int sshift = (rt * TBN) % 16;
        auto proj = [&](int i) -> int { int m = na - 1 + i; return m < 0 ? m + Np : (m >= Np ? m - Np : m); };   // i = 0 .. len + 1
        if (io) {
            for (int i = 0; i < 3 && i < len + 2; ++i) load_tile(proj(i), rt, i);
        }
        // A(i): inverse FFT along x + support / HIO of projection proj(i) in slot i % 3.  The last
        // stage and the update happen in registers (ghat_old requested before the tile is waited
        // for); the new state goes back to the slot AND stays in v for the mix of B(i - 1).
        c2 v[E0];
        int pend_tile = -1, pend_slot = 0;   // refill of the slot B stored from, issued one pass into the next A
        auto stepA = [&](int i) {
            const int s = i % 3, m = proj(i);
            float4* const tile = sm + s * tile_quads<N>();
            const float4* __restrict__ gh = gh_old + (size_t)m * istride + (size_t)rt * tile_quads<N>();
            // ghat_old: pulled into L2 now, into registers two passes later (keeps 32 registers free)
#pragma unroll
            for (int r = 0; r < E0; ++r) asm volatile("prefetch.global.L2 [%0];" ::"l"(gh + i0(r)));
            mbar_wait(full + s, (phase >> s) & 1u);
            phase ^= 1u << s;
            {
                c2 w[RL];
                load_transposed<N>(tile, w, q, j, rt);
                dft<RL, true>(w);
                __syncwarp();   // positions [64 b, 64 b + 64) of a tile belong to warp b in the two
#pragma unroll                  // inner stages (radix 8 x 8, 4 pairs): their exchanges stay inside a warp
                for (int r = 0; r < RL; ++r) st_quad(tile + iL(r), w[r]);
            }
            __syncwarp();
            c2 g0[E0];
#pragma unroll
            for (int r = 0; r < E0; ++r) g0[r] = from_quad(__ldg(gh + i0(r)));
            {
                c2 w[R1];
#pragma unroll
                for (int r = 0; r < R1; ++r) w[r] = from_quad(tile[i1(r)]);
                twiddle<R1, true>(w, tw1, q % 8);
                dft<R1, true>(w);
#pragma unroll
                for (int r = 0; r < R1; ++r) st_quad(tile + i1(r), w[r]);
            }
            __syncthreads();
            if (io && pend_tile >= 0) {   // the store of the last B has been read out by now: no one waits here
                bulk_wait_read0();
                load_tile(proj(pend_tile), rt, pend_slot);
            }
            pend_tile = -1;
#pragma unroll
            for (int r = 0; r < E0; ++r) v[r] = from_quad(tile[iS(r)]);
            stage0_inv(v);
            const uint16_t* __restrict__ sp = sup + s * N;
#pragma unroll
            for (int r = 0; r < E0; ++r) {
                const unsigned bits = inside_bits(mp, (unsigned)sp[p0(r)] >> (sshift + 2 * j0), v[r].re);
                const float2 ore = update_outside(mp, v[r].re, g0[r].re), oim = update_outside(mp, v[r].im, g0[r].im);
                v[r].re = make_float2((bits & 1) ? v[r].re.x : ore.x, (bits & 2) ? v[r].re.y : ore.y);
                v[r].im = make_float2((bits & 1) ? v[r].im.x : oim.x, (bits & 2) ? v[r].im.y : oim.y);
                st_quad(tile + i0(r), v[r]);
            }
            // no barrier: the quads written here are read back by this same thread (the mix of B(i))
        };
        // B(i): ghat_new(m_i) from gm (registers: g_new(m_{i-1})), slot i % 3 (g_new(m_i)) and v
        // (registers: g_new(m_{i+1})); forward FFT along x in place in slot i % 3, store; refill it
        // with the tile of m_{i+3}.  The quads read from the slot become the next gm.
        c2 gm[E0];
        auto stepB = [&](int i) {
            const int m = proj(i), s0 = i % 3;
            float4* const t0 = sm + s0 * tile_quads<N>();
            float4* __restrict__ gout = gh_new + (size_t)m * istride + (size_t)rt * tile_quads<N>();
            {
                c2 w[E0];
#pragma unroll
                for (int r = 0; r < E0; ++r) {
                    const int i2 = i0(r);
                    const c2 own = from_quad(t0[i2]);
                    w[r] = c2{pfma(a0, own.re, pmul(a1, padd(gm[r].re, v[r].re))), pfma(a0, own.im, pmul(a1, padd(gm[r].im, v[r].im)))};
                    gm[r] = own;
                    gout[i2] = to_quad(w[r]);
                }
                stage0_fwd(w);
#pragma unroll
                for (int r = 0; r < E0; ++r) st_quad(t0 + i0(r), w[r]);
            }
            __syncthreads();
            {
                c2 w[R1];
#pragma unroll
                for (int r = 0; r < R1; ++r) w[r] = from_quad(t0[i1(r)]);
                dft<R1, false>(w);
                twiddle<R1, false>(w, tw1, q % 8);
#pragma unroll
                for (int r = 0; r < R1; ++r) st_quad(t0 + i1(r), w[r]);
            }
            __syncwarp();
            {
                c2 w[RL];
#pragma unroll
                for (int r = 0; r < RL; ++r) w[r] = from_quad(t0[iL(r)]);
                dft<RL, false>(w);
                __syncwarp();
                store_transposed<N>(t0, w, q, j, rt);
            }
            fence_async_smem();
            __syncthreads();
            if (io) {
                tma_store_tile(&tm_out, rt, m, t0);
                bulk_commit();
            }
            pend_tile = (i + 3 <= len + 1) ? i + 3 : -1;
            pend_slot = s0;
        };
        // A(0) A(1) A(2) B(1) A(3) B(2) ... A(len + 1) B(len)   (one call site each: both bodies inline)
        for (int i = 0; i <= len + 1; ++i) {
            stepA(i);
            // a halo tile reached by wrapping round the end of the stack is used mirrored in x
            const bool mirror = mp.flip_seam && ((i == 0 && na == 0) || (i == len + 1 && nb == Np - 1));
            if (mirror) {
                __syncthreads();   // the new state of the halo tile is complete in its slot
                const float4* const th = sm + (i % 3) * tile_quads<N>();
#pragma unroll
                for (int r = 0; r < E0; ++r) v[r] = from_quad(th[i0m(r)]);
            }
            if (i == 0) {   // the first halo tile is only needed in registers: its slot takes the tile of m_3 at once
#pragma unroll
                for (int r = 0; r < E0; ++r) gm[r] = v[r];
                // A(0) wrote the halo's new state into slot 0 with ordinary stores: they must be ordered before the
                // asynchronous-proxy writes of the copy that refills the slot (a barrier alone does not order the two proxies)
                fence_async_smem();
                __syncthreads();   // every thread is done with slot 0
                if (io && 3 <= len + 1) load_tile(proj(3), rt, 0);
            }
            if (i >= 2) stepB(i - 1);
        }
        fence_async_smem();   // the ordinary stores of the last A (the halo's new state) before the next run's copies into the slots
        if (io) bulk_wait_read0();
        __syncthreads();   // the last store has been read out (warp 0 waited) before the next run reloads the slots
        u += len;
    }
}

}  // namespace cpra
