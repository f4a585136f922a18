// cpra_generic_kernels.cuh -- the kernels of cpra_generic.cuh (included by cpra_generic.cu only: they are not
// templates, so they must live in exactly one translation unit).
#pragma once
#include "cpra_generic.cuh"

namespace cpra {

// two lines (w, w + 1) as one packed value: the 16 bytes (re_w, im_w, re_w1, im_w1) of shared memory <-> c2
__device__ __forceinline__ c2 gen_ld2(const float2* p) { const float4 q = *reinterpret_cast<const float4*>(p); return c2{make_float2(q.x, q.z), make_float2(q.y, q.w)}; }
__device__ __forceinline__ void gen_st2(float2* p, c2 v) { *reinterpret_cast<float4*>(p) = make_float4(v.re.x, v.im.x, v.re.y, v.im.y); }

// r-point DFT of packed values: the butterfly networks of cpra_fft.cuh for r = 2, 4, 8; the definition
// out[p] = sum_q v[q] w_r^{pq} with the roots from the table for r = 3, 5, 7
template <int R, bool INV>
__device__ __forceinline__ void gen_small_dft(c2 (&v)[R], const float2* __restrict__ tw, int rstep)
{
    if constexpr (R == 2 || R == 4 || R == 8) {
        dft<R, INV>(v);
    } else {
        // odd prime R: X[p], X[R-p] = t -+ i u (forward) with t = v0 + sum_q cos(2 pi p q / R) (v_q + v_{R-q}),
        // u = sum_q sin(2 pi p q / R) (v_q - v_{R-q}), q = 1 .. (R-1)/2: real coefficients only
        constexpr int H = (R - 1) / 2;
        float2 cs[H], sn[H];          // cos, sin of 2 pi k / R, k = 1 .. H (the other roots by symmetry)
#pragma unroll
        for (int k = 1; k <= H; ++k) {
            const float2 w = tw[k * rstep];
            cs[k - 1] = bc(w.x);
            sn[k - 1] = bc(-w.y);
        }
        c2 A[H], B[H];
        c2 sum = v[0];
#pragma unroll
        for (int q = 1; q <= H; ++q) {
            A[q - 1] = cadd(v[q], v[R - q]);
            B[q - 1] = csub(v[q], v[R - q]);
            sum = cadd(sum, A[q - 1]);
        }
        const c2 v0 = v[0];
        v[0] = sum;
#pragma unroll
        for (int p = 1; p <= H; ++p) {
            c2 t = v0, u{make_float2(0.f, 0.f), make_float2(0.f, 0.f)};
#pragma unroll
            for (int q = 1; q <= H; ++q) {
                // cos, sin of 2 pi (p q mod R) / R: k > H is the mirror of R - k (same cosine, opposite sine)
                const int k = (p * q) % R, km = k <= H ? k : R - k;
                const float2 c = cs[km - 1], sg = k <= H ? sn[km - 1] : neg2(sn[km - 1]);
                t = c2{pfma(c, A[q - 1].re, t.re), pfma(c, A[q - 1].im, t.im)};
                u = c2{pfma(sg, B[q - 1].re, u.re), pfma(sg, B[q - 1].im, u.im)};
            }
            // -i u = (u.im, -u.re)
            const c2 lo{padd(t.re, u.im), psub(t.im, u.re)};     // t - i u
            const c2 hi{psub(t.re, u.im), padd(t.im, u.re)};     // t + i u
            v[p] = INV ? hi : lo;
            v[R - p] = INV ? lo : hi;
        }
    }
}

// ---- the tile in shared memory --------------------------------------------------------------------------------
// float2 index of line w at position x: the W / 2 pairs of a position are XOR-ed with key(x) (see cpra_generic.cuh)
struct GenTile {
    int W, W2m, ksh;
    __device__ __forceinline__ explicit GenTile(int W_) : W(W_), W2m(W_ / 2 - 1), ksh(W_ >= 16 ? 0 : (W_ == 8 ? 1 : 2)) {}
    __device__ __forceinline__ int pair(int x, int w2) const { return x * W + 2 * (w2 ^ ((x >> ksh) & W2m)); }      // 16-byte aligned
    __device__ __forceinline__ int line(int x, int w) const { return pair(x, w >> 1) + (w & 1); }
};

// one in-place stage of radix R on sub-transforms of length L (M = L / R): butterfly (blk, n2) of a pair of lines
// touches positions blk L + n2 + M q.  Forward: DFT, then output p times w_L^{n2 p}; inverse: input q times the
// conjugate first.  w_L^{m} = tw[m N / L].
template <int R, bool INV>
__device__ __forceinline__ void gen_stage(float2* __restrict__ a, const float2* __restrict__ tw, const GenGeo& g, int st)
{
    const int W = g.W, L = g.L[st], M = g.M[st], ts = g.ts[st], nb = g.nb[st];
    const GenTile t(W);
    const int W2 = W / 2, w2shift = 31 - __clz(W2);          // W / 2 is a power of two
    const float invM = g.invM[st];                           // b / M by reciprocal: (b + 0.5) / M is never within rounding of an integer
    for (int i = threadIdx.x; i < nb * W2; i += blockDim.x) {
        const int w2 = i & (W2 - 1), b = i >> w2shift;
        const int blk = (int)(((float)b + 0.5f) * invM), n2 = b - blk * M;
        const int base = blk * L + n2;
        int off[R];
        c2 v[R];
#pragma unroll
        for (int q = 0; q < R; ++q) {
            off[q] = t.pair(base + q * M, w2);
            v[q] = gen_ld2(a + off[q]);
            if (INV && q > 0 && M > 1) {
                const float2 w = tw[q * n2 * ts];             // q n2 < L: the index stays below N
                v[q] = cmulc(v[q], bc(w.x), bc(w.y));
            }
        }
        gen_small_dft<R, INV>(v, tw, nb);
#pragma unroll
        for (int q = 0; q < R; ++q) {
            if (!INV && q > 0 && M > 1) {
                const float2 w = tw[q * n2 * ts];
                v[q] = cmul(v[q], bc(w.x), bc(w.y));
            }
            gen_st2(a + off[q], v[q]);
        }
    }
}
template <bool INV>
__device__ __forceinline__ void gen_stage_any(float2* a, const float2* __restrict__ tw, const GenGeo& g, int st)
{
    switch (g.radix[st]) {
        case 8: gen_stage<8, INV>(a, tw, g, st); break;
        case 4: gen_stage<4, INV>(a, tw, g, st); break;
        case 2: gen_stage<2, INV>(a, tw, g, st); break;
        case 3: gen_stage<3, INV>(a, tw, g, st); break;
        case 5: gen_stage<5, INV>(a, tw, g, st); break;
        default: gen_stage<7, INV>(a, tw, g, st); break;
    }
}
// W lines of length N in the tile a, in place (a block barrier after every stage); tw[m] = e^{-2 pi i m / N} in shared memory
__device__ void gen_fft_fwd(float2* a, const float2* __restrict__ tw, const GenGeo& g)
{
    for (int f = 0; f < g.nf; ++f) {
        gen_stage_any<false>(a, tw, g, f);
        __syncthreads();
    }
}
__device__ void gen_fft_inv(float2* a, const float2* __restrict__ tw, const GenGeo& g)
{
    for (int f = g.nf - 1; f >= 0; --f) {
        gen_stage_any<true>(a, tw, g, f);
        __syncthreads();
    }
}

struct GenSmem {
    float2 *a, *tw;
    double* red;
    int* perm;   // pos(k), filled by the kernels that need it
    __device__ __forceinline__ GenSmem(unsigned char* sm, int N, int W)
    {
        a = reinterpret_cast<float2*>(sm);
        tw = a + (size_t)N * W;
        red = reinterpret_cast<double*>(tw + N);
        perm = reinterpret_cast<int*>(red + 32);
    }
};

// Row tiles: a warp takes whole lines (w = warp, warp + nw, ...: W >= the number of warps), the lanes run along x
// (coalesced), GEN_U steps of 32 at a time: all their global loads are issued before the first value is used.
constexpr int GEN_U = 4;
__device__ __forceinline__ void gen_prefetch_l2(const void* p) { asm volatile("prefetch.global.L2 [%0];" ::"l"(p)); }
__device__ __forceinline__ void gen_cp_async8(void* smem_dst, const void* gsrc)
{
    const unsigned d = (unsigned)__cvta_generic_to_shared(smem_dst);
    asm volatile("cp.async.ca.shared.global [%0], [%1], 8;" ::"r"(d), "l"(gsrc) : "memory");
}
__device__ __forceinline__ void gen_cp_async_wait() { asm volatile("cp.async.wait_all;" ::: "memory"); }

// Eq. (4) at pixel (y, x) of projection n on natural arrays, with the mirrored wrap of cpra_set_seam
__device__ __forceinline__ float2 gen_mix(const float2* __restrict__ g, const GenGeo& gg, const MixParams& mp, int n, int y, int x, bool fires)
{
    const int N = gg.N, Np = gg.Np;
    const size_t px = (size_t)N * N;
    const float2 own = g[(size_t)n * px + (size_t)y * N + x];
    if (!fires || (mp.K == 0 && mp.a[0] == 1.0f)) return own;
    float2 acc = make_float2(mp.a[0] * own.x, mp.a[0] * own.y);
    for (int k = 1; k <= mp.K; ++k) {
        float sx = 0.f, sy = 0.f;
        for (int sgn = -1; sgn <= 1; sgn += 2) {
            int m = n + sgn * k;
            const bool wrapped = m < 0 || m >= Np;
            if (m < 0) m += Np;
            if (m >= Np) m -= Np;
            const int xs = (wrapped && mp.flip_seam) ? ((N - x) % N) : x;
            const float2 v = g[(size_t)m * px + (size_t)y * N + xs];
            sx += v.x; sy += v.y;
        }
        acc.x = fmaf(mp.a[k], sx, acc.x);
        acc.y = fmaf(mp.a[k], sy, acc.y);
    }
    return acc;
}

// K1: mix + forward FFT along x of W rows; spectrum rows to scr ([n][y][position], see cpra_generic.cuh).  mask_mode:
// multiply by the support first (the slices of the assembly); ghat_out: also store the mixed input (for the update of K3).
__global__ void __launch_bounds__(GEN_NT, 4)
k_gen_row_fwd(const float2* __restrict__ cur, float2* __restrict__ scr, const float2* __restrict__ twg, const unsigned char* __restrict__ S,
              MixParams mp, GenGeo gg, int n0, int fires, int mask_mode, float2* __restrict__ ghat_out)
{
    extern __shared__ __align__(16) unsigned char smraw[];
    const int N = gg.N, W = gg.W, Np = gg.Np;
    GenSmem s(smraw, N, W);
    const GenTile t(W);
    const int tiles = (N + W - 1) / W;
    const int n = n0 + (int)(blockIdx.x / tiles), y0 = (int)(blockIdx.x % tiles) * W;
    const size_t px = (size_t)N * N;
    for (int i = threadIdx.x; i < N; i += blockDim.x) s.tw[i] = twg[i];
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5, nw = blockDim.x >> 5;
    const bool mixes = fires != 0 && !(mp.K == 0 && mp.a[0] == 1.0f);
    int mm = n - 1, mq = n + 1;                                  // the neighbours of the default coupling (K = 1)
    const bool wm = mm < 0, wq = mq >= Np;
    if (wm) mm += Np;
    if (wq) mq -= Np;
    const bool fm = wm && mp.flip_seam, fq = wq && mp.flip_seam;
    for (int w = wid; w < W; w += nw) {
        const int y = y0 + w;
        if (y >= N) {
            for (int x = lane; x < N; x += 32) s.a[t.line(x, w)] = make_float2(0.f, 0.f);
            continue;
        }
        const size_t row = (size_t)n * px + (size_t)y * N;
        if (!mixes && !mask_mode && !ghat_out) {
            // a plain copy: asynchronous, the whole line in flight at once
            for (int x = lane; x < N; x += 32) gen_cp_async8(s.a + t.line(x, w), cur + row + x);
        } else if (mixes && mp.K == 1) {
            // Eq. (4) with the default coupling: own + the two neighbours
            const float2* __restrict__ go = cur + row;
            const unsigned char* __restrict__ Sr = S + row;
            float2* __restrict__ ghr = ghat_out ? ghat_out + row : nullptr;
            const float2* __restrict__ gm = cur + (size_t)mm * px + (size_t)y * N;
            const float2* __restrict__ gq = cur + (size_t)mq * px + (size_t)y * N;
            for (int x0 = lane; x0 < N; x0 += 32 * GEN_U) {
                float2 o[GEN_U], a[GEN_U], b[GEN_U];
#pragma unroll
                for (int u = 0; u < GEN_U; ++u) {
                    const int x = x0 + 32 * u;
                    if (x < N) {
                        const int xm = x == 0 ? 0 : N - x;
                        o[u] = go[x];
                        a[u] = gm[fm ? xm : x];
                        b[u] = gq[fq ? xm : x];
                    }
                }
#pragma unroll
                for (int u = 0; u < GEN_U; ++u) {
                    const int x = x0 + 32 * u;
                    if (x < N) {
                        const float sx = (0.f + a[u].x) + b[u].x, sy = (0.f + a[u].y) + b[u].y;
                        float2 v = make_float2(fmaf(mp.a[1], sx, mp.a[0] * o[u].x), fmaf(mp.a[1], sy, mp.a[0] * o[u].y));
                        if (mask_mode && !Sr[x]) v = make_float2(0.f, 0.f);
                        if (ghr) ghr[x] = v;
                        s.a[t.line(x, w)] = v;
                    }
                }
            }
        } else {
            for (int x = lane; x < N; x += 32) {
                float2 v = gen_mix(cur, gg, mp, n, y, x, fires != 0);
                if (mask_mode && !S[row + x]) v = make_float2(0.f, 0.f);
                if (ghat_out) ghat_out[row + x] = v;
                s.a[t.line(x, w)] = v;
            }
        }
    }
    gen_cp_async_wait();
    __syncthreads();
    gen_fft_fwd(s.a, s.tw, gg);
    // position p of the transform goes to column p of the scratch row (position order)
    for (int w = wid; w < W; w += nw) {
        const int y = y0 + w;
        if (y >= N) continue;
        float2* __restrict__ out = scr + (size_t)n * px + (size_t)y * N;
        for (int x0 = lane; x0 < N; x0 += 32 * GEN_U) {
            float2 v[GEN_U];
#pragma unroll
            for (int u = 0; u < GEN_U; ++u) if (x0 + 32 * u < N) v[u] = s.a[t.line(x0 + 32 * u, w)];
#pragma unroll
            for (int u = 0; u < GEN_U; ++u) if (x0 + 32 * u < N) out[x0 + 32 * u] = v[u];
        }
    }
}

// K2: W columns: forward FFT along y, error metric + Fourier-modulus constraint, inverse FFT along y (unnormalised);
// mode 0 = all three, 1 = forward only (rows left in position order), 2 = inverse only (rows expected in position
// order).  The columns of scr are in position order (K1).  A: sqrt(I) in position order on both axes
// (A[pos(ky)][pos(kx)], k_gen_set_data), A < 0 = unmeasured.
// Modes 3 and 4 are the plain 1D transform along the slow axis with NATURAL order on both sides (the z pass of
// cpra_fft3): 3 = forward, 4 = inverse times `scale`.  "Image" n starts at scr + n istride, its rows are `pitch` apart.
// The mode is a template parameter: the loop's kernel (mode 0) carries nothing of the others.
template <int MODE>
__global__ void __launch_bounds__(GEN_NT, 4)
k_gen_col(float2* __restrict__ scr, const float* __restrict__ A, const float2* __restrict__ twg, double* __restrict__ partial,
          GenGeo gg, int n0, float scale, size_t istride, size_t pitch)
{
    constexpr int mode = MODE;
    constexpr bool ZM = MODE >= 3;
    extern __shared__ __align__(16) unsigned char smraw[];
    const int N = gg.N, W = gg.W;
    GenSmem s(smraw, N, W);
    const GenTile t(W);
    const int tiles = (N + W - 1) / W;
    const int n = n0 + (int)(blockIdx.x / tiles), tile = (int)(blockIdx.x % tiles), x0 = tile * W;
    const size_t px = (size_t)N * N;
    for (int i = threadIdx.x; i < N; i += blockDim.x) s.tw[i] = twg[i];
    // thread -> (pair of columns w2 of the tile, rows r0, r0 + rstep, ...): a row segment of W complex numbers is
    // contiguous, a pair of columns is 16 aligned bytes both in the scratch row and in the tile (N and W are even)
    const int W2 = W / 2, w2 = threadIdx.x & (W2 - 1), r0 = threadIdx.x / W2, rstep = blockDim.x / W2, cx = x0 + 2 * w2;
    float2* __restrict__ col0 = scr + (size_t)n * istride + cx;
    const float* __restrict__ A0 = A + (size_t)n * px + cx;
    if constexpr (ZM) {
        for (int i = threadIdx.x; i < N; i += blockDim.x) s.perm[i] = gen_pos(i, gg);
        __syncthreads();
    }
    // the tile arrives by asynchronous 16-byte copies (all of a thread's rows in flight at once); sqrt(I) of the tile is
    // requested into L2 meanwhile
    if (cx < N) {
        for (int y = r0; y < N; y += rstep) {
            const unsigned d = (unsigned)__cvta_generic_to_shared(s.a + t.pair(ZM && mode == 4 ? s.perm[y] : y, w2));
            asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(d), "l"(col0 + (size_t)y * pitch) : "memory");
        }
        if (mode == 0 && (w2 & 3) == 0)
            for (int y = r0; y < N; y += rstep) gen_prefetch_l2(A0 + (size_t)y * N);
    } else {
        for (int y = r0; y < N; y += rstep) *reinterpret_cast<float4*>(s.a + t.pair(y, w2)) = make_float4(0.f, 0.f, 0.f, 0.f);
    }
    gen_cp_async_wait();
    __syncthreads();
    if (mode != 2 && mode != 4) gen_fft_fwd(s.a, s.tw, gg);
    if (mode == 0) {
        // the modulus step of the power-of-two path (cpra_kernels.cuh) on the two columns of the pair
        float2 acc2 = make_float2(0.f, 0.f);
        constexpr int UA = 4;   // sqrt(I) of UA rows requested before the first is used
        for (int kb = r0; kb < N && cx < N; kb += UA * rstep) {
            float2 av[UA];
#pragma unroll
            for (int u = 0; u < UA; ++u) {
                const int ky = kb + u * rstep;
                av[u] = ky < N ? __ldg(reinterpret_cast<const float2*>(A0 + (size_t)ky * N)) : make_float2(-1.f, -1.f);
            }
#pragma unroll
            for (int u = 0; u < UA; ++u) {
                const int ky = kb + u * rstep;
                if (ky >= N) break;
                float2* q = s.a + t.pair(ky, w2);
                c2 v = gen_ld2(q);
                modulus_pair(v, av[u], scale, acc2);
                gen_st2(q, v);
            }
        }
        // fixed-order block reduction of the error numerator
        float acc = acc2.x + acc2.y;
        for (int o = 16; o > 0; o >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, o);
        if ((threadIdx.x & 31) == 0) s.red[threadIdx.x >> 5] = (double)acc;
        __syncthreads();
        if (threadIdx.x == 0) {
            double sum = 0.0;
            for (int w = 0; w < (int)blockDim.x / 32; ++w) sum += s.red[w];
            partial[(size_t)n * tiles + tile] = sum;
        }
    }
    if (mode != 1 && mode != 3) gen_fft_inv(s.a, s.tw, gg);
    if (cx < N) {
        if (ZM && mode >= 3) {
            const float f = mode == 4 ? scale : 1.0f;
            for (int y = r0; y < N; y += rstep) {
                const float4 q = *reinterpret_cast<const float4*>(s.a + t.pair(mode == 3 ? s.perm[y] : y, w2));
                *reinterpret_cast<float4*>(col0 + (size_t)y * pitch) = make_float4(q.x * f, q.y * f, q.z * f, q.w * f);
            }
        } else {
#pragma unroll 4
            for (int y = r0; y < N; y += rstep)
                *reinterpret_cast<float4*>(col0 + (size_t)y * pitch) = *reinterpret_cast<const float4*>(s.a + t.pair(y, w2));
        }
    }
}

// K3: inverse FFT along x of W rows (times `scale`) + support / update (cpra_set_update); hio = 0: plain
// scaled inverse transform.  ghat: the mixed input stored by K1, or NULL = re-mix from the previous state.
__global__ void __launch_bounds__(GEN_NT, 4)
k_gen_row_inv(const float2* __restrict__ scr, const float2* __restrict__ cur, float2* __restrict__ nxt, const float2* __restrict__ twg,
              const unsigned char* __restrict__ S, MixParams mp, GenGeo gg, int n0, int fires, int hio, float scale,
              const float2* __restrict__ ghat)
{
    extern __shared__ __align__(16) unsigned char smraw[];
    const int N = gg.N, W = gg.W;
    GenSmem s(smraw, N, W);
    const GenTile t(W);
    const int tiles = (N + W - 1) / W;
    const int n = n0 + (int)(blockIdx.x / tiles), y0 = (int)(blockIdx.x % tiles) * W;
    const size_t px = (size_t)N * N;
    for (int i = threadIdx.x; i < N; i += blockDim.x) s.tw[i] = twg[i];
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5, nw = blockDim.x >> 5;
    const size_t tbase = (size_t)n * px + (size_t)y0 * N;       // element (w, x) of the tile at tbase + w N + x
    // the spectrum rows (columns in position order, as K1 stored them) arrive by asynchronous copies, all in flight at once
    for (int w = wid; w < W; w += nw) {
        if (y0 + w < N) {
            const float2* __restrict__ in = scr + tbase + (size_t)w * N;
            for (int x = lane; x < N; x += 32) gen_cp_async8(s.a + t.line(x, w), in + x);
        } else {
            for (int x = lane; x < N; x += 32) s.a[t.line(x, w)] = make_float2(0.f, 0.f);
        }
    }
    if (hio) {
        // what the update will read after the transform (support bytes, stored ghat) is requested into L2 meanwhile
        const int rows = min(W, N - y0), el = rows * N;
        for (int i = threadIdx.x * 128; i < el; i += blockDim.x * 128) gen_prefetch_l2(S + tbase + i);
        if (ghat) for (int i = threadIdx.x * 16; i < el; i += blockDim.x * 16) gen_prefetch_l2(ghat + tbase + i);
    }
    gen_cp_async_wait();
    __syncthreads();
    gen_fft_inv(s.a, s.tw, gg);
    for (int w = wid; w < W; w += nw) {
        const int y = y0 + w;
        if (y >= N) continue;
        // the line's rows of the global arrays as pointers of their own: the loop below adds only x
        const size_t row = tbase + (size_t)w * N;
        const unsigned char* __restrict__ Sr = S + row;
        const float2* __restrict__ ghr = ghat ? ghat + row : nullptr;
        float2* __restrict__ outr = nxt + row;
        const bool use_gh = hio && ghat != nullptr;
        for (int x0 = lane; x0 < N; x0 += 32 * GEN_U) {
            float2 gp[GEN_U], gh[GEN_U];
            unsigned char sv[GEN_U];
#pragma unroll
            for (int u = 0; u < GEN_U; ++u) {
                const int x = x0 + 32 * u;
                gh[u] = make_float2(0.f, 0.f);
                sv[u] = 1;
                if (x < N) {
                    gp[u] = s.a[t.line(x, w)];
                    if (hio) sv[u] = Sr[x];
                    if (use_gh) gh[u] = ghr[x];
                }
            }
#pragma unroll
            for (int u = 0; u < GEN_U; ++u) {
                const int x = x0 + 32 * u;
                if (x >= N) continue;
                float2 g = make_float2(gp[u].x * scale, gp[u].y * scale);
                if (hio && (!sv[u] || (mp.positivity && g.x < 0.f))) {
                    const float2 h = ghat ? gh[u] : gen_mix(cur, gg, mp, n, y, x, fires != 0);
                    g = make_float2(fmaf(mp.c_gp, g.x, mp.c_ghat * h.x), fmaf(mp.c_gp, g.y, mp.c_ghat * h.y));
                }
                outr[x] = g;
            }
        }
    }
}

// A0: A = sqrt(max(I, 0)), mask folded in as A = -1, detector-centred -> native (ifftshift) -> position order on both
// axes (where the transforms of the loop leave frequency (ky, kx)); den_n
__global__ void k_gen_set_data(const float* __restrict__ I, const unsigned char* __restrict__ mask, float* __restrict__ A, double* __restrict__ den, GenGeo gg)
{
    const int N = gg.N, n = blockIdx.x, h = N / 2;
    double acc = 0.0;
    for (int i = threadIdx.x; i < N * N; i += blockDim.x) {
        const int yc = i / N, xc = i % N;
        const size_t src = (size_t)n * N * N + i;
        const float v = fmaxf(I[src], 0.f);
        const bool m = mask ? (mask[src] != 0) : true;
        A[(size_t)n * N * N + (size_t)gen_pos((yc + h) % N, gg) * N + gen_pos((xc + h) % N, gg)] = m ? sqrtf(v) : -1.f;
        if (m) acc += (double)v;
    }
    __shared__ double red[32];
    for (int o = 16; o > 0; o >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, o);
    if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = acc;
    __syncthreads();
    if (threadIdx.x == 0) {
        double t = 0.0;
        for (int w = 0; w < (int)blockDim.x / 32; ++w) t += red[w];
        den[n] = t;
    }
}
__global__ void k_gen_copy_support(const unsigned char* __restrict__ in, unsigned char* __restrict__ out, size_t total)
{
    const size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i < total) out[i] = in[i] ? 1 : 0;
}
__global__ void k_gen_get(const float2* __restrict__ st, const unsigned char* __restrict__ S, float2* __restrict__ out, size_t total, int masked)
{
    const size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= total) return;
    out[i] = (masked && !S[i]) ? make_float2(0.f, 0.f) : st[i];
}
// spectrum in position order [n][pos(kz)][pos(ku)] -> natural and transposed [n][ku][kz] (what k_assemble reads)
__global__ void k_gen_transpose(const float2* __restrict__ in, float2* __restrict__ out, GenGeo gg, size_t total)
{
    const size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= total) return;
    const int N = gg.N, kz = (int)(i % N), ku = (int)((i / N) % N);
    const size_t n = i / ((size_t)N * N);
    out[i] = in[(n * N + gen_pos(kz, gg)) * N + gen_pos(ku, gg)];
}
// natural [n][ky][kx] <-> position order [n][pos(ky)][pos(kx)]  (to_pos: into position order; else out of it).  One
// block per (n, GEN_PB consecutive rows of the position-order array): those rows and the natural rows they map to
// both move coalesced; the permutation along x goes through shared memory with the tables pos / its inverse built
// once per block.  Dynamic shared memory: GEN_PB N float2 + 2 N int.
// zperm (a cube of N planes, Step D): the planes are permuted too, natural plane n <-> plane pos(n) of the position-order array.
constexpr int GEN_PB = 4;
template <class T>
__global__ void k_gen_permute(const T* __restrict__ in, T* __restrict__ out, GenGeo gg, int to_pos, int zperm)
{
    extern __shared__ __align__(16) unsigned char pm[];
    const int N = gg.N;
    T* rows = reinterpret_cast<T*>(pm);
    int* pos = reinterpret_cast<int*>(rows + (size_t)GEN_PB * N);
    int* inv = pos + N;
    const int nb = (N + GEN_PB - 1) / GEN_PB;
    const int py0 = (int)(blockIdx.x % nb) * GEN_PB, nr = min(GEN_PB, N - py0);
    const size_t n = blockIdx.x / nb;                                  // plane of the position-order array
    const size_t nn = zperm ? (size_t)-1 : n;                          // plane of the natural array (zperm: inv[n], below)
    for (int k = threadIdx.x; k < N; k += blockDim.x) {
        const int p = gen_pos(k, gg);
        pos[k] = p;
        inv[p] = k;
    }
    __syncthreads();
    const size_t nnat = zperm ? (size_t)inv[n] : nn;
    if (to_pos) {
        for (int r = 0; r < nr; ++r) {
            const T* __restrict__ src = in + (nnat * N + inv[py0 + r]) * N;
            for (int x = threadIdx.x; x < N; x += blockDim.x) rows[r * N + x] = src[x];
        }
        __syncthreads();
        for (int r = 0; r < nr; ++r) {
            T* __restrict__ dst = out + (n * N + py0 + r) * N;
            for (int q = threadIdx.x; q < N; q += blockDim.x) dst[q] = rows[r * N + inv[q]];
        }
    } else {
        const T* __restrict__ src = in + (n * N + py0) * N;               // nr rows, contiguous
        for (int i = threadIdx.x; i < nr * N; i += blockDim.x) rows[i] = src[i];
        __syncthreads();
        for (int r = 0; r < nr; ++r) {
            T* __restrict__ dst = out + (nnat * N + inv[py0 + r]) * N;
            for (int x = threadIdx.x; x < N; x += blockDim.x) dst[x] = rows[r * N + pos[x]];
        }
    }
}
// ---- shrink-wrap (reading A23) on natural arrays ------------------------------------
// (|S g|, 0)
__global__ void k_gen_abs_supported(const float2* __restrict__ st, const unsigned char* __restrict__ S, float2* __restrict__ out, size_t total)
{
    const size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= total) return;
    const float2 v = st[i];
    out[i] = make_float2(S[i] ? sqrtf(v.x * v.x + v.y * v.y) : 0.f, 0.f);
}
// spectrum in position order *= exp(-2 pi^2 sigma^2 (ky^2 + kx^2) / N^2): the product of two entries of a table over the
// positions (tab[pos(k)] = exp(-2 pi^2 sigma^2 k^2 / N^2), k signed; built per block in shared memory), so the array is
// walked in its own order.  Dynamic shared memory: N floats.
__global__ void k_gen_gauss_filter(float2* __restrict__ scr, GenGeo gg, size_t total, float sigma)
{
    extern __shared__ float gtab[];
    const int N = gg.N;
    const double c = -2.0 * 9.86960440108935861883 * (double)sigma * (double)sigma / ((double)N * N);
    for (int k = threadIdx.x; k < N; k += blockDim.x) {
        const int ks = k < N / 2 ? k : k - N;
        gtab[gen_pos(k, gg)] = (float)exp(c * (double)ks * (double)ks);
    }
    __syncthreads();
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < total; i += (size_t)gridDim.x * blockDim.x) {
        const int px = (int)(i % N), py = (int)((i / N) % N);
        const float f = gtab[py] * gtab[px];
        float2 v = scr[i];
        v.x *= f; v.y *= f;
        scr[i] = v;
    }
}
// the cube's spectrum in position order on all three axes *= exp(-2 pi^2 sigma^2 |k|^2 / N^2)
__global__ void k_gen_gauss3(float2* __restrict__ scr, GenGeo gg, size_t n3, float sigma)
{
    extern __shared__ float gtab[];
    const int N = gg.N;
    const double c = -2.0 * 9.86960440108935861883 * (double)sigma * (double)sigma / ((double)N * N);
    for (int k = threadIdx.x; k < N; k += blockDim.x) {
        const int ks = k < N / 2 ? k : k - N;
        gtab[gen_pos(k, gg)] = (float)exp(c * (double)ks * (double)ks);
    }
    __syncthreads();
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n3; i += (size_t)gridDim.x * blockDim.x) {
        const int px = (int)(i % N), py = (int)((i / N) % N), pz = (int)(i / ((size_t)N * N));
        const float f = gtab[pz] * gtab[py] * gtab[px];
        float2 v = scr[i];
        v.x *= f; v.y *= f;
        scr[i] = v;
    }
}
// per-image maximum of the real part (one block per image)
__global__ void k_gen_image_max(const float2* __restrict__ st, float* __restrict__ mx, int N)
{
    const size_t px = (size_t)N * N;
    const float2* __restrict__ p = st + (size_t)blockIdx.x * px;
    float m = -3.402823466e38f;
    for (size_t i = threadIdx.x; i < px; i += blockDim.x) m = fmaxf(m, p[i].x);
    __shared__ float red[32];
    for (int o = 16; o > 0; o >>= 1) m = fmaxf(m, __shfl_xor_sync(0xffffffffu, m, o));
    if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = m;
    __syncthreads();
    if (threadIdx.x == 0) {
        for (int w = 1; w < (int)blockDim.x / 32; ++w) m = fmaxf(m, red[w]);
        mx[blockIdx.x] = m;
    }
}
// S <- [ b >= threshold max_n b ], max_n > 0; blurred (optional): b as natural floats
__global__ void k_gen_threshold(const float2* __restrict__ b, const float* __restrict__ mx, unsigned char* __restrict__ S,
                                float* __restrict__ blurred, int N, size_t total, float threshold)
{
    const size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= total) return;
    const float m = mx[i / ((size_t)N * N)];
    const float v = b[i].x;
    S[i] = (m > 0.f && v >= threshold * m) ? 1 : 0;
    if (blurred) blurred[i] = v;
}
// PRTF sums: scr = F2[avg_n] and A = sqrt(I), both in position order; acc[0..ns): sum of |G| / A over
// the measured pixels with A > 0 of ring s = round(|k|), acc[ns..2ns): their number
__global__ void k_gen_prtf_accumulate(const float2* __restrict__ scr, const float* __restrict__ A, double* __restrict__ acc, GenGeo gg, size_t total)
{
    extern __shared__ double sh[];   // 2 ns
    const int N = gg.N, ns = N / 2 + 1;
    for (int i = threadIdx.x; i < 2 * ns; i += blockDim.x) sh[i] = 0.0;
    __syncthreads();
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < total; i += (size_t)gridDim.x * blockDim.x) {
        const int ix = (int)(i % N), iy = (int)((i / N) % N);
        const size_t n = i / ((size_t)N * N);
        const int kx = ix < N / 2 ? ix : ix - N, ky = iy < N / 2 ? iy : iy - N;
        const int sh_i = (int)floor(sqrt((double)kx * kx + (double)ky * ky) + 0.5);
        if (sh_i >= ns) continue;
        const size_t o = (n * N + gen_pos(iy, gg)) * N + gen_pos(ix, gg);
        const float a = A[o];
        if (!(a > 0.f)) continue;
        const float2 G = scr[o];
        atomicAdd(&sh[sh_i], sqrt((double)G.x * G.x + (double)G.y * G.y) / (double)a);
        atomicAdd(&sh[ns + sh_i], 1.0);
    }
    __syncthreads();
    for (int i = threadIdx.x; i < 2 * ns; i += blockDim.x) if (sh[i] != 0.0) atomicAdd(&acc[i], sh[i]);
}

}  // namespace cpra
