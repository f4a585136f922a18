// cpra_kernels.cuh -- the CUDA kernels of the CPRA loop (sm_100a).  See DESIGN.md "Kernels".
//
// Internal HBM layouts (all chosen so that every global access of the three hot kernels is a run of
// 128 B per half-warp with lanes along the batch index of the tile):
//   state g   [n][rt][x][16]      rt = y/16, fast index y%16        ("row-tiled", 8 B elements)
//   scratch   [n][ct][py][16]     ct = px/16, fast index px%16      ("column-tiled"; py, px are
//                                  digit-reversed frequency positions, see cpra_fft.cuh)
//   A=sqrt(I) [n][ct][q][16][RL]  py = RL q + r: the RL values one thread needs are contiguous
//   support   [n][rt][x] u16      bit b = S(y = 16 rt + b, x)       (1 bit per pixel)
#pragma once
#include "cpra_fft.cuh"

namespace cpra {

constexpr int MAXK = 8;  // = CPRA_MAX_K
struct MixParams {
    int K;
    float a[MAXK + 1];
};

enum { MIX_NONE = 0, MIX_K1 = 1, MIX_GEN = 2, MIX_MASK = 3 };
enum { COL_FULL = 0, COL_FWD = 1, COL_INV = 2 };
enum { ROWINV_HIO = 0, ROWINV_PLAIN = 1 };

constexpr int ROW_PITCH = TB + 1;  // odd pitch: the transposing copies are conflict-free too
constexpr int COL_PITCH = TB;

template <int N> constexpr int row_smem_bytes() { return (N * ROW_PITCH + N) * (int)sizeof(float2); }
template <int N> constexpr int col_smem_bytes() { return (N * COL_PITCH + N) * (int)sizeof(float2); }

// The carousel mix of Eq. (4) evaluated at one element: `img` = offset of the
// element inside an image (same for every n), `istride` = elements per image.
template <int MODE>
struct MixLoader {
    const float2* __restrict__ c0;   // image n
    const float2* __restrict__ cm;   // image n-1 (mod Np)
    const float2* __restrict__ cp;   // image n+1 (mod Np)
    const float2* __restrict__ base; // image 0
    size_t istride;
    int n, Np;
    MixParams mp;

    __device__ __forceinline__ MixLoader(const float2* cur, size_t istride_, int n_, int Np_, const MixParams& mp_)
        : base(cur), istride(istride_), n(n_), Np(Np_), mp(mp_)
    {
        c0 = cur + (size_t)n_ * istride_;
        cm = cur + (size_t)(n_ == 0 ? Np_ - 1 : n_ - 1) * istride_;
        cp = cur + (size_t)(n_ == Np_ - 1 ? 0 : n_ + 1) * istride_;
    }
    __device__ __forceinline__ float2 operator()(size_t img) const
    {
        if constexpr (MODE == MIX_NONE || MODE == MIX_MASK) {
            return c0[img];
        } else if constexpr (MODE == MIX_K1) {
            const float2 a = c0[img], m = cm[img], p = cp[img];
            return make_float2(fmaf(mp.a[0], a.x, mp.a[1] * (m.x + p.x)), fmaf(mp.a[0], a.y, mp.a[1] * (m.y + p.y)));
        } else {
            const float2 a = c0[img];
            float2 acc = make_float2(mp.a[0] * a.x, mp.a[0] * a.y);
            for (int j = 1; j <= mp.K; ++j) {
                int nm = n - j; if (nm < 0) nm += Np;
                int np = n + j; if (np >= Np) np -= Np;
                const float2 m = base[(size_t)nm * istride + img], p = base[(size_t)np * istride + img];
                acc.x = fmaf(mp.a[j], m.x + p.x, acc.x);
                acc.y = fmaf(mp.a[j], m.y + p.y, acc.y);
            }
            return acc;
        }
    }
};

// ------------------------------------------------------------------------------------------------
// K1: mix (Eq. (4)) + forward FFT along x of 16 rows; writes the column-tiled scratch.
// grid = nimg * N/16 CTAs, n fastest (so that the three CTAs sharing a neighbour tile run together
// and the second and third read hit L2).
// ------------------------------------------------------------------------------------------------
template <int N, int NT, int MODE>
__global__ void __launch_bounds__(NT)
k_row_fwd(const float2* __restrict__ cur, float2* __restrict__ scr, const float2* __restrict__ twg,
          const uint16_t* __restrict__ S16, MixParams mp, int Np, int n0, int nimg)
{
    using RX = Radix<N>;
    constexpr int NRT = N / TB, NCT = N / TB, P = ROW_PITCH;
    extern __shared__ float2 sm[];
    float2* tile = sm;
    float2* tw = sm + N * P;
    const int n = n0 + (int)(blockIdx.x % (unsigned)nimg);
    const int rt = (int)(blockIdx.x / (unsigned)nimg);
    for (int i = threadIdx.x; i < N; i += NT) tw[i] = twg[i];

    const size_t toff = (size_t)rt * N * TB;  // tile offset inside an image
    const MixLoader<MODE> mix(cur, (size_t)N * N, n, Np, mp);
    const uint16_t* __restrict__ Srow = S16 + ((size_t)n * NRT + rt) * N;
    auto ld_g = [&](int x, int b) -> float2 {
        float2 v = mix(toff + (size_t)x * TB + b);
        if constexpr (MODE == MIX_MASK) {
            if (!((Srow[x] >> b) & 1)) v = make_float2(0.f, 0.f);
        }
        return v;
    };
    auto ld_s = [&](int p, int b) -> float2 { return tile[p * P + b]; };
    auto st_s = [&](int p, int b, float2 v) { tile[p * P + b] = v; };

    __syncthreads();
    fft_stage<N, RX::R0, N, false, NT, 2>(tw, ld_g, st_s);
    __syncthreads();
    fft_stage<N, RX::R1, N / RX::R0, false, NT, 1>(tw, ld_s, st_s);
    __syncthreads();
    if constexpr (RX::S == 3) {
        fft_stage<N, RX::R2, N / (RX::R0 * RX::R1), false, NT, 1>(tw, ld_s, st_s);
        __syncthreads();
    }
    // transposing copy-out: tile[px][row] -> scratch[n][ct][y = 16 rt + row][c]
    float2* __restrict__ dst = scr + (size_t)n * N * N + (size_t)rt * TB * TB;
#pragma unroll 4
    for (int e = threadIdx.x; e < N * TB; e += NT) {
        const int c = e % TB, bb = (e / TB) % TB, ct = e / (TB * TB);
        dst[(size_t)ct * N * TB + bb * TB + c] = tile[(ct * TB + c) * P + bb];
    }
}

// ------------------------------------------------------------------------------------------------
// K2: column pass on one [N][16] scratch tile: forward FFT along y, error metric + Fourier-modulus
// constraint in registers, inverse FFT along y, in place.
// A < 0 marks an unmeasured pixel (beamstop): left free.  `scale` (= 1/N^2, a power
// of two) is folded into the constraint.  partial[n][ct] = sum over the tile of (|G| - A)^2.
// ------------------------------------------------------------------------------------------------
template <int N, int NT, int MODE>
__global__ void __launch_bounds__(NT)
k_col(float2* __restrict__ scr, const float* __restrict__ Aperm, const float2* __restrict__ twg,
      double* __restrict__ partial, int n0, float scale)
{
    using RX = Radix<N>;
    constexpr int NCT = N / TB, P = COL_PITCH, RL = last_radix<N>();
    extern __shared__ float2 sm[];
    float2* tile = sm;
    float2* tw = sm + N * P;
    const int n = n0 + (int)(blockIdx.x / (unsigned)NCT);
    const int ct = (int)(blockIdx.x % (unsigned)NCT);
    for (int i = threadIdx.x; i < N; i += NT) tw[i] = twg[i];

    float2* __restrict__ g = scr + ((size_t)n * NCT + ct) * N * TB;
    auto ld_g = [&](int p, int b) -> float2 { return g[p * TB + b]; };
    auto st_g = [&](int p, int b, float2 v) { g[p * TB + b] = v; };
    auto ld_s = [&](int p, int b) -> float2 { return tile[p * P + b]; };
    auto st_s = [&](int p, int b, float2 v) { tile[p * P + b] = v; };
    __syncthreads();

    if constexpr (MODE == COL_FULL || MODE == COL_FWD) {
        fft_stage<N, RX::R0, N, false, NT, 2>(tw, ld_g, st_s);
        __syncthreads();
        if constexpr (RX::S == 3) {
            fft_stage<N, RX::R1, N / RX::R0, false, NT, 1>(tw, ld_s, st_s);
            __syncthreads();
        }
    }
    if constexpr (MODE == COL_FWD) {
        fft_stage<N, RL, RL, false, NT, 1>(tw, ld_s, st_g);
        return;
    }
    if constexpr (MODE == COL_FULL) {
        const float* __restrict__ At = Aperm + ((size_t)n * NCT + ct) * N * TB;
        float acc = 0.f;
        auto pw = [&](float2 (&v)[RL], int q, int b) {
            const float4* __restrict__ a4 = reinterpret_cast<const float4*>(At + ((size_t)q * TB + b) * RL);
            float a[RL];
#pragma unroll
            for (int r = 0; r < RL / 4; ++r) {
                const float4 t = a4[r];
                a[4 * r] = t.x; a[4 * r + 1] = t.y; a[4 * r + 2] = t.z; a[4 * r + 3] = t.w;
            }
#pragma unroll
            for (int r = 0; r < RL; ++r) {
                const float m2 = fmaf(v[r].x, v[r].x, v[r].y * v[r].y);
                float s = scale;                       // unmeasured: G' = G
                if (a[r] >= 0.f) {                     // measured
                    float rs = rsqrtf(m2);             // + one Newton step: ~1 ulp
                    const float h = 0.5f * m2 * rs;
                    rs = fmaf(rs, fmaf(-h, rs, 0.5f), rs);
                    const float mag = m2 * rs;
                    if (m2 > 0.f) {
                        const float d = mag - a[r];
                        acc = fmaf(d, d, acc);
                        s = a[r] * rs * scale;         // G' = A G / |G|
                    } else {                           // |G| = 0: phase 0 (reading A13)
                        acc = fmaf(a[r], a[r], acc);
                        v[r] = make_float2(1.f, 0.f);
                        s = a[r] * scale;
                    }
                }
                v[r].x *= s; v[r].y *= s;
            }
        };
        fft_stage_mid<N, RL, NT, 1>(ld_s, pw, st_s);
        // block reduction of the error numerator (fixed order: deterministic)
        __shared__ float red[32];
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, o);
        if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = acc;
        __syncthreads();
        if (threadIdx.x == 0) {
            double s = 0.0;
            for (int w = 0; w < NT / 32; ++w) s += (double)red[w];
            partial[(size_t)n * NCT + ct] = s;
        }
    }
    if constexpr (MODE == COL_INV) {
        fft_stage<N, RL, RL, true, NT, 2>(tw, ld_g, st_s);
        __syncthreads();
    }
    if constexpr (RX::S == 3) {
        fft_stage<N, RX::R1, N / RX::R0, true, NT, 1>(tw, ld_s, st_s);
        __syncthreads();
    }
    fft_stage<N, RX::R0, N, true, NT, 1>(tw, ld_s, st_g);
}

// ------------------------------------------------------------------------------------------------
// K3: inverse FFT along x of 16 rows + support / HIO update (PAPER.md:98 ref [22], :104):
//   S = 1: g <- g';  S = 0: g <- ghat - beta g'   (ghat = the mixed input of this iteration,
// recomputed from the previous state).  Writes the new state (ping-pong buffer).
// ------------------------------------------------------------------------------------------------
template <int N, int NT, int MODE, int MIXMODE>
__global__ void __launch_bounds__(NT)
k_row_inv(const float2* __restrict__ scr, const float2* __restrict__ cur, float2* __restrict__ nxt,
          const float2* __restrict__ twg, const uint16_t* __restrict__ S16, MixParams mp, float beta,
          float scale, int Np, int n0, int nimg)
{
    using RX = Radix<N>;
    constexpr int NRT = N / TB, P = ROW_PITCH, RL = last_radix<N>();
    extern __shared__ float2 sm[];
    float2* tile = sm;
    float2* tw = sm + N * P;
    const int n = n0 + (int)(blockIdx.x % (unsigned)nimg);
    const int rt = (int)(blockIdx.x / (unsigned)nimg);
    for (int i = threadIdx.x; i < N; i += NT) tw[i] = twg[i];

    // transposing copy-in: scratch[n][ct][y = 16 rt + row][c] -> tile[px = 16 ct + c][row]
    const float2* __restrict__ src = scr + (size_t)n * N * N + (size_t)rt * TB * TB;
#pragma unroll 8
    for (int e = threadIdx.x; e < N * TB; e += NT) {
        const int c = e % TB, bb = (e / TB) % TB, ct = e / (TB * TB);
        tile[(ct * TB + c) * P + bb] = src[(size_t)ct * N * TB + bb * TB + c];
    }
    __syncthreads();

    auto ld_s = [&](int p, int b) -> float2 { return tile[p * P + b]; };
    auto st_s = [&](int p, int b, float2 v) { tile[p * P + b] = v; };
    fft_stage<N, RL, RL, true, NT, 1>(tw, ld_s, st_s);
    __syncthreads();
    if constexpr (RX::S == 3) {
        fft_stage<N, RX::R1, N / RX::R0, true, NT, 1>(tw, ld_s, st_s);
        __syncthreads();
    }
    const size_t toff = (size_t)rt * N * TB;
    float2* __restrict__ out = nxt + (size_t)n * N * N + toff;
    if constexpr (MODE == ROWINV_PLAIN) {
        auto st_g = [&](int x, int b, float2 v) { out[(size_t)x * TB + b] = make_float2(v.x * scale, v.y * scale); };
        fft_stage<N, RX::R0, N, true, NT, 1>(tw, ld_s, st_g);
    } else {
        const MixLoader<MIXMODE> mix(cur, (size_t)N * N, n, Np, mp);
        const uint16_t* __restrict__ Srow = S16 + ((size_t)n * NRT + rt) * N;
        auto st_g = [&](int x, int b, float2 v) {
            const bool inside = (Srow[x] >> b) & 1;
            const float2 gh = mix(toff + (size_t)x * TB + b);
            float2 o;
            o.x = inside ? v.x : fmaf(-beta, v.x, gh.x);
            o.y = inside ? v.y : fmaf(-beta, v.y, gh.y);
            out[(size_t)x * TB + b] = o;
        };
        fft_stage<N, RX::R0, N, true, NT, 1>(tw, ld_s, st_g);
    }
}

// ------------------------------------------------------------------------------------------------
// One-off / layout kernels (not on the timed path)
// ------------------------------------------------------------------------------------------------
struct Geo {
    int N, Np, R0, R1, R2, RL;
};
__device__ __forceinline__ size_t st_idx(int N, int n, int y, int x)
{
    return (((size_t)n * (N / TB) + (y / TB)) * N + x) * TB + (y % TB);
}
__device__ __forceinline__ size_t sc_idx(int N, int n, int py, int px)
{
    return (((size_t)n * (N / TB) + (px / TB)) * N + py) * TB + (px % TB);
}
__device__ __forceinline__ size_t a_idx(int N, int RL, int n, int py, int px)
{
    return ((size_t)n * (N / TB) + (px / TB)) * N * TB + ((size_t)(py / RL) * TB + (px % TB)) * RL + (py % RL);
}

// A0: A = sqrt(max(I, 0)) (A14), mask folded in as A = -1, detector-centred ->
// native (ifftshift, A11) -> the permuted order of the FFT kernels; den_n = sum_{M=1} max(I, 0).
__global__ void k_set_data(const float* __restrict__ I, const unsigned char* __restrict__ mask,
                           float* __restrict__ Aperm, double* __restrict__ den, Geo g)
{
    const int n = blockIdx.x, N = g.N, h = N / 2;
    double acc = 0.0;
    for (int i = threadIdx.x; i < N * N; i += blockDim.x) {
        const int yc = i / N, xc = i % N;
        const size_t src = (size_t)n * N * N + i;
        const float v = fmaxf(I[src], 0.f);
        const bool m = mask ? (mask[src] != 0) : true;
        const int ky = (yc + h) % N, kx = (xc + h) % N;
        Aperm[a_idx(N, g.RL, n, fft_pos(ky, g.R0, g.R1, g.R2), fft_pos(kx, g.R0, g.R1, g.R2))] = m ? sqrtf(v) : -1.f;
        if (m) acc += (double)v;
    }
    __shared__ double red[32];
    for (int o = 16; o > 0; o >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, o);
    if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = acc;
    __syncthreads();
    if (threadIdx.x == 0) {
        double s = 0.0;
        for (int w = 0; w < (int)blockDim.x / 32; ++w) s += red[w];
        den[n] = s;
    }
}

// support u8 [n][y][x] -> bit-packed [n][rt][x] u16
__global__ void k_pack_support(const unsigned char* __restrict__ S, uint16_t* __restrict__ S16, int N, size_t total16)
{
    const size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;  // index into S16
    if (i >= total16) return;
    const int x = (int)(i % N);
    const size_t nr = i / N;  // n * NRT + rt
    const int rt = (int)(nr % (N / TB));
    const size_t n = nr / (N / TB);
    unsigned bits = 0;
    for (int b = 0; b < TB; ++b)
        if (S[(n * N + (size_t)(rt * TB + b)) * N + x]) bits |= 1u << b;
    S16[i] = (uint16_t)bits;
}

// natural [n][y][x] <-> row-tiled state; mode 1 of unpack multiplies by the support
__global__ void k_pack_state(const float2* __restrict__ in, float2* __restrict__ st, int N, size_t total)
{
    const size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;  // index into st (tiled)
    if (i >= total) return;
    const int b = (int)(i % TB);
    const int x = (int)((i / TB) % N);
    const size_t nr = i / ((size_t)TB * N);
    const int rt = (int)(nr % (N / TB));
    const size_t n = nr / (N / TB);
    st[i] = in[(n * N + (size_t)(rt * TB + b)) * N + x];
}
__global__ void k_unpack_state(const float2* __restrict__ st, const uint16_t* __restrict__ S16,
                               float2* __restrict__ out, int N, size_t total, int masked)
{
    const size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;  // index into out (natural)
    if (i >= total) return;
    const int x = (int)(i % N);
    const int y = (int)((i / N) % N);
    const int n = (int)(i / ((size_t)N * N));
    float2 v = st[st_idx(N, n, y, x)];
    if (masked && !((S16[((size_t)n * (N / TB) + y / TB) * N + x] >> (y % TB)) & 1)) v = make_float2(0.f, 0.f);
    out[i] = v;
}
// natural-order spectrum [n][ky][kx] <-> column-tiled permuted scratch
__global__ void k_unpack_spectrum(const float2* __restrict__ scr, float2* __restrict__ out, Geo g, size_t total)
{
    const size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= total) return;
    const int N = g.N;
    const int kx = (int)(i % N), ky = (int)((i / N) % N), n = (int)(i / ((size_t)N * N));
    out[i] = scr[sc_idx(N, n, fft_pos(ky, g.R0, g.R1, g.R2), fft_pos(kx, g.R0, g.R1, g.R2))];
}
__global__ void k_pack_spectrum(const float2* __restrict__ in, float2* __restrict__ scr, Geo g, size_t total)
{
    const size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= total) return;
    const int N = g.N;
    const int kx = (int)(i % N), ky = (int)((i / N) % N), n = (int)(i / ((size_t)N * N));
    scr[sc_idx(N, n, fft_pos(ky, g.R0, g.R1, g.R2), fft_pos(kx, g.R0, g.R1, g.R2))] = in[i];
}

// A3: E_n = sqrt(num_n / den_n), E = sqrt(sum num / sum den); one block, fixed order.
__global__ void k_finalize_error(const double* __restrict__ partial, const double* __restrict__ den,
                                 float* __restrict__ E, float* __restrict__ Eg, int Np, int NCT)
{
    double num = 0.0, dd = 0.0;
    for (int n = threadIdx.x; n < Np; n += blockDim.x) {
        double s = 0.0;
        for (int c = 0; c < NCT; ++c) s += partial[(size_t)n * NCT + c];
        const double d = den[n];
        if (E) E[n] = d > 0.0 ? (float)sqrt(s / d) : 0.f;
        num += s; dd += d;
    }
    __shared__ double rn[32], rd[32];
    for (int o = 16; o > 0; o >>= 1) {
        num += __shfl_xor_sync(0xffffffffu, num, o);
        dd += __shfl_xor_sync(0xffffffffu, dd, o);
    }
    if ((threadIdx.x & 31) == 0) { rn[threadIdx.x >> 5] = num; rd[threadIdx.x >> 5] = dd; }
    __syncthreads();
    if (threadIdx.x == 0 && Eg) {
        double a = 0.0, b = 0.0;
        for (int w = 0; w < (int)blockDim.x / 32; ++w) { a += rn[w]; b += rd[w]; }
        *Eg = b > 0.0 ? (float)sqrt(a / b) : 0.f;
    }
}

// ------------------------------------------------------------------------------------------------
// A7: Fourier-slice assembly (slice theorem PAPER.md:35-44; reading A17).
// scr holds E_n = F[S_n g_n] in the permuted column-tiled layout.  One thread per (ky, kx) computes
// the polar geometry in fp64 once, then walks kz.
//   uphi[U]      sorted unique ray directions in [0, 2 pi)
//   ustart[U+1]  contributors of unique ray u are rays[ustart[u] .. ustart[u+1])
//   rays[]       n | (neg << 30): the slice and whether the ray is its ku <= 0 half
// ------------------------------------------------------------------------------------------------
__global__ void k_assemble(const float2* __restrict__ scr, float2* __restrict__ vol, float* __restrict__ wgt,
                           const double* __restrict__ uphi, const int* __restrict__ ustart,
                           const int* __restrict__ rays, int U, Geo g, int zper)
{
    const int N = g.N, Np = g.Np, h = N / 2;
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= N * N) return;
    const int ix = i % N, iy = i / N;
    const int kx = ix < h ? ix : ix - N, ky = iy < h ? iy : iy - N;
    const double PI = 3.14159265358979323846264338327950288;
    const double rho = sqrt((double)kx * kx + (double)ky * ky);
    int mode = 0;  // 0: outside, 1: axis (rho = 0), 2: interpolate
    int ur[2] = {0, 0}, r0 = 0;
    double wphi[2] = {0.0, 0.0}, wr = 0.0;
    if (rho == 0.0) mode = 1;
    else if (rho <= (double)(h - 1)) {
        mode = 2;
        double phi = atan2((double)ky, (double)kx);
        if (phi < 0.0) phi += 2.0 * PI;
        int a = -1;
        for (int lo = 0, hi = U - 1; lo <= hi;) {
            const int mid = (lo + hi) / 2;
            if (uphi[mid] <= phi) { a = mid; lo = mid + 1; } else hi = mid - 1;
        }
        double pa, pb; int b;
        if (a < 0) { a = U - 1; pa = uphi[a] - 2.0 * PI; } else pa = uphi[a];
        b = a + 1;
        if (b >= U) { b = 0; pb = uphi[0] + 2.0 * PI; } else pb = uphi[b];
        const double wp = (pb > pa) ? (phi - pa) / (pb - pa) : 0.0;
        r0 = (int)floor(rho);
        wr = rho - (double)r0;
        ur[0] = a; ur[1] = b; wphi[0] = 1.0 - wp; wphi[1] = wp;
    }
    const int z0 = blockIdx.y * zper, z1 = min(N, z0 + zper);
    for (int iz = z0; iz < z1; ++iz) {
        const int kz = iz < h ? iz : iz - N;
        const int pz = fft_pos(iz, g.R0, g.R1, g.R2);
        double vr = 0.0, vi = 0.0;
        float w = 0.f;
        if (mode == 1) {
            const int pu = fft_pos(0, g.R0, g.R1, g.R2);
            for (int n = 0; n < Np; ++n) {
                const float2 e = scr[sc_idx(N, n, pz, pu)];
                const double sg = (iz & 1) ? -1.0 : 1.0;
                vr += sg * e.x; vi += sg * e.y;
            }
            vr /= Np; vi /= Np; w = 1.f;
        } else if (mode == 2) {
            for (int q = 0; q < 2; ++q) {
                if (wphi[q] == 0.0) continue;
                const int u = ur[q];
                const int c0 = ustart[u], c1 = ustart[u + 1];
                for (int rr = 0; rr < 2; ++rr) {
                    const double wrr = rr ? wr : 1.0 - wr;
                    if (wrr == 0.0) continue;
                    const int r = r0 + rr;
                    double sr = 0.0, si = 0.0;
                    for (int c = c0; c < c1; ++c) {
                        const int code = rays[c];
                        const int n = code & 0x3fffffff;
                        const int ku = (code >> 30) ? -r : r;
                        const int iu = ((ku % N) + N) % N;
                        const float2 e = scr[sc_idx(N, n, pz, fft_pos(iu, g.R0, g.R1, g.R2))];
                        const double sg = ((iz + iu) & 1) ? -1.0 : 1.0;   // origin -> centre pixel
                        sr += sg * e.x; si += sg * e.y;
                    }
                    vr += wphi[q] * wrr * sr / (c1 - c0);
                    vi += wphi[q] * wrr * si / (c1 - c0);
                }
            }
            w = 1.f;
        }
        if ((kx + ky + kz) & 1) { vr = -vr; vi = -vi; }
        const size_t o = ((size_t)iz * N + iy) * N + ix;
        vol[o] = make_float2((float)vr, (float)vi);
        if (wgt) wgt[o] = w;
    }
}

}  // namespace cpra
