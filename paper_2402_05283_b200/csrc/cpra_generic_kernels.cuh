// cpra_generic_kernels.cuh -- the kernels of cpra_generic.cuh (included by cpra_generic.cu only: they are not
// templates, so they must live in exactly one translation unit).
#pragma once
#include "cpra_generic.cuh"

namespace cpra {

__device__ __forceinline__ float2 cm(float2 a, float2 b) { return make_float2(a.x * b.x - a.y * b.y, a.x * b.y + a.y * b.x); }

// W lines of length N in a (stride W + 1), result in the returned buffer; tw[m] = e^{-2 pi i m / N} in shared memory
__device__ float2* gen_fft(float2* a, float2* b, const float2* __restrict__ tw, const GenGeo& g, bool inverse)
{
    const int N = g.N, W = g.W, Wp = gen_wp(W);
    int Ns = 1;
    for (int f = 0; f < g.nf; ++f) {
        const int r = g.radix[f], m = N / r, tstep = N / (Ns * r), rstep = N / r;
        for (int i = threadIdx.x; i < m * W; i += blockDim.x) {
            const int w = i % W, j = i / W, k = j % Ns;
            float2 v[8];
#pragma unroll
            for (int q = 0; q < 8; ++q) {
                if (q < r) {
                    float2 x = a[(j + q * m) * Wp + w];
                    if (q > 0 && k > 0) {
                        float2 t = tw[(q * k * tstep) % N];
                        if (inverse) t.y = -t.y;
                        x = cm(x, t);
                    }
                    v[q] = x;
                }
            }
            const int j0 = (j / Ns) * Ns * r + k;
#pragma unroll
            for (int p = 0; p < 8; ++p) {
                if (p < r) {
                    float2 acc = v[0];
#pragma unroll
                    for (int q = 1; q < 8; ++q) {
                        if (q < r) {
                            float2 t = tw[((p * q) % r) * rstep];
                            if (inverse) t.y = -t.y;
                            const float2 y = cm(v[q], t);
                            acc.x += y.x; acc.y += y.y;
                        }
                    }
                    b[(j0 + p * Ns) * Wp + w] = acc;
                }
            }
        }
        __syncthreads();
        float2* t = a; a = b; b = t;
        Ns *= r;
    }
    return a;
}

struct GenSmem {
    float2 *a, *b, *tw;
    double* red;
    __device__ __forceinline__ GenSmem(unsigned char* sm, int N, int W)
    {
        a = reinterpret_cast<float2*>(sm);
        b = a + (size_t)N * gen_wp(W);
        tw = b + (size_t)N * gen_wp(W);
        red = reinterpret_cast<double*>(tw + N);
    }
};

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

// K1: mix + forward FFT along x of W rows; spectrum rows to scr (natural [n][y][kx]).  mask_mode: multiply by the
// support first (the slices of the assembly); ghat_out: also store the mixed input (for the update of K3).
__global__ void __launch_bounds__(GEN_NT)
k_gen_row_fwd(const float2* __restrict__ cur, float2* __restrict__ scr, const float2* __restrict__ twg, const unsigned char* __restrict__ S,
              MixParams mp, GenGeo gg, int n0, int fires, int mask_mode, float2* __restrict__ ghat_out)
{
    extern __shared__ __align__(16) unsigned char smraw[];
    const int N = gg.N, W = gg.W, Wp = gen_wp(W);
    GenSmem s(smraw, N, W);
    const int tiles = (N + W - 1) / W;
    const int n = n0 + (int)(blockIdx.x / tiles), y0 = (int)(blockIdx.x % tiles) * W;
    const size_t px = (size_t)N * N;
    for (int i = threadIdx.x; i < N; i += blockDim.x) s.tw[i] = twg[i];
    for (int i = threadIdx.x; i < N * W; i += blockDim.x) {
        const int x = i % N, w = i / N, y = y0 + w;
        float2 v = make_float2(0.f, 0.f);
        if (y < N) {
            v = gen_mix(cur, gg, mp, n, y, x, fires != 0);
            if (mask_mode && !S[(size_t)n * px + (size_t)y * N + x]) v = make_float2(0.f, 0.f);
            if (ghat_out) ghat_out[(size_t)n * px + (size_t)y * N + x] = v;
        }
        s.a[x * Wp + w] = v;
    }
    __syncthreads();
    const float2* r = gen_fft(s.a, s.b, s.tw, gg, false);
    for (int i = threadIdx.x; i < N * W; i += blockDim.x) {
        const int x = i % N, w = i / N, y = y0 + w;
        if (y < N) scr[(size_t)n * px + (size_t)y * N + x] = r[x * Wp + w];
    }
}

// K2: W columns: forward FFT along y, error metric + Fourier-modulus constraint, inverse FFT along y (unnormalised);
// mode 0 = all three, 1 = forward only, 2 = inverse only.  A: natural native order, A < 0 = unmeasured.
__global__ void __launch_bounds__(GEN_NT)
k_gen_col(float2* __restrict__ scr, const float* __restrict__ A, const float2* __restrict__ twg, double* __restrict__ partial,
          GenGeo gg, int n0, int mode, float scale)
{
    extern __shared__ __align__(16) unsigned char smraw[];
    const int N = gg.N, W = gg.W, Wp = gen_wp(W);
    GenSmem s(smraw, N, W);
    const int tiles = (N + W - 1) / W;
    const int n = n0 + (int)(blockIdx.x / tiles), tile = (int)(blockIdx.x % tiles), x0 = tile * W;
    const size_t px = (size_t)N * N;
    for (int i = threadIdx.x; i < N; i += blockDim.x) s.tw[i] = twg[i];
    for (int i = threadIdx.x; i < N * W; i += blockDim.x) {
        const int w = i % W, y = i / W, x = x0 + w;
        s.a[y * Wp + w] = x < N ? scr[(size_t)n * px + (size_t)y * N + x] : make_float2(0.f, 0.f);
    }
    __syncthreads();
    float2* r = s.a;
    float2* other = s.b;
    if (mode != 2) { r = gen_fft(s.a, s.b, s.tw, gg, false); other = (r == s.a) ? s.b : s.a; }
    if (mode == 0) {
        double acc = 0.0;
        for (int i = threadIdx.x; i < N * W; i += blockDim.x) {
            const int w = i % W, ky = i / W, x = x0 + w;
            if (x >= N) continue;
            float2 G = r[ky * Wp + w];
            const float a = A[(size_t)n * px + (size_t)ky * N + x];
            float f = scale;
            if (a >= 0.f) {
                const float m2 = G.x * G.x + G.y * G.y;
                if (m2 >= 1.17549435e-38f) {
                    const float mag = sqrtf(m2);
                    const float d = mag - a;
                    acc += (double)d * (double)d;
                    f = a / mag * scale;
                } else {
                    acc += (double)a * (double)a;
                    G = make_float2(1.f, 0.f);
                    f = a * scale;
                }
            }
            r[ky * Wp + w] = make_float2(G.x * f, G.y * f);
        }
        // fixed-order block reduction of the error numerator
        for (int o = 16; o > 0; o >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, o);
        if ((threadIdx.x & 31) == 0) s.red[threadIdx.x >> 5] = acc;
        __syncthreads();
        if (threadIdx.x == 0) {
            double t = 0.0;
            for (int w = 0; w < (int)blockDim.x / 32; ++w) t += s.red[w];
            partial[(size_t)n * tiles + tile] = t;
        }
    }
    if (mode != 1) r = gen_fft(r, other, s.tw, gg, true);
    for (int i = threadIdx.x; i < N * W; i += blockDim.x) {
        const int w = i % W, y = i / W, x = x0 + w;
        if (x < N) scr[(size_t)n * px + (size_t)y * N + x] = r[y * Wp + w];
    }
}

// K3: inverse FFT along x of W rows (times `scale`) + support / update (cpra_set_update); hio = 0: plain
// scaled inverse transform.  ghat: the mixed input stored by K1, or NULL = re-mix from the previous state.
__global__ void __launch_bounds__(GEN_NT)
k_gen_row_inv(const float2* __restrict__ scr, const float2* __restrict__ cur, float2* __restrict__ nxt, const float2* __restrict__ twg,
              const unsigned char* __restrict__ S, MixParams mp, GenGeo gg, int n0, int fires, int hio, float scale,
              const float2* __restrict__ ghat)
{
    extern __shared__ __align__(16) unsigned char smraw[];
    const int N = gg.N, W = gg.W, Wp = gen_wp(W);
    GenSmem s(smraw, N, W);
    const int tiles = (N + W - 1) / W;
    const int n = n0 + (int)(blockIdx.x / tiles), y0 = (int)(blockIdx.x % tiles) * W;
    const size_t px = (size_t)N * N;
    for (int i = threadIdx.x; i < N; i += blockDim.x) s.tw[i] = twg[i];
    for (int i = threadIdx.x; i < N * W; i += blockDim.x) {
        const int x = i % N, w = i / N, y = y0 + w;
        s.a[x * Wp + w] = y < N ? scr[(size_t)n * px + (size_t)y * N + x] : make_float2(0.f, 0.f);
    }
    __syncthreads();
    const float2* r = gen_fft(s.a, s.b, s.tw, gg, true);
    for (int i = threadIdx.x; i < N * W; i += blockDim.x) {
        const int x = i % N, w = i / N, y = y0 + w;
        if (y >= N) continue;
        const size_t o = (size_t)n * px + (size_t)y * N + x;
        float2 gp = r[x * Wp + w];
        gp.x *= scale; gp.y *= scale;
        if (hio && !S[o]) {
            const float2 gh = ghat ? ghat[o] : gen_mix(cur, gg, mp, n, y, x, fires != 0);
            gp = make_float2(fmaf(mp.c_gp, gp.x, mp.c_ghat * gh.x), fmaf(mp.c_gp, gp.y, mp.c_ghat * gh.y));
        }
        nxt[o] = gp;
    }
}

// A0 on natural arrays: A = sqrt(max(I, 0)), mask folded in as A = -1, detector-centred -> native (ifftshift); den_n
__global__ void k_gen_set_data(const float* __restrict__ I, const unsigned char* __restrict__ mask, float* __restrict__ A, double* __restrict__ den, int N)
{
    const int n = blockIdx.x, h = N / 2;
    double acc = 0.0;
    for (int i = threadIdx.x; i < N * N; i += blockDim.x) {
        const int yc = i / N, xc = i % N;
        const size_t src = (size_t)n * N * N + i;
        const float v = fmaxf(I[src], 0.f);
        const bool m = mask ? (mask[src] != 0) : true;
        A[(size_t)n * N * N + (size_t)((yc + h) % N) * N + (xc + h) % N] = m ? sqrtf(v) : -1.f;
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
// natural spectrum [n][kz][ku] -> [n][ku][kz] (what k_assemble reads)
__global__ void k_gen_transpose(const float2* __restrict__ in, float2* __restrict__ out, int N, size_t total)
{
    const size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= total) return;
    const int kz = (int)(i % N), ku = (int)((i / N) % N);
    const size_t n = i / ((size_t)N * N);
    out[i] = in[(n * N + kz) * N + ku];
}

}  // namespace cpra
