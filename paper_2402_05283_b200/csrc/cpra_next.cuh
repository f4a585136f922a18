// cpra_next.cuh -- one-off kernels around the loop: shrink-wrap support update (f2), the
// episode bank and merge of Step C (f1).  Pointwise / reduction work on natural [n][y][x] arrays or through
// the index helpers of cpra_layout.cuh; none of it is on the timed path.  Reductions run in a fixed order in
// double precision: every result is deterministic.
#pragma once
#include "cpra_layout.cuh"

namespace cpra {

// ---------------------------------------------------------------------------------------------------
// f2: shrink-wrap (PAPER.md:82 "2D CSWA" ref [35], :104; reading A23)
//     b_n = G_sigma * |S_n g_n|,   S_n <- [ b_n >= threshold max b_n ]
// The blur is a product in Fourier space between the loop's own forward and inverse FFT kernels: |S g| is formed by the
// forward row pass as it loads the state (k_row_fwd<MIX_ABS>), the transfer function sits inside the column kernel.
// ---------------------------------------------------------------------------------------------------
// spectrum (scratch layout) *= exp(-2 pi^2 sigma^2 (ky^2 + kx^2) / N^2): the factor is the product of two entries of a table
// over the scratch POSITIONS, tab[pos(k)] = exp(-2 pi^2 sigma^2 k^2 / N^2), k signed, applied by k_col<COL_GAUSS> between its
// forward and inverse stages
__global__ void k_gauss_table(float* __restrict__ tab, Geo g, float sigma)
{
    const int N = g.N, k = blockIdx.x * blockDim.x + threadIdx.x;
    if (k >= N) return;
    const double c = -2.0 * 9.86960440108935861883 * (double)sigma * (double)sigma / ((double)N * N);
    const int ks = k < N / 2 ? k : k - N;
    tab[fft_pos(k, g.R0, g.R1, g.R2)] = (float)exp(c * (double)ks * (double)ks);
}
// per-image maximum of the real part of a state-layout stack (one block per image)
__global__ void k_image_max(const float4* __restrict__ st, float* __restrict__ mx, Geo g)
{
    const size_t nq = (size_t)g.N * g.N / 2;
    const float4* __restrict__ p = st + (size_t)blockIdx.x * nq;
    float m = -3.402823466e38f;
    for (size_t i = threadIdx.x; i < nq; i += blockDim.x) { const float4 v = p[i]; m = fmaxf(m, fmaxf(v.x, v.y)); }
    __shared__ float red[32];
    for (int o = 16; o > 0; o >>= 1) m = fmaxf(m, __shfl_xor_sync(0xffffffffu, m, o));
    if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = m;
    __syncthreads();
    if (threadIdx.x == 0) {
        for (int w = 1; w < (int)blockDim.x / 32; ++w) m = fmaxf(m, red[w]);
        mx[blockIdx.x] = m;
    }
}
// S16 word (n, y / 16, x): bit b = [ b(16 (y/16) + b, x) >= threshold * max_n ], max_n > 0
__global__ void k_threshold_pack(const float* __restrict__ st, const float* __restrict__ mx, uint16_t* __restrict__ S16,
                                 Geo g, size_t total16, float threshold)
{
    const size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= total16) return;
    const int N = g.N;
    const int x = (int)(i % N);
    const size_t nr = i / N;
    const int r16 = (int)(nr % (N / 16));
    const int n = (int)(nr / (N / 16));
    const float m = mx[n];
    const float t = threshold * m;
    unsigned bits = 0;
    for (int b = 0; b < 16; ++b)
        if (m > 0.f && st[st_idx(g, n, r16 * 16 + b, x)] >= t) bits |= 1u << b;
    S16[i] = (uint16_t)bits;
}
// bit-packed support -> u8 [n][y][x]
__global__ void k_unpack_support(const uint16_t* __restrict__ S16, unsigned char* __restrict__ S, int N, size_t total)
{
    const size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= total) return;
    const int x = (int)(i % N), y = (int)((i / N) % N);
    const size_t n = i / ((size_t)N * N);
    S[i] = (S16[(n * (N / 16) + y / 16) * N + x] >> (y % 16)) & 1;
}
// blurred image (real part of a state-layout stack) -> natural float [n][y][x] (diagnostic output of the shrink-wrap)
__global__ void k_unpack_real(const float* __restrict__ st, float* __restrict__ out, Geo g, size_t total)
{
    const size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= total) return;
    const int N = g.N;
    out[i] = st[st_idx(g, (int)(i / ((size_t)N * N)), (int)((i / N) % N), (int)(i % N))];
}

// ---------------------------------------------------------------------------------------------------
// f1: Step C.  The bank holds the N_l lowest-error episodes offered so far, natural
// [slot][n][y][x] complex fp32; an episode is the stack of supported estimates S_n g_n.
// ---------------------------------------------------------------------------------------------------
struct Bank {
    float2* ep;        // [NL][Np][N][N]
    double* E;         // [NL] reconstruction error of the kept episodes
    int* count;        // [1] episodes kept
    int* slot;         // [1] slot chosen by the last offer (-1: rejected)
    float* Ein;        // [2] staging for the offered error when it comes from the plan (E global)
    int* shift;        // [NL][Np][2] whole-pixel shifts (sy, sx) of the merge
    double* partial;   // [NL][MERGE_BLOCKS][4] partial inner products (c, c_T)
    int* twin;         // [NL]
    double* phase;     // [NL][2] unit factor conj(c)/|c| applied to the episode
    int* best;         // [1]
    int NL;
};
constexpr int MERGE_BLOCKS = 64;

// the rule of the bank: a free slot, else the worst kept episode if the offer is better (first worst on ties)
__global__ void k_offer_select(Bank b, const float* __restrict__ E_dev, double E_host)
{
    const double E = E_dev ? (double)*E_dev : E_host;
    int slot = -1;
    if (*b.count < b.NL) slot = (*b.count)++;
    else {
        int w = 0;
        for (int e = 1; e < b.NL; ++e) if (b.E[e] > b.E[w]) w = e;
        if (E < b.E[w]) slot = w;
    }
    if (slot >= 0) b.E[slot] = E;
    *b.slot = slot;
}
// copy the offered episode into the chosen slot: from a natural array, or from the plan's state (S g)
__global__ void k_offer_copy(Bank b, const float2* __restrict__ src, const float* __restrict__ st, const uint16_t* __restrict__ S16,
                             Geo g, size_t total)
{
    const int slot = *b.slot;
    if (slot < 0) return;
    const size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= total) return;
    float2 v;
    if (src) v = src[i];
    else {
        const int N = g.N;
        const int x = (int)(i % N), y = (int)((i / N) % N), n = (int)(i / ((size_t)N * N));
        v = ld_c(st, st_idx(g, n, y, x));
        if (!((S16[((size_t)n * (N / 16) + y / 16) * N + x] >> (y % 16)) & 1)) v = make_float2(0.f, 0.f);
    }
    b.ep[(size_t)slot * total + i] = v;
}

__device__ __forceinline__ double block_sum(double v, double* red)
{
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    __syncthreads();
    if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = v;
    __syncthreads();
    double s = 0.0;
    for (int w = 0; w < (int)blockDim.x / 32; ++w) s += red[w];
    return s;
}
// centre of mass of |O| about the centre pixel -> whole-pixel shift -round(com) (halves away from zero);
// one block per (episode, projection).  PAPER.md:64, reading A24.
__global__ void k_merge_com(Bank b, Geo g)
{
    const int e = blockIdx.x / g.Np, n = blockIdx.x % g.Np, N = g.N;
    if (e >= *b.count) return;
    __shared__ double red[32];
    const float2* __restrict__ o = b.ep + ((size_t)e * g.Np + n) * N * N;
    double m = 0.0, sy = 0.0, sx = 0.0;
    for (int i = threadIdx.x; i < N * N; i += blockDim.x) {
        const float2 v = o[i];
        const double w = sqrt((double)v.x * v.x + (double)v.y * v.y);
        m += w; sy += w * (double)(i / N - N / 2); sx += w * (double)(i % N - N / 2);
    }
    m = block_sum(m, red); sy = block_sum(sy, red); sx = block_sum(sx, red);
    if (threadIdx.x == 0) {
        const double cy = m > 0.0 ? sy / m : 0.0, cx = m > 0.0 ? sx / m : 0.0;
        b.shift[((size_t)e * g.Np + n) * 2] = -(int)(cy >= 0.0 ? floor(cy + 0.5) : -floor(-cy + 0.5));
        b.shift[((size_t)e * g.Np + n) * 2 + 1] = -(int)(cx >= 0.0 ? floor(cx + 0.5) : -floor(-cx + 0.5));
    }
}
__global__ void k_merge_best(Bank b)
{
    int w = 0;
    for (int e = 1; e < *b.count; ++e) if (b.E[e] < b.E[w]) w = e;
    *b.best = w;
}
__device__ __forceinline__ int wrapi(int a, int N) { return ((a % N) + N) % N; }
// inner products of the centred best episode with the centred episode e and with its twin T O = conj(O(-r)),
// on projection n_ref (or all of them, n_ref = -1): grid (MERGE_BLOCKS, NL)
__global__ void k_merge_inner(Bank b, Geo g, int n_ref)
{
    const int e = blockIdx.y, N = g.N, Np = g.Np;
    if (e >= *b.count) return;
    const int best = *b.best;
    __shared__ double red[32];
    double cr = 0.0, ci = 0.0, tr = 0.0, ti = 0.0;
    if (e != best) {
        const int n0 = n_ref < 0 ? 0 : n_ref, n1 = n_ref < 0 ? Np : n_ref + 1;
        const size_t px = (size_t)N * N, cnt = (size_t)(n1 - n0) * px;
        const size_t per = (cnt + gridDim.x - 1) / gridDim.x;
        const size_t i0 = (size_t)blockIdx.x * per, i1 = min(cnt, i0 + per);
        for (size_t i = i0 + threadIdx.x; i < i1; i += blockDim.x) {
            const int n = n0 + (int)(i / px), y = (int)((i % px) / N), x = (int)(i % N);
            const int* sb = b.shift + ((size_t)best * Np + n) * 2;
            const int* se = b.shift + ((size_t)e * Np + n) * 2;
            const float2 a = b.ep[((size_t)best * Np + n) * px + (size_t)wrapi(y - sb[0], N) * N + wrapi(x - sb[1], N)];
            const float2 v = b.ep[((size_t)e * Np + n) * px + (size_t)wrapi(y - se[0], N) * N + wrapi(x - se[1], N)];
            const float2 w = b.ep[((size_t)e * Np + n) * px + (size_t)wrapi(-y - se[0], N) * N + wrapi(-x - se[1], N)];
            cr += (double)a.x * v.x + (double)a.y * v.y;
            ci += (double)a.x * v.y - (double)a.y * v.x;
            tr += (double)a.x * w.x - (double)a.y * w.y;
            ti += -(double)a.x * w.y - (double)a.y * w.x;
        }
    }
    cr = block_sum(cr, red); ci = block_sum(ci, red); tr = block_sum(tr, red); ti = block_sum(ti, red);
    if (threadIdx.x == 0) {
        double* o = b.partial + ((size_t)e * gridDim.x + blockIdx.x) * 4;
        o[0] = cr; o[1] = ci; o[2] = tr; o[3] = ti;
    }
}
// twin iff |c_T| > |c|; the episode is multiplied by conj(c)/|c| of the chosen product (reading A25)
__global__ void k_merge_decide(Bank b)
{
    const int e = threadIdx.x;
    if (e >= *b.count) return;
    double cr = 0.0, ci = 0.0, tr = 0.0, ti = 0.0;
    for (int k = 0; k < MERGE_BLOCKS; ++k) {
        const double* o = b.partial + ((size_t)e * MERGE_BLOCKS + k) * 4;
        cr += o[0]; ci += o[1]; tr += o[2]; ti += o[3];
    }
    int twin = 0;
    double ur = 1.0, ui = 0.0;
    if (e != *b.best) {
        const double mc = sqrt(cr * cr + ci * ci), mt = sqrt(tr * tr + ti * ti);
        twin = mt > mc;
        const double m = twin ? mt : mc;
        if (m > 0.0) { ur = (twin ? tr : cr) / m; ui = -(twin ? ti : ci) / m; }
    }
    b.twin[e] = twin;
    b.phase[2 * e] = ur; b.phase[2 * e + 1] = ui;
}
// out_n = mean over the kept episodes of  u_e . (twin_e ? T : 1) shift_e O_e,n   -- one gather, no intermediate
__global__ void k_merge_average(Bank b, float2* __restrict__ out, Geo g, size_t total)
{
    const size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= total) return;
    const int N = g.N, Np = g.Np, L = *b.count;
    const size_t px = (size_t)N * N;
    const int x = (int)(i % N), y = (int)((i / N) % N), n = (int)(i / px);
    double sr = 0.0, si = 0.0;
    for (int e = 0; e < L; ++e) {
        const int* s = b.shift + ((size_t)e * Np + n) * 2;
        const int tw = b.twin[e];
        float2 v = b.ep[((size_t)e * Np + n) * px + (size_t)wrapi((tw ? -y : y) - s[0], N) * N + wrapi((tw ? -x : x) - s[1], N)];
        if (tw) v.y = -v.y;
        const double ur = b.phase[2 * e], ui = b.phase[2 * e + 1];
        sr += ur * (double)v.x - ui * (double)v.y;
        si += ur * (double)v.y + ui * (double)v.x;
    }
    out[i] = make_float2((float)(sr / L), (float)(si / L));
}

// ---------------------------------------------------------------------------------------------------
// f3: Step D's iterations (PAPER.md:72 ref [32]; reading A26) on natural-order N^3 arrays:
//     O = S3 . F3^-1[F];  F' = F3[O];  err = sqrt(sum_{W>0} |F' - E|^2 / sum_{W>0} |E|^2);  F = W > 0 ? E : F'
// The transforms are cpra_fft3; these are the pointwise steps with fixed-order double reductions.
// ---------------------------------------------------------------------------------------------------
// F = W > 0 ? E : 0; part[b] = sum over the block's slice of |E|^2 on the known voxels
__global__ void k_refine_init(const float2* __restrict__ E, const float* __restrict__ W, float2* __restrict__ F,
                              double* __restrict__ part, size_t n3)
{
    __shared__ double red[32];
    const size_t per = (n3 + gridDim.x - 1) / gridDim.x, i0 = (size_t)blockIdx.x * per, i1 = min(n3, i0 + per);
    double acc = 0.0;
    for (size_t i = i0 + threadIdx.x; i < i1; i += blockDim.x) {
        const bool known = W[i] > 0.f;
        const float2 e = E[i];
        F[i] = known ? e : make_float2(0.f, 0.f);
        if (known) acc += (double)e.x * e.x + (double)e.y * e.y;
    }
    acc = block_sum(acc, red);
    if (threadIdx.x == 0) part[blockIdx.x] = acc;
}
// T holds F'; on the known voxels the residual is accumulated and E is put back
__global__ void k_refine_replace(float2* __restrict__ T, const float2* __restrict__ E, const float* __restrict__ W,
                                 double* __restrict__ part, size_t n3)
{
    __shared__ double red[32];
    const size_t per = (n3 + gridDim.x - 1) / gridDim.x, i0 = (size_t)blockIdx.x * per, i1 = min(n3, i0 + per);
    double acc = 0.0;
    // four elements per pass, their loads issued together (the order of the additions is the element order, as before)
    for (size_t i = i0 + threadIdx.x; i < i1; i += (size_t)4 * blockDim.x) {
        float w[4];
        float2 e[4], t[4];
#pragma unroll
        for (int u = 0; u < 4; ++u) {
            const size_t k = i + (size_t)u * blockDim.x;
            w[u] = 0.f;
            if (k < i1) { w[u] = W[k]; e[u] = E[k]; t[u] = T[k]; }
        }
#pragma unroll
        for (int u = 0; u < 4; ++u) {
            if (w[u] > 0.f) {
                const double dr = (double)t[u].x - (double)e[u].x, di = (double)t[u].y - (double)e[u].y;
                acc += dr * dr + di * di;
                T[i + (size_t)u * blockDim.x] = e[u];
            }
        }
    }
    acc = block_sum(acc, red);
    if (threadIdx.x == 0) part[blockIdx.x] = acc;
}
// err = sqrt(sum num / sum den), one thread, fixed order
__global__ void k_refine_error(const double* __restrict__ num, const double* __restrict__ den, int nblk, float* __restrict__ err)
{
    double a = 0.0, b = 0.0;
    for (int i = 0; i < nblk; ++i) { a += num[i]; b += den[i]; }
    *err = b > 0.0 ? (float)sqrt(a / b) : 0.f;
}

// ---------------------------------------------------------------------------------------------------
// Step D's support (readings A29, A30), on natural [z][y][x] volumes.
// ---------------------------------------------------------------------------------------------------
// The visual hull of the 2D supports: S u8 [Np][N][N] (rows = z, columns = u), cs = (cos theta_n, sin theta_n) doubles.
// Voxel (z, y, x) stays iff for every n S_n[z][floor(u)] or S_n[z][floor(u) + 1] is set, u = c + (x - c) cos + (y - c) sin
// evaluated in double without contraction (the products and sums of the definition, one rounding each).
__global__ void k_backproject_support(const unsigned char* __restrict__ S, const double* __restrict__ cs, unsigned char* __restrict__ S3, int N, int Np)
{
    const size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    const size_t n3 = (size_t)N * N * N;
    if (i >= n3) return;
    const int x = (int)(i % N), y = (int)((i / N) % N), z = (int)(i / ((size_t)N * N)), c = N / 2;
    const double dx = (double)(x - c), dy = (double)(y - c);
    int in = 1;
    for (int n = 0; n < Np && in; ++n) {
        const double u = __dadd_rn(__dadd_rn((double)c, __dmul_rn(dx, cs[2 * n])), __dmul_rn(dy, cs[2 * n + 1]));
        const long u0 = (long)floor(u);
        const unsigned char* __restrict__ row = S + ((size_t)n * N + z) * N;
        const int a = (u0 >= 0 && u0 < N) ? row[u0] : 0, b = (u0 + 1 >= 0 && u0 + 1 < N) ? row[u0 + 1] : 0;
        in = a || b;
    }
    S3[i] = (unsigned char)in;
}
// (|O|, 0)
__global__ void k_abs3(const float2* __restrict__ O, float2* __restrict__ out, size_t n3)
{
    const size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n3) return;
    const float2 v = O[i];
    out[i] = make_float2(sqrtf(v.x * v.x + v.y * v.y), 0.f);
}
// maximum of the real part of every z plane (one block per plane), then of the planes (one block): mx[0]
__global__ void k_plane_max(const float2* __restrict__ v, float* __restrict__ mx, size_t px)
{
    const float2* __restrict__ p = v + (size_t)blockIdx.x * px;
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
__global__ void k_max_final(float* __restrict__ mx, int n)
{
    float m = -3.402823466e38f;
    for (int i = threadIdx.x; i < n; i += blockDim.x) m = fmaxf(m, mx[i]);
    __shared__ float red[32];
    for (int o = 16; o > 0; o >>= 1) m = fmaxf(m, __shfl_xor_sync(0xffffffffu, m, o));
    if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = m;
    __syncthreads();   // every thread has read its share of mx before mx[0] is overwritten
    if (threadIdx.x == 0) {
        for (int w = 1; w < (int)blockDim.x / 32; ++w) m = fmaxf(m, red[w]);
        mx[0] = m;
    }
}
// S3 <- [ b >= threshold max b ], max b = mx[0] > 0; blurred (optional): b
__global__ void k_threshold3(const float2* __restrict__ b, const float* __restrict__ mx, unsigned char* __restrict__ S3,
                             float* __restrict__ blurred, size_t n3, float threshold)
{
    const size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n3) return;
    const float m = mx[0], v = b[i].x;
    S3[i] = (m > 0.f && v >= threshold * m) ? 1 : 0;
    if (blurred) blurred[i] = v;
}

// Step D's iterations with the cube kept in the loop's own layouts (power-of-two N): the spectrum F, the assembled
// spectrum E and the weights W live quad by quad in the scratch layout with the planes in position order (k_pack_spectrum
// / k_pack_weight with zperm), so these run over quads: a = (x, z), b = (y, w) are the two complex numbers of a quad.
// F = E on the known voxels (W > 0), 0 elsewhere; part[block] = sum over the block's known voxels of |E|^2
__global__ void k_refine_init_q(const float4* __restrict__ E, const float2* __restrict__ W, float4* __restrict__ F,
                                double* __restrict__ part, size_t nq)
{
    __shared__ double red[32];
    const size_t per = (nq + gridDim.x - 1) / gridDim.x, i0 = (size_t)blockIdx.x * per, i1 = min(nq, i0 + per);
    double acc = 0.0;
    for (size_t i = i0 + threadIdx.x; i < i1; i += blockDim.x) {
        const float2 w = W[i];
        const float4 e = E[i];
        const bool ka = w.x > 0.f, kb = w.y > 0.f;
        if (ka) acc += (double)e.x * e.x + (double)e.z * e.z;
        if (kb) acc += (double)e.y * e.y + (double)e.w * e.w;
        F[i] = make_float4(ka ? e.x : 0.f, kb ? e.y : 0.f, ka ? e.z : 0.f, kb ? e.w : 0.f);
    }
    acc = block_sum(acc, red);
    if (threadIdx.x == 0) part[blockIdx.x] = acc;
}
// F holds F'; on the known voxels the residual |F' - E|^2 is accumulated and E is put back
__global__ void k_refine_replace_q(float4* __restrict__ F, const float4* __restrict__ E, const float2* __restrict__ W,
                                   double* __restrict__ part, size_t nq)
{
    __shared__ double red[32];
    const size_t per = (nq + gridDim.x - 1) / gridDim.x, i0 = (size_t)blockIdx.x * per, i1 = min(nq, i0 + per);
    double acc = 0.0;
    for (size_t i = i0 + threadIdx.x; i < i1; i += (size_t)2 * blockDim.x) {
        float2 w[2];
        float4 e[2], t[2];
#pragma unroll
        for (int u = 0; u < 2; ++u) {
            const size_t k = i + (size_t)u * blockDim.x;
            w[u] = make_float2(0.f, 0.f);
            if (k < i1) { w[u] = W[k]; e[u] = E[k]; t[u] = F[k]; }
        }
#pragma unroll
        for (int u = 0; u < 2; ++u) {
            const bool ka = w[u].x > 0.f, kb = w[u].y > 0.f;
            if (!(ka || kb)) continue;
            if (ka) { const double dr = (double)t[u].x - (double)e[u].x, di = (double)t[u].z - (double)e[u].z; acc += dr * dr + di * di; }
            if (kb) { const double dr = (double)t[u].y - (double)e[u].y, di = (double)t[u].w - (double)e[u].w; acc += dr * dr + di * di; }
            F[i + (size_t)u * blockDim.x] = make_float4(ka ? e[u].x : t[u].x, kb ? e[u].y : t[u].y, ka ? e[u].z : t[u].z, kb ? e[u].w : t[u].w);
        }
    }
    acc = block_sum(acc, red);
    if (threadIdx.x == 0) part[blockIdx.x] = acc;
}
// the cube's spectrum in the scratch layout, planes in position order, *= exp(-2 pi^2 sigma^2 |k|^2 / N^2): three entries of
// the table over positions (see k_gauss_table) per quad
__global__ void k_gauss3_q(float4* __restrict__ scr, Geo g, size_t nquads, float sigma)
{
    extern __shared__ float gtab[];
    const int N = g.N, tb = g.TB, np = tb / 2;
    const double c = -2.0 * 9.86960440108935861883 * (double)sigma * (double)sigma / ((double)N * N);
    for (int k = threadIdx.x; k < N; k += blockDim.x) {
        const int ks = k < N / 2 ? k : k - N;
        gtab[fft_pos(k, g.R0, g.R1, g.R2)] = (float)exp(c * (double)ks * (double)ks);
    }
    __syncthreads();
    const size_t per_image = (size_t)N * N / 2;
    for (size_t q = (size_t)blockIdx.x * blockDim.x + threadIdx.x; q < nquads; q += (size_t)gridDim.x * blockDim.x) {
        const int qi = (int)(q % per_image), pz = (int)(q / per_image);
        const int slot = qi % np, phys = (qi / np) % N, ct = qi / (np * N);
        const int py = ppos(phys, tb, ct & 1);
        const int px = ct * tb + 2 * sw(slot, py, np);
        const float f = gtab[pz] * gtab[py], fa = f * gtab[px], fb = f * gtab[px + 1];
        float4 v = scr[q];
        v.x *= fa; v.y *= fb; v.z *= fa; v.w *= fb;
        scr[q] = v;
    }
}
// mx[i] = mx[0] for all i < n (after k_max_final): the per-image thresholds of k_threshold_pack become one
__global__ void k_max_broadcast(float* __restrict__ mx, int n)
{
    const float m = mx[0];
    __syncthreads();
    for (int i = 1 + threadIdx.x; i < n; i += blockDim.x) mx[i] = m;
}

// ---------------------------------------------------------------------------------------------------
// f4: the paper's quality metrics: Fourier shell correlation and PRTF.
// Shell sums are accumulated per block in shared memory and added to the global shell accumulators with
// double atomics (the order of the additions varies from run to run at the 1e-16 level).
// ---------------------------------------------------------------------------------------------------
// acc[0..ns): Re sum F1 conj F2;  acc[ns..2ns): sum |F1|^2;  acc[2ns..3ns): sum |F2|^2;  shell = round(|k|) <= N/2
__global__ void k_fsc_accumulate(const float2* __restrict__ F1, const float2* __restrict__ F2, double* __restrict__ acc, int N)
{
    extern __shared__ double sh[];   // 3 ns
    const int ns = N / 2 + 1;
    for (int i = threadIdx.x; i < 3 * ns; i += blockDim.x) sh[i] = 0.0;
    __syncthreads();
    const size_t n3 = (size_t)N * N * N;
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n3; i += (size_t)gridDim.x * blockDim.x) {
        const int ix = (int)(i % N), iy = (int)((i / N) % N), iz = (int)(i / ((size_t)N * N));
        const int kx = ix < N / 2 ? ix : ix - N, ky = iy < N / 2 ? iy : iy - N, kz = iz < N / 2 ? iz : iz - N;
        const int s = (int)floor(sqrt((double)kx * kx + (double)ky * ky + (double)kz * kz) + 0.5);
        if (s >= ns) continue;
        const float2 a = F1[i], b = F2[i];
        atomicAdd(&sh[s], (double)a.x * b.x + (double)a.y * b.y);
        atomicAdd(&sh[ns + s], (double)a.x * a.x + (double)a.y * a.y);
        atomicAdd(&sh[2 * ns + s], (double)b.x * b.x + (double)b.y * b.y);
    }
    __syncthreads();
    for (int i = threadIdx.x; i < 3 * ns; i += blockDim.x) if (sh[i] != 0.0) atomicAdd(&acc[i], sh[i]);
}
__global__ void k_fsc_finalize(const double* __restrict__ acc, float* __restrict__ out, int ns)
{
    const int s = blockIdx.x * blockDim.x + threadIdx.x;
    if (s >= ns) return;
    const double d = sqrt(acc[ns + s] * acc[2 * ns + s]);
    out[s] = d > 0.0 ? (float)(acc[s] / d) : 0.f;
}
// PRTF: scr holds F2[avg_n] in the scratch layout, Aperm the measured amplitudes (A < 0: unmeasured);
// acc[0..ns): sum of |G| / A over the measured pixels with A > 0 of ring s, acc[ns..2ns): their number
__global__ void k_prtf_accumulate(const float* __restrict__ scr, const float* __restrict__ Aperm, double* __restrict__ acc, Geo g, size_t total)
{
    extern __shared__ double sh[];   // 2 ns
    const int N = g.N, ns = N / 2 + 1;
    for (int i = threadIdx.x; i < 2 * ns; i += blockDim.x) sh[i] = 0.0;
    __syncthreads();
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < total; i += (size_t)gridDim.x * blockDim.x) {
        const int ix = (int)(i % N), iy = (int)((i / N) % N), n = (int)(i / ((size_t)N * N));
        const int kx = ix < N / 2 ? ix : ix - N, ky = iy < N / 2 ? iy : iy - N;
        const int s = (int)floor(sqrt((double)kx * kx + (double)ky * ky) + 0.5);
        if (s >= ns) continue;
        const int py = fft_pos(iy, g.R0, g.R1, g.R2), px = fft_pos(ix, g.R0, g.R1, g.R2);
        const float A = Aperm[a_idx(g, n, py, px)];
        if (!(A > 0.f)) continue;
        const float2 G = ld_c(scr, sc_idx(g, n, py, px));
        atomicAdd(&sh[s], sqrt((double)G.x * G.x + (double)G.y * G.y) / (double)A);
        atomicAdd(&sh[ns + s], 1.0);
    }
    __syncthreads();
    for (int i = threadIdx.x; i < 2 * ns; i += blockDim.x) if (sh[i] != 0.0) atomicAdd(&acc[i], sh[i]);
}
__global__ void k_prtf_finalize(const double* __restrict__ acc, float* __restrict__ out, int ns)
{
    const int s = blockIdx.x * blockDim.x + threadIdx.x;
    if (s < ns) out[s] = acc[ns + s] > 0.0 ? (float)(acc[s] / acc[ns + s]) : 0.f;
}

// ---------------------------------------------------------------------------------------------------
// Consistency of one episode before Step D (reading A28): phase gauge (every projection of one
// object has the same total) and twin chain (neighbouring projections are similar), on a natural
// [n][y][x] complex fp32 stack, in place.  scratch: double [Np][8] = (s_re, s_im, c_re, c_im, d_re, d_im, -, -),
// c_n = <O_{n-1}, O_n>, d_n = <O_{n-1}, T O_n> on the raw data; flags: int [Np].
// ---------------------------------------------------------------------------------------------------
__global__ void k_align_sums(const float2* __restrict__ ep, double* __restrict__ scratch, int N)
{
    __shared__ double red[32];
    const int n = blockIdx.x;
    const size_t px = (size_t)N * N;
    const float2* __restrict__ o = ep + (size_t)n * px;
    const float2* __restrict__ a = n > 0 ? ep + (size_t)(n - 1) * px : nullptr;
    double sr = 0.0, si = 0.0, cr = 0.0, ci = 0.0, dr = 0.0, di = 0.0;
    for (int i = threadIdx.x; i < N * N; i += blockDim.x) {
        const float2 v = o[i];
        sr += v.x; si += v.y;
        if (a) {
            const int y = i / N, x = i % N;
            const float2 w = o[(size_t)((N - y) % N) * N + (N - x) % N];    // T O = conj of this
            const float2 u = a[i];
            cr += (double)u.x * v.x + (double)u.y * v.y;  ci += (double)u.x * v.y - (double)u.y * v.x;      // conj(u) v
            dr += (double)u.x * w.x - (double)u.y * w.y;  di += -(double)u.x * w.y - (double)u.y * w.x;     // conj(u) conj(w)
        }
    }
    sr = block_sum(sr, red); si = block_sum(si, red); cr = block_sum(cr, red); ci = block_sum(ci, red);
    dr = block_sum(dr, red); di = block_sum(di, red);
    if (threadIdx.x == 0) {
        double* s = scratch + (size_t)n * 8;
        s[0] = sr; s[1] = si; s[2] = cr; s[3] = ci; s[4] = dr; s[5] = di;
    }
}
// unit phases u_n = conj(s_n)/|s_n| (into scratch[n][6..7]); relative twin flags from
// Re<O'_{n-1}, O'_n> = Re(conj(u_{n-1}) u_n c_n)  and  Re<O'_{n-1}, T O'_n> = Re(conj(u_{n-1}) conj(u_n) d_n);
// absolute flags by walking away from n_ref
__global__ void k_align_decide(double* __restrict__ scratch, int* __restrict__ flags, int Np, int n_ref)
{
    if (threadIdx.x != 0 || blockIdx.x != 0) return;
    for (int n = 0; n < Np; ++n) {
        double* s = scratch + (size_t)n * 8;
        const double m = sqrt(s[0] * s[0] + s[1] * s[1]);
        s[6] = m > 0.0 ? s[0] / m : 1.0;
        s[7] = m > 0.0 ? -s[1] / m : 0.0;
    }
    auto rel = [&](int n) -> int {   // does projection n flip relative to n - 1?
        const double* a = scratch + (size_t)(n - 1) * 8;
        const double* b = scratch + (size_t)n * 8;
        // conj(u_a) u_b and conj(u_a) conj(u_b)
        const double pr = a[6] * b[6] + a[7] * b[7], pi = a[6] * b[7] - a[7] * b[6];
        const double qr = a[6] * b[6] - a[7] * b[7], qi = -a[6] * b[7] - a[7] * b[6];
        const double pp = pr * b[2] - pi * b[3];
        const double qq = qr * b[4] - qi * b[5];
        return qq > pp;
    };
    flags[n_ref] = 0;
    for (int n = n_ref + 1; n < Np; ++n) flags[n] = flags[n - 1] ^ rel(n);
    for (int n = n_ref - 1; n >= 0; --n) flags[n] = flags[n + 1] ^ rel(n + 1);
}
// O_n <- u_n O_n, then its twin where flagged; every thread owns a pixel and its mirror partner
__global__ void k_align_apply(float2* __restrict__ ep, const double* __restrict__ scratch, const int* __restrict__ flags, int N, size_t total)
{
    const size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= total) return;
    const size_t px = (size_t)N * N;
    const int n = (int)(i / px), y = (int)((i % px) / N), x = (int)(i % N);
    const size_t j = (size_t)n * px + (size_t)((N - y) % N) * N + (N - x) % N;
    if (j < i) return;                                  // the partner's thread does both
    const double ur = scratch[(size_t)n * 8 + 6], ui = scratch[(size_t)n * 8 + 7];
    auto rot = [&](float2 v) { return make_float2((float)(ur * v.x - ui * v.y), (float)(ur * v.y + ui * v.x)); };
    float2 a = rot(ep[i]), b = rot(ep[j]);
    if (flags[n]) { const float2 t = a; a = make_float2(b.x, -b.y); b = make_float2(t.x, -t.y); }
    ep[i] = a;
    if (j != i) ep[j] = b;
}

}  // namespace cpra
