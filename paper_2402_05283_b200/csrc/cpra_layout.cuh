// cpra_layout.cuh -- one-off kernels of the CPRA library (not on the timed path): conversions between
// the caller's natural [n][y][x] arrays and the internal tiled layouts of cpra_kernels.cuh, the
// error finalisation, and the Fourier-slice assembly.
#pragma once
#include "cpra_kernels.cuh"

namespace cpra {

// float index of the real part of element (n, y, x) of the row-tiled state; the imaginary part is 2
// floats further (quad = [re_a, re_b, im_a, im_b])
__device__ __forceinline__ size_t st_idx(const Geo& g, int n, int y, int x)
{
    const int tb = g.TB, np = tb / 2;
    return ((((size_t)n * (g.N / tb) + (y / tb)) * g.N + ppos(x, tb)) * np + (y % tb) / 2) * 4 + (y & 1);
}
// the same for element (n, py, px) of the column-tiled scratch
__device__ __forceinline__ size_t sc_idx(const Geo& g, int n, int py, int px)
{
    const int tb = g.TB, np = tb / 2;
    return ((((size_t)n * (g.N / tb) + (px / tb)) * g.N + ppos(py, tb, (px / tb) & 1)) * np + sw((px % tb) / 2, py, np)) * 4 + (px & 1);
}
__device__ __forceinline__ size_t a_idx(const Geo& g, int n, int py, int px)
{
    const int tb = g.TB, np = tb / 2, RL = g.RL;
    return ((((size_t)n * (g.N / tb) + (px / tb)) * (g.N / RL) + (py / RL)) * np + (px % tb) / 2) * (2 * RL) + (py % RL) * 2 + (px & 1);
}
__device__ __forceinline__ float2 ld_c(const float* __restrict__ a, size_t i) { return make_float2(a[i], a[i + 2]); }
__device__ __forceinline__ void st_c(float* __restrict__ a, size_t i, float2 v) { a[i] = v.x; a[i + 2] = v.y; }

// A0: A = sqrt(max(I, 0)) (A14), mask folded in as A = -1, detector-centred ->
// native (ifftshift, A11) -> the permuted order of the FFT kernels; den_n = sum_{M=1} max(I, 0).
// SET_DATA_SPLIT blocks per image, each a band of rows; the band sums go to part[n][band] and k_set_data_den adds
// them in band order (fixed order: deterministic).
constexpr int SET_DATA_SPLIT = 8;
__global__ void k_set_data(const float* __restrict__ I, const unsigned char* __restrict__ mask,
                           float* __restrict__ Aperm, double* __restrict__ part, Geo g)
{
    const int n = blockIdx.x / SET_DATA_SPLIT, band = blockIdx.x % SET_DATA_SPLIT, N = g.N, h = N / 2;
    const int rows = (N + SET_DATA_SPLIT - 1) / SET_DATA_SPLIT, y0 = band * rows, y1 = min(N, y0 + rows);
    double acc = 0.0;
    for (int i = y0 * N + threadIdx.x; i < y1 * N; i += blockDim.x) {
        const int yc = i / N, xc = i % N;
        const size_t src = (size_t)n * N * N + i;
        const float v = fmaxf(I[src], 0.f);
        const bool m = mask ? (mask[src] != 0) : true;
        const int ky = (yc + h) % N, kx = (xc + h) % N;
        Aperm[a_idx(g, n, fft_pos(ky, g.R0, g.R1, g.R2), fft_pos(kx, g.R0, g.R1, g.R2))] = m ? sqrtf(v) : -1.f;
        if (m) acc += (double)v;
    }
    __shared__ double red[32];
    for (int o = 16; o > 0; o >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, o);
    if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = acc;
    __syncthreads();
    if (threadIdx.x == 0) {
        double s = 0.0;
        for (int w = 0; w < (int)blockDim.x / 32; ++w) s += red[w];
        part[blockIdx.x] = s;
    }
}
__global__ void k_set_data_den(const double* __restrict__ part, double* __restrict__ den, int Np)
{
    const int n = blockIdx.x * blockDim.x + threadIdx.x;
    if (n >= Np) return;
    double s = 0.0;
    for (int b = 0; b < SET_DATA_SPLIT; ++b) s += part[n * SET_DATA_SPLIT + b];
    den[n] = s;
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

// position -> frequency (the inverse of fft_pos)
__host__ __device__ __forceinline__ int fft_unpos(int pos, int R0, int R1, int R2)
{
    const int k2 = pos % R2, k1 = (pos / R2) % R1, k0 = pos / (R2 * R1);
    return k0 + R0 * (k1 + R1 * k2);
}

// natural [n][y][x] <-> row-tiled state; `masked` multiplies by the support.  One thread per (n, row tile, x): it
// moves the TB rows of the tile at column x, i.e. TB coalesced 8-byte accesses on the natural side (the lanes run
// along x) and the TB / 2 quads of one position = 64 or 128 contiguous bytes on the tiled side.  units = Np (N / TB) N.
__global__ void k_pack_state(const float2* __restrict__ in, float* __restrict__ st, Geo g, size_t units)
{
    const size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= units) return;
    const int N = g.N, tb = g.TB, np = tb / 2;
    const int x = (int)(i % N);
    const size_t nrt = i / N;                        // n (N / TB) + rt
    const int rt = (int)(nrt % (N / tb));
    const size_t n = nrt / (N / tb);
    const float2* __restrict__ src = in + (n * N + (size_t)rt * tb) * N + x;
    float4* __restrict__ dst = reinterpret_cast<float4*>(st) + (nrt * N + ppos(x, tb)) * np;
#pragma unroll
    for (int j = 0; j < NPAIR; ++j) {
        if (j >= np) break;
        const float2 a = src[(size_t)(2 * j) * N], b = src[(size_t)(2 * j + 1) * N];
        dst[j] = make_float4(a.x, b.x, a.y, b.y);
    }
}
__global__ void k_unpack_state(const float* __restrict__ st, const uint16_t* __restrict__ S16,
                               float2* __restrict__ out, Geo g, size_t units, int masked)
{
    const size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= units) return;
    const int N = g.N, tb = g.TB, np = tb / 2;
    const int x = (int)(i % N);
    const size_t nrt = i / N;
    const int rt = (int)(nrt % (N / tb));
    const size_t n = nrt / (N / tb);
    const float4* __restrict__ src = reinterpret_cast<const float4*>(st) + (nrt * N + ppos(x, tb)) * np;
    float2* __restrict__ dst = out + (n * N + (size_t)rt * tb) * N + x;
    const int y0 = rt * tb;
    const unsigned bits = masked ? ((unsigned)S16[(n * (N / 16) + y0 / 16) * N + x] >> (y0 % 16)) : 0xffffu;
#pragma unroll
    for (int j = 0; j < NPAIR; ++j) {
        if (j >= np) break;
        const float4 q = src[j];
        dst[(size_t)(2 * j) * N] = ((bits >> (2 * j)) & 1) ? make_float2(q.x, q.z) : make_float2(0.f, 0.f);
        dst[(size_t)(2 * j + 1) * N] = ((bits >> (2 * j + 1)) & 1) ? make_float2(q.y, q.w) : make_float2(0.f, 0.f);
    }
}
// natural-order spectrum [n][ky][kx] <-> column-tiled permuted scratch.  One block per (n, group of PB consecutive
// scratch rows py): in every column tile those rows are PB x TB/2 quads = one contiguous piece (512 B at PB = TB = 8),
// read / written with the lanes along it; the permutation along x happens in shared memory (PB rows of N complex
// numbers), and each of the PB natural rows ky = unpos(py) moves coalesced.  PB divides 8.
__host__ __device__ __forceinline__ int spectrum_rows_per_block(int N) { return N <= 512 ? 8 : 4; }   // PB N 8 bytes <= 32 KiB
// fft_unpos with the radices (powers of two on this path) given as shifts: no division per element
__host__ __device__ __forceinline__ int ilog2_of(int v) { int l = 0; while ((1 << l) < v) ++l; return l; }
struct Unpos {
    int l1, l2, l0s;   // log2 R1, log2 R2, log2 (R2 R1)... and the shift of k2 in the result
    int R0, m1, m2;
    __device__ __forceinline__ explicit Unpos(const Geo& g)
        : l1(ilog2_of(g.R1)), l2(ilog2_of(g.R2)), l0s(0), R0(g.R0), m1(g.R1 - 1), m2(g.R2 - 1) {}
    __device__ __forceinline__ int operator()(int pos) const
    {
        const int k2 = pos & m2, k1 = (pos >> l2) & m1, k0 = pos >> (l2 + l1);
        return k0 + R0 * (k1 + (k2 << l1));
    }
};
__global__ void k_unpack_spectrum(const float* __restrict__ scr, float2* __restrict__ out, Geo g)
{
    extern __shared__ __align__(16) float2 rowbuf[];
    const int N = g.N, tb = g.TB, np = tb / 2, nct = N / tb, PB = spectrum_rows_per_block(N);
    const int py0 = (int)(blockIdx.x % (N / PB)) * PB;
    const size_t n = blockIdx.x / (N / PB);
    const float4* __restrict__ src = reinterpret_cast<const float4*>(scr);
    const Unpos unpos(g);
    const int lnp = ilog2_of(np), lpb = ilog2_of(PB);
    for (int t = threadIdx.x; t < PB * np * nct; t += blockDim.x) {
        const int slot = t & (np - 1), pp = (t >> lnp) & (PB - 1), ct = t >> (lnp + lpb);
        const int py = ppos(py0 + pp, tb, ct & 1);                  // the row stored at physical row py0 + pp (ppos is an involution)
        const float4 v = src[((n * nct + ct) * N + py0 + pp) * np + slot];
        const int px = ct * tb + 2 * sw(slot, py, np);               // slot = j ^ s is its own inverse
        float2* __restrict__ row = rowbuf + (py - py0) * N;
        row[unpos(px)] = make_float2(v.x, v.z);
        row[unpos(px + 1)] = make_float2(v.y, v.w);
    }
    __syncthreads();
    for (int r = 0; r < PB; ++r) {
        float2* __restrict__ dst = out + (n * N + fft_unpos(py0 + r, g.R0, g.R1, g.R2)) * N;
        for (int x = threadIdx.x; x < N; x += blockDim.x) dst[x] = rowbuf[r * N + x];
    }
}
// zperm (a cube of N planes, Step D): plane n of the natural array goes to plane pos(n) of the scratch
__global__ void k_pack_spectrum(const float2* __restrict__ in, float* __restrict__ scr, Geo g, int zperm = 0)
{
    extern __shared__ __align__(16) float2 rowbuf[];
    const int N = g.N, tb = g.TB, np = tb / 2, nct = N / tb, PB = spectrum_rows_per_block(N);
    const int py0 = (int)(blockIdx.x % (N / PB)) * PB;
    const size_t n = blockIdx.x / (N / PB);
    const size_t nd = zperm ? (size_t)fft_pos((int)n, g.R0, g.R1, g.R2) : n;
    for (int r = 0; r < PB; ++r) {
        const float2* __restrict__ src = in + (n * N + fft_unpos(py0 + r, g.R0, g.R1, g.R2)) * N;
        for (int x = threadIdx.x; x < N; x += blockDim.x) rowbuf[r * N + x] = src[x];
    }
    __syncthreads();
    float4* __restrict__ dst = reinterpret_cast<float4*>(scr);
    const Unpos unpos(g);
    const int lnp = ilog2_of(np), lpb = ilog2_of(PB);
    for (int t = threadIdx.x; t < PB * np * nct; t += blockDim.x) {
        const int slot = t & (np - 1), pp = (t >> lnp) & (PB - 1), ct = t >> (lnp + lpb);
        const int py = ppos(py0 + pp, tb, ct & 1);
        const int px = ct * tb + 2 * sw(slot, py, np);
        const float2* __restrict__ row = rowbuf + (py - py0) * N;
        const float2 a = row[unpos(px)], b = row[unpos(px + 1)];
        dst[((nd * nct + ct) * N + py0 + pp) * np + slot] = make_float4(a.x, b.x, a.y, b.y);
    }
}
// the weights of Step D, float [kz][ky][kx] natural -> one float2 (w_a, w_b) per quad of the scratch layout, planes in
// position order: what k_pack_spectrum(zperm) does to the spectrum they belong to
__global__ void k_pack_weight(const float* __restrict__ in, float2* __restrict__ wq, Geo g)
{
    extern __shared__ __align__(16) float wrow[];
    const int N = g.N, tb = g.TB, np = tb / 2, nct = N / tb, PB = spectrum_rows_per_block(N);
    const int py0 = (int)(blockIdx.x % (N / PB)) * PB;
    const size_t n = blockIdx.x / (N / PB);
    const size_t nd = (size_t)fft_pos((int)n, g.R0, g.R1, g.R2);
    for (int r = 0; r < PB; ++r) {
        const float* __restrict__ src = in + (n * N + fft_unpos(py0 + r, g.R0, g.R1, g.R2)) * N;
        for (int x = threadIdx.x; x < N; x += blockDim.x) wrow[r * N + x] = src[x];
    }
    __syncthreads();
    const Unpos unpos(g);
    const int lnp = ilog2_of(np), lpb = ilog2_of(PB);
    for (int t = threadIdx.x; t < PB * np * nct; t += blockDim.x) {
        const int slot = t & (np - 1), pp = (t >> lnp) & (PB - 1), ct = t >> (lnp + lpb);
        const int py = ppos(py0 + pp, tb, ct & 1);
        const int px = ct * tb + 2 * sw(slot, py, np);
        const float* __restrict__ row = wrow + (py - py0) * N;
        wq[((nd * nct + ct) * N + py0 + pp) * np + slot] = make_float2(row[unpos(px)], row[unpos(px + 1)]);
    }
}
// spectrum of the assembly: column-tiled permuted scratch -> natural order, TRANSPOSED: Et[n][ku][kz],
// kz fastest, so that the gather kernel, which walks kz for fixed (n, ku), streams contiguous memory
__global__ void k_unpack_spectrum_T(const float* __restrict__ scr, float2* __restrict__ Et, Geo g, size_t total)
{
    const size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= total) return;
    const int N = g.N;
    const int kz = (int)(i % N), ku = (int)((i / N) % N), n = (int)(i / ((size_t)N * N));
    Et[i] = ld_c(scr, sc_idx(g, n, fft_pos(kz, g.R0, g.R1, g.R2), fft_pos(ku, g.R0, g.R1, g.R2)));
}
__global__ void k_pack_spectrum(const float2* __restrict__ in, float* __restrict__ scr, Geo g, size_t total)
{
    const size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= total) return;
    const int N = g.N;
    const int kx = (int)(i % N), ky = (int)((i / N) % N), n = (int)(i / ((size_t)N * N));
    st_c(scr, sc_idx(g, n, fft_pos(ky, g.R0, g.R1, g.R2), fft_pos(kx, g.R0, g.R1, g.R2)), in[i]);
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
// Et holds E_n = F[S_n g_n] in natural order, [n][ku][kz] (k_unpack_spectrum_T).  One thread per
// (ky, kx) computes the polar geometry in fp64 once, then walks kz: each of its taps is a contiguous
// stream.
//   uphi[U]      sorted unique ray directions in [0, 2 pi)
//   ustart[U+1]  contributors of unique ray u are rays[ustart[u] .. ustart[u+1])
//   rays[]       n | (neg << 30): the slice and whether the ray is its ku <= 0 half
// ------------------------------------------------------------------------------------------------
__global__ void k_assemble(const float2* __restrict__ Et, float2* __restrict__ vol, float* __restrict__ wgt,
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
        double vr = 0.0, vi = 0.0;
        float w = 0.f;
        if (mode == 1) {
            for (int n = 0; n < Np; ++n) {
                const float2 e = __ldg(Et + (size_t)n * N * N + iz);
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
                        const float2 e = __ldg(Et + ((size_t)n * N + iu) * N + iz);
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

// ------------------------------------------------------------------------------------------------
// A7, round 2: the same gather (same arithmetic, same results) laid out for the memory system.
//   k_assemble_geo     one thread per (ky, kx): the polar geometry in fp64, once, into a table
//   k_unpack_tile_T    scratch column tile -> Et[n][ku][kz]: the tile is read as it lies in HBM and every output
//                      row (all kz of one ku) is written contiguously
//   k_assemble_gather  a block = 32 kx x 32 kz at one ky; the lanes of a warp run along kz, so every tap is one
//                      coalesced 256-byte read of Et, and the tile leaves through shared memory as contiguous kx
//                      rows of the volume.  kz tiles are the slowest grid index: the 1/16 of Et that one kz tile
//                      touches stays in L2 while all (ky, kx) are served from it.
// ------------------------------------------------------------------------------------------------
struct AsmGeo {
    int mode;        // 0: outside (rho > N/2 - 1), 1: axis (rho = 0), 2: interpolate
    int ua, ub;      // bracketing unique rays
    int r0;          // floor(rho)
    double wp, wr;   // angular weight of ray ub, radial weight of sample r0 + 1
};
__global__ void k_assemble_geo(AsmGeo* __restrict__ geo, const double* __restrict__ uphi, int U, int N)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= N * N) return;
    const int h = N / 2, ix = i % N, iy = i / N;
    const int kx = ix < h ? ix : ix - N, ky = iy < h ? iy : iy - N;
    const double PI = 3.14159265358979323846264338327950288;
    const double rho = sqrt((double)kx * kx + (double)ky * ky);
    AsmGeo g;
    g.mode = 0; g.ua = g.ub = 0; g.r0 = 0; g.wp = 0.0; g.wr = 0.0;
    if (rho == 0.0) g.mode = 1;
    else if (rho <= (double)(h - 1)) {
        g.mode = 2;
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
        g.wp = (pb > pa) ? (phi - pa) / (pb - pa) : 0.0;
        g.r0 = (int)floor(rho);
        g.wr = rho - (double)g.r0;
        g.ua = a; g.ub = b;
    }
    geo[i] = g;
}

// one block per scratch column tile (n, ct): TB columns x N positions, contiguous in HBM
__global__ void k_unpack_tile_T(const float4* __restrict__ scr, float2* __restrict__ Et, Geo g)
{
    extern __shared__ __align__(16) float4 tile[];   // N * TB/2 quads, as in HBM
    const int N = g.N, tb = g.TB, np = tb / 2, nct = N / tb;
    const int n = blockIdx.x / nct, ct = blockIdx.x % nct;
    const float4* __restrict__ src = scr + ((size_t)n * nct + ct) * (size_t)N * np;
    for (int i = threadIdx.x; i < N * np; i += blockDim.x) tile[i] = src[i];
    __syncthreads();
    const float* __restrict__ t = reinterpret_cast<const float*>(tile);
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5, nw = blockDim.x >> 5;
    for (int c = wid; c < tb; c += nw) {
        const int ku = fft_unpos(ct * tb + c, g.R0, g.R1, g.R2);
        float2* __restrict__ out = Et + ((size_t)n * N + ku) * N;
        for (int kz = lane; kz < N; kz += 32) {
            const int py = fft_pos(kz, g.R0, g.R1, g.R2);
            const int q = (ppos(py, tb, ct & 1) * np + sw(c / 2, py, np)) * 4 + (c & 1);
            out[kz] = make_float2(t[q], t[q + 2]);
        }
    }
}

__global__ void __launch_bounds__(256)
k_assemble_gather(const float2* __restrict__ Et, float2* __restrict__ vol, float* __restrict__ wgt, const AsmGeo* __restrict__ geo,
                  const int* __restrict__ ustart, const int* __restrict__ rays, int N, int Np)
{
    __shared__ float2 tv[32][33];
    __shared__ float tw[32];
    const int xt = N / 32;                                   // kx tiles per row
    const int iz0 = (int)(blockIdx.x / ((unsigned)xt * N)) * 32;     // kz tile: slowest
    const int rem = (int)(blockIdx.x % ((unsigned)xt * N));
    const int iy = rem / xt, ix0 = (rem % xt) * 32;
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    const int iz = iz0 + lane, h = N / 2;
    const int ky = iy < h ? iy : iy - N, kz = iz < h ? iz : iz - N;
    for (int c = wid; c < 32; c += 8) {
        const int ix = ix0 + c, kx = ix < h ? ix : ix - N;
        const AsmGeo g = geo[iy * N + ix];
        double vr = 0.0, vi = 0.0;
        float w = 0.f;
        if (g.mode == 1) {
            const double sg = (iz & 1) ? -1.0 : 1.0;
            for (int n = 0; n < Np; ++n) {
                const float2 e = __ldg(Et + (size_t)n * N * N + iz);
                vr += sg * e.x; vi += sg * e.y;
            }
            vr /= Np; vi /= Np; w = 1.f;
        } else if (g.mode == 2) {
#pragma unroll
            for (int q = 0; q < 2; ++q) {
                const double wq = q ? g.wp : 1.0 - g.wp;
                if (wq == 0.0) continue;
                const int u = q ? g.ub : g.ua;
                const int c0 = ustart[u], c1 = ustart[u + 1];
#pragma unroll
                for (int rr = 0; rr < 2; ++rr) {
                    const double wrr = rr ? g.wr : 1.0 - g.wr;
                    if (wrr == 0.0) continue;
                    const int r = g.r0 + rr;                 // 0 <= r <= N/2 - 1
                    double sr = 0.0, si = 0.0;
                    for (int cc = c0; cc < c1; ++cc) {
                        const int code = rays[cc];
                        const int n = code & 0x3fffffff;
                        const int iu = ((code >> 30) && r) ? N - r : r;      // -r mod N
                        const float2 e = __ldg(Et + ((size_t)n * N + iu) * N + iz);
                        const bool neg = (iz + iu) & 1;                      // origin -> centre pixel
                        sr += neg ? -(double)e.x : (double)e.x;
                        si += neg ? -(double)e.y : (double)e.y;
                    }
                    const double wt = wq * wrr / (double)(c1 - c0);
                    vr += wt * sr;
                    vi += wt * si;
                }
            }
            w = 1.f;
        }
        if ((kx + ky + kz) & 1) { vr = -vr; vi = -vi; }
        tv[lane][c] = make_float2((float)vr, (float)vi);
        if (lane == 0) tw[c] = w;
    }
    __syncthreads();
    // rows of 32 consecutive kx: contiguous in the volume
    for (int z = wid; z < 32; z += 8) {
        const size_t o = ((size_t)(iz0 + z) * N + iy) * N + ix0 + lane;
        vol[o] = tv[z][lane];
        if (wgt) wgt[o] = tw[lane];
    }
}

}  // namespace cpra
