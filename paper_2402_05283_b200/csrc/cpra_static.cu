// cpra_static.cu -- cpra_fsc_static: the Fourier shell correlation (include/cpra.h) for callers
// that cannot allocate device memory (code under CUDA graph capture, serving loops, harnesses that forbid cudaMalloc).
// It needs no plan and no workspace: the shell accumulators, which cpra_fsc keeps in the caller's workspace, live in
// a file-scope __device__ array of fixed size.  Every GPU that loads libcpra.so holds that array until the process
// exits (CPRA_FSC_STATIC_SCRATCH_BYTES = 12312 bytes).
//
// The array's name in HOST code is a host-side stand-in for the symbol, not a device address: its device address is
// asked for once per device with cudaGetSymbolAddress (with that device current) and that pointer is what the
// kernels get.  All calls share the array and it keeps the last call's sums: every call clears it first, on the
// caller's stream, and two calls that overlap on the GPU (different streams, no dependency) race on it.
#include <cuda_runtime.h>
#include <mutex>
#include "../../include/cpra.h"

namespace {

constexpr int MAX_NS = CPRA_FSC_STATIC_MAX_N / 2 + 1;
static_assert(sizeof(double) * 3 * MAX_NS == CPRA_FSC_STATIC_SCRATCH_BYTES, "the header states the size of the array");

// [0, ns): Re sum F1 conj F2;  [ns, 2 ns): sum |F1|^2;  [2 ns, 3 ns): sum |F2|^2
static __device__ __align__(256) double g_fsc_static_scratch[3 * MAX_NS];

constexpr int MAX_DEVICES = 64;
std::mutex g_lock;
double* g_scratch_ptr[MAX_DEVICES];   // device address of g_fsc_static_scratch on device d (nullptr: not asked yet)
int g_sms[MAX_DEVICES];

// set-up, once per device, with that device current
int scratch_of_current_device(double** ptr, int* sms)
{
    int dev = -1;
    if (cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev >= MAX_DEVICES) return CPRA_ERR_CUDA;
    std::lock_guard<std::mutex> hold(g_lock);
    if (!g_scratch_ptr[dev]) {
        double* a = nullptr;
        if (cudaGetSymbolAddress((void**)&a, g_fsc_static_scratch) != cudaSuccess || !a) return CPRA_ERR_CUDA;
        int n = 0;
        if (cudaDeviceGetAttribute(&n, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess || n < 1) return CPRA_ERR_CUDA;
        g_scratch_ptr[dev] = a;
        g_sms[dev] = n;
    }
    *ptr = g_scratch_ptr[dev];
    *sms = g_sms[dev];
    return CPRA_OK;
}

__global__ void k_fsc_static_clear(double* __restrict__ acc, int n)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n) acc[i] = 0.0;
}

// the shell sums of cpra_fsc's k_fsc_accumulate, into the static array (acc = its device address)
__global__ void k_fsc_static_accumulate(const float2* __restrict__ F1, const float2* __restrict__ F2, double* __restrict__ acc, int N)
{
    __shared__ double sh[3 * MAX_NS];
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

__global__ void k_fsc_static_finalize(const double* __restrict__ acc, float* __restrict__ out, int ns)
{
    const int s = blockIdx.x * blockDim.x + threadIdx.x;
    if (s >= ns) return;
    const double d = sqrt(acc[ns + s] * acc[2 * ns + s]);
    out[s] = d > 0.0 ? (float)(acc[s] / d) : 0.f;
}

}  // namespace

extern "C" int cpra_fsc_static(int N, const float* d_F1, const float* d_F2, float* d_out, void* stream)
{
    if (!d_F1 || !d_F2 || !d_out || N < 2 || (N & 1)) return CPRA_ERR_INVALID_ARG;
    if (N > CPRA_FSC_STATIC_MAX_N) return CPRA_ERR_UNSUPPORTED_SIZE;   // the static array holds N / 2 + 1 <= 513 shells
    double* acc = nullptr;
    int sms = 0;
    if (int rc = scratch_of_current_device(&acc, &sms)) return rc;
    cudaStream_t st = (cudaStream_t)stream;
    const int ns = N / 2 + 1;
    k_fsc_static_clear<<<(3 * ns + 255) / 256, 256, 0, st>>>(acc, 3 * ns);
    k_fsc_static_accumulate<<<4 * sms, 256, 0, st>>>((const float2*)d_F1, (const float2*)d_F2, acc, N);
    k_fsc_static_finalize<<<(ns + 127) / 128, 128, 0, st>>>(acc, d_out, ns);
    return cudaGetLastError() == cudaSuccess ? CPRA_OK : CPRA_ERR_CUDA;
}
