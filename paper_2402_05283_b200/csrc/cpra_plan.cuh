// cpra_plan.cuh -- the plan object behind include/cpra.h and the per-size launch logic.
// Host code only decides what to enqueue; every step of the path runs in the kernels of cpra_kernels.cuh
// / cpra_walk.cuh / cpra_image.cuh.  The kernels of one image size N are instantiated in ONE translation
// unit (cpra_inst.cu compiled with -DCPRA_INST_N=<N>: `template struct Launch<N>`), so that the sizes
// build in parallel; cpra_api.cu sees `extern template` declarations only.
#pragma once
#include <algorithm>
#include <cmath>
#include <cstring>
#include <new>
#include <vector>

#include "../../include/cpra.h"
#include <cuda.h>

#include "cpra_image.cuh"
#include "cpra_cluster.cuh"
#include "cpra_walk.cuh"
#include "cpra_generic.cuh"

struct cpra_plan_s {
    int N = 0, Np = 0;
    unsigned flags = 0;
    cudaStream_t stream = nullptr;
    cpra::Geo geo{};
    // workspace carve-up
    char* ws = nullptr;
    size_t ws_bytes = 0;
    float2* tw = nullptr;
    float* A = nullptr;
    uint16_t* S16 = nullptr;
    float4* st[2] = {nullptr, nullptr};
    float4* scr = nullptr;
    float4* scr2 = nullptr;   // second spectrum buffer: k_row_walk reads one and writes the other
    CUtensorMap tm_scr[2];    // TMA descriptors of scr and scr2 for k_row_walk
    bool have_tmap = false;
    double* partial = nullptr;
    double* den = nullptr;
    double* uphi = nullptr;
    int* ustart = nullptr;
    int* rays = nullptr;
    float* mx = nullptr;      // per-image maxima of the shrink-wrap update
    double* shell = nullptr;  // shell sums of cpra_fsc / cpra_prtf
    double* align = nullptr;  // scratch of cpra_align_episode
    int cur = 0;
    // parameters / state
    int K = 1;
    float alpha[cpra::MAXK + 1] = {0};
    int n_ei = 1;
    int update = CPRA_UPDATE_HIO;
    int flip_seam = 0;        // cpra_set_seam
    int positivity = 0;       // cpra_set_positivity
    int walk_ctas = 0;        // cpra_set_walk_ctas: CTAs per SM of the fused row kernel (0 = library default)
    // sizes that are not powers of two (cpra_generic.cuh): natural-layout buffers in the same workspace
    bool generic = false;
    cpra::GenGeo gg{};
    unsigned char* S8 = nullptr;   // support, u8 [Np][N][N]
    int cluster = 0;          // cpra_set_cluster: CTAs per image of the whole-image kernel (0 = library default, -1 = never)
    // Step C bank (cpra_merge_*): caller-owned device buffer
    char* bank_buf = nullptr;
    size_t bank_bytes = 0;
    int bank_NL = 0;
    long t = 0;
    bool have_data = false, have_support = false, have_estimate = false, have_error = false;
    bool attrs_set = false;
    std::vector<double> angles;
    std::vector<float2> h_tw;
    std::vector<double> h_uphi;
    std::vector<int> h_ustart, h_rays;
    std::vector<double> h_cs;         // (cos theta_n, sin theta_n) of cpra_backproject_support
    long launches = 0;
    int chunk = 0;  // images per L2-resident chunk; 0 = all
    int sms = 148;     // SMs of the device
    bool walk = true;  // use k_row_walk where the plan allows it (CPRA_FLAG_NO_WALK switches it off)
    // per-kernel-class timing (cpra_profile): event pairs around every launch of the loop
    bool profiling = false;
    std::vector<cudaEvent_t> ev;      // 2 * PROF_PAIRS events, created on first use
    std::vector<int> ev_cls;          // class of each recorded pair
    double prof_ms[CPRA_PROFILE_CLASSES] = {0};
    long prof_n[CPRA_PROFILE_CLASSES] = {0};
};


namespace cpra {

inline size_t align256(size_t x) { return (x + 255) & ~(size_t)255; }

struct Carve {
    size_t off = 0;
    size_t take(size_t bytes) { const size_t o = off; off = align256(off + bytes); return o; }
};

struct Layout {
    size_t tw, A, S16, S8, st0, st1, scr, scr2, partial, den, uphi, ustart, rays, mx, shell, align, total;
};

inline Layout layout_of(int N, int Np, bool generic = false)
{
    const size_t px = (size_t)Np * N * N;
    Carve c;
    Layout L;
    L.tw = c.take(sizeof(float2) * 1024);   // >= tw_count<N>() for every N
    L.A = c.take(sizeof(float) * px);
    L.S16 = c.take(px / 8);
    L.S8 = c.take(generic ? px : 0);   // sizes that are not powers of two keep the support as bytes
    L.st0 = c.take(sizeof(float2) * px);
    L.st1 = c.take(sizeof(float2) * px);
    L.scr = c.take(sizeof(float2) * px);
    L.scr2 = c.take(sizeof(float2) * px);
    L.partial = c.take(sizeof(double) * (size_t)Np * std::max(N / 4 + 1, 8));   // >= N / Radix<N>::TB (or ceil(N / W)) tiles per image, >= SET_DATA_SPLIT
    L.den = c.take(sizeof(double) * Np);
    L.uphi = c.take(sizeof(double) * 2 * Np);
    L.ustart = c.take(sizeof(int) * (2 * (size_t)Np + 1));
    L.rays = c.take(sizeof(int) * 2 * (size_t)Np);
    L.mx = c.take(sizeof(float) * (size_t)Np);
    L.shell = c.take(sizeof(double) * 3 * (size_t)(N / 2 + 1));   // shell sums of cpra_fsc / cpra_prtf
    L.align = c.take(sizeof(double) * 9 * (size_t)Np);   // cpra_align_episode: sums, inner products, phases, flags
    L.total = c.off;
    return L;
}

inline bool is_pow2(int n) { return n > 0 && (n & (n - 1)) == 0; }

// per-stage twiddle tables of cpra_fft.cuh: (wr, wi), w = exp(-2 pi i n2 r / L), computed in double
// and rounded once
template <int N>
void build_twiddles(std::vector<float2>& t)
{
    using RX = Radix<N>;
    const double PI = 3.14159265358979323846264338327950288;
    t.clear();
    auto stage = [&](int L, int R) {
        const int M = L / R;
        for (int n2 = 0; n2 < M; ++n2)
            for (int r = 1; r < R; ++r) {
                const double a = -2.0 * PI * (double)(n2 * r) / (double)L;
                t.push_back(make_float2((float)std::cos(a), (float)std::sin(a)));
            }
    };
    stage(N, RX::R0);
    if (RX::S == 3) stage(N / RX::R0, RX::R1);
    t.resize(1024, make_float2(0.f, 0.f));
}

// every launch of a size-templated kernel goes through Launch<N> (explicitly instantiated per N)
// the one-CTA-per-image kernel exists for the 16-wide two-stage plans
template <int N> constexpr bool image_ok() { return N <= 128 && Radix<N>::S == 2 && tile_batch<N>() == TB; }

template <int N>
struct Launch {
    static int set_attrs();
    static int row_fwd(cpra_plan_s* p, const float4* cur, int mode, int n0, int nimg, float4* ghat_out = nullptr);
    static int col(cpra_plan_s* p, int mode, int n0, int nimg, float scale, float4* scr = nullptr, const float* table = nullptr);
    static int row_inv(cpra_plan_s* p, const float4* cur, float4* nxt, bool hio, int mode, float beta, float scale, int n0, int nimg,
                       const float4* scr = nullptr, const float4* ghat_in = nullptr);
    static int walk(cpra_plan_s* p, const float4* scr_in, float4* scr_out, const float4* gh_old, float4* gh_new, float beta, bool fires);
    static int iterate_walk(cpra_plan_s* p, int k, float beta, float scale);
    static int image(cpra_plan_s* p, const float4* cur, float4* nxt, int mode, float beta, float scale);
    static int fftz(cpra_plan_s* p, float2* vol, int sign);
    static int fftz_scr(cpra_plan_s* p, float4* scr, int sign, float scale);   // the cube in the scratch layout (Np == N)
    static int image_cl(cpra_plan_s* p, const float4* cur, float4* nxt, int mode, float beta, float scale, int C);
    static bool image_cl_ok(int C);
    static bool has_image() { return image_ok<N>(); }
};

#define CPRA_DISPATCH_N(N_, ...)                                                     \
    switch (N_) {                                                                    \
        case 16:   { constexpr int NN = 16;   __VA_ARGS__; break; }                  \
        case 32:   { constexpr int NN = 32;   __VA_ARGS__; break; }                  \
        case 64:   { constexpr int NN = 64;   __VA_ARGS__; break; }                  \
        case 128:  { constexpr int NN = 128;  __VA_ARGS__; break; }                  \
        case 256:  { constexpr int NN = 256;  __VA_ARGS__; break; }                  \
        case 512:  { constexpr int NN = 512;  __VA_ARGS__; break; }                  \
        case 1024: { constexpr int NN = 1024; __VA_ARGS__; break; }                  \
        default: return CPRA_ERR_UNSUPPORTED_SIZE;                                   \
    }

template <class F>
cudaError_t allow_smem(F* f, int bytes)
{
    return cudaFuncSetAttribute(reinterpret_cast<const void*>(f), cudaFuncAttributeMaxDynamicSharedMemorySize, bytes);
}

template <int N, int C, class ACC>
void set_attrs_cl(ACC& acc)
{
    if constexpr (cl_ok<N, C>()) {
        constexpr int SMB = cl_smem_bytes<N, C>();
        acc(allow_smem(k_image_cl<N, C, MIX_NONE>, SMB));
        acc(allow_smem(k_image_cl<N, C, MIX_K1>, SMB));
        acc(allow_smem(k_image_cl<N, C, MIX_GEN>, SMB));
        // cluster launches get the smallest shared-memory carveout that fits ONE block unless told otherwise
        acc(cudaFuncSetAttribute(reinterpret_cast<const void*>(k_image_cl<N, C, MIX_NONE>), cudaFuncAttributePreferredSharedMemoryCarveout, cudaSharedmemCarveoutMaxShared));
        acc(cudaFuncSetAttribute(reinterpret_cast<const void*>(k_image_cl<N, C, MIX_K1>), cudaFuncAttributePreferredSharedMemoryCarveout, cudaSharedmemCarveoutMaxShared));
        acc(cudaFuncSetAttribute(reinterpret_cast<const void*>(k_image_cl<N, C, MIX_GEN>), cudaFuncAttributePreferredSharedMemoryCarveout, cudaSharedmemCarveoutMaxShared));
        if constexpr (C > 8) {
            acc(cudaFuncSetAttribute(reinterpret_cast<const void*>(k_image_cl<N, C, MIX_NONE>), cudaFuncAttributeNonPortableClusterSizeAllowed, 1));
            acc(cudaFuncSetAttribute(reinterpret_cast<const void*>(k_image_cl<N, C, MIX_K1>), cudaFuncAttributeNonPortableClusterSizeAllowed, 1));
            acc(cudaFuncSetAttribute(reinterpret_cast<const void*>(k_image_cl<N, C, MIX_GEN>), cudaFuncAttributeNonPortableClusterSizeAllowed, 1));
        }
    }
}

template <int N>
int Launch<N>::set_attrs()
{
    static_assert(tw_count<N>() <= 1024, "twiddle region of the workspace too small");
    cudaError_t e = cudaSuccess;
    auto acc = [&](cudaError_t r) { if (e == cudaSuccess) e = r; };
    constexpr int SM = smem_bytes<N>();
    acc(allow_smem(k_row_fwd<N, MIX_NONE>, SM));
    acc(allow_smem(k_row_fwd<N, MIX_K1>, SM));
    acc(allow_smem(k_row_fwd<N, MIX_GEN>, SM));
    acc(allow_smem(k_row_fwd<N, MIX_MASK>, SM));
    acc(allow_smem(k_row_fwd<N, MIX_ABS>, SM));
    acc(allow_smem(k_col<N, COL_FULL>, SM));
    acc(allow_smem(k_col<N, COL_FWD>, SM));
    acc(allow_smem(k_col<N, COL_INV>, SM));
    acc(allow_smem(k_col<N, COL_GAUSS>, SM));
    acc(allow_smem(k_row_inv<N, ROWINV_PLAIN, MIX_NONE>, SM));
    acc(allow_smem(k_row_inv<N, ROWINV_HIO, MIX_NONE>, SM));
    acc(allow_smem(k_row_inv<N, ROWINV_HIO, MIX_K1>, SM));
    acc(allow_smem(k_row_inv<N, ROWINV_HIO, MIX_GEN>, SM));
    if constexpr (walk_ok<N>()) acc(allow_smem(k_row_walk<N>, walk_smem_bytes<N>()));
    set_attrs_cl<N, 1>(acc); set_attrs_cl<N, 2>(acc); set_attrs_cl<N, 4>(acc); set_attrs_cl<N, 8>(acc); set_attrs_cl<N, 16>(acc);
    acc(allow_smem(k_fft_z<N, false>, SM));
    acc(allow_smem(k_fft_z<N, true>, SM));
    acc(allow_smem(k_fft_z_scr<N, false>, SM));
    acc(allow_smem(k_fft_z_scr<N, true>, SM));
    if constexpr (image_ok<N>()) {
        constexpr int ISM = image_smem_bytes<N>();
        acc(allow_smem(k_image<N, MIX_NONE>, ISM));
        acc(allow_smem(k_image<N, MIX_K1>, ISM));
        acc(allow_smem(k_image<N, MIX_GEN>, ISM));
    }
    return e == cudaSuccess ? CPRA_OK : CPRA_ERR_CUDA;
}

inline MixParams mix_params(const cpra_plan_s* p, float beta = 0.f)
{
    MixParams mp;
    mp.K = p->K;
    for (int j = 0; j <= MAXK; ++j) mp.a[j] = j <= p->K ? p->alpha[j] : 0.f;
    // coefficients of the update outside the support (cpra_set_update)
    if (p->update == CPRA_UPDATE_RAAR) { mp.c_ghat = beta; mp.c_gp = 1.0f - 2.0f * beta; }
    else if (p->update == CPRA_UPDATE_ER) { mp.c_ghat = 0.f; mp.c_gp = 0.f; }
    else { mp.c_ghat = 1.0f; mp.c_gp = -beta; }
    mp.flip_seam = p->flip_seam;
    mp.positivity = p->positivity;
    return mp;
}

constexpr int PROF_PAIRS = 2048;

// fold the recorded event pairs into the per-class sums (synchronises the stream)
inline int prof_drain(cpra_plan_s* p)
{
    if (p->ev_cls.empty()) return CPRA_OK;
    if (cudaStreamSynchronize(p->stream) != cudaSuccess) return CPRA_ERR_CUDA;
    for (size_t i = 0; i < p->ev_cls.size(); ++i) {
        float ms = 0.f;
        if (cudaEventElapsedTime(&ms, p->ev[2 * i], p->ev[2 * i + 1]) != cudaSuccess) return CPRA_ERR_CUDA;
        p->prof_ms[p->ev_cls[i]] += (double)ms;
        p->prof_n[p->ev_cls[i]] += 1;
    }
    p->ev_cls.clear();
    return CPRA_OK;
}

struct ProfScope {
    cpra_plan_s* p;
    bool on;
    size_t slot = 0;
    ProfScope(cpra_plan_s* p_, int cls) : p(p_), on(p_->profiling)
    {
        if (!on) return;
        if (p->ev.empty()) {
            p->ev.resize(2 * PROF_PAIRS);
            for (auto& e : p->ev) cudaEventCreate(&e);
        }
        if (p->ev_cls.size() == PROF_PAIRS) prof_drain(p);
        slot = p->ev_cls.size();
        p->ev_cls.push_back(cls);
        cudaEventRecord(p->ev[2 * slot], p->stream);
    }
    ~ProfScope() { if (on) cudaEventRecord(p->ev[2 * slot + 1], p->stream); }
};

inline int check_launch(cpra_plan_s* p, int n = 1)
{
    p->launches += n;
    return cudaGetLastError() == cudaSuccess ? CPRA_OK : CPRA_ERR_CUDA;
}

// mix mode of one iteration: does the carousel fire, and which kernel variant serves it
inline int mix_mode(const cpra_plan_s* p, bool fires)
{
    if (!fires) return MIX_NONE;
    if (p->K == 0) return p->alpha[0] == 1.0f ? MIX_NONE : MIX_GEN;
    return p->K == 1 ? MIX_K1 : MIX_GEN;
}

template <int N>
int Launch<N>::row_fwd(cpra_plan_s* p, const float4* cur, int mode, int n0, int nimg, float4* ghat_out)
{
    constexpr int NT = Radix<N>::NT;
    const dim3 grid((unsigned)nimg * (N / tile_batch<N>()));
    const int smem = smem_bytes<N>();
    const MixParams mp = mix_params(p);
    ProfScope prof(p, CPRA_PROFILE_ROW_FWD);
#define ROWFWD(M) k_row_fwd<N, M><<<grid, NT, smem, p->stream>>>(cur, p->tm_scr[0], p->tw, p->S16, mp, p->Np, n0, nimg, ghat_out)
    switch (mode) {
        case MIX_NONE: ROWFWD(MIX_NONE); break;
        case MIX_K1: ROWFWD(MIX_K1); break;
        case MIX_GEN: ROWFWD(MIX_GEN); break;
        case MIX_ABS: ROWFWD(MIX_ABS); break;
        default: ROWFWD(MIX_MASK); break;
    }
#undef ROWFWD
    return check_launch(p);
}

template <int N>
int Launch<N>::col(cpra_plan_s* p, int mode, int n0, int nimg, float scale, float4* scr, const float* table)
{
    constexpr int NT = Radix<N>::NT;
    const dim3 grid((unsigned)nimg * (N / tile_batch<N>()));
    const int smem = smem_bytes<N>();
    ProfScope prof(p, CPRA_PROFILE_COL);
    if (!scr) scr = p->scr;
    switch (mode) {
        case COL_FULL: k_col<N, COL_FULL><<<grid, NT, smem, p->stream>>>(scr, p->A, p->tw, p->partial, n0, scale); break;
        case COL_FWD: k_col<N, COL_FWD><<<grid, NT, smem, p->stream>>>(scr, p->A, p->tw, p->partial, n0, scale); break;
        case COL_GAUSS: k_col<N, COL_GAUSS><<<grid, NT, smem, p->stream>>>(scr, table, p->tw, p->partial, n0, scale); break;
        default: k_col<N, COL_INV><<<grid, NT, smem, p->stream>>>(scr, p->A, p->tw, p->partial, n0, scale); break;
    }
    return check_launch(p);
}

template <int N>
int Launch<N>::row_inv(cpra_plan_s* p, const float4* cur, float4* nxt, bool hio, int mode, float beta, float scale, int n0, int nimg,
                       const float4* scr, const float4* ghat_in)
{
    constexpr int NT = Radix<N>::NT;
    const dim3 grid((unsigned)nimg * (N / tile_batch<N>()));
    const int smem = smem_bytes<N>();
    const MixParams mp = mix_params(p, beta);
    ProfScope prof(p, CPRA_PROFILE_ROW_INV);
    if (!scr) scr = p->scr;
#define ROWINV(H, M) k_row_inv<N, H, M><<<grid, NT, smem, p->stream>>>(p->tm_scr[scr == p->scr ? 0 : 1], cur, nxt, p->tw, p->S16, mp, beta, scale, p->Np, n0, nimg, ghat_in)
    if (!hio) ROWINV(ROWINV_PLAIN, MIX_NONE);
    else if (mode == MIX_NONE) ROWINV(ROWINV_HIO, MIX_NONE);
    else if (mode == MIX_K1) ROWINV(ROWINV_HIO, MIX_K1);
    else ROWINV(ROWINV_HIO, MIX_GEN);
#undef ROWINV
    return check_launch(p);
}

// TMA descriptor of a spectrum buffer as the contiguous tensor [n][ct][rt][split][inner floats], box =
// all column tiles of one row tile (see tma_load_tile).  cuTensorMapEncodeTiled is fetched through the runtime, so that the
// library does not link against the driver.
inline bool encode_scratch_tmap(CUtensorMap* tm, void* base, int N, int Np, int tb)
{
    typedef CUresult (*Encode)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*, const cuuint64_t*,
                               const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave, CUtensorMapSwizzle,
                               CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
    void* fn = nullptr;
    cudaDriverEntryPointQueryResult q;
    if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &q) != cudaSuccess || q != cudaDriverEntryPointSuccess || !fn) {
        (void)cudaGetLastError();
        return false;
    }
    const cuuint64_t blk = (cuuint64_t)tb * tb * 2, nt = (cuuint64_t)(N / tb);   // floats per block, tiles per side
    const cuuint64_t inner = blk < 256 ? blk : 256, split = blk / inner;          // box dimensions are limited to 256
    const cuuint64_t dims[5] = {inner, split, nt, nt, (cuuint64_t)Np};
    const cuuint64_t strides[4] = {inner * 4, blk * 4, blk * 4 * nt, blk * 4 * nt * nt};
    const cuuint32_t box[5] = {(cuuint32_t)inner, (cuuint32_t)split, 1u, (cuuint32_t)nt, 1u};
    const cuuint32_t estr[5] = {1u, 1u, 1u, 1u, 1u};
    return ((Encode)fn)(tm, CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 5, base, dims, strides, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE,
                        CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_NONE, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS;
}

// K3 of one iteration fused with K1 of the next (cpra_walk.cuh): walk_ctas_per_sm CTAs per SM, each a run of tiles
template <int N>
int Launch<N>::walk(cpra_plan_s* p, const float4* scr_in, float4* scr_out, const float4* gh_old, float4* gh_new, float beta, bool fires)
{
    if constexpr (walk_ok<N>()) {
        const int total = (N / tile_batch<N>()) * p->Np;
        const int per_sm = p->walk_ctas > 0 ? p->walk_ctas : walk_ctas_per_sm<N>();   // what the kernel's registers / shared memory allow
        const int ctas = std::min(total, per_sm * p->sms);
        const int per = (total + ctas - 1) / ctas;
        const dim3 grid((unsigned)((total + per - 1) / per));
        MixParams mp = mix_params(p, beta);
        if (!fires) { mp.a[0] = 1.0f; mp.a[1] = 0.0f; }   // no mix before the next iteration (n_ei > 1): ghat = g exactly
        ProfScope prof(p, CPRA_PROFILE_WALK);
        const CUtensorMap& tin = p->tm_scr[scr_in == p->scr ? 0 : 1];
        const CUtensorMap& tout = p->tm_scr[scr_out == p->scr ? 0 : 1];
        k_row_walk<N><<<grid, walk_threads<N>(), walk_smem_bytes<N>(), p->stream>>>(tin, tout, gh_old, gh_new, p->tw, p->S16, mp, beta, p->Np, per);
        return check_launch(p);
    } else {
        return CPRA_ERR_UNSUPPORTED_SIZE;
    }
}

// k iterations with the walking kernel: K1 (storing ghat) -> [K2 -> walk] x (k - 1) -> K2 -> K3 (reading ghat).
// With n_ei > 1 the walk of an iteration that is not followed by a mix runs with weights (1, 0).
template <int N>
int Launch<N>::iterate_walk(cpra_plan_s* p, int k, float beta, float scale)
{
    float4* g = p->st[p->cur];
    float4* other = p->st[p->cur ^ 1];
    // does the carousel mix open iteration t (reading A3); never for the uncoupled loop (K = 0, alpha_0 = 1)
    auto fires = [&](long t) { return p->K == 1 && (t % p->n_ei) == 0; };
    int rc = row_fwd(p, g, fires(p->t) ? MIX_K1 : MIX_NONE, 0, p->Np, other);
    float4 *sin = p->scr, *sout = p->scr2, *gh_old = other, *gh_new = g;
    for (int it = 0; it < k && rc == CPRA_OK; ++it) {
        rc = col(p, COL_FULL, 0, p->Np, scale, sin);
        if (rc != CPRA_OK) break;
        if (it == k - 1) {
            rc = row_inv(p, gh_old, gh_new, true, MIX_K1, beta, 1.0f, 0, p->Np, sin, gh_old);
        } else {
            rc = walk(p, sin, sout, gh_old, gh_new, beta, fires(p->t + it + 1));
            std::swap(sin, sout);
            std::swap(gh_old, gh_new);
        }
    }
    if (rc != CPRA_OK) return rc;
    p->cur = (gh_new == p->st[0]) ? 0 : 1;
    p->t += k;
    p->have_error = true;
    return CPRA_OK;
}

// the whole iteration of every projection in one launch (N <= 128, cpra_image.cuh)
template <int N>
int Launch<N>::image(cpra_plan_s* p, const float4* cur, float4* nxt, int mode, float beta, float scale)
{
    if constexpr (image_ok<N>()) {
        constexpr int NT = image_threads<N>(), ISM = image_smem_bytes<N>();
        const dim3 grid((unsigned)p->Np);
        const MixParams mp = mix_params(p, beta);
        ProfScope prof(p, CPRA_PROFILE_IMAGE);
#define IMG(M) k_image<N, M><<<grid, NT, ISM, p->stream>>>(cur, nxt, p->A, p->tw, p->S16, p->partial, mp, beta, scale, p->Np, 0)
        if (mode == MIX_NONE) IMG(MIX_NONE);
        else if (mode == MIX_K1) IMG(MIX_K1);
        else IMG(MIX_GEN);
#undef IMG
        return check_launch(p);
    } else {
        return CPRA_ERR_UNSUPPORTED_SIZE;
    }
}

// z lines of a natural-order N^3 cube, in place (sign = -1 forward, +1 inverse scaled by 1/N)
template <int N>
int Launch<N>::fftz(cpra_plan_s* p, float2* vol, int sign)
{
    const dim3 grid((unsigned)(N / tile_batch<N>()), (unsigned)N);
    if (sign < 0) k_fft_z<N, false><<<grid, Radix<N>::NT, smem_bytes<N>(), p->stream>>>(vol, p->tw, 1.0f);
    else k_fft_z<N, true><<<grid, Radix<N>::NT, smem_bytes<N>(), p->stream>>>(vol, p->tw, 1.0f / (float)N);
    return check_launch(p);
}

template <int N>
int Launch<N>::fftz_scr(cpra_plan_s* p, float4* scr, int sign, float scale)
{
    const dim3 grid((unsigned)N, (unsigned)(N / tile_batch<N>()));
    if (sign < 0) k_fft_z_scr<N, false><<<grid, Radix<N>::NT, smem_bytes<N>(), p->stream>>>(scr, p->tw, scale);
    else k_fft_z_scr<N, true><<<grid, Radix<N>::NT, smem_bytes<N>(), p->stream>>>(scr, p->tw, scale);
    return check_launch(p);
}

// the whole iteration of every projection in one launch, C CTAs per image (cpra_cluster.cuh); cluster launch
// with programmatic stream serialization (the next launch's prologue overlaps this one's tail)
template <int N, int C>
int launch_image_cl(cpra_plan_s* p, const float4* cur, float4* nxt, int mode, float beta, float scale)
{
    if constexpr (cl_ok<N, C>()) {
        const MixParams mp = mix_params(p, beta);
        ProfScope prof(p, CPRA_PROFILE_IMAGE);
        cudaLaunchConfig_t cfg = {};
        cfg.gridDim = dim3((unsigned)p->Np * C);
        cfg.blockDim = dim3(cl_threads<N, C>());
        cfg.dynamicSmemBytes = cl_smem_bytes<N, C>();
        cfg.stream = p->stream;
        cudaLaunchAttribute at[2];
        at[0].id = cudaLaunchAttributeClusterDimension;
        at[0].val.clusterDim.x = C; at[0].val.clusterDim.y = 1; at[0].val.clusterDim.z = 1;
        at[1].id = cudaLaunchAttributeProgrammaticStreamSerialization;
        at[1].val.programmaticStreamSerializationAllowed = 1;
        cfg.attrs = at;
        cfg.numAttrs = 2;
        float4* gh = p->scr;   // the FFT scratch is free on this path: it holds ghat
        cudaError_t e;
        if (mode == MIX_NONE) e = cudaLaunchKernelEx(&cfg, k_image_cl<N, C, MIX_NONE>, cur, nxt, gh, (const float*)p->A, (const float2*)p->tw, (const uint16_t*)p->S16, p->partial, mp, beta, scale, p->Np);
        else if (mode == MIX_K1) e = cudaLaunchKernelEx(&cfg, k_image_cl<N, C, MIX_K1>, cur, nxt, gh, (const float*)p->A, (const float2*)p->tw, (const uint16_t*)p->S16, p->partial, mp, beta, scale, p->Np);
        else e = cudaLaunchKernelEx(&cfg, k_image_cl<N, C, MIX_GEN>, cur, nxt, gh, (const float*)p->A, (const float2*)p->tw, (const uint16_t*)p->S16, p->partial, mp, beta, scale, p->Np);
        p->launches += 1;
        return e == cudaSuccess ? CPRA_OK : CPRA_ERR_CUDA;
    } else {
        return CPRA_ERR_UNSUPPORTED_SIZE;
    }
}
template <int N>
int Launch<N>::image_cl(cpra_plan_s* p, const float4* cur, float4* nxt, int mode, float beta, float scale, int C)
{
    switch (C) {
        case 1: return launch_image_cl<N, 1>(p, cur, nxt, mode, beta, scale);
        case 2: return launch_image_cl<N, 2>(p, cur, nxt, mode, beta, scale);
        case 4: return launch_image_cl<N, 4>(p, cur, nxt, mode, beta, scale);
        case 8: return launch_image_cl<N, 8>(p, cur, nxt, mode, beta, scale);
        case 16: return launch_image_cl<N, 16>(p, cur, nxt, mode, beta, scale);
        default: return CPRA_ERR_UNSUPPORTED_SIZE;
    }
}
template <int N>
bool Launch<N>::image_cl_ok(int C)
{
    return (C == 1 && cl_ok<N, 1>()) || (C == 2 && cl_ok<N, 2>()) || (C == 4 && cl_ok<N, 4>()) || (C == 8 && cl_ok<N, 8>()) ||
           (C == 16 && cl_ok<N, 16>());
}

// host side of cpra_generic.cuh (cpra_generic.cu)
bool gen_supported(int N);
void gen_make_geo(int N, int Np, GenGeo& g, std::vector<float2>& tw);
int gen_set_attrs();
int gen_set_data(cpra_plan_s* p, const float* d_I, const unsigned char* d_mask);
int gen_set_support(cpra_plan_s* p, const unsigned char* d_S);
int gen_set_estimate(cpra_plan_s* p, const float* d_g0);
int gen_set_estimate_spectrum(cpra_plan_s* p, const float* d_G0);
int gen_iterate(cpra_plan_s* p, int k, float beta);
int gen_prereconstruct(cpra_plan_s* p, int n, int k, float beta);
int gen_get_projections(cpra_plan_s* p, int which, float* d_out);
int gen_fft2(cpra_plan_s* p, const float* d_in, float* d_out, int sign);
int gen_slices(cpra_plan_s* p, float2* Et);
int gen_fftz(cpra_plan_s* p, float2* vol, int sign);                        // natural [z][y][x], in place
int gen_shrinkwrap(cpra_plan_s* p, float sigma, float threshold, float* d_blurred);
int gen_prtf_sums(cpra_plan_s* p, const float* d_avg, double* acc);
int gen_cube_to_pos(cpra_plan_s* p, const float2* in, float2* out);          // Step D in position order (cpra_generic.cu)
int gen_cube_to_pos_f(cpra_plan_s* p, const float* in, float* out);
int gen_cube_inverse(cpra_plan_s* p, float2* O, bool with_support, const float2* finite);
int gen_cube_forward(cpra_plan_s* p, const float2* O);
int gen_cube_gauss(cpra_plan_s* p, float sigma);   // E_n = F[S_n g_n], natural, transposed to [n][ku][kz]

#define CPRA_FOR_EACH_N(X) X(16) X(32) X(64) X(128) X(256) X(512) X(1024)
#ifndef CPRA_INST_N
#define CPRA_EXTERN_LAUNCH(N_) extern template struct Launch<N_>;
CPRA_FOR_EACH_N(CPRA_EXTERN_LAUNCH)
#undef CPRA_EXTERN_LAUNCH
#endif

}  // namespace cpra
