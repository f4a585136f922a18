// cpra_api.cu -- the C ABI of libcpra.so (include/cpra.h): plan, workspace, launch logic.
// Host code only decides what to enqueue; every step of the path runs in the kernels of
// cpra_kernels.cuh.  There is no CPU fallback.
#include <algorithm>
#include <cmath>
#include <cstdlib>
#include <cstring>
#include <new>
#include <vector>

#include "../../include/cpra.h"
#include "cpra_layout.cuh"
#include <cuda.h>

#include "cpra_image.cuh"
#include "cpra_walk.cuh"

using namespace cpra;

struct cpra_plan_s {
    int N = 0, Np = 0;
    unsigned flags = 0;
    cudaStream_t stream = nullptr;
    Geo geo{};
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
    int cur = 0;
    // parameters / state
    int K = 1;
    float alpha[MAXK + 1] = {0};
    int n_ei = 1;
    int update = CPRA_UPDATE_HIO;
    long t = 0;
    bool have_data = false, have_support = false, have_estimate = false, have_error = false;
    bool attrs_set = false;
    std::vector<double> angles;
    std::vector<float2> h_tw;
    std::vector<double> h_uphi;
    std::vector<int> h_ustart, h_rays;
    long launches = 0;
    int chunk = 0;  // images per L2-resident chunk; 0 = all
    int sms = 148;     // SMs of the device
    bool walk = true;  // use k_row_walk where the plan allows it (CPRA_WALK=0 switches it off)
    // per-kernel-class timing (cpra_profile): event pairs around every launch of the loop
    bool profiling = false;
    std::vector<cudaEvent_t> ev;      // 2 * PROF_PAIRS events, created on first use
    std::vector<int> ev_cls;          // class of each recorded pair
    double prof_ms[CPRA_PROFILE_CLASSES] = {0};
    long prof_n[CPRA_PROFILE_CLASSES] = {0};
};

namespace {

size_t align256(size_t x) { return (x + 255) & ~(size_t)255; }

struct Carve {
    size_t off = 0;
    size_t take(size_t bytes) { const size_t o = off; off = align256(off + bytes); return o; }
};

struct Layout {
    size_t tw, A, S16, st0, st1, scr, scr2, partial, den, uphi, ustart, rays, total;
};

Layout layout_of(int N, int Np)
{
    const size_t px = (size_t)Np * N * N;
    Carve c;
    Layout L;
    L.tw = c.take(sizeof(float2) * 1024);   // >= tw_count<N>() for every N
    L.A = c.take(sizeof(float) * px);
    L.S16 = c.take(px / 8);
    L.st0 = c.take(sizeof(float2) * px);
    L.st1 = c.take(sizeof(float2) * px);
    L.scr = c.take(sizeof(float2) * px);
    L.scr2 = c.take(sizeof(float2) * px);
    L.partial = c.take(sizeof(double) * (size_t)Np * (N / 8));   // >= N / Radix<N>::TB tiles per image
    L.den = c.take(sizeof(double) * Np);
    L.uphi = c.take(sizeof(double) * 2 * Np);
    L.ustart = c.take(sizeof(int) * (2 * (size_t)Np + 1));
    L.rays = c.take(sizeof(int) * 2 * (size_t)Np);
    L.total = c.off;
    return L;
}

bool is_pow2(int n) { return n > 0 && (n & (n - 1)) == 0; }

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

template <int N>
int set_attrs()
{
    static_assert(tw_count<N>() <= 1024, "twiddle region of the workspace too small");
    cudaError_t e = cudaSuccess;
    auto acc = [&](cudaError_t r) { if (e == cudaSuccess) e = r; };
    constexpr int SM = smem_bytes<N>();
    acc(allow_smem(k_row_fwd<N, MIX_NONE>, SM));
    acc(allow_smem(k_row_fwd<N, MIX_K1>, SM));
    acc(allow_smem(k_row_fwd<N, MIX_GEN>, SM));
    acc(allow_smem(k_row_fwd<N, MIX_MASK>, SM));
    acc(allow_smem(k_col<N, COL_FULL>, SM));
    acc(allow_smem(k_col<N, COL_FWD>, SM));
    acc(allow_smem(k_col<N, COL_INV>, SM));
    acc(allow_smem(k_row_inv<N, ROWINV_PLAIN, MIX_NONE>, SM));
    acc(allow_smem(k_row_inv<N, ROWINV_HIO, MIX_NONE>, SM));
    acc(allow_smem(k_row_inv<N, ROWINV_HIO, MIX_K1>, SM));
    acc(allow_smem(k_row_inv<N, ROWINV_HIO, MIX_GEN>, SM));
    if constexpr (walk_ok<N>()) acc(allow_smem(k_row_walk<N>, walk_smem_bytes<N>()));
    if constexpr (N <= 128) {
        constexpr int ISM = image_smem_bytes<N>();
        acc(allow_smem(k_image<N, MIX_NONE>, ISM));
        acc(allow_smem(k_image<N, MIX_K1>, ISM));
        acc(allow_smem(k_image<N, MIX_GEN>, ISM));
    }
    return e == cudaSuccess ? CPRA_OK : CPRA_ERR_CUDA;
}

MixParams mix_params(const cpra_plan_s* p, float beta = 0.f)
{
    MixParams mp;
    mp.K = p->K;
    for (int j = 0; j <= MAXK; ++j) mp.a[j] = j <= p->K ? p->alpha[j] : 0.f;
    // coefficients of the update outside the support (cpra_set_update)
    if (p->update == CPRA_UPDATE_RAAR) { mp.c_ghat = beta; mp.c_gp = 1.0f - 2.0f * beta; }
    else if (p->update == CPRA_UPDATE_ER) { mp.c_ghat = 0.f; mp.c_gp = 0.f; }
    else { mp.c_ghat = 1.0f; mp.c_gp = -beta; }
    return mp;
}

constexpr int PROF_PAIRS = 2048;

// fold the recorded event pairs into the per-class sums (synchronises the stream)
int prof_drain(cpra_plan_s* p)
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

int check_launch(cpra_plan_s* p, int n = 1)
{
    p->launches += n;
    return cudaGetLastError() == cudaSuccess ? CPRA_OK : CPRA_ERR_CUDA;
}

// mix mode of one iteration: does the carousel fire, and which kernel variant serves it
int mix_mode(const cpra_plan_s* p, bool fires)
{
    if (!fires) return MIX_NONE;
    if (p->K == 0) return p->alpha[0] == 1.0f ? MIX_NONE : MIX_GEN;
    return p->K == 1 ? MIX_K1 : MIX_GEN;
}

template <int N>
int launch_row_fwd(cpra_plan_s* p, const float4* cur, int mode, int n0, int nimg, float4* ghat_out = nullptr)
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
        default: ROWFWD(MIX_MASK); break;
    }
#undef ROWFWD
    return check_launch(p);
}

template <int N>
int launch_col(cpra_plan_s* p, int mode, int n0, int nimg, float scale, float4* scr = nullptr)
{
    constexpr int NT = Radix<N>::NT;
    const dim3 grid((unsigned)nimg * (N / tile_batch<N>()));
    const int smem = smem_bytes<N>();
    ProfScope prof(p, CPRA_PROFILE_COL);
    if (!scr) scr = p->scr;
    switch (mode) {
        case COL_FULL: k_col<N, COL_FULL><<<grid, NT, smem, p->stream>>>(scr, p->A, p->tw, p->partial, n0, scale); break;
        case COL_FWD: k_col<N, COL_FWD><<<grid, NT, smem, p->stream>>>(scr, p->A, p->tw, p->partial, n0, scale); break;
        default: k_col<N, COL_INV><<<grid, NT, smem, p->stream>>>(scr, p->A, p->tw, p->partial, n0, scale); break;
    }
    return check_launch(p);
}

template <int N>
int launch_row_inv(cpra_plan_s* p, const float4* cur, float4* nxt, bool hio, int mode, float beta, float scale, int n0, int nimg,
                   const float4* scr = nullptr, const float4* ghat_in = nullptr)
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
bool encode_scratch_tmap(CUtensorMap* tm, void* base, int N, int Np, int tb)
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

// K3 of one iteration fused with K1 of the next (cpra_walk.cuh): 2 CTAs per SM, each a run of tiles
template <int N>
int launch_walk(cpra_plan_s* p, const float4* scr_in, float4* scr_out, const float4* gh_old, float4* gh_new, float beta, bool fires)
{
    if constexpr (walk_ok<N>()) {
        const int total = (N / tile_batch<N>()) * p->Np;
        const int ctas = std::min(total, 2 * p->sms);
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
int iterate_walk(cpra_plan_s* p, int k, float beta, float scale)
{
    float4* g = p->st[p->cur];
    float4* other = p->st[p->cur ^ 1];
    auto fires = [&](long t) { return (t % p->n_ei) == 0; };   // does the carousel mix open iteration t (reading A3)
    int rc = launch_row_fwd<N>(p, g, fires(p->t) ? MIX_K1 : MIX_NONE, 0, p->Np, other);
    float4 *sin = p->scr, *sout = p->scr2, *gh_old = other, *gh_new = g;
    for (int it = 0; it < k && rc == CPRA_OK; ++it) {
        rc = launch_col<N>(p, COL_FULL, 0, p->Np, scale, sin);
        if (rc != CPRA_OK) break;
        if (it == k - 1) {
            rc = launch_row_inv<N>(p, gh_old, gh_new, true, MIX_K1, beta, 1.0f, 0, p->Np, sin, gh_old);
        } else {
            rc = launch_walk<N>(p, sin, sout, gh_old, gh_new, beta, fires(p->t + it + 1));
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
int launch_image(cpra_plan_s* p, const float4* cur, float4* nxt, int mode, float beta, float scale)
{
    if constexpr (N <= 128) {
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

int ready(const cpra_plan_s* p) { return p->ws ? CPRA_OK : CPRA_ERR_WORKSPACE; }

unsigned blocks_for(size_t total, int nt) { return (unsigned)((total + nt - 1) / nt); }

// sorted unique ray directions of the assembly (step (ii))
void build_rays(cpra_plan_s* p)
{
    const double PI = 3.14159265358979323846264338327950288;
    struct Ray { double phi; int n, neg; };
    std::vector<Ray> rays;
    rays.reserve(2 * (size_t)p->Np);
    for (int n = 0; n < p->Np; ++n)
        for (int neg = 0; neg < 2; ++neg) {
            double ph = std::fmod(p->angles[n] + (neg ? PI : 0.0), 2.0 * PI);
            if (ph < 0.0) ph += 2.0 * PI;
            if (ph >= 2.0 * PI - 1e-9) ph = 0.0;
            rays.push_back({ph, n, neg});
        }
    std::sort(rays.begin(), rays.end(), [](const Ray& a, const Ray& b) { return a.phi < b.phi || (a.phi == b.phi && a.n < b.n); });
    p->h_uphi.clear(); p->h_ustart.clear(); p->h_rays.clear();
    for (size_t i = 0; i < rays.size(); ++i) {
        if (p->h_uphi.empty() || rays[i].phi - p->h_uphi.back() > 1e-9) {
            p->h_ustart.push_back((int)i);
            p->h_uphi.push_back(rays[i].phi);
        }
        p->h_rays.push_back(rays[i].n | (rays[i].neg << 30));
    }
    p->h_ustart.push_back((int)rays.size());
}

}  // namespace

extern "C" {

const char* cpra_status_string(int s)
{
    switch (s) {
        case CPRA_OK: return "CPRA_OK";
        case CPRA_ERR_INVALID_ARG: return "CPRA_ERR_INVALID_ARG";
        case CPRA_ERR_UNSUPPORTED_SIZE: return "CPRA_ERR_UNSUPPORTED_SIZE";
        case CPRA_ERR_NOT_READY: return "CPRA_ERR_NOT_READY";
        case CPRA_ERR_WORKSPACE: return "CPRA_ERR_WORKSPACE";
        case CPRA_ERR_CUDA: return "CPRA_ERR_CUDA";
        case CPRA_ERR_INVALID_VALUE: return "CPRA_ERR_INVALID_VALUE";
        default: return "CPRA_ERR_UNKNOWN";
    }
}

int cpra_plan(cpra_plan_t* out, int N, int Np, unsigned flags, void* cuda_stream)
{
    if (!out) return CPRA_ERR_INVALID_ARG;
    *out = nullptr;
    if (!is_pow2(N) || N < 16 || N > 1024 || Np < 1 || Np >= (1 << 30)) return CPRA_ERR_UNSUPPORTED_SIZE;
    cpra_plan_s* p = new (std::nothrow) cpra_plan_s;
    if (!p) return CPRA_ERR_INVALID_ARG;
    p->N = N; p->Np = Np; p->flags = flags;
    p->stream = (cudaStream_t)cuda_stream;
    int R0 = 1, R1 = 1, R2 = 1, RL = 1, TBN = 16;
    { auto f = [&]() -> int { CPRA_DISPATCH_N(N, R0 = Radix<NN>::R0; R1 = Radix<NN>::R1; R2 = Radix<NN>::R2; RL = last_radix<NN>(); TBN = tile_batch<NN>()); return 0; }; f(); }
    p->geo = Geo{N, Np, R0, R1, R2, RL, TBN};
    // reading A2: the paper's example weights
    if (Np >= 3) { p->K = 1; p->alpha[0] = 0.6f; p->alpha[1] = 0.2f; }
    else { p->K = 0; p->alpha[0] = 1.0f; }
    p->n_ei = 1;
    p->angles.assign(Np, 0.0);
    { auto f = [&]() -> int { CPRA_DISPATCH_N(N, build_twiddles<NN>(p->h_tw)); return 0; }; f(); }
    if (const char* e = std::getenv("CPRA_CHUNK")) p->chunk = std::max(0, std::atoi(e));
    if (const char* e = std::getenv("CPRA_WALK")) p->walk = std::atoi(e) != 0;
    {
        int dev = 0, sms = 0;
        if (cudaGetDevice(&dev) == cudaSuccess &&
            cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) == cudaSuccess && sms > 0)
            p->sms = sms;
        (void)cudaGetLastError();
    }
    *out = p;
    return CPRA_OK;
}

int cpra_destroy(cpra_plan_t p)
{
    if (!p) return CPRA_ERR_INVALID_ARG;
    for (auto& e : p->ev) cudaEventDestroy(e);
    delete p;
    return CPRA_OK;
}

int cpra_workspace_bytes(cpra_plan_t p, size_t* bytes)
{
    if (!p || !bytes) return CPRA_ERR_INVALID_ARG;
    *bytes = layout_of(p->N, p->Np).total;
    return CPRA_OK;
}

int cpra_bind_workspace(cpra_plan_t p, void* d_ws, size_t bytes)
{
    if (!p || !d_ws) return CPRA_ERR_INVALID_ARG;
    const Layout L = layout_of(p->N, p->Np);
    if (bytes < L.total || ((uintptr_t)d_ws & 255)) return CPRA_ERR_WORKSPACE;
    char* w = (char*)d_ws;
    p->ws = w; p->ws_bytes = bytes;
    p->tw = (float2*)(w + L.tw);
    p->A = (float*)(w + L.A);
    p->S16 = (uint16_t*)(w + L.S16);
    p->st[0] = (float4*)(w + L.st0);
    p->st[1] = (float4*)(w + L.st1);
    p->scr = (float4*)(w + L.scr);
    p->scr2 = (float4*)(w + L.scr2);
    p->partial = (double*)(w + L.partial);
    p->den = (double*)(w + L.den);
    p->uphi = (double*)(w + L.uphi);
    p->ustart = (int*)(w + L.ustart);
    p->rays = (int*)(w + L.rays);
    p->cur = 0;
    p->have_data = p->have_support = p->have_estimate = p->have_error = false;
    if (!p->attrs_set) {
        int rc = CPRA_OK;
        { auto f = [&]() -> int { CPRA_DISPATCH_N(p->N, rc = set_attrs<NN>()); return 0; }; f(); }
        if (rc != CPRA_OK) { p->ws = nullptr; return rc; }
        p->attrs_set = true;
    }
    p->have_tmap = false;
    p->have_tmap = encode_scratch_tmap(&p->tm_scr[0], p->scr, p->N, p->Np, p->geo.TB) &&
                   encode_scratch_tmap(&p->tm_scr[1], p->scr2, p->N, p->Np, p->geo.TB);
    if (!p->have_tmap) { p->ws = nullptr; return CPRA_ERR_CUDA; }   // the row kernels move their tiles by TMA tensor copies
    if (cudaMemcpyAsync(p->tw, p->h_tw.data(), sizeof(float2) * p->h_tw.size(), cudaMemcpyHostToDevice, p->stream) != cudaSuccess) {
        p->ws = nullptr;
        return CPRA_ERR_CUDA;
    }
    return CPRA_OK;
}

int cpra_set_data(cpra_plan_t p, const float* d_I, const unsigned char* d_mask, const double* h_angles)
{
    if (!p || !d_I) return CPRA_ERR_INVALID_ARG;
    if (int rc = ready(p)) return rc;
    for (int n = 0; n < p->Np; ++n) p->angles[n] = h_angles ? h_angles[n] : 0.0;
    k_set_data<<<p->Np, 256, 0, p->stream>>>(d_I, d_mask, p->A, p->den, p->geo);
    if (int rc = check_launch(p)) return rc;
    p->have_data = true;
    p->have_error = false;
    return CPRA_OK;
}

int cpra_set_support(cpra_plan_t p, const unsigned char* d_S)
{
    if (!p || !d_S) return CPRA_ERR_INVALID_ARG;
    if (int rc = ready(p)) return rc;
    const size_t total16 = (size_t)p->Np * p->N * p->N / TB;
    k_pack_support<<<blocks_for(total16, 256), 256, 0, p->stream>>>(d_S, p->S16, p->N, total16);
    if (int rc = check_launch(p)) return rc;
    p->have_support = true;
    return CPRA_OK;
}

int cpra_set_carousel(cpra_plan_t p, int K, const double* h_alpha, int n_ei)
{
    if (!p || !h_alpha || K < 0 || K > CPRA_MAX_K || 2 * K + 1 > p->Np || n_ei < 1) return CPRA_ERR_INVALID_ARG;
    for (int j = 0; j <= K; ++j)
        if (!std::isfinite(h_alpha[j])) return CPRA_ERR_INVALID_ARG;
    p->K = K;
    for (int j = 0; j <= MAXK; ++j) p->alpha[j] = j <= K ? (float)h_alpha[j] : 0.f;
    p->n_ei = n_ei;
    return CPRA_OK;
}

int cpra_set_update(cpra_plan_t p, int rule)
{
    if (!p || (rule != CPRA_UPDATE_HIO && rule != CPRA_UPDATE_RAAR && rule != CPRA_UPDATE_ER)) return CPRA_ERR_INVALID_ARG;
    p->update = rule;
    return CPRA_OK;
}

int cpra_set_estimate(cpra_plan_t p, const float* d_g0)
{
    if (!p || !d_g0) return CPRA_ERR_INVALID_ARG;
    if (int rc = ready(p)) return rc;
    const size_t total = (size_t)p->Np * p->N * p->N;
    k_pack_state<<<blocks_for(total, 256), 256, 0, p->stream>>>((const float2*)d_g0, (float*)p->st[p->cur], p->geo, total);
    if (int rc = check_launch(p)) return rc;
    p->t = 0;
    p->have_estimate = true;
    p->have_error = false;
    return CPRA_OK;
}

int cpra_get_iteration(cpra_plan_t p, long* t)
{
    if (!p || !t) return CPRA_ERR_INVALID_ARG;
    *t = p->t;
    return CPRA_OK;
}

int cpra_set_iteration(cpra_plan_t p, long t)
{
    if (!p || t < 0) return CPRA_ERR_INVALID_ARG;
    p->t = t;
    return CPRA_OK;
}

int cpra_set_chunk(cpra_plan_t p, int images)
{
    if (!p || images < 0) return CPRA_ERR_INVALID_ARG;
    p->chunk = images;
    return CPRA_OK;
}

int cpra_iterate(cpra_plan_t p, int k, float beta)
{
    if (!p || k < 0 || !std::isfinite(beta)) return CPRA_ERR_INVALID_ARG;
    if (int rc = ready(p)) return rc;
    if (!p->have_data || !p->have_support || !p->have_estimate) return CPRA_ERR_NOT_READY;
    const float scale = 1.0f / ((float)p->N * (float)p->N);
    const int chunk = (p->chunk > 0 && !(p->flags & CPRA_FLAG_NO_CHUNKING)) ? std::min(p->chunk, p->Np) : p->Np;
    // the walking kernel serves the default carousel (K = 1 every iteration) on plans with 8-row tiles
    if (k > 0 && p->walk && p->have_tmap && chunk == p->Np && p->K == 1 && p->Np >= 3) {
        int rc = CPRA_ERR_UNSUPPORTED_SIZE;
        { auto f = [&]() -> int { CPRA_DISPATCH_N(p->N, if constexpr (walk_ok<NN>()) rc = iterate_walk<NN>(p, k, beta, scale)); return 0; }; f(); }
        if (rc != CPRA_ERR_UNSUPPORTED_SIZE) return rc;
    }
    for (int it = 0; it < k; ++it) {
        const int mode = mix_mode(p, (p->t % p->n_ei) == 0);
        const float4* cur = p->st[p->cur];
        float4* nxt = p->st[p->cur ^ 1];
        if (p->N <= 128 && !(p->flags & CPRA_FLAG_FORCE_MULTIPASS)) {
            int rc = CPRA_OK;
            { auto f = [&]() -> int { CPRA_DISPATCH_N(p->N, rc = launch_image<NN>(p, cur, nxt, mode, beta, scale)); return 0; }; f(); }
            if (rc != CPRA_OK) return rc;
            p->cur ^= 1;
            p->t += 1;
            p->have_error = true;
            continue;
        }
        for (int n0 = 0; n0 < p->Np; n0 += chunk) {
            const int nimg = std::min(chunk, p->Np - n0);
            int rc = CPRA_OK;
            { auto f = [&]() -> int {
                CPRA_DISPATCH_N(p->N,
                    rc = launch_row_fwd<NN>(p, cur, mode, n0, nimg);
                    if (rc == CPRA_OK) rc = launch_col<NN>(p, COL_FULL, n0, nimg, scale);
                    if (rc == CPRA_OK) rc = launch_row_inv<NN>(p, cur, nxt, true, mode, beta, 1.0f, n0, nimg));
                return 0; }; f(); }
            if (rc != CPRA_OK) return rc;
        }
        p->cur ^= 1;
        p->t += 1;
        p->have_error = true;
    }
    return CPRA_OK;
}

int cpra_get_error(cpra_plan_t p, float* d_E, float* d_Eglobal)
{
    if (!p) return CPRA_ERR_INVALID_ARG;
    if (int rc = ready(p)) return rc;
    if (!p->have_error) return CPRA_ERR_NOT_READY;
    if (!d_E && !d_Eglobal) return CPRA_OK;
    k_finalize_error<<<1, 256, 0, p->stream>>>(p->partial, p->den, d_E, d_Eglobal, p->Np, p->N / p->geo.TB);
    return check_launch(p);
}

int cpra_get_projections(cpra_plan_t p, int which, float* d_out)
{
    if (!p || !d_out || (which != CPRA_ITERATE && which != CPRA_SUPPORTED)) return CPRA_ERR_INVALID_ARG;
    if (int rc = ready(p)) return rc;
    if (!p->have_estimate || (which == CPRA_SUPPORTED && !p->have_support)) return CPRA_ERR_NOT_READY;
    const size_t total = (size_t)p->Np * p->N * p->N;
    k_unpack_state<<<blocks_for(total, 256), 256, 0, p->stream>>>((const float*)p->st[p->cur], p->S16, (float2*)d_out, p->geo, total, which == CPRA_SUPPORTED);
    return check_launch(p);
}

int cpra_fft2(cpra_plan_t p, const float* d_in, float* d_out, int sign)
{
    if (!p || !d_in || !d_out || (sign != 1 && sign != -1)) return CPRA_ERR_INVALID_ARG;
    if (int rc = ready(p)) return rc;
    const size_t total = (size_t)p->Np * p->N * p->N;
    float4* tmp = p->st[p->cur ^ 1];
    const unsigned nb = blocks_for(total, 256);
    int rc = CPRA_OK;
    if (sign < 0) {
        k_pack_state<<<nb, 256, 0, p->stream>>>((const float2*)d_in, (float*)tmp, p->geo, total);
        if ((rc = check_launch(p))) return rc;
        { auto f = [&]() -> int {
            CPRA_DISPATCH_N(p->N,
                rc = launch_row_fwd<NN>(p, tmp, MIX_NONE, 0, p->Np);
                if (rc == CPRA_OK) rc = launch_col<NN>(p, COL_FWD, 0, p->Np, 1.0f));
            return 0; }; f(); }
        if (rc) return rc;
        k_unpack_spectrum<<<nb, 256, 0, p->stream>>>((const float*)p->scr, (float2*)d_out, p->geo, total);
        return check_launch(p);
    }
    k_pack_spectrum<<<nb, 256, 0, p->stream>>>((const float2*)d_in, (float*)p->scr, p->geo, total);
    if ((rc = check_launch(p))) return rc;
    const float scale = 1.0f / ((float)p->N * (float)p->N);
    { auto f = [&]() -> int {
        CPRA_DISPATCH_N(p->N,
            rc = launch_col<NN>(p, COL_INV, 0, p->Np, 1.0f);
            if (rc == CPRA_OK) rc = launch_row_inv<NN>(p, tmp, tmp, false, MIX_NONE, 0.f, scale, 0, p->Np));
        return 0; }; f(); }
    if (rc) return rc;
    k_unpack_state<<<nb, 256, 0, p->stream>>>((const float*)tmp, p->S16, (float2*)d_out, p->geo, total, 0);
    return check_launch(p);
}

int cpra_assemble_3d(cpra_plan_t p, float* d_vol, float* d_weight)
{
    if (!p || !d_vol) return CPRA_ERR_INVALID_ARG;
    if (int rc = ready(p)) return rc;
    if (!p->have_data || !p->have_support || !p->have_estimate) return CPRA_ERR_NOT_READY;
    build_rays(p);
    const int U = (int)p->h_uphi.size();
    if (cudaMemcpyAsync(p->uphi, p->h_uphi.data(), sizeof(double) * U, cudaMemcpyHostToDevice, p->stream) != cudaSuccess ||
        cudaMemcpyAsync(p->ustart, p->h_ustart.data(), sizeof(int) * (U + 1), cudaMemcpyHostToDevice, p->stream) != cudaSuccess ||
        cudaMemcpyAsync(p->rays, p->h_rays.data(), sizeof(int) * p->h_rays.size(), cudaMemcpyHostToDevice, p->stream) != cudaSuccess)
        return CPRA_ERR_CUDA;
    // (i) E_n = F[S_n g_n] into the scratch
    int rc = CPRA_OK;
    { auto f = [&]() -> int {
        CPRA_DISPATCH_N(p->N,
            rc = launch_row_fwd<NN>(p, p->st[p->cur], MIX_MASK, 0, p->Np);
            if (rc == CPRA_OK) rc = launch_col<NN>(p, COL_FWD, 0, p->Np, 1.0f));
        return 0; }; f(); }
    if (rc) return rc;
    // (ii)-(iv) gather
    const int N = p->N;
    const int zsplit = std::max(1, std::min(N, 4096 / std::max(1, (N * N) / 256)));
    const int zper = (N + zsplit - 1) / zsplit;
    const dim3 grid(blocks_for((size_t)N * N, 128), (unsigned)((N + zper - 1) / zper));
    const size_t total = (size_t)p->Np * N * N;
    k_unpack_spectrum_T<<<blocks_for(total, 256), 256, 0, p->stream>>>((const float*)p->scr, (float2*)p->scr2, p->geo, total);
    if (int rc2 = check_launch(p)) return rc2;
    k_assemble<<<grid, 128, 0, p->stream>>>((const float2*)p->scr2, (float2*)d_vol, d_weight, p->uphi, p->ustart, p->rays, U, p->geo, zper);
    return check_launch(p);
}

int cpra_host_staging_bytes(cpra_plan_t p, size_t* bytes)
{
    if (!p || !bytes) return CPRA_ERR_INVALID_ARG;
    const size_t px = (size_t)p->Np * p->N * p->N;
    *bytes = align256(px * 8) + align256(px * 4) + 2 * align256(px) + align256(sizeof(float) * (p->Np + 1));
    return CPRA_OK;
}

int cpra_reconstruct_host(cpra_plan_t p, void* d_stage, size_t stage_bytes, const float* h_I,
                          const unsigned char* h_mask, const double* h_angles, const unsigned char* h_S,
                          const float* h_g0, int k, float beta, float* h_out, float* h_E, float* h_Eglobal)
{
    if (!p || !d_stage || !h_I || !h_S || !h_g0 || k < 0) return CPRA_ERR_INVALID_ARG;
    size_t need = 0;
    cpra_host_staging_bytes(p, &need);
    if (stage_bytes < need || ((uintptr_t)d_stage & 255)) return CPRA_ERR_WORKSPACE;
    if (int rc = ready(p)) return rc;
    const size_t px = (size_t)p->Np * p->N * p->N;
    char* s = (char*)d_stage;
    float* d_g = (float*)s;                          s += align256(px * 8);
    float* d_I = (float*)s;                          s += align256(px * 4);
    unsigned char* d_M = (unsigned char*)s;          s += align256(px);
    unsigned char* d_S = (unsigned char*)s;          s += align256(px);
    float* d_E = (float*)s;
    auto H2D = [&](void* d, const void* h, size_t b) { return cudaMemcpyAsync(d, h, b, cudaMemcpyHostToDevice, p->stream) == cudaSuccess; };
    auto D2H = [&](void* h, const void* d, size_t b) { return cudaMemcpyAsync(h, d, b, cudaMemcpyDeviceToHost, p->stream) == cudaSuccess; };
    if (!H2D(d_I, h_I, px * 4) || (h_mask && !H2D(d_M, h_mask, px)) || !H2D(d_S, h_S, px) || !H2D(d_g, h_g0, px * 8)) return CPRA_ERR_CUDA;
    int rc;
    if ((rc = cpra_set_data(p, d_I, h_mask ? d_M : nullptr, h_angles))) return rc;
    if ((rc = cpra_set_support(p, d_S))) return rc;
    if ((rc = cpra_set_estimate(p, d_g))) return rc;
    if ((rc = cpra_iterate(p, k, beta))) return rc;
    if (h_out) {
        if ((rc = cpra_get_projections(p, CPRA_ITERATE, d_g))) return rc;
        if (!D2H(h_out, d_g, px * 8)) return CPRA_ERR_CUDA;
    }
    if ((h_E || h_Eglobal) && k > 0) {
        if ((rc = cpra_get_error(p, d_E, d_E + p->Np))) return rc;
        if (h_E && !D2H(h_E, d_E, sizeof(float) * p->Np)) return CPRA_ERR_CUDA;
        if (h_Eglobal && !D2H(h_Eglobal, d_E + p->Np, sizeof(float))) return CPRA_ERR_CUDA;
    }
    return cudaStreamSynchronize(p->stream) == cudaSuccess ? CPRA_OK : CPRA_ERR_CUDA;
}

int cpra_profile(cpra_plan_t p, int enable)
{
    if (!p) return CPRA_ERR_INVALID_ARG;
    if (!enable && p->profiling) { if (int rc = prof_drain(p)) return rc; }
    p->profiling = enable != 0;
    return CPRA_OK;
}

int cpra_profile_read(cpra_plan_t p, double* h_ms, long* h_launches)
{
    if (!p || !h_ms || !h_launches) return CPRA_ERR_INVALID_ARG;
    if (int rc = prof_drain(p)) return rc;
    for (int c = 0; c < CPRA_PROFILE_CLASSES; ++c) {
        h_ms[c] = p->prof_ms[c]; h_launches[c] = p->prof_n[c];
        p->prof_ms[c] = 0.0; p->prof_n[c] = 0;
    }
    return CPRA_OK;
}

int cpra_launch_count(cpra_plan_t p, long* count)
{
    if (!p || !count) return CPRA_ERR_INVALID_ARG;
    *count = p->launches;
    return CPRA_OK;
}

}  // extern "C"
