// cpra_api.cu -- the C ABI of libcpra.so (include/cpra.h): plan, workspace, what to enqueue.
// The kernels are launched through cpra::Launch<N> (cpra_plan.cuh, instantiated per size in cpra_inst.cu).
// There is no CPU fallback.
#include "cpra_plan.cuh"
#include "cpra_layout.cuh"
#include "cpra_next.cuh"

using namespace cpra;

namespace {

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

// the caller-owned bank buffer of Step C, carved up (cpra_merge_bytes states the size)
struct BankLayout { size_t ep, E, phase, partial, shift, twin, ints, Ein, total; };
BankLayout bank_layout(int N, int Np, int NL)
{
    const size_t px = (size_t)Np * N * N;
    Carve c;
    BankLayout L;
    L.ep = c.take(sizeof(float2) * px * NL);
    L.E = c.take(sizeof(double) * NL);
    L.phase = c.take(sizeof(double) * 2 * NL);
    L.partial = c.take(sizeof(double) * 4 * MERGE_BLOCKS * NL);
    L.shift = c.take(sizeof(int) * 2 * (size_t)Np * NL);
    L.twin = c.take(sizeof(int) * NL);
    L.ints = c.take(sizeof(int) * 4);
    L.Ein = c.take(sizeof(float) * 2);
    L.total = c.off;
    return L;
}
Bank bank_of(const cpra_plan_s* p)
{
    const BankLayout L = bank_layout(p->N, p->Np, p->bank_NL);
    char* w = p->bank_buf;
    Bank b;
    b.ep = (float2*)(w + L.ep); b.E = (double*)(w + L.E); b.phase = (double*)(w + L.phase);
    b.partial = (double*)(w + L.partial); b.shift = (int*)(w + L.shift); b.twin = (int*)(w + L.twin);
    b.count = (int*)(w + L.ints); b.slot = b.count + 1; b.best = b.count + 2;
    b.Ein = (float*)(w + L.Ein);
    b.NL = p->bank_NL;
    return b;
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
    const bool generic = !is_pow2(N) && gen_supported(N);
    if ((!is_pow2(N) && !generic) || N < 16 || N > 1024 || Np < 1 || Np >= (1 << 30)) return CPRA_ERR_UNSUPPORTED_SIZE;
    if (flags & ~CPRA_FLAG_ALL) return CPRA_ERR_INVALID_ARG;
    cpra_plan_s* p = new (std::nothrow) cpra_plan_s;
    if (!p) return CPRA_ERR_INVALID_ARG;
    p->N = N; p->Np = Np; p->flags = flags;
    p->stream = (cudaStream_t)cuda_stream;
    p->generic = generic;
    int R0 = 1, R1 = 1, R2 = 1, RL = 1, TBN = 16;
    if (!generic) { auto f = [&]() -> int { CPRA_DISPATCH_N(N, R0 = Radix<NN>::R0; R1 = Radix<NN>::R1; R2 = Radix<NN>::R2; RL = last_radix<NN>(); TBN = tile_batch<NN>()); return 0; }; f(); }
    p->geo = Geo{N, Np, R0, R1, R2, RL, generic ? gen_lines_per_tile(N) : TBN};   // (generic: TB = lines per tile, for the error partials only)
    // reading A2: the paper's example weights
    if (Np >= 3) { p->K = 1; p->alpha[0] = 0.6f; p->alpha[1] = 0.2f; }
    else { p->K = 0; p->alpha[0] = 1.0f; }
    p->n_ei = 1;
    p->angles.assign(Np, 0.0);
    if (generic) gen_make_geo(N, Np, p->gg, p->h_tw);
    else { auto f = [&]() -> int { CPRA_DISPATCH_N(N, build_twiddles<NN>(p->h_tw)); return 0; }; f(); }
    p->walk = !(flags & CPRA_FLAG_NO_WALK);
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
    *bytes = layout_of(p->N, p->Np, p->generic).total;
    return CPRA_OK;
}

int cpra_bind_workspace(cpra_plan_t p, void* d_ws, size_t bytes)
{
    if (!p || !d_ws) return CPRA_ERR_INVALID_ARG;
    const Layout L = layout_of(p->N, p->Np, p->generic);
    if (bytes < L.total || ((uintptr_t)d_ws & 255)) return CPRA_ERR_WORKSPACE;
    char* w = (char*)d_ws;
    p->ws = w; p->ws_bytes = bytes;
    p->tw = (float2*)(w + L.tw);
    p->A = (float*)(w + L.A);
    p->S16 = (uint16_t*)(w + L.S16);
    p->S8 = (unsigned char*)(w + L.S8);
    p->st[0] = (float4*)(w + L.st0);
    p->st[1] = (float4*)(w + L.st1);
    p->scr = (float4*)(w + L.scr);
    p->scr2 = (float4*)(w + L.scr2);
    p->partial = (double*)(w + L.partial);
    p->den = (double*)(w + L.den);
    p->uphi = (double*)(w + L.uphi);
    p->ustart = (int*)(w + L.ustart);
    p->rays = (int*)(w + L.rays);
    p->mx = (float*)(w + L.mx);
    p->shell = (double*)(w + L.shell);
    p->align = (double*)(w + L.align);
    p->cur = 0;
    p->have_data = p->have_support = p->have_estimate = p->have_error = false;
    if (!p->attrs_set) {
        int rc = CPRA_OK;
        if (p->generic) rc = gen_set_attrs();
        else { auto f = [&]() -> int { CPRA_DISPATCH_N(p->N, rc = Launch<NN>::set_attrs()); return 0; }; f(); }
        if (rc != CPRA_OK) { p->ws = nullptr; return rc; }
        p->attrs_set = true;
    }
    p->have_tmap = false;
    if (!p->generic) {
        p->have_tmap = encode_scratch_tmap(&p->tm_scr[0], p->scr, p->N, p->Np, p->geo.TB) &&
                       encode_scratch_tmap(&p->tm_scr[1], p->scr2, p->N, p->Np, p->geo.TB);
        if (!p->have_tmap) { p->ws = nullptr; return CPRA_ERR_CUDA; }   // the row kernels move their tiles by TMA tensor copies
    }
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
    if (p->generic) { if (int rc = gen_set_data(p, d_I, d_mask)) return rc; }
    else {
        static_assert(SET_DATA_SPLIT <= 8, "the band sums use the error scratch: Np max(N / 4 + 1, 8) doubles (layout_of)");
        double* part = p->partial;
        k_set_data<<<p->Np * SET_DATA_SPLIT, 256, 0, p->stream>>>(d_I, d_mask, p->A, part, p->geo);
        if (int rc = check_launch(p)) return rc;
        k_set_data_den<<<blocks_for(p->Np, 128), 128, 0, p->stream>>>(part, p->den, p->Np);
        if (int rc = check_launch(p)) return rc;
    }
    p->have_data = true;
    p->have_error = false;
    return CPRA_OK;
}

int cpra_set_support(cpra_plan_t p, const unsigned char* d_S)
{
    if (!p || !d_S) return CPRA_ERR_INVALID_ARG;
    if (int rc = ready(p)) return rc;
    if (p->generic) { if (int rc = gen_set_support(p, d_S)) return rc; }
    else {
        const size_t total16 = (size_t)p->Np * p->N * p->N / TB;
        k_pack_support<<<blocks_for(total16, 256), 256, 0, p->stream>>>(d_S, p->S16, p->N, total16);
        if (int rc = check_launch(p)) return rc;
    }
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
    if (p->generic) { if (int rc = gen_set_estimate(p, d_g0)) return rc; }
    else {
        k_pack_state<<<blocks_for(total / (p->geo.TB), 256), 256, 0, p->stream>>>((const float2*)d_g0, (float*)p->st[p->cur], p->geo, total / p->geo.TB);
        if (int rc = check_launch(p)) return rc;
    }
    p->t = 0;
    p->have_estimate = true;
    p->have_error = false;
    return CPRA_OK;
}

int cpra_set_estimate_spectrum(cpra_plan_t p, const float* d_G0)
{
    if (!p || !d_G0) return CPRA_ERR_INVALID_ARG;
    if (int rc = ready(p)) return rc;
    int rc = CPRA_OK;
    const float scale = 1.0f / ((float)p->N * (float)p->N);
    if (p->generic) {
        if ((rc = gen_set_estimate_spectrum(p, d_G0))) return rc;
    } else {
        // cpra_fft2's inverse path with the state buffer as its destination: no natural-order copy in between
        const int PB = spectrum_rows_per_block(p->N);
        k_pack_spectrum<<<(unsigned)((size_t)p->Np * (p->N / PB)), 256, sizeof(float2) * p->N * PB, p->stream>>>((const float2*)d_G0, (float*)p->scr, p->geo);
        if ((rc = check_launch(p))) return rc;
        float4* g = p->st[p->cur];
        { auto f = [&]() -> int {
            CPRA_DISPATCH_N(p->N,
                rc = Launch<NN>::col(p, COL_INV, 0, p->Np, 1.0f);
                if (rc == CPRA_OK) rc = Launch<NN>::row_inv(p, g, g, false, MIX_NONE, 0.f, scale, 0, p->Np));
            return 0; }; f(); }
        if (rc) return rc;
    }
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
    if (p->generic) return gen_iterate(p, k, beta);
    const float scale = 1.0f / ((float)p->N * (float)p->N);
    const int chunk = (p->chunk > 0 && !(p->flags & CPRA_FLAG_NO_CHUNKING)) ? std::min(p->chunk, p->Np) : p->Np;
    // the walking kernel serves the default carousel (K = 1) and the uncoupled loop (K = 0 with alpha_0 = 1: the batched
    // pre-reconstructions of Step A) on plans with 8-row tiles
    const bool uncoupled = p->K == 0 && p->alpha[0] == 1.0f;
    if (k > 0 && p->walk && p->cluster <= 0 && p->have_tmap && chunk == p->Np && (p->K == 1 || uncoupled) && p->Np >= 3) {
        int rc = CPRA_ERR_UNSUPPORTED_SIZE;
        { auto f = [&]() -> int { CPRA_DISPATCH_N(p->N, if constexpr (walk_ok<NN>()) rc = Launch<NN>::iterate_walk(p, k, beta, scale)); return 0; }; f(); }
        if (rc != CPRA_ERR_UNSUPPORTED_SIZE) return rc;
    }
    // whole-image kernel on a cluster of C CTAs per projection (cpra_set_cluster; cpra_cluster.cuh)
    int C = p->cluster;
    // library default (measured, B200): at N = 64 the clustered kernel with programmatic dependent launch beats
    // the one-CTA-per-image kernel (N_p = 32: 6.9 us per iteration with 4 CTAs per image against 9.3; N_p = 180:
    // 12.0 with 2 against 12.9); at N = 128 and 256 it does not
    if (C == 0 && p->N == 64) C = (4 * p->Np <= 2 * p->sms) ? 4 : 2;
    if (C > 0) {
        bool ok = false;
        { auto f = [&]() -> int { CPRA_DISPATCH_N(p->N, ok = Launch<NN>::image_cl_ok(C)); return 0; }; f(); }
        if (!ok || (p->flags & CPRA_FLAG_FORCE_MULTIPASS) || chunk != p->Np) C = 0;
    }
    bool have_image = false;
    { auto f = [&]() -> int { CPRA_DISPATCH_N(p->N, have_image = Launch<NN>::has_image()); return 0; }; f(); }
    for (int it = 0; it < k; ++it) {
        const int mode = mix_mode(p, (p->t % p->n_ei) == 0);
        const float4* cur = p->st[p->cur];
        float4* nxt = p->st[p->cur ^ 1];
        if (C > 0) {
            int rc = CPRA_OK;
            { auto f = [&]() -> int { CPRA_DISPATCH_N(p->N, rc = Launch<NN>::image_cl(p, cur, nxt, mode, beta, scale, C)); return 0; }; f(); }
            if (rc != CPRA_OK) return rc;
            p->cur ^= 1;
            p->t += 1;
            p->have_error = true;
            continue;
        }
        if (have_image && !(p->flags & CPRA_FLAG_FORCE_MULTIPASS)) {
            int rc = CPRA_OK;
            { auto f = [&]() -> int { CPRA_DISPATCH_N(p->N, rc = Launch<NN>::image(p, cur, nxt, mode, beta, scale)); return 0; }; f(); }
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
                    rc = Launch<NN>::row_fwd(p, cur, mode, n0, nimg);
                    if (rc == CPRA_OK) rc = Launch<NN>::col(p, COL_FULL, n0, nimg, scale);
                    if (rc == CPRA_OK) rc = Launch<NN>::row_inv(p, cur, nxt, true, mode, beta, 1.0f, n0, nimg));
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
    k_finalize_error<<<1, 256, 0, p->stream>>>(p->partial, p->den, d_E, d_Eglobal, p->Np, (p->N + p->geo.TB - 1) / p->geo.TB);
    return check_launch(p);
}

int cpra_get_projections(cpra_plan_t p, int which, float* d_out)
{
    if (!p || !d_out || (which != CPRA_ITERATE && which != CPRA_SUPPORTED)) return CPRA_ERR_INVALID_ARG;
    if (int rc = ready(p)) return rc;
    if (!p->have_estimate || (which == CPRA_SUPPORTED && !p->have_support)) return CPRA_ERR_NOT_READY;
    if (p->generic) return gen_get_projections(p, which, d_out);
    const size_t total = (size_t)p->Np * p->N * p->N;
    k_unpack_state<<<blocks_for(total / p->geo.TB, 256), 256, 0, p->stream>>>((const float*)p->st[p->cur], p->S16, (float2*)d_out, p->geo, total / p->geo.TB,
                                                                           which == CPRA_SUPPORTED);
    return check_launch(p);
}

int cpra_fft2(cpra_plan_t p, const float* d_in, float* d_out, int sign)
{
    if (!p || !d_in || !d_out || (sign != 1 && sign != -1)) return CPRA_ERR_INVALID_ARG;
    if (int rc = ready(p)) return rc;
    if (p->generic) return gen_fft2(p, d_in, d_out, sign);
    const size_t total = (size_t)p->Np * p->N * p->N;
    float4* tmp = p->st[p->cur ^ 1];
    const size_t units = total / p->geo.TB;                              // (n, row tile, x) of the state conversions
    const int PB = spectrum_rows_per_block(p->N);                        // scratch rows per block of the spectrum conversions
    const unsigned rows = (unsigned)((size_t)p->Np * (p->N / PB));
    const int rowt = 256, rowsm = (int)sizeof(float2) * p->N * PB;
    int rc = CPRA_OK;
    if (sign < 0) {
        k_pack_state<<<blocks_for(units, 256), 256, 0, p->stream>>>((const float2*)d_in, (float*)tmp, p->geo, units);
        if ((rc = check_launch(p))) return rc;
        { auto f = [&]() -> int {
            CPRA_DISPATCH_N(p->N,
                rc = Launch<NN>::row_fwd(p, tmp, MIX_NONE, 0, p->Np);
                if (rc == CPRA_OK) rc = Launch<NN>::col(p, COL_FWD, 0, p->Np, 1.0f));
            return 0; }; f(); }
        if (rc) return rc;
        k_unpack_spectrum<<<rows, rowt, rowsm, p->stream>>>((const float*)p->scr, (float2*)d_out, p->geo);
        return check_launch(p);
    }
    k_pack_spectrum<<<rows, rowt, rowsm, p->stream>>>((const float2*)d_in, (float*)p->scr, p->geo);
    if ((rc = check_launch(p))) return rc;
    const float scale = 1.0f / ((float)p->N * (float)p->N);
    { auto f = [&]() -> int {
        CPRA_DISPATCH_N(p->N,
            rc = Launch<NN>::col(p, COL_INV, 0, p->Np, 1.0f);
            if (rc == CPRA_OK) rc = Launch<NN>::row_inv(p, tmp, tmp, false, MIX_NONE, 0.f, scale, 0, p->Np));
        return 0; }; f(); }
    if (rc) return rc;
    k_unpack_state<<<blocks_for(units, 256), 256, 0, p->stream>>>((const float*)tmp, p->S16, (float2*)d_out, p->geo, units, 0);
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
    const int N = p->N;
    const size_t total = (size_t)p->Np * N * N;
    // the gather with the lanes along kz needs whole 32 x 32 tiles and room for its geometry table (N^2 x 32 B in the
    // spare state buffer); anything else takes the one-thread-per-(ky, kx) gather
    const bool tiled = (N % 32 == 0) && (size_t)p->Np * sizeof(float2) >= sizeof(AsmGeo);
    // (i) E_n = F[S_n g_n], natural order, transposed to Et[n][ku][kz] in the second scratch
    if (p->generic) {
        if (int rc = gen_slices(p, (float2*)p->scr2)) return rc;
    } else {
        int rc = CPRA_OK;
        { auto f = [&]() -> int {
            CPRA_DISPATCH_N(p->N,
                rc = Launch<NN>::row_fwd(p, p->st[p->cur], MIX_MASK, 0, p->Np);
                if (rc == CPRA_OK) rc = Launch<NN>::col(p, COL_FWD, 0, p->Np, 1.0f));
            return 0; }; f(); }
        if (rc) return rc;
        const int tile_smem = N * (p->geo.TB / 2) * 16;
        if (tile_smem <= 48 * 1024)
            k_unpack_tile_T<<<(unsigned)(p->Np * (N / p->geo.TB)), 256, tile_smem, p->stream>>>(p->scr, (float2*)p->scr2, p->geo);
        else
            k_unpack_spectrum_T<<<blocks_for(total, 256), 256, 0, p->stream>>>((const float*)p->scr, (float2*)p->scr2, p->geo, total);
        if (int rc2 = check_launch(p)) return rc2;
    }
    // (ii)-(iv) gather
    if (tiled) {
        AsmGeo* geo = (AsmGeo*)p->st[p->cur ^ 1];
        k_assemble_geo<<<blocks_for((size_t)N * N, 128), 128, 0, p->stream>>>(geo, p->uphi, U, N);
        if (int rc2 = check_launch(p)) return rc2;
        k_assemble_gather<<<(unsigned)((N / 32) * N * (N / 32)), 256, 0, p->stream>>>((const float2*)p->scr2, (float2*)d_vol, d_weight, geo,
                                                                                     p->ustart, p->rays, N, p->Np);
        return check_launch(p);
    }
    const int zsplit = std::max(1, std::min(N, 4096 / std::max(1, (N * N) / 256)));
    const int zper = (N + zsplit - 1) / zsplit;
    const dim3 grid(blocks_for((size_t)N * N, 128), (unsigned)((N + zper - 1) / zper));
    k_assemble<<<grid, 128, 0, p->stream>>>((const float2*)p->scr2, (float2*)d_vol, d_weight, p->uphi, p->ustart, p->rays, U, p->geo, zper);
    return check_launch(p);
}

int cpra_set_cluster(cpra_plan_t p, int ctas_per_image)
{
    if (!p || ctas_per_image < -1 || ctas_per_image > 16) return CPRA_ERR_INVALID_ARG;
    p->cluster = ctas_per_image;
    return CPRA_OK;
}

int cpra_set_walk_ctas(cpra_plan_t p, int per_sm)
{
    if (!p || per_sm < 0 || per_sm > 8) return CPRA_ERR_INVALID_ARG;
    p->walk_ctas = per_sm;
    return CPRA_OK;
}

int cpra_set_positivity(cpra_plan_t p, int on)
{
    if (!p || (on != 0 && on != 1)) return CPRA_ERR_INVALID_ARG;
    p->positivity = on;
    return CPRA_OK;
}

int cpra_set_seam(cpra_plan_t p, int flip)
{
    if (!p || (flip != 0 && flip != 1)) return CPRA_ERR_INVALID_ARG;
    p->flip_seam = flip;
    return CPRA_OK;
}

int cpra_get_support(cpra_plan_t p, unsigned char* d_S)
{
    if (!p || !d_S) return CPRA_ERR_INVALID_ARG;
    if (int rc = ready(p)) return rc;
    if (!p->have_support) return CPRA_ERR_NOT_READY;
    const size_t total = (size_t)p->Np * p->N * p->N;
    if (p->generic)
        return cudaMemcpyAsync(d_S, p->S8, total, cudaMemcpyDeviceToDevice, p->stream) == cudaSuccess ? CPRA_OK : CPRA_ERR_CUDA;
    k_unpack_support<<<blocks_for(total, 256), 256, 0, p->stream>>>(p->S16, d_S, p->N, total);
    return check_launch(p);
}

int cpra_shrinkwrap(cpra_plan_t p, float sigma, float threshold, float* d_blurred)
{
    if (!p || !(sigma >= 0.f) || !(threshold >= 0.f) || !std::isfinite(sigma) || !std::isfinite(threshold)) return CPRA_ERR_INVALID_ARG;
    if (int rc = ready(p)) return rc;
    if (!p->have_support || !p->have_estimate) return CPRA_ERR_NOT_READY;
    if (p->generic) return gen_shrinkwrap(p, sigma, threshold, d_blurred);
    const size_t total = (size_t)p->Np * p->N * p->N;
    float4* tmp = p->st[p->cur ^ 1];
    // |S g| (formed by the row pass as it loads the state) -> forward 2D FT -> Gaussian transfer function -> inverse 2D FT ->
    // per-image maximum -> threshold
    int rc = CPRA_OK;
    // the transfer function as a table over the scratch positions (the shell scratch: 12 N bytes are there), applied between
    // the forward and the inverse column pass inside one kernel
    float* tab = (float*)p->shell;
    k_gauss_table<<<blocks_for(p->N, 128), 128, 0, p->stream>>>(tab, p->geo, sigma);
    if ((rc = check_launch(p))) return rc;
    const float scale = 1.0f / ((float)p->N * (float)p->N);
    { auto f = [&]() -> int {
        CPRA_DISPATCH_N(p->N,
            rc = Launch<NN>::row_fwd(p, p->st[p->cur], MIX_ABS, 0, p->Np);
            if (rc == CPRA_OK) rc = Launch<NN>::col(p, COL_GAUSS, 0, p->Np, 1.0f, nullptr, tab);
            if (rc == CPRA_OK) rc = Launch<NN>::row_inv(p, tmp, tmp, false, MIX_NONE, 0.f, scale, 0, p->Np));
        return 0; }; f(); }
    if (rc) return rc;
    k_image_max<<<p->Np, 256, 0, p->stream>>>(tmp, p->mx, p->geo);
    if ((rc = check_launch(p))) return rc;
    if (d_blurred) {
        k_unpack_real<<<blocks_for(total, 256), 256, 0, p->stream>>>((const float*)tmp, d_blurred, p->geo, total);
        if ((rc = check_launch(p))) return rc;
    }
    const size_t total16 = total / 16;
    k_threshold_pack<<<blocks_for(total16, 256), 256, 0, p->stream>>>((const float*)tmp, p->mx, p->S16, p->geo, total16, threshold);
    return check_launch(p);
}

int cpra_prereconstruct(cpra_plan_t p, int n, int k, float beta)
{
    if (!p || n < 0 || n >= p->Np || k < 0 || !std::isfinite(beta)) return CPRA_ERR_INVALID_ARG;
    if (int rc = ready(p)) return rc;
    if (!p->have_data || !p->have_support || !p->have_estimate) return CPRA_ERR_NOT_READY;
    if (k == 0) return CPRA_OK;
    if (p->generic) return gen_prereconstruct(p, n, k, beta);
    const float scale = 1.0f / ((float)p->N * (float)p->N);
    // the conventional 2D iteration on projection n alone: no mix, the three tile kernels on a one-image grid;
    // the image ping-pongs between the two state buffers, the other projections stay where they are
    int rc = CPRA_OK, src = p->cur;
    for (int it = 0; it < k && rc == CPRA_OK; ++it) {
        const float4* cur = p->st[src];
        float4* nxt = p->st[src ^ 1];
        { auto f = [&]() -> int {
            CPRA_DISPATCH_N(p->N,
                rc = Launch<NN>::row_fwd(p, cur, MIX_NONE, n, 1);
                if (rc == CPRA_OK) rc = Launch<NN>::col(p, COL_FULL, n, 1, scale);
                if (rc == CPRA_OK) rc = Launch<NN>::row_inv(p, cur, nxt, true, MIX_NONE, beta, 1.0f, n, 1));
            return 0; }; f(); }
        src ^= 1;
    }
    if (rc) return rc;
    if (src != p->cur) {
        const size_t ib = sizeof(float2) * (size_t)p->N * p->N;
        if (cudaMemcpyAsync((char*)p->st[p->cur] + ib * n, (const char*)p->st[src] + ib * n, ib, cudaMemcpyDeviceToDevice, p->stream) != cudaSuccess)
            return CPRA_ERR_CUDA;
    }
    p->have_error = false;   // the error partials of projection n now belong to the pre-reconstruction
    return CPRA_OK;
}

int cpra_merge_bytes(cpra_plan_t p, int NL, size_t* bytes)
{
    if (!p || !bytes || NL < 1 || NL > 1024) return CPRA_ERR_INVALID_ARG;
    *bytes = bank_layout(p->N, p->Np, NL).total;
    return CPRA_OK;
}

int cpra_merge_bind(cpra_plan_t p, void* d_buf, size_t bytes, int NL)
{
    if (!p || !d_buf || NL < 1 || NL > 1024) return CPRA_ERR_INVALID_ARG;
    const BankLayout L = bank_layout(p->N, p->Np, NL);
    if (bytes < L.total || ((uintptr_t)d_buf & 255)) return CPRA_ERR_WORKSPACE;
    p->bank_buf = (char*)d_buf; p->bank_bytes = bytes; p->bank_NL = NL;
    // everything but the episodes themselves starts at zero (count = 0: the bank is empty)
    if (cudaMemsetAsync(p->bank_buf + L.E, 0, L.total - L.E, p->stream) != cudaSuccess) return CPRA_ERR_CUDA;
    return CPRA_OK;
}

int cpra_merge_offer(cpra_plan_t p, const float* d_episode, double E)
{
    if (!p) return CPRA_ERR_INVALID_ARG;
    if (!p->bank_buf) return CPRA_ERR_NOT_READY;
    const Bank b = bank_of(p);
    const size_t total = (size_t)p->Np * p->N * p->N;
    if (!d_episode) {
        if (int rc = ready(p)) return rc;
        if (!p->have_estimate || !p->have_support || !p->have_error) return CPRA_ERR_NOT_READY;
        k_finalize_error<<<1, 256, 0, p->stream>>>(p->partial, p->den, nullptr, b.Ein, p->Np, (p->N + p->geo.TB - 1) / p->geo.TB);
        if (int rc = check_launch(p)) return rc;
        k_offer_select<<<1, 1, 0, p->stream>>>(b, b.Ein, 0.0);
    } else {
        if (!std::isfinite(E)) return CPRA_ERR_INVALID_ARG;
        k_offer_select<<<1, 1, 0, p->stream>>>(b, nullptr, E);
    }
    if (int rc = check_launch(p)) return rc;
    if (!d_episode && p->generic) {
        // natural state: S g into the other state buffer (free between calls), then offered like a caller's episode
        float2* tmp = (float2*)p->st[p->cur ^ 1];
        if (int rc = gen_get_projections(p, CPRA_SUPPORTED, (float*)tmp)) return rc;
        k_offer_copy<<<blocks_for(total, 256), 256, 0, p->stream>>>(b, tmp, nullptr, p->S16, p->geo, total);
        return check_launch(p);
    }
    k_offer_copy<<<blocks_for(total, 256), 256, 0, p->stream>>>(b, (const float2*)d_episode, d_episode ? nullptr : (const float*)p->st[p->cur],
                                                                 p->S16, p->geo, total);
    return check_launch(p);
}

int cpra_merge_errors(cpra_plan_t p, double* d_E, int* d_count)
{
    if (!p || (!d_E && !d_count)) return CPRA_ERR_INVALID_ARG;
    if (!p->bank_buf) return CPRA_ERR_NOT_READY;
    const Bank b = bank_of(p);
    if (d_E && cudaMemcpyAsync(d_E, b.E, sizeof(double) * p->bank_NL, cudaMemcpyDeviceToDevice, p->stream) != cudaSuccess) return CPRA_ERR_CUDA;
    if (d_count && cudaMemcpyAsync(d_count, b.count, sizeof(int), cudaMemcpyDeviceToDevice, p->stream) != cudaSuccess) return CPRA_ERR_CUDA;
    return CPRA_OK;
}

int cpra_merge_get(cpra_plan_t p, int slot, float* d_episode)
{
    if (!p || !d_episode || slot < 0) return CPRA_ERR_INVALID_ARG;
    if (!p->bank_buf) return CPRA_ERR_NOT_READY;
    if (slot >= p->bank_NL) return CPRA_ERR_INVALID_ARG;
    const Bank b = bank_of(p);
    const size_t total = (size_t)p->Np * p->N * p->N;
    if (cudaMemcpyAsync(d_episode, b.ep + (size_t)slot * total, sizeof(float2) * total, cudaMemcpyDeviceToDevice, p->stream) != cudaSuccess) return CPRA_ERR_CUDA;
    return CPRA_OK;
}

int cpra_merge_finish(cpra_plan_t p, int n_ref, float* d_out, int* d_shifts, int* d_twins)
{
    if (!p || !d_out || n_ref < -1 || n_ref >= p->Np) return CPRA_ERR_INVALID_ARG;
    if (!p->bank_buf) return CPRA_ERR_NOT_READY;
    const Bank b = bank_of(p);
    const size_t total = (size_t)p->Np * p->N * p->N;
    k_merge_com<<<(unsigned)(p->bank_NL * p->Np), 256, 0, p->stream>>>(b, p->geo);
    if (int rc = check_launch(p)) return rc;
    k_merge_best<<<1, 1, 0, p->stream>>>(b);
    if (int rc = check_launch(p)) return rc;
    k_merge_inner<<<dim3(MERGE_BLOCKS, (unsigned)p->bank_NL), 256, 0, p->stream>>>(b, p->geo, n_ref);
    if (int rc = check_launch(p)) return rc;
    k_merge_decide<<<1, 1024, 0, p->stream>>>(b);
    if (int rc = check_launch(p)) return rc;
    k_merge_average<<<blocks_for(total, 256), 256, 0, p->stream>>>(b, (float2*)d_out, p->geo, total);
    if (int rc = check_launch(p)) return rc;
    if (d_shifts && cudaMemcpyAsync(d_shifts, b.shift, sizeof(int) * 2 * (size_t)p->Np * p->bank_NL, cudaMemcpyDeviceToDevice, p->stream) != cudaSuccess) return CPRA_ERR_CUDA;
    if (d_twins && cudaMemcpyAsync(d_twins, b.twin, sizeof(int) * p->bank_NL, cudaMemcpyDeviceToDevice, p->stream) != cudaSuccess) return CPRA_ERR_CUDA;
    return CPRA_OK;
}

int cpra_align_episode(cpra_plan_t p, float* d_episode, int n_ref, int* d_flips)
{
    if (!p || !d_episode || n_ref < 0 || n_ref >= p->Np) return CPRA_ERR_INVALID_ARG;
    if (int rc = ready(p)) return rc;
    const size_t total = (size_t)p->Np * p->N * p->N;
    int* flags = (int*)(p->align + (size_t)8 * p->Np);
    k_align_sums<<<p->Np, 256, 0, p->stream>>>((const float2*)d_episode, p->align, p->N);
    if (int rc = check_launch(p)) return rc;
    k_align_decide<<<1, 32, 0, p->stream>>>(p->align, flags, p->Np, n_ref);
    if (int rc = check_launch(p)) return rc;
    k_align_apply<<<blocks_for(total, 256), 256, 0, p->stream>>>((float2*)d_episode, p->align, flags, p->N, total);
    if (int rc = check_launch(p)) return rc;
    if (d_flips && cudaMemcpyAsync(d_flips, flags, sizeof(int) * p->Np, cudaMemcpyDeviceToDevice, p->stream) != cudaSuccess) return CPRA_ERR_CUDA;
    return CPRA_OK;
}

}  // extern "C"

namespace {
// Step D's iterations for a power-of-two N with the cube kept in the loop's own layouts: O in the row-tiled state, the
// spectra F (scratch), E (second scratch) and the weights (spare state buffer) quad by quad in the scratch layout with the
// planes in position order.  An iteration is z pass (inverse) -> column pass -> row pass with the support as an ER update
// (outside the support 0) -> row pass -> column pass -> z pass -> replace: no natural-order copy in between.
// every >= 1: the support update of cpra_refine_3d_sw, with the blur run through the same kernels (F is parked in d_obj).
int refine_3d_tiled(cpra_plan_s* p, const float* d_E, const float* d_W, const unsigned char* d_S3_in, unsigned char* d_S3_out, int k, int every,
                    float sigma, float threshold, float* d_obj, float* d_err, float* d_blurred)
{
    const int N = p->N;
    const size_t n3 = (size_t)N * N * N, nq = n3 / 2, total16 = n3 / 16, units = n3 / p->geo.TB;
    const int nblk = (int)std::min<size_t>(2048, (size_t)p->Np * (N / 8) / 2);
    if (nblk < 1) return CPRA_ERR_UNSUPPORTED_SIZE;
    float4* O = p->st[p->cur];                       // the object, row-tiled
    float2* Wq = (float2*)p->st[p->cur ^ 1];         // (w_a, w_b) per quad
    float4* F = p->scr;                              // the spectrum the transforms work on
    float4* Eq = p->scr2;                            // the assembled spectrum
    double* num = p->partial;
    double* den = p->partial + nblk;
    const int PB = spectrum_rows_per_block(N);
    const unsigned rows = (unsigned)((size_t)N * (N / PB));
    const int saved_update = p->update;
    const auto saved_positivity = p->positivity;
    int rc = CPRA_OK;
    auto launch = [&]() { return (rc = check_launch(p)) == CPRA_OK; };
    auto run = [&](auto&& f) { f(); return rc == CPRA_OK; };
    auto dispatch = [&](auto&& body) { auto f = [&]() -> int { CPRA_DISPATCH_N(N, body(std::integral_constant<int, NN>{})); return 0; }; f(); };
    (void)run;
    // layouts: support bits, E and W quad by quad with the planes in position order; O starts as zeros (it is only ever
    // multiplied by 0 before the first row pass overwrites it)
    k_pack_support<<<blocks_for(total16, 256), 256, 0, p->stream>>>(d_S3_in, p->S16, N, total16);
    if (!launch()) return rc;
    k_pack_spectrum<<<rows, 256, sizeof(float2) * N * PB, p->stream>>>((const float2*)d_E, (float*)Eq, p->geo, 1);
    if (!launch()) return rc;
    // (the row pass reads the weights' buffer as the "previous state" it multiplies by 0: all of it must be finite)
    if (cudaMemsetAsync(Wq, 0, sizeof(float2) * n3, p->stream) != cudaSuccess) return CPRA_ERR_CUDA;
    k_pack_weight<<<rows, 256, sizeof(float) * N * PB, p->stream>>>(d_W, Wq, p->geo);
    if (!launch()) return rc;
    if (cudaMemsetAsync(O, 0, sizeof(float2) * n3, p->stream) != cudaSuccess) return CPRA_ERR_CUDA;
    k_refine_init_q<<<nblk, 256, 0, p->stream>>>(Eq, Wq, F, den, nq);
    if (!launch()) return rc;
    const float inv3 = 1.0f / ((float)N * (float)N * (float)N);
    p->update = CPRA_UPDATE_ER;                      // the support step: inside g', outside 0
    p->positivity = 0;                               // (Step D has no positivity step: reading A26)
    for (int it = 0; it < k && rc == CPRA_OK; ++it) {
        // O = S3 . F3^-1[F]
        dispatch([&](auto nn) {
            constexpr int NN = decltype(nn)::value;
            rc = Launch<NN>::fftz_scr(p, F, +1, inv3);
            if (rc == CPRA_OK) rc = Launch<NN>::col(p, COL_INV, 0, N, 1.0f);
            if (rc == CPRA_OK) rc = Launch<NN>::row_inv(p, (const float4*)Wq, O, true, MIX_NONE, 0.f, 1.0f, 0, N, nullptr, (const float4*)Wq);
            // F' = F3[O]
            if (rc == CPRA_OK) rc = Launch<NN>::row_fwd(p, O, MIX_NONE, 0, N);
            if (rc == CPRA_OK) rc = Launch<NN>::col(p, COL_FWD, 0, N, 1.0f);
            if (rc == CPRA_OK) rc = Launch<NN>::fftz_scr(p, F, -1, 1.0f);
        });
        if (rc) break;
        k_refine_replace_q<<<nblk, 256, 0, p->stream>>>(F, Eq, Wq, num, nq);
        if (!launch()) break;
        if (d_err) {
            k_refine_error<<<1, 1, 0, p->stream>>>(num, den, nblk, d_err + it);
            if (!launch()) break;
        }
        if (every >= 1 && (it + 1) % every == 0 && it + 1 < k) {
            // S3 <- [ G_sigma * |O| >= threshold max ] (readings A23, A30) through the same kernels; F waits in d_obj
            if (cudaMemcpyAsync(d_obj, F, sizeof(float2) * n3, cudaMemcpyDeviceToDevice, p->stream) != cudaSuccess) { rc = CPRA_ERR_CUDA; break; }
            dispatch([&](auto nn) {
                constexpr int NN = decltype(nn)::value;
                rc = Launch<NN>::row_fwd(p, O, MIX_ABS, 0, N);                      // |S3 O| formed as the row pass loads O
                if (rc == CPRA_OK) rc = Launch<NN>::col(p, COL_FWD, 0, N, 1.0f);
                if (rc == CPRA_OK) rc = Launch<NN>::fftz_scr(p, F, -1, 1.0f);
            });
            if (rc) break;
            k_gauss3_q<<<8 * p->sms, 256, sizeof(float) * N, p->stream>>>(F, p->geo, nq, sigma);
            if (!launch()) break;
            dispatch([&](auto nn) {
                constexpr int NN = decltype(nn)::value;
                rc = Launch<NN>::fftz_scr(p, F, +1, inv3);
                if (rc == CPRA_OK) rc = Launch<NN>::col(p, COL_INV, 0, N, 1.0f);
                if (rc == CPRA_OK) rc = Launch<NN>::row_inv(p, O, O, false, MIX_NONE, 0.f, 1.0f, 0, N);
            });
            if (rc) break;
            k_image_max<<<N, 256, 0, p->stream>>>(O, p->mx, p->geo);
            if (!launch()) break;
            k_max_final<<<1, 256, 0, p->stream>>>(p->mx, N);
            if (!launch()) break;
            k_max_broadcast<<<1, 256, 0, p->stream>>>(p->mx, N);
            if (!launch()) break;
            if (d_blurred) {
                k_unpack_real<<<blocks_for(n3, 256), 256, 0, p->stream>>>((const float*)O, d_blurred, p->geo, n3);
                if (!launch()) break;
            }
            k_threshold_pack<<<blocks_for(total16, 256), 256, 0, p->stream>>>((const float*)O, p->mx, p->S16, p->geo, total16, threshold);
            if (!launch()) break;
            if (d_S3_out) {
                k_unpack_support<<<blocks_for(n3, 256), 256, 0, p->stream>>>(p->S16, d_S3_out, N, n3);
                if (!launch()) break;
            }
            if (cudaMemcpyAsync(F, d_obj, sizeof(float2) * n3, cudaMemcpyDeviceToDevice, p->stream) != cudaSuccess) { rc = CPRA_ERR_CUDA; break; }
        }
    }
    p->update = saved_update;
    p->positivity = saved_positivity;
    if (rc == CPRA_OK) {
        k_unpack_state<<<blocks_for(units, 256), 256, 0, p->stream>>>((const float*)O, p->S16, (float2*)d_obj, p->geo, units, 0);
        rc = check_launch(p);
    }
    p->have_estimate = false;   // the state buffers, the scratch and the packed support were used
    p->have_support = false;
    p->have_error = false;
    return rc;
}

// The same for the sizes that are not powers of two: the cube's spectrum, the assembled spectrum and the weights in position
// order on all three axes (scratch, second scratch, spare state buffer), the object natural in the state buffer.  An
// iteration is z pass -> column pass -> row pass with the support as an ER update -> row pass -> column pass -> z pass ->
// replace; the natural-order path needed two conversions and a copy more per iteration.
int refine_3d_pos(cpra_plan_s* p, const float* d_E, const float* d_W, const unsigned char* d_S3_in, unsigned char* d_S3_out, int k, int every,
                  float sigma, float threshold, float* d_obj, float* d_err, float* d_blurred)
{
    const int N = p->N;
    const size_t n3 = (size_t)N * N * N;
    const int nblk = (int)std::min<size_t>(2048, (size_t)p->Np * (N / 8) / 2);
    if (nblk < 1) return CPRA_ERR_UNSUPPORTED_SIZE;
    float2* O = (float2*)p->st[p->cur];
    float* Wp = (float*)p->st[p->cur ^ 1];
    float2* F = (float2*)p->scr;
    float2* Ep = (float2*)p->scr2;
    double* num = p->partial;
    double* den = p->partial + nblk;
    const int saved_update = p->update;
    const auto saved_positivity = p->positivity;
    int rc = CPRA_OK;
    auto launch = [&]() { return (rc = check_launch(p)) == CPRA_OK; };
    if (cudaMemcpyAsync(p->S8, d_S3_in, n3, cudaMemcpyDeviceToDevice, p->stream) != cudaSuccess) return CPRA_ERR_CUDA;
    // (the weights' buffer doubles as the finite "previous state" that the ER update multiplies by 0: clear all of it)
    if (cudaMemsetAsync(Wp, 0, sizeof(float2) * n3, p->stream) != cudaSuccess) return CPRA_ERR_CUDA;
    if ((rc = gen_cube_to_pos(p, (const float2*)d_E, Ep))) return rc;
    if ((rc = gen_cube_to_pos_f(p, d_W, Wp))) return rc;
    k_refine_init<<<nblk, 256, 0, p->stream>>>(Ep, Wp, F, den, n3);
    if (!launch()) return rc;
    p->update = CPRA_UPDATE_ER;
    p->positivity = 0;                               // (Step D has no positivity step: reading A26)
    for (int it = 0; it < k && rc == CPRA_OK; ++it) {
        if ((rc = gen_cube_inverse(p, O, true, (const float2*)Wp))) break;       // O = S3 . F3^-1[F]
        if ((rc = gen_cube_forward(p, O))) break;                                 // F' = F3[O]
        k_refine_replace<<<nblk, 256, 0, p->stream>>>(F, Ep, Wp, num, n3);
        if (!launch()) break;
        if (d_err) {
            k_refine_error<<<1, 1, 0, p->stream>>>(num, den, nblk, d_err + it);
            if (!launch()) break;
        }
        if (every >= 1 && (it + 1) % every == 0 && it + 1 < k) {
            // S3 <- [ G_sigma * |O| >= threshold max ] through the same transforms; F waits in d_obj
            if (cudaMemcpyAsync(d_obj, F, sizeof(float2) * n3, cudaMemcpyDeviceToDevice, p->stream) != cudaSuccess) { rc = CPRA_ERR_CUDA; break; }
            k_abs3<<<blocks_for(n3, 256), 256, 0, p->stream>>>(O, O, n3);
            if (!launch()) break;
            if ((rc = gen_cube_forward(p, O))) break;
            if ((rc = gen_cube_gauss(p, sigma))) break;
            if ((rc = gen_cube_inverse(p, O, false, nullptr))) break;
            k_plane_max<<<N, 256, 0, p->stream>>>(O, p->mx, (size_t)N * N);
            if (!launch()) break;
            k_max_final<<<1, 256, 0, p->stream>>>(p->mx, N);
            if (!launch()) break;
            k_threshold3<<<blocks_for(n3, 256), 256, 0, p->stream>>>(O, p->mx, p->S8, d_blurred, n3, threshold);
            if (!launch()) break;
            if (d_S3_out && cudaMemcpyAsync(d_S3_out, p->S8, n3, cudaMemcpyDeviceToDevice, p->stream) != cudaSuccess) { rc = CPRA_ERR_CUDA; break; }
            if (cudaMemcpyAsync(F, d_obj, sizeof(float2) * n3, cudaMemcpyDeviceToDevice, p->stream) != cudaSuccess) { rc = CPRA_ERR_CUDA; break; }
        }
    }
    p->update = saved_update;
    p->positivity = saved_positivity;
    if (rc == CPRA_OK && cudaMemcpyAsync(d_obj, O, sizeof(float2) * n3, cudaMemcpyDeviceToDevice, p->stream) != cudaSuccess) rc = CPRA_ERR_CUDA;
    p->have_estimate = false;
    p->have_support = false;
    p->have_error = false;
    return rc;
}
}  // namespace

extern "C" {

int cpra_fft3(cpra_plan_t p, const float* d_in, float* d_out, int sign)
{
    if (!p || !d_in || !d_out || (sign != 1 && sign != -1)) return CPRA_ERR_INVALID_ARG;
    if (p->Np != p->N) return CPRA_ERR_INVALID_ARG;   // a cube is a stack of N slices of N x N
    int rc = cpra_fft2(p, d_in, d_out, sign);          // the (y, x) transforms of all z slices
    if (rc) return rc;
    if (p->generic) return gen_fftz(p, (float2*)d_out, sign);
    { auto f = [&]() -> int { CPRA_DISPATCH_N(p->N, rc = Launch<NN>::fftz(p, (float2*)d_out, sign)); return 0; }; f(); }
    return rc;
}

int cpra_refine_3d(cpra_plan_t p, const float* d_E, const float* d_W, const unsigned char* d_S3, int k, float* d_obj, float* d_err)
{
    if (!p || !d_E || !d_W || !d_S3 || !d_obj || k < 1) return CPRA_ERR_INVALID_ARG;
    if (p->Np != p->N) return CPRA_ERR_INVALID_ARG;
    if (int rc = ready(p)) return rc;
    if (!p->generic) return refine_3d_tiled(p, d_E, d_W, d_S3, nullptr, k, 0, 0.f, 0.f, d_obj, d_err, nullptr);
    return refine_3d_pos(p, d_E, d_W, d_S3, nullptr, k, 0, 0.f, 0.f, d_obj, d_err, nullptr);
}

int cpra_refine_3d_sw(cpra_plan_t p, const float* d_E, const float* d_W, unsigned char* d_S3, int k, int every, float sigma, float threshold,
                      float* d_obj, float* d_err, float* d_blurred)
{
    if (!p || !d_E || !d_W || !d_S3 || !d_obj || k < 1 || !(sigma >= 0.f) || !(threshold >= 0.f) || !std::isfinite(sigma) ||
        !std::isfinite(threshold))
        return CPRA_ERR_INVALID_ARG;
    if (p->Np != p->N) return CPRA_ERR_INVALID_ARG;
    if (int rc = ready(p)) return rc;
    if (!p->generic) return refine_3d_tiled(p, d_E, d_W, d_S3, d_S3, k, every, sigma, threshold, d_obj, d_err, d_blurred);
    return refine_3d_pos(p, d_E, d_W, d_S3, d_S3, k, every, sigma, threshold, d_obj, d_err, d_blurred);
}

int cpra_backproject_support(cpra_plan_t p, unsigned char* d_S3)
{
    if (!p || !d_S3) return CPRA_ERR_INVALID_ARG;
    if (int rc = ready(p)) return rc;
    if (!p->have_support) return CPRA_ERR_NOT_READY;
    const size_t total = (size_t)p->Np * p->N * p->N, n3 = (size_t)p->N * p->N * p->N;
    // the 2D supports as bytes: this path's own copy, or unpacked into the second scratch
    const unsigned char* S = p->S8;
    if (!p->generic) {
        unsigned char* u8 = (unsigned char*)p->scr2;
        k_unpack_support<<<blocks_for(total, 256), 256, 0, p->stream>>>(p->S16, u8, p->N, total);
        if (int rc = check_launch(p)) return rc;
        S = u8;
    }
    p->h_cs.resize(2 * (size_t)p->Np);
    for (int n = 0; n < p->Np; ++n) { p->h_cs[2 * n] = std::cos(p->angles[n]); p->h_cs[2 * n + 1] = std::sin(p->angles[n]); }
    double* cs = p->align;   // 9 Np doubles of scratch, free between calls
    if (cudaMemcpyAsync(cs, p->h_cs.data(), sizeof(double) * 2 * p->Np, cudaMemcpyHostToDevice, p->stream) != cudaSuccess) return CPRA_ERR_CUDA;
    k_backproject_support<<<blocks_for(n3, 256), 256, 0, p->stream>>>(S, cs, d_S3, p->N, p->Np);
    return check_launch(p);
}

int cpra_fsc(cpra_plan_t p, const float* d_F1, const float* d_F2, float* d_out)
{
    if (!p || !d_F1 || !d_F2 || !d_out) return CPRA_ERR_INVALID_ARG;
    if (p->Np != p->N) return CPRA_ERR_INVALID_ARG;
    if (int rc = ready(p)) return rc;
    const int ns = p->N / 2 + 1;
    double* acc = p->shell;
    if (cudaMemsetAsync(acc, 0, sizeof(double) * 3 * ns, p->stream) != cudaSuccess) return CPRA_ERR_CUDA;
    k_fsc_accumulate<<<4 * p->sms, 256, sizeof(double) * 3 * ns, p->stream>>>((const float2*)d_F1, (const float2*)d_F2, acc, p->N);
    if (int rc = check_launch(p)) return rc;
    k_fsc_finalize<<<blocks_for(ns, 128), 128, 0, p->stream>>>(acc, d_out, ns);
    return check_launch(p);
}

int cpra_prtf(cpra_plan_t p, const float* d_avg, float* d_out)
{
    if (!p || !d_avg || !d_out) return CPRA_ERR_INVALID_ARG;
    if (int rc = ready(p)) return rc;
    if (!p->have_data) return CPRA_ERR_NOT_READY;
    const size_t total = (size_t)p->Np * p->N * p->N;
    const int ns = p->N / 2 + 1;
    if (p->generic) {
        if (int rc = gen_prtf_sums(p, d_avg, p->shell)) return rc;
        k_prtf_finalize<<<blocks_for(ns, 128), 128, 0, p->stream>>>(p->shell, d_out, ns);
        return check_launch(p);
    }
    float4* tmp = p->st[p->cur ^ 1];
    k_pack_state<<<blocks_for(total / p->geo.TB, 256), 256, 0, p->stream>>>((const float2*)d_avg, (float*)tmp, p->geo, total / p->geo.TB);
    int rc = check_launch(p);
    if (rc) return rc;
    { auto f = [&]() -> int {
        CPRA_DISPATCH_N(p->N,
            rc = Launch<NN>::row_fwd(p, tmp, MIX_NONE, 0, p->Np);
            if (rc == CPRA_OK) rc = Launch<NN>::col(p, COL_FWD, 0, p->Np, 1.0f));
        return 0; }; f(); }
    if (rc) return rc;
    double* acc = p->shell;
    if (cudaMemsetAsync(acc, 0, sizeof(double) * 2 * ns, p->stream) != cudaSuccess) return CPRA_ERR_CUDA;
    k_prtf_accumulate<<<4 * p->sms, 256, sizeof(double) * 2 * ns, p->stream>>>((const float*)p->scr, p->A, acc, p->geo, total);
    if ((rc = check_launch(p))) return rc;
    k_prtf_finalize<<<blocks_for(ns, 128), 128, 0, p->stream>>>(acc, d_out, ns);
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
