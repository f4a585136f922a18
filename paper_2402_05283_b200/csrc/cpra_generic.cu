// cpra_generic.cu -- host side of the path for sizes that are not powers of two (cpra_generic.cuh).
#include "cpra_plan.cuh"
#include "cpra_generic_kernels.cuh"

namespace cpra {

bool gen_supported(int N)
{
    if (N < 16 || N > 1024 || (N & 1)) return false;
    int n = N;
    for (int f : {2, 3, 5, 7}) while (n % f == 0) n /= f;
    return n == 1;
}

// stages: 8s, then 4 / 2, then 3s, 5s, 7s (an odd radix last: the stage with contiguous positions is then free of
// bank conflicts); W = lines per tile; tw[m] = e^{-2 pi i m / N}
void gen_make_geo(int N, int Np, GenGeo& g, std::vector<float2>& tw)
{
    g.N = N; g.Np = Np; g.W = gen_lines_per_tile(N); g.nf = 0;
    int n = N;
    while (n % 8 == 0) { g.radix[g.nf++] = 8; n /= 8; }
    if (n % 4 == 0) { g.radix[g.nf++] = 4; n /= 4; }
    if (n % 2 == 0) { g.radix[g.nf++] = 2; n /= 2; }
    for (int f : {3, 5, 7}) while (n % f == 0) { g.radix[g.nf++] = f; n /= f; }
    for (int s = 0, L = N; s < g.nf; ++s) {
        g.L[s] = L; g.M[s] = L / g.radix[s]; g.ts[s] = N / L; g.nb[s] = N / g.radix[s]; g.invM[s] = 1.0f / (float)g.M[s];
        L /= g.radix[s];
    }
    const double PI = 3.14159265358979323846264338327950288;
    tw.assign(1024, make_float2(0.f, 0.f));
    for (int m = 0; m < N; ++m) {
        const double a = -2.0 * PI * (double)m / (double)N;
        tw[m] = make_float2((float)std::cos(a), (float)std::sin(a));
    }
}

int gen_set_attrs()
{
    cudaError_t e = cudaSuccess;
    auto acc = [&](cudaError_t r) { if (e == cudaSuccess) e = r; };
    const int SM = 200 * 1024;
    acc(allow_smem(k_gen_row_fwd, SM));
    acc(allow_smem(k_gen_col<0>, SM));
    acc(allow_smem(k_gen_col<1>, SM));
    acc(allow_smem(k_gen_col<2>, SM));
    acc(allow_smem(k_gen_col<3>, SM));
    acc(allow_smem(k_gen_col<4>, SM));
    acc(allow_smem(k_gen_row_inv, SM));
    // as much shared memory as the SM has, whatever one block asks for (the default carveout fits fewer blocks)
    acc(cudaFuncSetAttribute(reinterpret_cast<const void*>(k_gen_row_fwd), cudaFuncAttributePreferredSharedMemoryCarveout, cudaSharedmemCarveoutMaxShared));
    acc(cudaFuncSetAttribute(reinterpret_cast<const void*>(k_gen_col<0>), cudaFuncAttributePreferredSharedMemoryCarveout, cudaSharedmemCarveoutMaxShared));
    acc(cudaFuncSetAttribute(reinterpret_cast<const void*>(k_gen_col<1>), cudaFuncAttributePreferredSharedMemoryCarveout, cudaSharedmemCarveoutMaxShared));
    acc(cudaFuncSetAttribute(reinterpret_cast<const void*>(k_gen_col<2>), cudaFuncAttributePreferredSharedMemoryCarveout, cudaSharedmemCarveoutMaxShared));
    acc(cudaFuncSetAttribute(reinterpret_cast<const void*>(k_gen_col<3>), cudaFuncAttributePreferredSharedMemoryCarveout, cudaSharedmemCarveoutMaxShared));
    acc(cudaFuncSetAttribute(reinterpret_cast<const void*>(k_gen_col<4>), cudaFuncAttributePreferredSharedMemoryCarveout, cudaSharedmemCarveoutMaxShared));
    acc(cudaFuncSetAttribute(reinterpret_cast<const void*>(k_gen_row_inv), cudaFuncAttributePreferredSharedMemoryCarveout, cudaSharedmemCarveoutMaxShared));
    return e == cudaSuccess ? CPRA_OK : CPRA_ERR_CUDA;
}

namespace {
unsigned gblocks(size_t total, int nt) { return (unsigned)((total + nt - 1) / nt); }
int tiles_of(const cpra_plan_s* p) { return (p->gg.N + p->gg.W - 1) / p->gg.W; }
int smem_of(const cpra_plan_s* p) { return (int)gen_smem_bytes(p->gg.N, p->gg.W); }

int row_fwd(cpra_plan_s* p, const float2* cur, int n0, int nimg, bool fires, bool mask, float2* ghat_out)
{
    ProfScope prof(p, CPRA_PROFILE_ROW_FWD);
    k_gen_row_fwd<<<(unsigned)(nimg * tiles_of(p)), GEN_NT, smem_of(p), p->stream>>>(cur, (float2*)p->scr, p->tw, p->S8, mix_params(p), p->gg, n0,
                                                                                      fires ? 1 : 0, mask ? 1 : 0, ghat_out);
    return check_launch(p);
}
int col(cpra_plan_s* p, int n0, int nimg, int mode, float scale)
{
    ProfScope prof(p, CPRA_PROFILE_COL);
    const unsigned grid = (unsigned)(nimg * tiles_of(p));
    const size_t px = (size_t)p->N * p->N, N = (size_t)p->N;
    if (mode == 0) k_gen_col<0><<<grid, GEN_NT, smem_of(p), p->stream>>>((float2*)p->scr, p->A, p->tw, p->partial, p->gg, n0, scale, px, N);
    else if (mode == 1) k_gen_col<1><<<grid, GEN_NT, smem_of(p), p->stream>>>((float2*)p->scr, p->A, p->tw, p->partial, p->gg, n0, scale, px, N);
    else k_gen_col<2><<<grid, GEN_NT, smem_of(p), p->stream>>>((float2*)p->scr, p->A, p->tw, p->partial, p->gg, n0, scale, px, N);
    return check_launch(p);
}
int permute(cpra_plan_s* p, const float2* in, float2* out, int to_pos, int zperm = 0)
{
    const int N = p->N, nb = (N + GEN_PB - 1) / GEN_PB;
    const size_t sm = sizeof(float2) * GEN_PB * N + sizeof(int) * 2 * N;
    k_gen_permute<float2><<<(unsigned)(p->Np * nb), 256, sm, p->stream>>>(in, out, p->gg, to_pos, zperm);
    return check_launch(p);
}
// the z pass on the cube held in p->scr with its planes in position order (modes 1 / 2 of the column kernel with rows one
// plane apart): forward natural z -> position order, inverse position order -> natural z
int zpass_pos(cpra_plan_s* p, int sign)
{
    const size_t N = (size_t)p->N;
    const unsigned grid = (unsigned)(p->N * tiles_of(p));
    if (sign < 0) k_gen_col<1><<<grid, GEN_NT, smem_of(p), p->stream>>>((float2*)p->scr, nullptr, p->tw, nullptr, p->gg, 0, 1.0f, N, N * N);
    else k_gen_col<2><<<grid, GEN_NT, smem_of(p), p->stream>>>((float2*)p->scr, nullptr, p->tw, nullptr, p->gg, 0, 1.0f, N, N * N);
    return check_launch(p);
}
int row_inv(cpra_plan_s* p, const float2* cur, float2* nxt, int n0, int nimg, bool fires, bool hio, float beta, float scale, const float2* ghat)
{
    ProfScope prof(p, CPRA_PROFILE_ROW_INV);
    k_gen_row_inv<<<(unsigned)(nimg * tiles_of(p)), GEN_NT, smem_of(p), p->stream>>>((const float2*)p->scr, cur, nxt, p->tw, p->S8, mix_params(p, beta),
                                                                                      p->gg, n0, fires ? 1 : 0, hio ? 1 : 0, scale, ghat);
    return check_launch(p);
}
}  // namespace

int gen_set_data(cpra_plan_s* p, const float* d_I, const unsigned char* d_mask)
{
    k_gen_set_data<<<p->Np, 256, 0, p->stream>>>(d_I, d_mask, p->A, p->den, p->gg);
    return check_launch(p);
}
int gen_set_support(cpra_plan_s* p, const unsigned char* d_S)
{
    const size_t total = (size_t)p->Np * p->N * p->N;
    k_gen_copy_support<<<gblocks(total, 256), 256, 0, p->stream>>>(d_S, p->S8, total);
    return check_launch(p);
}
int gen_set_estimate(cpra_plan_s* p, const float* d_g0)
{
    const size_t total = (size_t)p->Np * p->N * p->N;
    return cudaMemcpyAsync(p->st[p->cur], d_g0, sizeof(float2) * total, cudaMemcpyDeviceToDevice, p->stream) == cudaSuccess ? CPRA_OK : CPRA_ERR_CUDA;
}
// g0 = F^-1[G0], G0 natural, straight into the state buffer
int gen_set_estimate_spectrum(cpra_plan_s* p, const float* d_G0)
{
    int rc = permute(p, (const float2*)d_G0, (float2*)p->scr, 1);
    if (rc == CPRA_OK) rc = col(p, 0, p->Np, 2, 1.0f);
    float2* g = (float2*)p->st[p->cur];
    if (rc == CPRA_OK) rc = row_inv(p, g, g, 0, p->Np, false, false, 0.f, 1.0f / ((float)p->N * (float)p->N), nullptr);
    return rc;
}
int gen_get_projections(cpra_plan_s* p, int which, float* d_out)
{
    const size_t total = (size_t)p->Np * p->N * p->N;
    k_gen_get<<<gblocks(total, 256), 256, 0, p->stream>>>((const float2*)p->st[p->cur], p->S8, (float2*)d_out, total, which == CPRA_SUPPORTED);
    return check_launch(p);
}

// one iteration = K1 (mix + row FFT, ghat stored when the mix fires) -> K2 -> K3, for all projections
int gen_iterate(cpra_plan_s* p, int k, float beta)
{
    const float scale = 1.0f / ((float)p->N * (float)p->N);
    for (int it = 0; it < k; ++it) {
        const bool fires = (p->t % p->n_ei) == 0 && !(p->K == 0 && p->alpha[0] == 1.0f);
        const float2* cur = (const float2*)p->st[p->cur];
        float2* nxt = (float2*)p->st[p->cur ^ 1];
        float2* gh = fires ? (float2*)p->scr2 : nullptr;
        int rc = row_fwd(p, cur, 0, p->Np, fires, false, gh);
        if (rc == CPRA_OK) rc = col(p, 0, p->Np, 0, scale);
        if (rc == CPRA_OK) rc = row_inv(p, cur, nxt, 0, p->Np, false, true, beta, 1.0f, fires ? gh : cur);
        if (rc != CPRA_OK) return rc;
        p->cur ^= 1;
        p->t += 1;
        p->have_error = true;
    }
    return CPRA_OK;
}

int gen_prereconstruct(cpra_plan_s* p, int n, int k, float beta)
{
    const float scale = 1.0f / ((float)p->N * (float)p->N);
    int src = p->cur, rc = CPRA_OK;
    for (int it = 0; it < k && rc == CPRA_OK; ++it) {
        const float2* cur = (const float2*)p->st[src];
        float2* nxt = (float2*)p->st[src ^ 1];
        rc = row_fwd(p, cur, n, 1, false, false, nullptr);
        if (rc == CPRA_OK) rc = col(p, n, 1, 0, scale);
        if (rc == CPRA_OK) rc = row_inv(p, cur, nxt, n, 1, false, true, beta, 1.0f, cur);
        src ^= 1;
    }
    if (rc) return rc;
    if (src != p->cur) {
        const size_t ib = sizeof(float2) * (size_t)p->N * p->N;
        if (cudaMemcpyAsync((char*)p->st[p->cur] + ib * n, (const char*)p->st[src] + ib * n, ib, cudaMemcpyDeviceToDevice, p->stream) != cudaSuccess)
            return CPRA_ERR_CUDA;
    }
    p->have_error = false;
    return CPRA_OK;
}

int gen_fft2(cpra_plan_s* p, const float* d_in, float* d_out, int sign)
{
    const size_t total = (size_t)p->Np * p->N * p->N;
    float2* tmp = (float2*)p->st[p->cur ^ 1];
    int rc;
    if (sign < 0) {
        if ((rc = row_fwd(p, (const float2*)d_in, 0, p->Np, false, false, nullptr))) return rc;
        if ((rc = col(p, 0, p->Np, 1, 1.0f))) return rc;
        return permute(p, (const float2*)p->scr, (float2*)d_out, 0);
    }
    if ((rc = permute(p, (const float2*)d_in, (float2*)p->scr, 1))) return rc;
    if ((rc = col(p, 0, p->Np, 2, 1.0f))) return rc;
    if ((rc = row_inv(p, tmp, tmp, 0, p->Np, false, false, 0.f, 1.0f / ((float)p->N * (float)p->N), nullptr))) return rc;
    return cudaMemcpyAsync(d_out, tmp, sizeof(float2) * total, cudaMemcpyDeviceToDevice, p->stream) == cudaSuccess ? CPRA_OK : CPRA_ERR_CUDA;
}

// the z pass of cpra_fft3 on a natural [z][y][x] volume, in place: for every y, the W-column tiles of the [z][x] slice
// (rows N^2 apart) through the column kernel's natural-order modes; inverse: times 1 / N
int gen_fftz(cpra_plan_s* p, float2* vol, int sign)
{
    const size_t N = (size_t)p->N;
    const unsigned grid = (unsigned)(p->N * tiles_of(p));
    if (sign < 0) k_gen_col<3><<<grid, GEN_NT, smem_of(p), p->stream>>>(vol, nullptr, p->tw, nullptr, p->gg, 0, 1.0f, N, N * N);
    else k_gen_col<4><<<grid, GEN_NT, smem_of(p), p->stream>>>(vol, nullptr, p->tw, nullptr, p->gg, 0, 1.0f / (float)p->N, N, N * N);
    return check_launch(p);
}

// shrink-wrap (cpra_shrinkwrap): b_n = G_sigma * |S_n g_n| through this path's own transforms, S_n <- [b_n >= threshold max b_n]
int gen_shrinkwrap(cpra_plan_s* p, float sigma, float threshold, float* d_blurred)
{
    const size_t total = (size_t)p->Np * p->N * p->N;
    float2* tmp = (float2*)p->st[p->cur ^ 1];
    k_gen_abs_supported<<<gblocks(total, 256), 256, 0, p->stream>>>((const float2*)p->st[p->cur], p->S8, tmp, total);
    int rc = check_launch(p);
    if (rc == CPRA_OK) rc = row_fwd(p, tmp, 0, p->Np, false, false, nullptr);
    if (rc == CPRA_OK) rc = col(p, 0, p->Np, 1, 1.0f);
    if (rc) return rc;
    k_gen_gauss_filter<<<8 * p->sms, 256, sizeof(float) * p->N, p->stream>>>((float2*)p->scr, p->gg, total, sigma);
    if ((rc = check_launch(p))) return rc;
    if ((rc = col(p, 0, p->Np, 2, 1.0f))) return rc;
    if ((rc = row_inv(p, tmp, tmp, 0, p->Np, false, false, 0.f, 1.0f / ((float)p->N * (float)p->N), nullptr))) return rc;
    k_gen_image_max<<<p->Np, 256, 0, p->stream>>>(tmp, p->mx, p->N);
    if ((rc = check_launch(p))) return rc;
    k_gen_threshold<<<gblocks(total, 256), 256, 0, p->stream>>>(tmp, p->mx, p->S8, d_blurred, p->N, total, threshold);
    return check_launch(p);
}

// the shell sums of cpra_prtf into acc (2 (N / 2 + 1) doubles, cleared here)
int gen_prtf_sums(cpra_plan_s* p, const float* d_avg, double* acc)
{
    const size_t total = (size_t)p->Np * p->N * p->N;
    const int ns = p->N / 2 + 1;
    int rc = row_fwd(p, (const float2*)d_avg, 0, p->Np, false, false, nullptr);
    if (rc == CPRA_OK) rc = col(p, 0, p->Np, 1, 1.0f);
    if (rc) return rc;
    if (cudaMemsetAsync(acc, 0, sizeof(double) * 2 * ns, p->stream) != cudaSuccess) return CPRA_ERR_CUDA;
    k_gen_prtf_accumulate<<<4 * p->sms, 256, sizeof(double) * 2 * ns, p->stream>>>((const float2*)p->scr, p->A, acc, p->gg, total);
    return check_launch(p);
}

// ---- Step D's iterations with the cube in position order on all three axes (cpra_refine_3d on this path; Np == N) ----
// natural cube -> position order (complex / float)
int gen_cube_to_pos(cpra_plan_s* p, const float2* in, float2* out) { return permute(p, in, out, 1, 1); }
int gen_cube_to_pos_f(cpra_plan_s* p, const float* in, float* out)
{
    const int N = p->N, nb = (N + GEN_PB - 1) / GEN_PB;
    const size_t sm = sizeof(float) * GEN_PB * N + sizeof(int) * 2 * N;
    k_gen_permute<float><<<(unsigned)(N * nb), 256, sm, p->stream>>>(in, out, p->gg, 1, 1);
    return check_launch(p);
}
// O = [support .] F3^-1[spectrum in p->scr] / N^3, natural order: z pass, column pass, row pass; with_support: the row pass
// applies the plan's support bytes as an ER update (outside 0), `finite` = any buffer of N^3 finite complex numbers (it is
// read as the previous state and multiplied by 0)
int gen_cube_inverse(cpra_plan_s* p, float2* O, bool with_support, const float2* finite)
{
    const float inv3 = 1.0f / ((float)p->N * (float)p->N * (float)p->N);
    int rc = zpass_pos(p, +1);
    if (rc == CPRA_OK) rc = col(p, 0, p->N, 2, 1.0f);
    if (rc == CPRA_OK) rc = row_inv(p, finite, O, 0, p->N, false, with_support, 0.f, inv3, with_support ? finite : nullptr);
    return rc;
}
// spectrum of the natural cube O into p->scr, position order
int gen_cube_forward(cpra_plan_s* p, const float2* O)
{
    int rc = row_fwd(p, O, 0, p->N, false, false, nullptr);
    if (rc == CPRA_OK) rc = col(p, 0, p->N, 1, 1.0f);
    if (rc == CPRA_OK) rc = zpass_pos(p, -1);
    return rc;
}
int gen_cube_gauss(cpra_plan_s* p, float sigma)
{
    const size_t n3 = (size_t)p->N * p->N * p->N;
    k_gen_gauss3<<<8 * p->sms, 256, sizeof(float) * p->N, p->stream>>>((float2*)p->scr, p->gg, n3, sigma);
    return check_launch(p);
}

int gen_slices(cpra_plan_s* p, float2* Et)
{
    const size_t total = (size_t)p->Np * p->N * p->N;
    int rc = row_fwd(p, (const float2*)p->st[p->cur], 0, p->Np, false, true, nullptr);
    if (rc == CPRA_OK) rc = col(p, 0, p->Np, 1, 1.0f);
    if (rc) return rc;
    k_gen_transpose<<<gblocks(total, 256), 256, 0, p->stream>>>((const float2*)p->scr, Et, p->gg, total);
    return check_launch(p);
}

}  // namespace cpra
