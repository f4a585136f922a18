/*
 * oracle/cpra_oracle.c -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * A plain, slow, obviously-correct CPU implementation of the CPRA iteration loop
 * (arXiv 2402.05283, "Real time 3D coherent X-ray diffraction imaging"), written from
 * /root/reference/PAPER.md (cited as P:<line>) and the readings listed in DESIGN.md.
 * It is the parity oracle for the CUDA path and shares NO code with it.  Only tests/,
 * __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may load it.
 *
 * Precision: every real number is `real` = double (liboracle.so).  The same source compiled with
 * -DORACLE_REAL=float (liboracle_f32.so) is used ONLY to show how far an fp32 state drifts from
 * the fp64 one over 20 iterations ("hard parts"); it is never the reference.
 *
 * What is computed, in the paper's order (one call oracle_iterate(k, beta) repeats k times):
 *   1. carousel mix, Eq. (4):  ghat_n = sum_{j=-K..K} alpha_|j| g_{(n+j) mod Np}
 *      (Jacobi: all right-hand sides from the state before the step; fires iff t mod n_ei == 0)
 *   2. forward 2D FT, Eq. (3):     G_n = F[ghat_n]      (e^{-2 pi i ...}, unnormalised)
 *   3. error:                      num_n = sum_{M=1} (|G_n| - A_n)^2, E_n = sqrt(num_n/den_n)
 *   4. Fourier-modulus constraint, P:13, P:25, P:98:
 *                                        measured: G' = A G/|G| (G' = A if |G| = 0); masked: G' = G
 *   5. inverse 2D FT:              g'_n = F^-1[G'_n]    (e^{+2 pi i ...} / N^2)
 *   6. support / HIO, P:98 ref [22], P:104 (beta):
 *                                        S=1: g_n <- g'_n ;  S=0: g_n <- ghat_n - beta g'_n
 *   7. t <- t + 1
 * plus the one-shot Fourier-slice assembly of Step D's first sentence; the
 * interpolation scheme is the polar bilinear gather of DESIGN.md (reading A17: the paper only says
 * "interpolate").  Its steps are pinned (geometry, centring, duplicate rays, and the weights: exact on a
 * spectrum bilinear in angle and radius); how close the scheme comes to the continuous transform is a
 * property of the method, measured on an analytic Gaussian, not a parity matter.
 *
 * Pins (tests/test_oracle_*.py): brute-force O(N^4) DFT below (separate code path), numpy.fft,
 * Parseval, shift theorem, Fourier-slice identity, idempotence of the two projections, closed-form
 * HIO decay, circulant eigenvalues of the mix, fixed point of the true object, error closed forms;
 * the feedback operand of step 6 under coupling (one-hot stack, nothing measured: (1 - beta) alpha
 * outside the support), the clamp of negative intensities (|F[g']| = 0 there), and the averaging of
 * duplicate rays in the assembly (slices with different constant spectra on a 360 degree scan).
 * A multi-iteration trajectory is the composition of these pinned steps; the composition itself is pinned by the
 * closed-form decay over k iterations, the fixed points and the split-call identity, not by an external trajectory.
 *
 * Around the loop (each function below cites its passage and is pinned in tests/test_oracle_next.py):
 * seam flip, blur / shrink-wrap, Step A, centre of mass / bank / merge (Step C), phase gauge and twin chain of an
 * episode, the 3D transform and Step D's iterations, the 3D support as the back-projection of the 2D supports and its
 * re-thresholding, FSC / PRTF, positivity.  Sizes that are not powers of two use the O(N^2)
 * definition of the 1D transform, in 2D and in 3D.
 *
 * Layout: images row-major [n][y][x], x fastest; complex = interleaved (re, im).  All I/O arrays of
 * this library are double / interleaved double regardless of `real`.
 */
#include <math.h>
#include <stdlib.h>
#include <string.h>

#ifndef ORACLE_REAL
#define ORACLE_REAL double
#endif
typedef ORACLE_REAL real;
typedef struct { real re, im; } cplx;

#define ORACLE_OK 0
#define ORACLE_ERR_INVALID_ARG (-1)
#define ORACLE_ERR_UNSUPPORTED_SIZE (-2)
#define ORACLE_ERR_NOT_READY (-3)

static const double PI = 3.14159265358979323846264338327950288;

/* ------------------------------------------------------------------------------------------ */
/* Fourier transforms                                                                          */
/* ------------------------------------------------------------------------------------------ */

/* Textbook iterative radix-2 decimation-in-time FFT, in place, N a power of two.
 * tw[m] = e^{sign 2 pi i m / N}, m = 0..N/2-1 (computed in double by twiddle_table, rounded once).
 * sign = -1: X[k] = sum_x x[x] e^{-2 pi i k x / N};  sign = +1: e^{+...}; never scaled here. */
static void fft1d(cplx* a, int N, const cplx* tw)
{
    /* bit-reversal permutation */
    for (int i = 1, j = 0; i < N; ++i) {
        int bit = N >> 1;
        for (; j & bit; bit >>= 1) j ^= bit;
        j ^= bit;
        if (i < j) { cplx t = a[i]; a[i] = a[j]; a[j] = t; }
    }
    for (int len = 2; len <= N; len <<= 1) {
        const int half = len >> 1, step = N / len;
        for (int i = 0; i < N; i += len) {
            for (int k = 0; k < half; ++k) {
                const real wr = tw[k * step].re, wi = tw[k * step].im;   /* e^{sign 2 pi i k/len} */
                const cplx u = a[i + k], v = a[i + k + half];
                const real tr = v.re * wr - v.im * wi;
                const real ti = v.re * wi + v.im * wr;
                a[i + k].re = u.re + tr;        a[i + k].im = u.im + ti;
                a[i + k + half].re = u.re - tr; a[i + k + half].im = u.im - ti;
            }
        }
    }
}

static cplx* twiddle_table(int N, int sign)
{
    cplx* tw = (cplx*)malloc(sizeof(cplx) * (size_t)(N / 2 + 1));
    for (int m = 0; m < N / 2; ++m) {
        const double ang = sign * 2.0 * PI * (double)m / (double)N;
        tw[m].re = (real)cos(ang); tw[m].im = (real)sin(ang);
    }
    return tw;
}

static int is_pow2(int N);

/* N not a power of two (the paper's own detector sizes, P:82 N = 160, P:98 N = 700): the 1D transform is
 * the definition itself, X[k] = sum_x x[x] e^{sign 2 pi i k x / N}, O(N^2) per line, with the N roots of
 * unity computed in double and rounded once.  tmp: N scratch elements. */
static void dft1d_direct(cplx* a, int N, const cplx* root, cplx* tmp)
{
    for (int k = 0; k < N; ++k) {
        real sr = 0, si = 0;
        for (int x = 0; x < N; ++x) {
            const cplx w = root[(int)(((long)k * x) % N)];
            sr += a[x].re * w.re - a[x].im * w.im;
            si += a[x].re * w.im + a[x].im * w.re;
        }
        tmp[k].re = sr; tmp[k].im = si;
    }
    for (int k = 0; k < N; ++k) a[k] = tmp[k];
}
static cplx* root_table(int N, int sign)
{
    cplx* r = (cplx*)malloc(sizeof(cplx) * (size_t)N);
    for (int m = 0; m < N; ++m) {
        const double ang = sign * 2.0 * PI * (double)m / (double)N;
        r[m].re = (real)cos(ang); r[m].im = (real)sin(ang);
    }
    return r;
}

/* 2D transform of one N x N image, in place: all rows, then all columns (Eq. (3) is a
 * separable double sum).  sign=+1 additionally divides by N^2 (P:19 inverse FT; reading A10). */
static void fft2d(cplx* img, int N, int sign)
{
    cplx* col = (cplx*)malloc(sizeof(cplx) * (size_t)N);
    if (!is_pow2(N)) {
        cplx* root = root_table(N, sign);
        cplx* tmp = (cplx*)malloc(sizeof(cplx) * (size_t)N);
        for (int y = 0; y < N; ++y) dft1d_direct(img + (size_t)y * N, N, root, tmp);
        for (int x = 0; x < N; ++x) {
            for (int y = 0; y < N; ++y) col[y] = img[(size_t)y * N + x];
            dft1d_direct(col, N, root, tmp);
            for (int y = 0; y < N; ++y) img[(size_t)y * N + x] = col[y];
        }
        free(root); free(tmp); free(col);
        if (sign > 0) {
            const real s = (real)(1.0 / ((double)N * (double)N));
            for (size_t i = 0; i < (size_t)N * N; ++i) { img[i].re *= s; img[i].im *= s; }
        }
        return;
    }
    cplx* tw = twiddle_table(N, sign);
    for (int y = 0; y < N; ++y) fft1d(img + (size_t)y * N, N, tw);
    for (int x = 0; x < N; ++x) {
        for (int y = 0; y < N; ++y) col[y] = img[(size_t)y * N + x];
        fft1d(col, N, tw);
        for (int y = 0; y < N; ++y) img[(size_t)y * N + x] = col[y];
    }
    free(col); free(tw);
    if (sign > 0) {
        const real s = (real)(1.0 / ((double)N * (double)N));
        for (size_t i = 0; i < (size_t)N * N; ++i) { img[i].re *= s; img[i].im *= s; }
    }
}

/* Brute-force definition, O(N^4), its own code path (no FFT, no shared twiddle logic), always in
 * double: out[ky][kx] = sum_{y,x} in[y][x] e^{sign 2 pi i (ky y + kx x)/N}  (/N^2 if sign=+1). */
int oracle_dft2_naive(const double* in, double* out, int N, int sign)
{
    if (!in || !out || N < 1 || (sign != 1 && sign != -1)) return ORACLE_ERR_INVALID_ARG;
    for (int ky = 0; ky < N; ++ky)
        for (int kx = 0; kx < N; ++kx) {
            double sr = 0.0, si = 0.0;
            for (int y = 0; y < N; ++y)
                for (int x = 0; x < N; ++x) {
                    const long m = ((long)ky * y + (long)kx * x) % N;
                    const double ang = sign * 2.0 * PI * (double)m / (double)N;
                    const double c = cos(ang), s = sin(ang);
                    const double ar = in[2 * ((size_t)y * N + x)], ai = in[2 * ((size_t)y * N + x) + 1];
                    sr += ar * c - ai * s;
                    si += ar * s + ai * c;
                }
            if (sign > 0) { sr /= (double)N * N; si /= (double)N * N; }
            out[2 * ((size_t)ky * N + kx)] = sr;
            out[2 * ((size_t)ky * N + kx) + 1] = si;
        }
    return ORACLE_OK;
}

static int is_pow2(int N) { return N > 0 && (N & (N - 1)) == 0; }

/* Exported FFT of a stack of `count` images (double I/O), the routine the loop itself uses. */
int oracle_fft2(const double* in, double* out, int N, int count, int sign)
{
    if (!in || !out || N < 2 || count < 0 || (sign != 1 && sign != -1)) return ORACLE_ERR_INVALID_ARG;
    const size_t px = (size_t)N * N;
    #pragma omp parallel for schedule(dynamic, 1)
    for (int n = 0; n < count; ++n) {
        cplx* buf = (cplx*)malloc(sizeof(cplx) * px);
        for (size_t i = 0; i < px; ++i) {
            buf[i].re = (real)in[2 * (n * px + i)];
            buf[i].im = (real)in[2 * (n * px + i) + 1];
        }
        fft2d(buf, N, sign);
        for (size_t i = 0; i < px; ++i) {
            out[2 * (n * px + i)] = (double)buf[i].re;
            out[2 * (n * px + i) + 1] = (double)buf[i].im;
        }
        free(buf);
    }
    return ORACLE_OK;
}

/* ------------------------------------------------------------------------------------------ */
/* The three pointwise operators, as the loop uses them                                        */
/* ------------------------------------------------------------------------------------------ */

/* Eq. (4), reading A1 (weights on n+-1, n+-2, ...; periodic in n) and A4 (Jacobi):
 * out_n = sum_{j=-K}^{K} alpha_|j| in_{(n+j) mod Np}.  in and out must not alias. */
static void mix_stack(const cplx* in, cplx* out, int Np, size_t px, int K, const real* alpha, int N, int flip_seam)
{
    #pragma omp parallel for schedule(static)
    for (int n = 0; n < Np; ++n) {
        cplx* o = out + (size_t)n * px;
        for (size_t i = 0; i < px; ++i) { o[i].re = 0; o[i].im = 0; }
        for (int j = -K; j <= K; ++j) {
            const int m = ((n + j) % Np + Np) % Np;
            const real a = alpha[j < 0 ? -j : j];
            const cplx* s = in + (size_t)m * px;
            /* Reading A5b (seam of a [0, 180) scan): projection n + Np is projection n seen from the
             * other side, P(theta + 180)(z, u) = P(theta)(z, -u) (rotation about one axis), so
             * a neighbour reached by wrapping ONCE round the end of the stack is read mirrored in u about
             * the centre pixel N/2: u -> (N - u) mod N.  (2K + 1 <= Np: never more than one wrap.) */
            const int wrapped = (n + j < 0) || (n + j >= Np);
            if (flip_seam && wrapped) {
                for (int y = 0; y < N; ++y)
                    for (int x = 0; x < N; ++x) {
                        const cplx v = s[(size_t)y * N + (size_t)((N - x) % N)];
                        o[(size_t)y * N + x].re += a * v.re; o[(size_t)y * N + x].im += a * v.im;
                    }
            } else {
                for (size_t i = 0; i < px; ++i) { o[i].re += a * s[i].re; o[i].im += a * s[i].im; }
            }
        }
    }
}

/* Fourier-modulus constraint on one image in native order (only |E|^2 = I is
 * measured; beamstop pixels are unmeasured).  Readings A12 (masked: G' = G) and A13
 * (|G| = 0: phase 0).  Returns num = sum_{M=1} (|G| - A)^2 of the INPUT G (error, reading A9). */
static double modulus_image(cplx* G, const real* A, const unsigned char* M, size_t px)
{
    double num = 0.0;
    for (size_t i = 0; i < px; ++i) {
        if (!M[i]) continue;
        const real mag = (real)sqrt((double)(G[i].re * G[i].re + G[i].im * G[i].im));
        const real d = mag - A[i];
        num += (double)(d * d);
        if (mag > 0) {
            const real s = A[i] / mag;
            G[i].re *= s; G[i].im *= s;
        } else {
            G[i].re = A[i]; G[i].im = 0;
        }
    }
    return num;
}

/* Support / HIO update on one image (Fienup's hybrid input-output, P:98 ref [22]; beta P:104;
 * readings A6, A7: fixed support, no positivity, complex componentwise):
 *   S=1: g <- g' ;  S=0: g <- ghat - beta g'.   ghat is overwritten with the new g. */
/* `pos` (oracle_set_positivity): a pixel inside the support with Re g' < 0 counts as outside. */
static void hio_image(cplx* ghat, const cplx* gp, const unsigned char* S, size_t px, real beta, int pos)
{
    for (size_t i = 0; i < px; ++i) {
        if (S[i] && !(pos && gp[i].re < 0)) { ghat[i] = gp[i]; }
        else { ghat[i].re -= beta * gp[i].re; ghat[i].im -= beta * gp[i].im; }
    }
}

/* The other real-space updates the paper uses or names (reading A22 of DESIGN.md), same support
 * constraint, no positivity:
 *   RAAR (ref [38], beta P:104):  x <- (beta/2)(R_S R_M + I) x + (1 - beta) P_M x,  R = 2P - I,
 *        P_M x = g', P_S = multiplication by S.  Written out:  S=1: g';  S=0: beta ghat + (1 - 2 beta) g'.
 *   ER (error reduction, the plain alternating projection P_S P_M):  S=1: g';  S=0: 0. */
#define ORACLE_UPDATE_HIO 0
#define ORACLE_UPDATE_RAAR 1
#define ORACLE_UPDATE_ER 2
static void raar_image(cplx* ghat, const cplx* gp, const unsigned char* S, size_t px, real beta, int pos)
{
    for (size_t i = 0; i < px; ++i) {
        if (S[i] && !(pos && gp[i].re < 0)) { ghat[i] = gp[i]; }
        else {
            ghat[i].re = beta * ghat[i].re + ((real)1 - (real)2 * beta) * gp[i].re;
            ghat[i].im = beta * ghat[i].im + ((real)1 - (real)2 * beta) * gp[i].im;
        }
    }
}
static void er_image(cplx* ghat, const cplx* gp, const unsigned char* S, size_t px, int pos)
{
    for (size_t i = 0; i < px; ++i) {
        if (S[i] && !(pos && gp[i].re < 0)) { ghat[i] = gp[i]; }
        else { ghat[i].re = 0; ghat[i].im = 0; }
    }
}

/* ------------------------------------------------------------------------------------------ */
/* Plan / state                                                                                */
/* ------------------------------------------------------------------------------------------ */
typedef struct oracle_plan_s {
    int N, Np;
    size_t px;
    real* A;              /* [Np][N][N] sqrt(max(I,0)), native (unshifted) order */
    unsigned char* M;     /* [Np][N][N] 1 = measured, native order */
    unsigned char* S;     /* [Np][N][N] 1 = inside the support */
    double* den;          /* [Np] sum_{M=1} I */
    double* angles;       /* [Np] */
    cplx* g;              /* state */
    cplx* tmp;            /* mixed copy ghat */
    int K; real alpha[64]; int n_ei;
    int positivity;       /* oracle_set_positivity */
    int flip_seam;        /* reading A5b: mirror the neighbours taken across the ends of the stack */
    /* Step C bank (oracle_merge_*): the N_l lowest-error episodes offered so far */
    int NL, bank_count; cplx* bank; double* bank_E;
    int update;   /* ORACLE_UPDATE_*; HIO by default */
    long t;
    double* E; double Eglobal;
    int have_data, have_support, have_estimate, have_error;
} oracle_plan_s;
typedef oracle_plan_s* oracle_plan_t;

int oracle_plan(oracle_plan_t* out, int N, int Np)
{
    if (!out) return ORACLE_ERR_INVALID_ARG;
    if (N < 2 || N > 4096 || (N & 1) || Np < 1) return ORACLE_ERR_UNSUPPORTED_SIZE;   /* even N: the centre pixel is N/2 */
    oracle_plan_t p = (oracle_plan_t)calloc(1, sizeof(*p));
    p->N = N; p->Np = Np; p->px = (size_t)N * N;
    const size_t tot = p->px * (size_t)Np;
    p->A = (real*)calloc(tot, sizeof(real));
    p->M = (unsigned char*)calloc(tot, 1);
    p->S = (unsigned char*)calloc(tot, 1);
    p->den = (double*)calloc((size_t)Np, sizeof(double));
    p->angles = (double*)calloc((size_t)Np, sizeof(double));
    p->g = (cplx*)calloc(tot, sizeof(cplx));
    p->tmp = (cplx*)calloc(tot, sizeof(cplx));
    p->E = (double*)calloc((size_t)Np, sizeof(double));
    /* reading A2: the paper's example weights */
    p->K = 1; p->alpha[0] = (real)0.6; p->alpha[1] = (real)0.2; p->n_ei = 1;
    *out = p;
    return ORACLE_OK;
}

int oracle_destroy(oracle_plan_t p)
{
    if (!p) return ORACLE_ERR_INVALID_ARG;
    free(p->A); free(p->M); free(p->S); free(p->den); free(p->angles);
    free(p->g); free(p->tmp); free(p->E); free(p->bank); free(p->bank_E); free(p);
    return ORACLE_OK;
}

/* I: [Np][N][N] detector-centred (DC at index N/2); mask likewise, NULL = all measured.
 * A = sqrt(max(I,0)) (reading A14), moved to native order (ifftshift, reading A11);
 * den_n = sum_{M=1} I_n (clamped I). */
int oracle_set_data(oracle_plan_t p, const double* I, const unsigned char* mask, const double* angles)
{
    if (!p || !I) return ORACLE_ERR_INVALID_ARG;
    const int N = p->N, h = N / 2;
    for (int n = 0; n < p->Np; ++n) {
        double den = 0.0;
        for (int y = 0; y < N; ++y)
            for (int x = 0; x < N; ++x) {
                const size_t src = (size_t)n * p->px + (size_t)y * N + x;              /* centred */
                const size_t dst = (size_t)n * p->px + (size_t)((y + h) % N) * N + ((x + h) % N);
                const double v = I[src] > 0.0 ? I[src] : 0.0;
                const unsigned char m = mask ? (mask[src] ? 1 : 0) : 1;
                p->A[dst] = (real)sqrt(v);
                p->M[dst] = m;
                if (m) den += v;
            }
        p->den[n] = den;
        p->angles[n] = angles ? angles[n] : 0.0;
    }
    p->have_data = 1;
    return ORACLE_OK;
}

int oracle_set_support(oracle_plan_t p, const unsigned char* S)
{
    if (!p || !S) return ORACLE_ERR_INVALID_ARG;
    const size_t tot = p->px * (size_t)p->Np;
    for (size_t i = 0; i < tot; ++i) p->S[i] = S[i] ? 1 : 0;
    p->have_support = 1;
    return ORACLE_OK;
}

int oracle_set_carousel(oracle_plan_t p, int K, const double* alpha, int n_ei)
{
    if (!p || !alpha || K < 0 || K > 63 || 2 * K + 1 > p->Np || n_ei < 1) return ORACLE_ERR_INVALID_ARG;
    p->K = K;
    for (int j = 0; j <= K; ++j) p->alpha[j] = (real)alpha[j];    /* reading A2: not renormalised */
    p->n_ei = n_ei;
    return ORACLE_OK;
}

/* real-space update rule of step 6: ORACLE_UPDATE_HIO (default), _RAAR, _ER */
int oracle_set_update(oracle_plan_t p, int rule)
{
    if (!p || rule < 0 || rule > 2) return ORACLE_ERR_INVALID_ARG;
    p->update = rule;
    return ORACLE_OK;
}

/* g0: interleaved complex double [Np][N][N]; resets t = 0. */
int oracle_set_estimate(oracle_plan_t p, const double* g0)
{
    if (!p || !g0) return ORACLE_ERR_INVALID_ARG;
    const size_t tot = p->px * (size_t)p->Np;
    for (size_t i = 0; i < tot; ++i) { p->g[i].re = (real)g0[2 * i]; p->g[i].im = (real)g0[2 * i + 1]; }
    p->t = 0; p->have_estimate = 1; p->have_error = 0;
    return ORACLE_OK;
}

int oracle_set_iteration(oracle_plan_t p, long t) { if (!p || t < 0) return ORACLE_ERR_INVALID_ARG; p->t = t; return ORACLE_OK; }
long oracle_get_iteration(oracle_plan_t p) { return p ? p->t : -1; }

int oracle_iterate(oracle_plan_t p, int k, double beta_d)
{
    if (!p || k < 0 || !isfinite(beta_d)) return ORACLE_ERR_INVALID_ARG;
    if (!p->have_data || !p->have_support || !p->have_estimate) return ORACLE_ERR_NOT_READY;
    const real beta = (real)beta_d;
    const size_t px = p->px;
    const int N = p->N, Np = p->Np;
    for (int it = 0; it < k; ++it) {
        /* 1. mix (Eq. (4)) at the start of an episode; otherwise ghat = g */
        const int do_mix = (p->t % p->n_ei) == 0;
        if (do_mix) {
            mix_stack(p->g, p->tmp, Np, px, p->K, p->alpha, N, p->flip_seam);
            cplx* sw = p->g; p->g = p->tmp; p->tmp = sw;            /* p->g now holds ghat */
        }
        double numtot = 0.0, dentot = 0.0;
        #pragma omp parallel for schedule(dynamic, 1) reduction(+:numtot, dentot)
        for (int n = 0; n < Np; ++n) {
            cplx* ghat = p->g + (size_t)n * px;
            cplx* G = (cplx*)malloc(sizeof(cplx) * px);
            memcpy(G, ghat, sizeof(cplx) * px);
            fft2d(G, N, -1);                                                     /* 2 */
            const double num = modulus_image(G, p->A + (size_t)n * px, p->M + (size_t)n * px, px); /* 3, 4 */
            fft2d(G, N, +1);                                                     /* 5 */
            if (p->update == ORACLE_UPDATE_RAAR) raar_image(ghat, G, p->S + (size_t)n * px, px, beta, p->positivity);
            else if (p->update == ORACLE_UPDATE_ER) er_image(ghat, G, p->S + (size_t)n * px, px, p->positivity);
            else hio_image(ghat, G, p->S + (size_t)n * px, px, beta, p->positivity);            /* 6 */
            free(G);
            p->E[n] = p->den[n] > 0.0 ? sqrt(num / p->den[n]) : 0.0;
            numtot += num; dentot += p->den[n];
        }
        p->Eglobal = dentot > 0.0 ? sqrt(numtot / dentot) : 0.0;
        p->have_error = 1;
        p->t += 1;                                                               /* 7 */
    }
    return ORACLE_OK;
}

int oracle_get_error(oracle_plan_t p, double* E, double* Eglobal)
{
    if (!p) return ORACLE_ERR_INVALID_ARG;
    if (!p->have_error) return ORACLE_ERR_NOT_READY;
    if (E) memcpy(E, p->E, sizeof(double) * (size_t)p->Np);
    if (Eglobal) *Eglobal = p->Eglobal;
    return ORACLE_OK;
}

/* which = 0: the iterate g; which = 1: S.g (the estimate restricted to the support). */
int oracle_get_projections(oracle_plan_t p, int which, double* out)
{
    if (!p || !out || (which != 0 && which != 1)) return ORACLE_ERR_INVALID_ARG;
    if (!p->have_estimate) return ORACLE_ERR_NOT_READY;
    const size_t tot = p->px * (size_t)p->Np;
    for (size_t i = 0; i < tot; ++i) {
        const int keep = which == 0 || p->S[i];
        out[2 * i] = keep ? (double)p->g[i].re : 0.0;
        out[2 * i + 1] = keep ? (double)p->g[i].im : 0.0;
    }
    return ORACLE_OK;
}

/* Stand-alone entry points for the pins: the very functions the loop calls. */
int oracle_mix(const double* in, double* out, int N, int Np, int K, const double* alpha)
{
    if (!in || !out || !alpha || K < 0 || K > 63 || 2 * K + 1 > Np) return ORACLE_ERR_INVALID_ARG;
    const size_t px = (size_t)N * N, tot = px * Np;
    cplx* a = (cplx*)malloc(sizeof(cplx) * tot); cplx* b = (cplx*)malloc(sizeof(cplx) * tot);
    real al[64];
    for (int j = 0; j <= K; ++j) al[j] = (real)alpha[j];
    for (size_t i = 0; i < tot; ++i) { a[i].re = (real)in[2 * i]; a[i].im = (real)in[2 * i + 1]; }
    mix_stack(a, b, Np, px, K, al, N, 0);
    for (size_t i = 0; i < tot; ++i) { out[2 * i] = b[i].re; out[2 * i + 1] = b[i].im; }
    free(a); free(b);
    return ORACLE_OK;
}

/* G (native order, interleaved double, in place), A and M native order; returns num via *num. */
int oracle_modulus(double* G, const double* A, const unsigned char* M, int N, double* num)
{
    if (!G || !A || !M) return ORACLE_ERR_INVALID_ARG;
    const size_t px = (size_t)N * N;
    cplx* g = (cplx*)malloc(sizeof(cplx) * px); real* a = (real*)malloc(sizeof(real) * px);
    for (size_t i = 0; i < px; ++i) { g[i].re = (real)G[2 * i]; g[i].im = (real)G[2 * i + 1]; a[i] = (real)A[i]; }
    const double s = modulus_image(g, a, M, px);
    for (size_t i = 0; i < px; ++i) { G[2 * i] = g[i].re; G[2 * i + 1] = g[i].im; }
    if (num) *num = s;
    free(g); free(a);
    return ORACLE_OK;
}

/* ghat (in place -> new g), gp = g', S. */
int oracle_hio(double* ghat, const double* gp, const unsigned char* S, int N, double beta)
{
    if (!ghat || !gp || !S) return ORACLE_ERR_INVALID_ARG;
    const size_t px = (size_t)N * N;
    cplx* a = (cplx*)malloc(sizeof(cplx) * px); cplx* b = (cplx*)malloc(sizeof(cplx) * px);
    for (size_t i = 0; i < px; ++i) {
        a[i].re = (real)ghat[2 * i]; a[i].im = (real)ghat[2 * i + 1];
        b[i].re = (real)gp[2 * i]; b[i].im = (real)gp[2 * i + 1];
    }
    hio_image(a, b, S, px, (real)beta, 0);
    for (size_t i = 0; i < px; ++i) { ghat[2 * i] = a[i].re; ghat[2 * i + 1] = a[i].im; }
    free(a); free(b);
    return ORACLE_OK;
}

/* ------------------------------------------------------------------------------------------ */
/* Fourier-slice assembly (first sentence of Step D; Fourier slice theorem P:35-44)      */
/* ------------------------------------------------------------------------------------------ */
/*
 * Geometry (reading A18): rotation about z, arrays O[z][y][x], P_n[z][u],
 *   x = u cos(th) - s sin(th), y = u sin(th) + s cos(th)  =>
 *   F2[P_n](kz, ku) = F3[O](kz, ky = ku sin(th_n), kx = ku cos(th_n)).
 * Steps (reading A17 -- the paper only says "interpolate"):
 *  (i)   E_n = F2[S_n g_n]; multiply by (-1)^(kz+ku): moves the real-space origin to the centre
 *        pixel (N/2, N/2), so that the spectrum of a centred object is smooth.
 *  (ii)  every slice is two rays from the origin: direction th_n (ku >= 0) and th_n + pi
 *        (ku <= 0).  Sort the 2 Np directions on [0, 2 pi); directions closer than 1e-9 rad are
 *        one ray whose samples are the mean of the contributors.
 *  (iii) voxel (kz,ky,kx), signed integer frequencies in [-N/2, N/2): rho = sqrt(kx^2+ky^2),
 *        phi = atan2(ky,kx) mod 2 pi.  rho > N/2-1: value 0, weight 0.  rho = 0: mean of all
 *        slices' DC sample at that kz.  Otherwise bilinear in (phi, rho) between the two rays
 *        bracketing phi (periodic) and the radial samples floor(rho), floor(rho)+1; weight 1.
 *  (iv)  multiply by (-1)^(kx+ky+kz), store at native indices (k mod N): comparable to fftn(O)
 *        of an object centred at (N/2,N/2,N/2).
 * vol: interleaved complex double [N][N][N] (kz,ky,kx); weight: [N][N][N] double or NULL.
 */
typedef struct { double phi; int n; int neg; } ray_t;
static int ray_cmp(const void* a, const void* b)
{
    const ray_t* x = (const ray_t*)a; const ray_t* y = (const ray_t*)b;
    if (x->phi < y->phi) return -1;
    if (x->phi > y->phi) return 1;
    return (x->n > y->n) - (x->n < y->n);
}

int oracle_assemble_3d(oracle_plan_t p, double* vol, double* weight)
{
    if (!p || !vol) return ORACLE_ERR_INVALID_ARG;
    if (!p->have_estimate || !p->have_support || !p->have_data) return ORACLE_ERR_NOT_READY;
    const int N = p->N, Np = p->Np, h = N / 2;
    const size_t px = p->px;

    /* (i) spectra of the supported estimates, origin moved to the centre pixel */
    cplx* E = (cplx*)malloc(sizeof(cplx) * px * (size_t)Np);
    #pragma omp parallel for schedule(dynamic, 1)
    for (int n = 0; n < Np; ++n) {
        cplx* e = E + (size_t)n * px;
        for (size_t i = 0; i < px; ++i) {
            const size_t gi = (size_t)n * px + i;
            if (p->S[gi]) e[i] = p->g[gi]; else { e[i].re = 0; e[i].im = 0; }
        }
        fft2d(e, N, -1);
        for (int kz = 0; kz < N; ++kz)
            for (int ku = 0; ku < N; ++ku)
                if ((kz + ku) & 1) { e[(size_t)kz * N + ku].re = -e[(size_t)kz * N + ku].re;
                                     e[(size_t)kz * N + ku].im = -e[(size_t)kz * N + ku].im; }
    }

    /* (ii) rays: sorted unique directions, each with its contributors [start, start+count) */
    const int R2 = 2 * Np;
    ray_t* rays = (ray_t*)malloc(sizeof(ray_t) * (size_t)R2);
    for (int n = 0; n < Np; ++n)
        for (int neg = 0; neg < 2; ++neg) {
            double ph = fmod(p->angles[n] + (neg ? PI : 0.0), 2.0 * PI);
            if (ph < 0.0) ph += 2.0 * PI;
            if (ph >= 2.0 * PI - 1e-9) ph = 0.0;          /* 2 pi is the direction 0 */
            rays[2 * n + neg].phi = ph; rays[2 * n + neg].n = n; rays[2 * n + neg].neg = neg;
        }
    qsort(rays, (size_t)R2, sizeof(ray_t), ray_cmp);
    int* ustart = (int*)malloc(sizeof(int) * (size_t)(R2 + 1));
    double* uphi = (double*)malloc(sizeof(double) * (size_t)R2);
    int U = 0;
    for (int i = 0; i < R2; ++i) {
        if (U == 0 || rays[i].phi - uphi[U - 1] > 1e-9) { ustart[U] = i; uphi[U] = rays[i].phi; ++U; }
    }
    ustart[U] = R2;

    /* (iii)+(iv) gather */
    #pragma omp parallel for schedule(static)
    for (int iz = 0; iz < N; ++iz) {
        const int kz = iz < h ? iz : iz - N;
        for (int iy = 0; iy < N; ++iy) {
            const int ky = iy < h ? iy : iy - N;
            for (int ix = 0; ix < N; ++ix) {
                const int kx = ix < h ? ix : ix - N;
                const size_t o = ((size_t)iz * N + iy) * N + ix;
                const double rho = sqrt((double)kx * kx + (double)ky * ky);
                double vr = 0.0, vi = 0.0, w = 0.0;
                if (rho == 0.0) {
                    for (int n = 0; n < Np; ++n) { vr += E[(size_t)n * px + (size_t)iz * N].re; vi += E[(size_t)n * px + (size_t)iz * N].im; }
                    vr /= Np; vi /= Np; w = 1.0;
                } else if (rho <= (double)(h - 1)) {
                    double phi = atan2((double)ky, (double)kx);
                    if (phi < 0.0) phi += 2.0 * PI;
                    /* bracket: largest a with uphi[a] <= phi (periodic) */
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
                    const int r0 = (int)floor(rho);
                    const double wr = rho - (double)r0;
                    const int ur[2] = { a, b };
                    const double wphi[2] = { 1.0 - wp, wp };
                    for (int q = 0; q < 2; ++q) {
                        if (wphi[q] == 0.0) continue;
                        const int u = ur[q];
                        const int cnt = ustart[u + 1] - ustart[u];
                        for (int rr = 0; rr < 2; ++rr) {
                            const double wrr = rr ? wr : 1.0 - wr;
                            if (wrr == 0.0) continue;
                            const int r = r0 + rr;
                            double sr = 0.0, si = 0.0;
                            for (int c = ustart[u]; c < ustart[u + 1]; ++c) {
                                const int ku = rays[c].neg ? -r : r;
                                const int iu = ((ku % N) + N) % N;
                                const cplx e = E[(size_t)rays[c].n * px + (size_t)iz * N + iu];
                                sr += e.re; si += e.im;
                            }
                            vr += wphi[q] * wrr * sr / cnt;
                            vi += wphi[q] * wrr * si / cnt;
                        }
                    }
                    w = 1.0;
                }
                if ((kx + ky + kz) & 1) { vr = -vr; vi = -vi; }
                vol[2 * o] = vr; vol[2 * o + 1] = vi;
                if (weight) weight[o] = w;
            }
        }
    }
    free(E); free(rays); free(ustart); free(uphi);
    return ORACLE_OK;
}

/* ------------------------------------------------------------------------------------------ */
/* seam of a 180 degree scan, shrink-wrap                                    */
/* ------------------------------------------------------------------------------------------ */

/* flip = 1: neighbours taken across the ends of the stack are mirrored in u (see mix_stack). */
int oracle_set_positivity(oracle_plan_t p, int on)
{
    if (!p || (on != 0 && on != 1)) return ORACLE_ERR_INVALID_ARG;
    p->positivity = on;
    return ORACLE_OK;
}

int oracle_set_seam(oracle_plan_t p, int flip)
{
    if (!p || (flip != 0 && flip != 1)) return ORACLE_ERR_INVALID_ARG;
    p->flip_seam = flip;
    return ORACLE_OK;
}

/* Eq. (4) with the seam flag, stand-alone (for the pins). */
int oracle_mix_seam(const double* in, double* out, int N, int Np, int K, const double* alpha, int flip)
{
    if (!in || !out || !alpha || K < 0 || K > 63 || 2 * K + 1 > Np) return ORACLE_ERR_INVALID_ARG;
    const size_t px = (size_t)N * N, tot = px * Np;
    cplx* a = (cplx*)malloc(sizeof(cplx) * tot); cplx* b = (cplx*)malloc(sizeof(cplx) * tot);
    real al[64];
    for (int j = 0; j <= K; ++j) al[j] = (real)alpha[j];
    for (size_t i = 0; i < tot; ++i) { a[i].re = (real)in[2 * i]; a[i].im = (real)in[2 * i + 1]; }
    mix_stack(a, b, Np, px, K, al, N, flip);
    for (size_t i = 0; i < tot; ++i) { out[2 * i] = b[i].re; out[2 * i + 1] = b[i].im; }
    free(a); free(b);
    return ORACLE_OK;
}

/* Periodic Gaussian blur of a real image, width sigma pixels, done in Fourier space:
 * B = F^-1[ F[a] . exp(-2 pi^2 sigma^2 (ky^2 + kx^2) / N^2) ], ky, kx signed integer frequencies
 * (the transform of a Gaussian of standard deviation sigma sampled on the N-periodic grid). */
static void blur_image(const real* a, real* b, int N, double sigma)
{
    const size_t px = (size_t)N * N;
    cplx* w = (cplx*)malloc(sizeof(cplx) * px);
    for (size_t i = 0; i < px; ++i) { w[i].re = a[i]; w[i].im = 0; }
    fft2d(w, N, -1);
    for (int iy = 0; iy < N; ++iy) {
        const int ky = iy < N / 2 ? iy : iy - N;
        for (int ix = 0; ix < N; ++ix) {
            const int kx = ix < N / 2 ? ix : ix - N;
            const real f = (real)exp(-2.0 * PI * PI * sigma * sigma * ((double)ky * ky + (double)kx * kx) / ((double)N * N));
            w[(size_t)iy * N + ix].re *= f; w[(size_t)iy * N + ix].im *= f;
        }
    }
    fft2d(w, N, +1);
    for (size_t i = 0; i < px; ++i) b[i] = w[i].re;
    free(w);
}

int oracle_blur(const double* in, double* out, int N, double sigma)
{
    if (!in || !out || N < 2 || (N & 1) || !(sigma >= 0.0)) return ORACLE_ERR_INVALID_ARG;   /* any even N (fft2d: reading A20) */
    const size_t px = (size_t)N * N;
    real* a = (real*)malloc(sizeof(real) * px); real* b = (real*)malloc(sizeof(real) * px);
    for (size_t i = 0; i < px; ++i) a[i] = (real)in[i];
    blur_image(a, b, N, sigma);
    for (size_t i = 0; i < px; ++i) out[i] = (double)b[i];
    free(a); free(b);
    return ORACLE_OK;
}

/* Shrink-wrap support update ("2D CSWA" ref [35]; "an extra 2D CSWA iteration to obtain a
 * tighter space constraint"), reading A23: for every projection
 *     b_n = G_sigma * |S_n g_n|   (the current estimate restricted to the current support, blurred),
 *     S_n <- [ b_n >= threshold . max_pixels b_n ]        (all zero if the maximum is not positive).
 * blurred (optional, [Np][N][N] double) receives b_n so that a comparison can set aside the pixels
 * whose b_n lies within rounding of the threshold. */
int oracle_shrinkwrap(oracle_plan_t p, double sigma, double threshold, double* blurred)
{
    if (!p || !(sigma >= 0.0) || !(threshold >= 0.0)) return ORACLE_ERR_INVALID_ARG;
    if (!p->have_support || !p->have_estimate) return ORACLE_ERR_NOT_READY;
    const int N = p->N;
    const size_t px = p->px;
    #pragma omp parallel for schedule(dynamic, 1)
    for (int n = 0; n < p->Np; ++n) {
        real* a = (real*)malloc(sizeof(real) * px); real* b = (real*)malloc(sizeof(real) * px);
        for (size_t i = 0; i < px; ++i) {
            const size_t gi = (size_t)n * px + i;
            a[i] = p->S[gi] ? (real)sqrt((double)(p->g[gi].re * p->g[gi].re + p->g[gi].im * p->g[gi].im)) : (real)0;
        }
        blur_image(a, b, N, sigma);
        real m = b[0];
        for (size_t i = 1; i < px; ++i) if (b[i] > m) m = b[i];
        for (size_t i = 0; i < px; ++i) {
            p->S[(size_t)n * px + i] = (m > 0 && b[i] >= (real)threshold * m) ? 1 : 0;
            if (blurred) blurred[(size_t)n * px + i] = (double)b[i];
        }
        free(a); free(b);
    }
    return ORACLE_OK;
}

int oracle_get_support(oracle_plan_t p, unsigned char* S)
{
    if (!p || !S) return ORACLE_ERR_INVALID_ARG;
    if (!p->have_support) return ORACLE_ERR_NOT_READY;
    memcpy(S, p->S, p->px * (size_t)p->Np);
    return ORACLE_OK;
}

/* ------------------------------------------------------------------------------------------ */
/* Step A (pre-reconstruction) and Step C (repeating and merging)           */
/* ------------------------------------------------------------------------------------------ */

/* Step A: "Pre-reconstruct a single PO ... via the conventional 2D CXDI algorithm": k iterations of
 * steps 2-6 of the loop on projection n alone (no mix: a single PO has no neighbours in Step A); the
 * other projections and the iteration counter t are untouched. */
int oracle_prereconstruct(oracle_plan_t p, int n, int k, double beta_d)
{
    if (!p || n < 0 || n >= p->Np || k < 0 || !isfinite(beta_d)) return ORACLE_ERR_INVALID_ARG;
    if (!p->have_data || !p->have_support || !p->have_estimate) return ORACLE_ERR_NOT_READY;
    const real beta = (real)beta_d;
    const size_t px = p->px;
    cplx* ghat = p->g + (size_t)n * px;
    cplx* G = (cplx*)malloc(sizeof(cplx) * px);
    for (int it = 0; it < k; ++it) {
        memcpy(G, ghat, sizeof(cplx) * px);
        fft2d(G, p->N, -1);
        (void)modulus_image(G, p->A + (size_t)n * px, p->M + (size_t)n * px, px);
        fft2d(G, p->N, +1);
        if (p->update == ORACLE_UPDATE_RAAR) raar_image(ghat, G, p->S + (size_t)n * px, px, beta, p->positivity);
        else if (p->update == ORACLE_UPDATE_ER) er_image(ghat, G, p->S + (size_t)n * px, px, p->positivity);
        else hio_image(ghat, G, p->S + (size_t)n * px, px, beta, p->positivity);
    }
    free(G);
    return ORACLE_OK;
}

/* Centre of mass of one PO about the centre pixel (N/2, N/2), mass = |O| ("we move the mass center
 * of each PO by Delta r_n = - int O'_n(r) r dv"; the printed integral lacks its normalisation; reading A24:
 * com = sum |O| r / sum |O|, r = (y - N/2, x - N/2)).  com = 0 for an empty image. */
static void center_of_mass(const cplx* o, int N, double* cy, double* cx)
{
    double m = 0.0, sy = 0.0, sx = 0.0;
    for (int y = 0; y < N; ++y)
        for (int x = 0; x < N; ++x) {
            const cplx v = o[(size_t)y * N + x];
            const double w = sqrt((double)v.re * v.re + (double)v.im * v.im);
            m += w; sy += w * (double)(y - N / 2); sx += w * (double)(x - N / 2);
        }
    *cy = m > 0.0 ? sy / m : 0.0;
    *cx = m > 0.0 ? sx / m : 0.0;
}
int oracle_center_of_mass(const double* img, int N, double* cy, double* cx)
{
    if (!img || !cy || !cx || N < 1) return ORACLE_ERR_INVALID_ARG;
    const size_t px = (size_t)N * N;
    cplx* a = (cplx*)malloc(sizeof(cplx) * px);
    for (size_t i = 0; i < px; ++i) { a[i].re = (real)img[2 * i]; a[i].im = (real)img[2 * i + 1]; }
    center_of_mass(a, N, cy, cx);
    free(a);
    return ORACLE_OK;
}
/* whole-pixel shift that brings the centre of mass to the centre pixel: -round(com), halves away from 0 */
static int shift_of(double com) { return -(int)(com >= 0.0 ? floor(com + 0.5) : -floor(-com + 0.5)); }

/* Step C.  The bank keeps the N_l episodes of lowest reconstruction error among those offered
 * ("We select a certain number N_l < N_r of the best reconstructed episodes, which have the lowest
 * reconstruction error").  An episode is the stack of supported estimates S_n g_n (what Step D consumes). */
int oracle_merge_begin(oracle_plan_t p, int NL)
{
    if (!p || NL < 1) return ORACLE_ERR_INVALID_ARG;
    free(p->bank); free(p->bank_E);
    p->NL = NL; p->bank_count = 0;
    p->bank = (cplx*)calloc((size_t)NL * p->Np * p->px, sizeof(cplx));
    p->bank_E = (double*)calloc((size_t)NL, sizeof(double));
    return ORACLE_OK;
}

/* Offer an episode with reconstruction error E: `episode` = interleaved complex double [Np][N][N], or
 * NULL = the plan's own S.g with the global error of its last iteration (E is then ignored).  It takes a
 * free slot, else replaces the worst kept episode if E is lower than that one's (the first worst on ties). */
int oracle_merge_offer(oracle_plan_t p, const double* episode, double E)
{
    if (!p || !p->bank) return ORACLE_ERR_INVALID_ARG;
    if (!episode) {
        if (!p->have_estimate || !p->have_support || !p->have_error) return ORACLE_ERR_NOT_READY;
        E = p->Eglobal;
    }
    int slot = -1;
    if (p->bank_count < p->NL) slot = p->bank_count++;
    else {
        int w = 0;
        for (int e = 1; e < p->NL; ++e) if (p->bank_E[e] > p->bank_E[w]) w = e;
        if (E < p->bank_E[w]) slot = w;
    }
    if (slot < 0) return ORACLE_OK;
    const size_t tot = p->px * (size_t)p->Np;
    cplx* dst = p->bank + (size_t)slot * tot;
    for (size_t i = 0; i < tot; ++i) {
        if (episode) { dst[i].re = (real)episode[2 * i]; dst[i].im = (real)episode[2 * i + 1]; }
        else if (p->S[i]) dst[i] = p->g[i];
        else { dst[i].re = 0; dst[i].im = 0; }
    }
    p->bank_E[slot] = E;
    return ORACLE_OK;
}

/* errors of the kept episodes, in slot order; returns how many are kept through *count */
int oracle_merge_errors(oracle_plan_t p, double* E, int* count)
{
    if (!p || !p->bank || !count) return ORACLE_ERR_INVALID_ARG;
    *count = p->bank_count;
    if (E) for (int e = 0; e < p->bank_count; ++e) E[e] = p->bank_E[e];
    return ORACLE_OK;
}

/* The merge itself, in the paper's order:
 *  1. every PO of every kept episode is moved by a whole number of pixels (circularly) so that its centre
 *     of mass sits on the centre pixel:  O'(y, x) = O(y - sy, x - sx),  s = -round(com)
 *  2. b = the kept episode of lowest error (first on ties).  For every other episode e, on ONE PO n_ref
 *     ("one of the POs in this best episode and the same number PO in other episodes"; n_ref = -1:
 *     summed over all POs): c = <O_b, O_e> = sum conj(O_b) O_e and c_T = <O_b, T O_e> with the twin
 *     T O(r) = conj(O(-r)) about the centre pixel -- the image with the same Fourier modulus (P:70 prints
 *     O(-r); that is the twin of a real object, conj(O(-r)) that of a complex one: reading A25).
 *     An iterate without reality constraint carries a free global phase, so "Euclidean distance" is read
 *     as the distance minimised over that phase, ||a||^2 + ||b||^2 - 2 |<a, b>| (reading A25): the twin is
 *     taken iff |c_T| > |c|, and the episode is multiplied by conj(c)/|c| (1 if c = 0) of the chosen one.
 *  3. out_n = mean over the kept episodes of the corrected POs
 * out: interleaved complex double [Np][N][N].  shifts (optional): int [kept][Np][2] (sy, sx);
 * twins (optional): int [kept] (1 = twin taken). */
int oracle_merge_finish(oracle_plan_t p, int n_ref, double* out, int* shifts, int* twins)
{
    if (!p || !p->bank || !out || n_ref < -1 || n_ref >= p->Np) return ORACLE_ERR_INVALID_ARG;
    if (p->bank_count < 1) return ORACLE_ERR_NOT_READY;
    const int N = p->N, Np = p->Np, L = p->bank_count;
    const size_t px = p->px, tot = px * (size_t)Np;
    /* 1. centre-of-mass shifts */
    cplx* tmp = (cplx*)malloc(sizeof(cplx) * px);
    for (int e = 0; e < L; ++e)
        for (int n = 0; n < Np; ++n) {
            cplx* o = p->bank + (size_t)e * tot + (size_t)n * px;
            double cy, cx;
            center_of_mass(o, N, &cy, &cx);
            const int sy = shift_of(cy), sx = shift_of(cx);
            if (shifts) { shifts[((size_t)e * Np + n) * 2] = sy; shifts[((size_t)e * Np + n) * 2 + 1] = sx; }
            memcpy(tmp, o, sizeof(cplx) * px);
            for (int y = 0; y < N; ++y)
                for (int x = 0; x < N; ++x)
                    o[(size_t)y * N + x] = tmp[(size_t)(((y - sy) % N + N) % N) * N + (size_t)(((x - sx) % N + N) % N)];
        }
    /* 2. twin and global phase against the best episode */
    int b = 0;
    for (int e = 1; e < L; ++e) if (p->bank_E[e] < p->bank_E[b]) b = e;
    for (int e = 0; e < L; ++e) {
        if (twins) twins[e] = 0;
        if (e == b) continue;
        double cr = 0.0, ci = 0.0, tr = 0.0, ti = 0.0;
        for (int n = (n_ref < 0 ? 0 : n_ref); n <= (n_ref < 0 ? Np - 1 : n_ref); ++n) {
            const cplx* ob = p->bank + (size_t)b * tot + (size_t)n * px;
            const cplx* oe = p->bank + (size_t)e * tot + (size_t)n * px;
            for (int y = 0; y < N; ++y)
                for (int x = 0; x < N; ++x) {
                    const cplx a = ob[(size_t)y * N + x];
                    const cplx v = oe[(size_t)y * N + x];
                    const cplx w = oe[(size_t)((N - y) % N) * N + (size_t)((N - x) % N)];   /* T: conj of this */
                    cr += (double)a.re * v.re + (double)a.im * v.im;      /* conj(a) v */
                    ci += (double)a.re * v.im - (double)a.im * v.re;
                    tr += (double)a.re * w.re - (double)a.im * w.im;      /* conj(a) conj(w) */
                    ti += -(double)a.re * w.im - (double)a.im * w.re;
                }
        }
        const double mc = sqrt(cr * cr + ci * ci), mt = sqrt(tr * tr + ti * ti);
        const int twin = mt > mc;
        const double m = twin ? mt : mc;
        const double ur = m > 0.0 ? (twin ? tr : cr) / m : 1.0, ui = m > 0.0 ? -(twin ? ti : ci) / m : 0.0;   /* conj(c)/|c| */
        if (twins) twins[e] = twin;
        for (int n = 0; n < Np; ++n) {
            cplx* o = p->bank + (size_t)e * tot + (size_t)n * px;
            memcpy(tmp, o, sizeof(cplx) * px);
            for (int y = 0; y < N; ++y)
                for (int x = 0; x < N; ++x) {
                    cplx v = tmp[(size_t)y * N + x];
                    if (twin) { v = tmp[(size_t)((N - y) % N) * N + (size_t)((N - x) % N)]; v.im = -v.im; }
                    o[(size_t)y * N + x].re = (real)(ur * v.re - ui * v.im);
                    o[(size_t)y * N + x].im = (real)(ur * v.im + ui * v.re);
                }
        }
    }
    free(tmp);
    /* 3. average */
    for (size_t i = 0; i < tot; ++i) {
        double sr = 0.0, si = 0.0;
        for (int e = 0; e < L; ++e) { sr += (double)p->bank[(size_t)e * tot + i].re; si += (double)p->bank[(size_t)e * tot + i].im; }
        out[2 * i] = sr / L; out[2 * i + 1] = si / L;
    }
    return ORACLE_OK;
}

/* Consistency of the projections of ONE episode before Step D (reading A28 -- an addition of this build, not the
 * paper's: the paper relies on the carousel coupling alone).  Two freedoms of an unconstrained complex
 * iterate survive the loop projection by projection, and both are fixed by facts of the forward model:
 *  (1) global phase: every projection of one object has the same total, sum_px P_n = sum_voxels O (line
 *      integrals), so each PO is multiplied by the unit factor that makes its total real and positive
 *      (conj(s_n)/|s_n|, s_n = sum_px O_n; left alone if s_n = 0);
 *  (2) twin: neighbouring projections are similar, so, walking away from projection n_ref in both directions,
 *      PO n is replaced by its twin conj(O_n(-r)) iff that is closer to the already decided neighbour:
 *      Re<a, T O_n> > Re<a, O_n>.  (The twin keeps a real positive total, so (1) stays satisfied.)
 * ep: interleaved complex double [Np][N][N], in place.  flips (optional): int [Np]. */
int oracle_align_episode(double* ep, int N, int Np, int n_ref, int* flips)
{
    if (!ep || N < 1 || Np < 1 || n_ref < 0 || n_ref >= Np) return ORACLE_ERR_INVALID_ARG;
    const size_t px = (size_t)N * N;
    for (int n = 0; n < Np; ++n) {
        double* o = ep + 2 * (size_t)n * px;
        double sr = 0.0, si = 0.0;
        for (size_t i = 0; i < px; ++i) { sr += o[2 * i]; si += o[2 * i + 1]; }
        const double m = sqrt(sr * sr + si * si);
        if (m > 0.0) {
            const double ur = sr / m, ui = -si / m;
            for (size_t i = 0; i < px; ++i) {
                const double a = o[2 * i], b = o[2 * i + 1];
                o[2 * i] = ur * a - ui * b; o[2 * i + 1] = ur * b + ui * a;
            }
        }
    }
    double* tmp = (double*)malloc(sizeof(double) * 2 * px);
    if (flips) for (int n = 0; n < Np; ++n) flips[n] = 0;
    for (int dir = 1; dir >= -1; dir -= 2)
        for (int n = n_ref + dir; n >= 0 && n < Np; n += dir) {
            const double* a = ep + 2 * (size_t)(n - dir) * px;      /* the decided neighbour */
            double* o = ep + 2 * (size_t)n * px;
            double pp = 0.0, qq = 0.0;
            for (int y = 0; y < N; ++y)
                for (int x = 0; x < N; ++x) {
                    const size_t i = (size_t)y * N + x, j = (size_t)((N - y) % N) * N + (size_t)((N - x) % N);
                    pp += a[2 * i] * o[2 * i] + a[2 * i + 1] * o[2 * i + 1];          /* Re conj(a) o      */
                    qq += a[2 * i] * o[2 * j] - a[2 * i + 1] * o[2 * j + 1];          /* Re conj(a) conj(o(-r)) */
                }
            if (qq > pp) {
                memcpy(tmp, o, sizeof(double) * 2 * px);
                for (int y = 0; y < N; ++y)
                    for (int x = 0; x < N; ++x) {
                        const size_t i = (size_t)y * N + x, j = (size_t)((N - y) % N) * N + (size_t)((N - x) % N);
                        o[2 * i] = tmp[2 * j]; o[2 * i + 1] = -tmp[2 * j + 1];
                    }
                if (flips) flips[n] = 1;
            }
        }
    free(tmp);
    return ORACLE_OK;
}

/* ------------------------------------------------------------------------------------------ */
/* the 3D transform of Step D ("3D FTs as a set of 2D FTs")     */
/* ------------------------------------------------------------------------------------------ */
/* vol [N][N][N] interleaved complex double (z, y, x), in -> out (may alias): all x lines, all y lines,
 * all z lines with the textbook fft1d.  sign = -1 forward, unnormalised; +1 inverse, / N^3. */
int oracle_fft3(const double* in, double* out, int N, int sign)
{
    if (!in || !out || N < 2 || (N & 1) || (sign != 1 && sign != -1)) return ORACLE_ERR_INVALID_ARG;
    const size_t n3 = (size_t)N * N * N;
    cplx* v = (cplx*)malloc(sizeof(cplx) * n3);
    for (size_t i = 0; i < n3; ++i) { v[i].re = (real)in[2 * i]; v[i].im = (real)in[2 * i + 1]; }
    /* the 1D transform of a line: the radix-2 FFT for a power of two, the O(N^2) definition otherwise (reading A20,
     * as in fft2d) */
    const int p2 = is_pow2(N);
    cplx* tw = p2 ? twiddle_table(N, sign) : root_table(N, sign);
    #pragma omp parallel
    {
        cplx* line = (cplx*)malloc(sizeof(cplx) * (size_t)N);
        cplx* tmp = (cplx*)malloc(sizeof(cplx) * (size_t)N);
        #pragma omp for schedule(static)
        for (int z = 0; z < N; ++z)
            for (int y = 0; y < N; ++y) {
                cplx* l = v + ((size_t)z * N + y) * N;
                if (p2) fft1d(l, N, tw); else dft1d_direct(l, N, tw, tmp);
            }
        #pragma omp for schedule(static)
        for (int z = 0; z < N; ++z)
            for (int x = 0; x < N; ++x) {
                for (int y = 0; y < N; ++y) line[y] = v[((size_t)z * N + y) * N + x];
                if (p2) fft1d(line, N, tw); else dft1d_direct(line, N, tw, tmp);
                for (int y = 0; y < N; ++y) v[((size_t)z * N + y) * N + x] = line[y];
            }
        #pragma omp for schedule(static)
        for (int y = 0; y < N; ++y)
            for (int x = 0; x < N; ++x) {
                for (int z = 0; z < N; ++z) line[z] = v[((size_t)z * N + y) * N + x];
                if (p2) fft1d(line, N, tw); else dft1d_direct(line, N, tw, tmp);
                for (int z = 0; z < N; ++z) v[((size_t)z * N + y) * N + x] = line[z];
            }
        free(line); free(tmp);
    }
    free(tw);
    const double sc = sign > 0 ? 1.0 / ((double)N * N * N) : 1.0;
    for (size_t i = 0; i < n3; ++i) { out[2 * i] = (double)v[i].re * sc; out[2 * i + 1] = (double)v[i].im * sc; }
    free(v);
    return ORACLE_OK;
}

/* Step D's iterations ("We proceed with a tomographic approach, which is like conventional 3D CXDI but
 * using E(q) obtained via the steps A-C ... Typically, only a single random guess and N_i^3D (around 50)
 * iterations are sufficient [32]"; ref [32] alternates between the known Fourier samples and the real-space
 * constraint).  Reading A26: with F_0 = E on the known voxels (W > 0) and 0 elsewhere, k times
 *     O    = S3 . F3^-1[F]                          real-space constraint: the 3D support (no positivity: complex O)
 *     F'   = F3[O]
 *     err  = sqrt( sum_{W>0} |F' - E|^2 / sum_{W>0} |E|^2 )
 *     F    = E where W > 0, F' elsewhere            the assembled spectrum is put back on the voxels it covers
 * E: interleaved complex double [N][N][N] (native order, as oracle_assemble_3d writes it), W: double [N][N][N],
 * S3: u8 [N][N][N]; obj (out): the object after the last support step; err (optional): k doubles. */
int oracle_refine_3d(const double* E, const double* W, const unsigned char* S3, int N, int k, double* obj, double* err)
{
    if (!E || !W || !S3 || !obj || N < 2 || (N & 1) || k < 1) return ORACLE_ERR_INVALID_ARG;
    const size_t n3 = (size_t)N * N * N;
    double* F = (double*)malloc(sizeof(double) * 2 * n3);
    double* T = (double*)malloc(sizeof(double) * 2 * n3);
    double den = 0.0;
    for (size_t i = 0; i < n3; ++i) {
        const int known = W[i] > 0.0;
        F[2 * i] = known ? E[2 * i] : 0.0; F[2 * i + 1] = known ? E[2 * i + 1] : 0.0;
        if (known) den += E[2 * i] * E[2 * i] + E[2 * i + 1] * E[2 * i + 1];
    }
    for (int it = 0; it < k; ++it) {
        oracle_fft3(F, obj, N, +1);
        for (size_t i = 0; i < n3; ++i) if (!S3[i]) { obj[2 * i] = 0.0; obj[2 * i + 1] = 0.0; }
        oracle_fft3(obj, T, N, -1);
        double num = 0.0;
        for (size_t i = 0; i < n3; ++i) {
            if (W[i] > 0.0) {
                const double dr = T[2 * i] - E[2 * i], di = T[2 * i + 1] - E[2 * i + 1];
                num += dr * dr + di * di;
                F[2 * i] = E[2 * i]; F[2 * i + 1] = E[2 * i + 1];
            } else { F[2 * i] = T[2 * i]; F[2 * i + 1] = T[2 * i + 1]; }
        }
        if (err) err[it] = den > 0.0 ? sqrt(num / den) : 0.0;
    }
    free(F); free(T);
    return ORACLE_OK;
}

/* Step D with the support update of P:104 ("We shrink the 3D space constraint every 5 iterations, leading to a tighter
 * 3D space constraint close to the shape of the object at the end"; reading A30): oracle_refine_3d's iteration, and after
 * every `every`-th iteration that is not the last the 3D analogue of the 2D shrink-wrap (reading A23):
 *     b = G_sigma * |O|   (Gaussian of standard deviation sigma voxels, as a product with exp(-2 pi^2 sigma^2 |k|^2 / N^2)
 *                          between a forward and an inverse 3D transform; the real part is kept)
 *     S3 <- [ b >= threshold . max b ]      (all zero if the maximum is not positive)
 * S3 is updated in place; blurred (optional, N^3 doubles) receives the b of the LAST update, so that a comparison can
 * set aside the voxels within rounding of the threshold.  every < 1: never (= oracle_refine_3d). */
int oracle_refine_3d_sw(const double* E, const double* W, unsigned char* S3, int N, int k, int every, double sigma, double threshold,
                        double* obj, double* err, double* blurred)
{
    if (!E || !W || !S3 || !obj || N < 2 || (N & 1) || k < 1 || !(sigma >= 0.0) || !(threshold >= 0.0)) return ORACLE_ERR_INVALID_ARG;
    const size_t n3 = (size_t)N * N * N;
    double* F = (double*)malloc(sizeof(double) * 2 * n3);
    double* T = (double*)malloc(sizeof(double) * 2 * n3);
    double den = 0.0;
    for (size_t i = 0; i < n3; ++i) {
        const int known = W[i] > 0.0;
        F[2 * i] = known ? E[2 * i] : 0.0; F[2 * i + 1] = known ? E[2 * i + 1] : 0.0;
        if (known) den += E[2 * i] * E[2 * i] + E[2 * i + 1] * E[2 * i + 1];
    }
    for (int it = 0; it < k; ++it) {
        oracle_fft3(F, obj, N, +1);
        for (size_t i = 0; i < n3; ++i) if (!S3[i]) { obj[2 * i] = 0.0; obj[2 * i + 1] = 0.0; }
        oracle_fft3(obj, T, N, -1);
        double num = 0.0;
        for (size_t i = 0; i < n3; ++i) {
            if (W[i] > 0.0) {
                const double dr = T[2 * i] - E[2 * i], di = T[2 * i + 1] - E[2 * i + 1];
                num += dr * dr + di * di;
                F[2 * i] = E[2 * i]; F[2 * i + 1] = E[2 * i + 1];
            } else { F[2 * i] = T[2 * i]; F[2 * i + 1] = T[2 * i + 1]; }
        }
        if (err) err[it] = den > 0.0 ? sqrt(num / den) : 0.0;
        if (every >= 1 && (it + 1) % every == 0 && it + 1 < k) {
            for (size_t i = 0; i < n3; ++i) { T[2 * i] = sqrt(obj[2 * i] * obj[2 * i] + obj[2 * i + 1] * obj[2 * i + 1]); T[2 * i + 1] = 0.0; }
            oracle_fft3(T, T, N, -1);
            for (int iz = 0; iz < N; ++iz) {
                const int kz = iz < N / 2 ? iz : iz - N;
                for (int iy = 0; iy < N; ++iy) {
                    const int ky = iy < N / 2 ? iy : iy - N;
                    for (int ix = 0; ix < N; ++ix) {
                        const int kx = ix < N / 2 ? ix : ix - N;
                        const double f = exp(-2.0 * PI * PI * sigma * sigma * ((double)kz * kz + (double)ky * ky + (double)kx * kx) / ((double)N * N));
                        const size_t i = ((size_t)iz * N + iy) * N + ix;
                        T[2 * i] *= f; T[2 * i + 1] *= f;
                    }
                }
            }
            oracle_fft3(T, T, N, +1);
            double m = T[0];
            for (size_t i = 1; i < n3; ++i) if (T[2 * i] > m) m = T[2 * i];
            for (size_t i = 0; i < n3; ++i) {
                S3[i] = (m > 0.0 && T[2 * i] >= threshold * m) ? 1 : 0;
                if (blurred) blurred[i] = T[2 * i];
            }
        }
    }
    free(F); free(T);
    return ORACLE_OK;
}

/* The 3D support of Step D from the 2D supports ("We project the 2D space constrains back to the 3D space to
 * form a relatively tight 3D space constraint"; reading A29).  The projections are line integrals along the direction
 * perpendicular to the rotation axis z: voxel (z, y, x) falls on detector row z at column
 *     u_n = c + (x - c) cos theta_n + (y - c) sin theta_n,        c = N / 2,
 * and it stays in the 3D support iff in EVERY projection n its footprint touches the 2D support:
 * S_n[z][floor(u_n)] or S_n[z][floor(u_n) + 1] is set (columns outside the detector count as outside).
 * S3: u8 [N][N][N] (z, y, x) out. */
int oracle_backproject_support(oracle_plan_t p, unsigned char* S3)
{
    if (!p || !S3) return ORACLE_ERR_INVALID_ARG;
    if (!p->have_support) return ORACLE_ERR_NOT_READY;
    const int N = p->N, c = N / 2;
    #pragma omp parallel for schedule(static)
    for (int z = 0; z < N; ++z)
        for (int y = 0; y < N; ++y)
            for (int x = 0; x < N; ++x) {
                int in = 1;
                for (int n = 0; n < p->Np && in; ++n) {
                    const double u = (double)c + (double)(x - c) * cos(p->angles[n]) + (double)(y - c) * sin(p->angles[n]);
                    const long u0 = (long)floor(u);
                    const unsigned char* row = p->S + (size_t)n * p->px + (size_t)z * N;
                    const int a = (u0 >= 0 && u0 < N) ? row[u0] : 0, b = (u0 + 1 >= 0 && u0 + 1 < N) ? row[u0 + 1] : 0;
                    in = a || b;
                }
                S3[((size_t)z * N + y) * N + x] = (unsigned char)in;
            }
    return ORACLE_OK;
}

/* ------------------------------------------------------------------------------------------ */
/* the paper's quality metrics (PRTF, FSC, cut-off at 0.5)   */
/* ------------------------------------------------------------------------------------------ */
/* Fourier shell correlation of two 3D spectra (native order, interleaved complex double [N][N][N]):
 *   FSC(s) = Re sum_{shell s} F1 conj(F2) / sqrt( sum_{shell s} |F1|^2 . sum_{shell s} |F2|^2 ),
 * shell s = round(|k|) over signed integer frequencies, s = 0 .. N/2 (voxels beyond N/2 are left out);
 * 0 where a shell has no energy.  out: N/2 + 1 doubles. */
int oracle_fsc(const double* F1, const double* F2, int N, double* out)
{
    if (!F1 || !F2 || !out || N < 2) return ORACLE_ERR_INVALID_ARG;
    const int ns = N / 2 + 1;
    double* acc = (double*)calloc((size_t)3 * ns, sizeof(double));
    for (int iz = 0; iz < N; ++iz)
        for (int iy = 0; iy < N; ++iy)
            for (int ix = 0; ix < N; ++ix) {
                const int kz = iz < N / 2 ? iz : iz - N, ky = iy < N / 2 ? iy : iy - N, kx = ix < N / 2 ? ix : ix - N;
                const int sh = (int)floor(sqrt((double)kx * kx + (double)ky * ky + (double)kz * kz) + 0.5);
                if (sh >= ns) continue;
                const size_t i = ((size_t)iz * N + iy) * N + ix;
                acc[sh] += F1[2 * i] * F2[2 * i] + F1[2 * i + 1] * F2[2 * i + 1];
                acc[ns + sh] += F1[2 * i] * F1[2 * i] + F1[2 * i + 1] * F1[2 * i + 1];
                acc[2 * ns + sh] += F2[2 * i] * F2[2 * i] + F2[2 * i + 1] * F2[2 * i + 1];
            }
    for (int sh = 0; sh < ns; ++sh) {
        const double d = sqrt(acc[ns + sh] * acc[2 * ns + sh]);
        out[sh] = d > 0.0 ? acc[sh] / d : 0.0;
    }
    free(acc);
    return ORACLE_OK;
}

/* Phase retrieval transfer function of an (averaged) episode against the measured amplitudes of the plan:
 *   PRTF(s) = mean over n and over the measured pixels (M = 1, A > 0) of ring s of  |F2[avg_n](k)| / A_n(k),
 * ring s = round(|k|) in the detector plane, s = 0 .. N/2; 0 for an empty ring.  avg: interleaved complex
 * double [Np][N][N] (e.g. the output of oracle_merge_finish); out: N/2 + 1 doubles. */
int oracle_prtf(oracle_plan_t p, const double* avg, double* out)
{
    if (!p || !avg || !out) return ORACLE_ERR_INVALID_ARG;
    if (!p->have_data) return ORACLE_ERR_NOT_READY;
    const int N = p->N, ns = N / 2 + 1;
    const size_t px = p->px;
    double* sum = (double*)calloc((size_t)ns, sizeof(double));
    double* cnt = (double*)calloc((size_t)ns, sizeof(double));
    cplx* G = (cplx*)malloc(sizeof(cplx) * px);
    for (int n = 0; n < p->Np; ++n) {
        for (size_t i = 0; i < px; ++i) { G[i].re = (real)avg[2 * (n * px + i)]; G[i].im = (real)avg[2 * (n * px + i) + 1]; }
        fft2d(G, N, -1);
        for (int iy = 0; iy < N; ++iy)
            for (int ix = 0; ix < N; ++ix) {
                const size_t i = (size_t)iy * N + ix;
                const double A = (double)p->A[n * px + i];
                if (!p->M[n * px + i] || !(A > 0.0)) continue;
                const int ky = iy < N / 2 ? iy : iy - N, kx = ix < N / 2 ? ix : ix - N;
                const int sh = (int)floor(sqrt((double)kx * kx + (double)ky * ky) + 0.5);
                if (sh >= ns) continue;
                sum[sh] += sqrt((double)G[i].re * G[i].re + (double)G[i].im * G[i].im) / A;
                cnt[sh] += 1.0;
            }
    }
    for (int sh = 0; sh < ns; ++sh) out[sh] = cnt[sh] > 0.0 ? sum[sh] / cnt[sh] : 0.0;
    free(sum); free(cnt); free(G);
    return ORACLE_OK;
}

const char* oracle_real_name(void) { return sizeof(real) == 8 ? "f64" : "f32"; }
