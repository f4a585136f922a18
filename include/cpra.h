/*
 * cpra.h -- C ABI of the B200-native CPRA iteration loop (libcpra.so).
 *
 * The library runs the data-parallel hot path of the carousel phase retrieval algorithm of
 * "Real time 3D coherent X-ray diffraction imaging" (arXiv 2402.05283): all N_p two-dimensional
 * projection reconstructions advance together, one iteration being
 *     carousel mix (Eq. (4))  ->  forward 2D FT  ->  error + Fourier-modulus constraint
 *                             ->  inverse 2D FT  ->  support / HIO update,
 * plus a one-shot Fourier-slice assembly of the retrieved projections into the N^3 spectrum.
 * Citations "P:<line>" are lines of the paper text; "A<k>" are the readings
 * of ambiguous passages listed in DESIGN.md.
 *
 * Conventions
 *   - n = 0..Np-1 projections (the paper counts from 1); pixel (y, x), row-major, x fastest;
 *     complex = interleaved (re, im) fp32; N a power of two in [16, 1024], or any even N in [16, 1024] whose
 *     prime factors are 2, 3, 5, 7 (the paper's detectors: 160; 700): every call serves both kinds.
 *   - Pointer names: d_* = DEVICE pointers (the caller's allocator, e.g. torch data_ptr());
 *     h_* = HOST pointers.  The library never allocates device memory: every internal buffer lives
 *     in the workspace the caller binds (cpra_workspace_bytes / cpra_bind_workspace).
 *   - Ownership: the caller owns every buffer it passes.  set_* calls copy / precompute into the
 *     workspace; the caller's buffer may be reused as soon as the plan's stream has passed the call.
 *   - Asynchrony: every call only enqueues work on the plan's CUDA stream (no host sync, no D2H),
 *     except cpra_reconstruct_host, which synchronises the stream before it returns.
 *   - Errors: every call returns CPRA_OK (0) or a negative code; nothing throws, aborts or prints.
 *     Errors detectable at enqueue time are returned at once; a kernel fault surfaces as
 *     CPRA_ERR_CUDA from a later call.
 *   - There is no CPU fallback: without a CUDA device every compute call returns CPRA_ERR_CUDA.
 */
#ifndef CPRA_H
#define CPRA_H

#include <stddef.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct cpra_plan_s* cpra_plan_t; /* opaque */

enum {
    CPRA_OK = 0,
    CPRA_ERR_INVALID_ARG = -1,      /* NULL pointer, k < 0, bad K / n_ei / beta, bad `which` */
    CPRA_ERR_UNSUPPORTED_SIZE = -2, /* N outside [16, 1024], odd, or with a prime factor above 7; or Np < 1 */
    CPRA_ERR_NOT_READY = -3,        /* call made before the state it needs exists */
    CPRA_ERR_WORKSPACE = -4,        /* workspace missing, too small or misaligned */
    CPRA_ERR_CUDA = -5,             /* a CUDA runtime call or an earlier kernel failed */
    CPRA_ERR_INVALID_VALUE = -6     /* reserved (input value checks; not performed) */
};

/* Largest half-width K of the carousel weights accepted by cpra_set_carousel. */
#define CPRA_MAX_K 8

/* `which` of cpra_get_projections */
#define CPRA_ITERATE 0   /* the iterate g_n */
#define CPRA_SUPPORTED 1 /* S_n * g_n */

/* plan flags */
#define CPRA_FLAG_DEFAULT 0u
#define CPRA_FLAG_FORCE_MULTIPASS 1u /* never use the one-CTA-per-image shared-memory kernel (N <= 128) */
#define CPRA_FLAG_NO_CHUNKING 2u     /* run every pass over all Np images (no L2-resident chunking) */
#define CPRA_FLAG_NO_WALK 4u         /* never fuse the inverse row pass of iteration t with the forward row pass of
                                        t + 1 (k_row_walk): every iteration runs the three tile kernels.  Same
                                        arithmetic per pixel; for tests and for timing the two structures */
#define CPRA_FLAG_ALL 7u             /* every defined bit; any other bit makes cpra_plan fail with INVALID_ARG */

/*
 * Create a plan for Np projections of N x N pixels ("a scattered intensity map ... of N x N
 * pixels is collected" for each of the N_p angles).  `cuda_stream` is a cudaStream_t (NULL = the
 * legacy default stream); all later work of this plan is enqueued on it.  Host-only: no device work.
 * Defaults: carousel weights alpha = (0.6, 0.2), K = 1, n_ei = 1 (K = 0, alpha_0 = 1 if Np < 3).
 * Every behaviour switch of the library is a flag bit or a call of this header: the library reads
 * no environment variable.
 * Errors: INVALID_ARG (out NULL, undefined flag bits), UNSUPPORTED_SIZE.
 */
int cpra_plan(cpra_plan_t* out, int N, int Np, unsigned flags, void* cuda_stream);

/* Bytes of device workspace this plan needs (a multiple of 256).  Host-only. */
int cpra_workspace_bytes(cpra_plan_t plan, size_t* bytes);

/*
 * Hand the plan its device workspace: `bytes` >= cpra_workspace_bytes, d_ws 256-byte aligned.  The
 * caller keeps ownership and must keep it alive until cpra_destroy.  Uploads the twiddle table.
 * Errors: INVALID_ARG, WORKSPACE (too small / misaligned), CUDA.
 */
int cpra_bind_workspace(cpra_plan_t plan, void* d_ws, size_t bytes);

/*
 * The measured data (I_n = |E_n|^2 for each angle; a beamstop leaves the central
 * pixels unmeasured).
 *   d_I      [Np][N][N] fp32 intensities, detector-centred (zero frequency at index (N/2, N/2)).
 *   d_mask   [Np][N][N] u8, 1 = measured, 0 = unmeasured (left free by the modulus constraint,
 *            A12); NULL = everything measured.
 *   h_angles [Np] doubles on the HOST, rotation angle theta_n about z in radians; used only
 *            by cpra_assemble_3d; NULL = all zero.
 * Precomputes A = sqrt(max(I, 0)) (A14) in the library's internal frequency order with the mask
 * folded in, and den_n = sum over measured pixels of I_n (the error normalisation, A9).
 * Errors: INVALID_ARG (d_I NULL), WORKSPACE (not bound), CUDA.
 */
int cpra_set_data(cpra_plan_t plan, const float* d_I, const unsigned char* d_mask, const double* h_angles);

/*
 * The real-space constraint ("space constraints"): d_S [Np][N][N] u8, non-zero = inside
 * the support of projection n.  Stored bit-packed.  Errors: INVALID_ARG, WORKSPACE, CUDA.
 */
int cpra_set_support(cpra_plan_t plan, const unsigned char* d_S);

/*
 * Carousel coupling, Eq. (4) (readings A1-A4): at the start of iteration t, iff
 * t mod n_ei == 0,   ghat_n = sum_{j=-K..K} alpha_|j| g_{(n+j) mod Np}   (Jacobi, periodic in n);
 * otherwise ghat_n = g_n.  h_alpha: K+1 doubles on the HOST (alpha_0 .. alpha_K), used as given
 * (not renormalised).  K = 0 with alpha_0 = 1 switches the coupling off.
 * Errors: INVALID_ARG (NULL, K < 0, K > CPRA_MAX_K, 2K+1 > Np, n_ei < 1).
 */
int cpra_set_carousel(cpra_plan_t plan, int K, const double* h_alpha, int n_ei);

/*
 * The starting estimate ("random initial guess"; A15): d_g0 interleaved complex fp32
 * [Np][N][N], objects centred at pixel (N/2, N/2).  Resets the iteration counter t to 0.
 * Errors: INVALID_ARG, WORKSPACE, CUDA.
 */
int cpra_set_estimate(cpra_plan_t plan, const float* d_g0);

/*
 * The starting estimate given as its spectrum: g0 = F^-1[G0] (inverse 2D FT of every projection, e^{+2 pi i ...} / N^2),
 * d_G0 interleaved complex fp32 [Np][N][N] in native frequency order (zero frequency at index (0, 0)).  What a random
 * start is made of ("random initial guess"; A15: G0 = M sqrt(I) e^{i phi}, phi uniform): the same result as
 * cpra_fft2(+1) followed by cpra_set_estimate, without the natural-order copy in between.  Resets t to 0.
 * Uses the FFT scratch.  Errors: INVALID_ARG, WORKSPACE, CUDA.
 */
int cpra_set_estimate_spectrum(cpra_plan_t plan, const float* d_G0);

/* Iteration counter t (iterations since cpra_set_estimate); settable for exact resume with n_ei > 1. */
int cpra_get_iteration(cpra_plan_t plan, long* t);
int cpra_set_iteration(cpra_plan_t plan, long t);

/*
 * Run k iterations of the loop (Step B of the paper, all Np projections at once) with
 * HIO feedback beta (P:98 ref [22]).  One iteration, in the paper's order:
 *   1. ghat = mix(g) as set by cpra_set_carousel                       (Eq. (4))
 *   2. G_n  = F[ghat_n], forward 2D FT, e^{-2 pi i ...}, unnormalised  (Eq. (3), A10)
 *   3. num_n = sum_{measured} (|G_n| - A_n)^2                          (A9)
 *   4. measured: G'_n = A_n G_n/|G_n| (G'_n = A_n where |G_n| = 0, A13); unmeasured: G'_n = G_n
 *   5. g'_n = F^-1[G'_n], e^{+2 pi i ...} / N^2
 *   6. S_n = 1: g_n <- g'_n;  S_n = 0: g_n <- ghat_n - beta g'_n       (HIO, complex, A6/A7)
 *   7. t <- t + 1
 * k = 0 is a valid no-op.  iterate(k1) followed by iterate(k2) equals iterate(k1 + k2) bit for bit.
 * Errors: INVALID_ARG (k < 0, beta not finite), NOT_READY (data, support or estimate missing),
 * WORKSPACE, CUDA.
 */
int cpra_iterate(cpra_plan_t plan, int k, float beta);

/*
 * Real-space update rule of step 6 (default CPRA_UPDATE_HIO).  The paper's reconstructions use HIO
 * (P:98 ref [22]) and RAAR with beta = 0.9 (P:98 ref [38]); all keep g' inside the support and
 * differ outside it (reading A22):
 *   CPRA_UPDATE_HIO   S_n = 0:  g_n <- ghat_n - beta g'_n
 *   CPRA_UPDATE_RAAR  S_n = 0:  g_n <- beta ghat_n + (1 - 2 beta) g'_n
 *   CPRA_UPDATE_ER    S_n = 0:  g_n <- 0                  (error reduction; beta unused)
 * Takes effect from the next cpra_iterate call.  Errors: INVALID_ARG.
 */
#define CPRA_UPDATE_HIO 0
#define CPRA_UPDATE_RAAR 1
#define CPRA_UPDATE_ER 2
int cpra_set_update(cpra_plan_t plan, int rule);

/*
 * Reconstruction error of the LAST iteration run (evaluated on its input, before the modulus
 * step; A9): d_E [Np] fp32, E_n = sqrt(num_n / den_n) (0 where den_n = 0); d_Eglobal [1] fp32,
 * sqrt(sum_n num_n / sum_n den_n).  Either pointer may be NULL.  Device-side reduction, fixed
 * summation order (deterministic).  Errors: NOT_READY (no iteration run yet), CUDA.
 */
int cpra_get_error(cpra_plan_t plan, float* d_E, float* d_Eglobal);

/*
 * The projected objects O'_n: d_out interleaved complex fp32 [Np][N][N];
 * which = CPRA_ITERATE: g_n; which = CPRA_SUPPORTED: S_n g_n.
 * Errors: INVALID_ARG, NOT_READY (no estimate; SUPPORTED also needs the support), CUDA.
 */
int cpra_get_projections(cpra_plan_t plan, int which, float* d_out);

/*
 * Fourier-slice assembly (first sentence of Step D; Fourier slice theorem P:35-44):
 * E_n = F[S_n g_n] are placed as central slices of the 3D spectrum (rotation about z by
 * theta_n: F2[P_n](kz, ku) = F3[O](kz, ky = ku sin theta_n, kx = ku cos theta_n)) and every voxel
 * is interpolated bilinearly in (angle, radius) between the two bracketing slices (A17; the paper
 * only says "interpolate").  d_vol: interleaved complex fp32 [N][N][N] (kz, ky, kx), native FFT
 * order, comparable with the 3D FT of an object centred at (N/2, N/2, N/2); voxels with
 * sqrt(kx^2+ky^2) > N/2-1 are zero.  d_weight: fp32 [N][N][N], 1 where a value was written, 0
 * elsewhere; may be NULL.  One-shot, outside the timed loop.  Needs data (for the angles), support
 * and an estimate -- NOT an iteration: assembling the starting estimate is allowed (the slices are
 * then F[S g0]).  Overwrites the FFT scratch only; the loop state is untouched.
 * Errors: INVALID_ARG, NOT_READY (data, support or estimate missing), CUDA.
 */
int cpra_assemble_3d(cpra_plan_t plan, float* d_vol, float* d_weight);

/*
 * Diagnostic: the library's own 2D FFT of a stack, natural order in and out.  d_in, d_out:
 * interleaved complex fp32 [Np][N][N]; sign = -1 forward (unnormalised), +1 inverse (/N^2).
 * Uses the same kernels as the loop (row pass, column pass); overwrites the FFT scratch only.
 * Errors: INVALID_ARG, WORKSPACE, CUDA.
 */
int cpra_fft2(cpra_plan_t plan, const float* d_in, float* d_out, int sign);

/* ---------------------------------------------------------------------------------------------------
 * Around the loop: the steps of the paper's procedure that wrap the iteration.
 * All of them enqueue on the plan's stream; none synchronises or copies to the host.
 * ------------------------------------------------------------------------------------------------- */

/*
 * Seam of a scan over [0, 180 degrees) (reading A5b).  The paper's stack is "periodic" in n
 * (P:54); with one rotation axis the projection at theta + 180 degrees is the projection at
 * theta mirrored in u, so true periodicity needs the neighbour that is reached by wrapping round the end
 * of the stack to be read mirrored: pixel (y, x) of it is taken at (y, (N - x) mod N).  flip = 0 (default):
 * literal wrap (exact for a [0, 360) scan); flip = 1: mirrored wrap.  Takes effect from the next
 * cpra_iterate.  Errors: INVALID_ARG.
 */
int cpra_set_seam(cpra_plan_t plan, int flip);

/*
 * Positivity in the real-space step (the conventional companion of the support constraint for
 * real, non-negative objects): with on = 1 a pixel INSIDE the support whose modulus-constrained estimate has
 * Re g' < 0 is updated like a pixel outside it (HIO: ghat - beta g'; RAAR / ER accordingly).  Default 0: support
 * only (reading A7: the headline object is complex).  The decision is a sign test in fp32, so it is not
 * continuous in the data: two arithmetics agree on it except at pixels with |Re g'| within rounding of zero.
 * Errors: INVALID_ARG.
 */
int cpra_set_positivity(cpra_plan_t plan, int on);

/*
 * Shrink-wrap update of the support ("2D CSWA" ref [35]; "At the end of each episode, we perform
 * an extra 2D CSWA iteration to obtain a tighter space constraint"; reading A23).  For every n:
 *     b_n = G_sigma * |S_n g_n|     periodic Gaussian blur, sigma in pixels, of the supported estimate
 *     S_n <- [ b_n >= threshold * max over the pixels of b_n ]      (empty if that maximum is <= 0)
 * d_blurred: optional fp32 [Np][N][N], receives b_n (so that a caller can see how close to the threshold a
 * pixel was); may be NULL.  Uses the FFT scratch and the spare state buffer; the iterate is untouched.
 * Errors: INVALID_ARG (sigma or threshold negative / not finite), NOT_READY (support or estimate missing), CUDA.
 */
int cpra_shrinkwrap(cpra_plan_t plan, float sigma, float threshold, float* d_blurred);

/* The current support as u8 [Np][N][N] (1 = inside).  Errors: INVALID_ARG, NOT_READY, CUDA. */
int cpra_get_support(cpra_plan_t plan, unsigned char* d_S);

/*
 * Step A: "Pre-reconstruct a single PO ... via the conventional 2D CXDI algorithm", k iterations of
 * steps 2-6 of cpra_iterate on projection n alone (no carousel mix: one PO has no neighbours yet).  The other
 * projections and the iteration counter are untouched; cpra_get_error is NOT_READY until the next cpra_iterate.
 * Errors: INVALID_ARG (n out of range, k < 0, beta not finite), NOT_READY, WORKSPACE, CUDA.
 */
int cpra_prereconstruct(cpra_plan_t plan, int n, int k, float beta);

/*
 * Step C: "Repeat step A and B multiple times ... We select a certain number N_l < N_r of the best
 * reconstructed episodes, which have the lowest reconstruction error", align them and average.
 * The bank of kept episodes lives in a caller-owned DEVICE buffer (cpra_merge_bytes; 256-byte aligned):
 * N_l stacks of complex fp32 [Np][N][N] plus a few hundred bytes per episode.
 *   cpra_merge_bind    attach the buffer and empty the bank.
 *   cpra_merge_offer   offer one episode: d_episode = complex fp32 [Np][N][N] with its error E, or NULL = the
 *                      plan's own supported estimate S_n g_n with the global error of its last iteration (E
 *                      ignored; needs an iteration).  It takes a free slot, else replaces the worst kept episode
 *                      if its error is lower (decided on the device, no host sync).
 *   cpra_merge_errors  d_E: double [N_l] errors in slot order (first *d_count are valid); d_count: int [1].
 *   cpra_merge_get     copy the episode of one slot out (for moving banks between GPUs).
 *   cpra_merge_finish  the merge, in the paper's order (readings A24, A25):
 *        1. every PO of every kept episode is shifted circularly by a whole number of pixels, -round(com),
 *           com = sum |O| r / sum |O| about the centre pixel ("we move the mass center of each PO");
 *        2. against the kept episode of lowest error, on projection n_ref (n_ref = -1: all projections): the
 *           episode or its twin conj(O(-r)) is taken, whichever has the larger |<O_best, .>| -- the smaller
 *           Euclidean distance once the free global phase of an unconstrained iterate is taken out -- and is
 *           multiplied by that unit phase;
 *        3. d_out [Np][N][N] complex fp32 = the mean of the corrected episodes.
 *        d_shifts: optional int [N_l][Np][2] (sy, sx); d_twins: optional int [N_l].
 * Errors: INVALID_ARG, WORKSPACE (buffer too small / misaligned), NOT_READY (no bank bound; offer from the plan
 * before an iteration), CUDA.
 */
int cpra_merge_bytes(cpra_plan_t plan, int n_keep, size_t* bytes);
int cpra_merge_bind(cpra_plan_t plan, void* d_buf, size_t bytes, int n_keep);
int cpra_merge_offer(cpra_plan_t plan, const float* d_episode, double E);
int cpra_merge_errors(cpra_plan_t plan, double* d_E, int* d_count);
int cpra_merge_get(cpra_plan_t plan, int slot, float* d_episode);
int cpra_merge_finish(cpra_plan_t plan, int n_ref, float* d_out, int* d_shifts, int* d_twins);

/*
 * Consistency of the projections of ONE episode before Step D (reading A28 -- an addition of this
 * library, not a step the paper states: the paper relies on the carousel coupling alone).  An iterate
 * without reality constraint keeps, projection by projection, a free global phase and the twin ambiguity; both are
 * fixed from facts of the forward model, in place on d_episode (complex fp32 [Np][N][N], e.g. cpra_merge_finish's
 * output):
 *   1. every projection of one object has the same total (line integrals), so each PO is multiplied by the
 *      unit phase that makes its total real and positive;
 *   2. neighbouring projections are similar, so, walking away from projection n_ref in both directions, PO n
 *      is replaced by its twin conj(O_n(-r)) iff the twin is closer to its already decided neighbour.
 * d_flips: optional int [Np], 1 where the twin was taken.  Errors: INVALID_ARG, WORKSPACE, CUDA.
 */
int cpra_align_episode(cpra_plan_t plan, float* d_episode, int n_ref, int* d_flips);

/*
 * Step D ("performing 3D FTs as a set of 2D FTs"): the 3D transform of a cube, on a plan created
 * with Np == N.  d_in, d_out: complex fp32 [N][N][N] (z, y, x), natural order, may not alias; sign = -1
 * forward (unnormalised), +1 inverse (/ N^3).  The (y, x) transforms of the N slices run through the loop's
 * own kernels (as cpra_fft2), the z lines through one more pass.  With sign = +1 on the output of
 * cpra_assemble_3d this gives the object O(r) centred at (N/2, N/2, N/2).
 * Errors: INVALID_ARG (Np != N), WORKSPACE, CUDA.
 */
int cpra_fft3(cpra_plan_t plan, const float* d_in, float* d_out, int sign);

/*
 * Step D's iterations ("a tomographic approach, which is like conventional 3D CXDI but using E(q) ... a
 * single random guess and N_i^3D (around 50) iterations are sufficient [32]"; reading A26), on a plan
 * created with Np == N.  With F = E on the voxels the slices cover (d_W > 0) and 0 elsewhere, k times:
 *     O = S3 . F3^-1[F];   F' = F3[O];   err_it = sqrt(sum_{W>0} |F' - E|^2 / sum_{W>0} |E|^2);   F = W > 0 ? E : F'
 *   d_E   complex fp32 [N][N][N], the assembled spectrum (cpra_assemble_3d's d_vol)
 *   d_W   fp32 [N][N][N], > 0 where E is known (cpra_assemble_3d's d_weight)
 *   d_S3  u8 [N][N][N], the 3D support (1 = inside), in the object's frame (centre at (N/2, N/2, N/2))
 *   d_obj complex fp32 [N][N][N] out: the object after the last support step
 *   d_err fp32 [k] out or NULL
 * Uses the plan's state buffers, both spectrum buffers and its packed support as scratch: a loop state and a support
 * held by this plan are lost (Step D runs on its own plan).  The cube stays in the library's internal layouts between
 * the transforms of an iteration; only d_E, d_W, d_S3 and d_obj are natural-order arrays.
 * Errors: INVALID_ARG (Np != N, k < 1, NULL), WORKSPACE, CUDA.
 */
int cpra_refine_3d(cpra_plan_t plan, const float* d_E, const float* d_W, const unsigned char* d_S3, int k,
                   float* d_obj, float* d_err);

/*
 * cpra_refine_3d with the support update of P:104 ("We shrink the 3D space constraint every 5 iterations, leading to a
 * tighter 3D space constraint close to the shape of the object at the end"; reading A30): after every
 * `every`-th iteration that is not the last, the 3D analogue of cpra_shrinkwrap,
 *     b = G_sigma * |O|  (product with exp(-2 pi^2 sigma^2 |k|^2 / N^2) between a forward and an inverse 3D transform),
 *     S3 <- [ b >= threshold . max b ]   (all zero if the maximum is not positive).
 *   d_S3       u8 [N][N][N] IN and OUT: the support the iterations start from; on return the support of the last update
 *   every      >= 1: update after iterations every, 2 every, ... (< k);  < 1: never (= cpra_refine_3d)
 *   sigma      standard deviation of the Gaussian in voxels, >= 0;  threshold: fraction of the maximum, >= 0
 *   d_blurred  fp32 [N][N][N] out or NULL: the b of the last update (diagnostic; untouched if no update ran)
 * Other arguments, scratch use and the plan (Np == N) as for cpra_refine_3d; the second spectrum buffer is used too.
 * Errors: INVALID_ARG (as cpra_refine_3d; sigma or threshold negative / not finite), WORKSPACE, CUDA.
 */
int cpra_refine_3d_sw(cpra_plan_t plan, const float* d_E, const float* d_W, unsigned char* d_S3, int k, int every, float sigma,
                      float threshold, float* d_obj, float* d_err, float* d_blurred);

/*
 * The 3D support of Step D from the 2D supports ("We project the 2D space constrains back to the 3D space to form
 * a relatively tight 3D space constraint"; reading A29): the visual hull.  With the geometry of the projections
 * (rotation about z; image rows = z, columns = u; the angles of cpra_set_data) voxel (z, y, x) lands on row z at
 *     u_n = c + (x - c) cos theta_n + (y - c) sin theta_n,   c = N / 2,
 * and stays iff in EVERY projection n S_n[z][floor(u_n)] or S_n[z][floor(u_n) + 1] is set (columns outside the detector
 * count as outside).  u_n is evaluated in double, one rounding per product and sum.
 *   d_S3  u8 [N][N][N] (z, y, x) out, caller-owned.
 * Uses the plan's current 2D supports (cpra_set_support, or the last cpra_shrinkwrap) and the second spectrum buffer.
 * Errors: INVALID_ARG, NOT_READY (no support), WORKSPACE, CUDA.
 */
int cpra_backproject_support(cpra_plan_t plan, unsigned char* d_S3);

/*
 * The paper's quality metrics ("PRTF", "FSC", resolution at the 0.5 cut-off).
 *   cpra_fsc   Fourier shell correlation of two 3D spectra d_F1, d_F2 (complex fp32 [N][N][N], native order; a
 *              plan with Np == N):  FSC(s) = Re sum_s F1 conj(F2) / sqrt(sum_s |F1|^2 sum_s |F2|^2), shell
 *              s = round(|k|) over signed integer frequencies, s = 0 .. N/2; 0 for a shell without energy.
 *   cpra_prtf  phase retrieval transfer function of an averaged episode d_avg (complex fp32 [Np][N][N], e.g.
 *              cpra_merge_finish's output) against the measured amplitudes of cpra_set_data:
 *              PRTF(s) = mean over n and the measured pixels with A > 0 of ring s of |F2[avg_n]| / A_n.
 *   d_out: fp32 [N/2 + 1].  Shell sums are double atomics: reproducible to ~1e-15, not bit for bit.
 * cpra_prtf uses the FFT scratch and the spare state buffer; the loop state is untouched.
 * Errors: INVALID_ARG (cpra_fsc: Np != N), NOT_READY (cpra_prtf without data), CUDA.
 */
int cpra_fsc(cpra_plan_t plan, const float* d_F1, const float* d_F2, float* d_out);
int cpra_prtf(cpra_plan_t plan, const float* d_avg, float* d_out);

/*
 * cpra_fsc for callers that cannot allocate device memory (code under CUDA graph capture, serving loops, harnesses
 * that forbid cudaMalloc): the same Fourier shell correlation (same kernels' arithmetic, same
 * result up to the order of the double atomics), but with no plan and no workspace.  The shell accumulators live in
 * a file-scope __device__ array of CPRA_FSC_STATIC_SCRATCH_BYTES inside libcpra.so, which every GPU that loads the
 * library holds until the process exits; the call allocates nothing (no cudaMalloc / cudaFree, no allocating
 * library routine; the array's device address is looked up once per device, on the first call made with that device
 * current).
 *   N        grid size, even, 2 <= N <= CPRA_FSC_STATIC_MAX_N; a larger N is refused with UNSUPPORTED_SIZE
 *   d_F1/2   DEVICE complex fp32 [N][N][N], native order (caller-owned, read only)
 *   d_out    DEVICE fp32 [N/2 + 1] (caller-owned)
 *   stream   a cudaStream_t of the current device (NULL = default stream); the call is asynchronous on it
 * All calls share the one array, which keeps the sums of the last call: every call clears it first, on its stream.
 * Two calls that overlap on the GPU (different streams without a dependency, or two host threads on two streams)
 * race on it and both results are undefined; calls on one stream, or otherwise ordered, are safe.
 * Errors: INVALID_ARG (NULL, N odd or < 2), UNSUPPORTED_SIZE (N > CPRA_FSC_STATIC_MAX_N), CUDA.
 */
#define CPRA_FSC_STATIC_MAX_N 1024
#define CPRA_FSC_STATIC_SCRATCH_BYTES 12312 /* 3 * (CPRA_FSC_STATIC_MAX_N / 2 + 1) doubles */
int cpra_fsc_static(int N, const float* d_F1, const float* d_F2, float* d_out, void* stream);

/*
 * End-to-end convenience with HOST buffers (pinned memory recommended): uploads the inputs,
 * runs k iterations, downloads the result and synchronises the plan's stream.
 *   h_I [Np][N][N] fp32, h_mask [Np][N][N] u8 or NULL, h_angles [Np] or NULL, h_S [Np][N][N] u8,
 *   h_g0 [Np][N][N] complex fp32  ->  h_out [Np][N][N] complex fp32 (the iterate; may be NULL),
 *   h_E [Np] fp32 or NULL, h_Eglobal [1] fp32 or NULL.
 * d_stage: DEVICE staging buffer of at least cpra_host_staging_bytes (caller-owned, 256-aligned).
 * Errors: as the calls it is made of.
 */
int cpra_host_staging_bytes(cpra_plan_t plan, size_t* bytes);
int cpra_reconstruct_host(cpra_plan_t plan, void* d_stage, size_t stage_bytes,
                          const float* h_I, const unsigned char* h_mask, const double* h_angles,
                          const unsigned char* h_S, const float* h_g0, int k, float beta,
                          float* h_out, float* h_E, float* h_Eglobal);

/* Tuning knob: process the Np images in chunks of `images` (K1, K2, K3 per chunk) so that a chunk's
 * intermediate spectrum stays in the 126 MB L2 between the three passes; 0 = one chunk (all images).
 * Results are bit-identical for every chunk size.  Errors: INVALID_ARG. */
int cpra_set_chunk(cpra_plan_t plan, int images);

/* Tuning knob: run every iteration as ONE launch of the whole-image kernel with each projection spread over
 * the shared memories of a thread-block cluster of `ctas_per_image` CTAs (1, 2, 4, 8 or 16; N <= 256 and
 * N / 16 divisible by it; ignored where the plan does not allow it).  0 = the library's own choice (default),
 * -1 = never.  Results agree with the other kernel paths to rounding (same stages, same arithmetic per pixel).
 * Errors: INVALID_ARG. */
int cpra_set_cluster(cpra_plan_t plan, int ctas_per_image);

/* Tuning knob: CTAs per SM of the fused inverse-row / forward-row kernel (k_row_walk).  Each CTA walks a run
 * of consecutive projections for one row tile and transforms the two tiles next to its run a second time, so
 * more CTAs mean more parallelism and shorter runs (more duplicated work).  0 = the library's choice (default:
 * 2 at N = 512, 4 at N = 256); values above what registers and shared memory allow only shorten the runs.
 * Results do not depend on it.  Errors: INVALID_ARG. */
int cpra_set_walk_ctas(cpra_plan_t plan, int per_sm);

/*
 * Per-kernel timing for the roofline report (bench.py): while enabled, every kernel launch of
 * cpra_iterate is bracketed by CUDA events on the plan's stream, summed per kernel class.
 * cpra_profile_read synchronises the stream, writes the accumulated milliseconds and launch counts
 * (HOST arrays of CPRA_PROFILE_CLASSES entries) and resets them.  Not for use inside a timed
 * throughput measurement: the event records sit between the launches.
 * Errors: INVALID_ARG, CUDA.
 */
#define CPRA_PROFILE_ROW_FWD 0 /* mix + forward row FFT */
#define CPRA_PROFILE_COL 1     /* forward column FFT + error + modulus + inverse column FFT */
#define CPRA_PROFILE_ROW_INV 2 /* inverse row FFT + support / HIO */
#define CPRA_PROFILE_IMAGE 3   /* N <= 128: the whole iteration of a projection in one kernel */
#define CPRA_PROFILE_WALK 4    /* inverse row FFT + HIO of iteration t fused with mix + forward row FFT of t + 1 */
#define CPRA_PROFILE_CLASSES 5
int cpra_profile(cpra_plan_t plan, int enable);
int cpra_profile_read(cpra_plan_t plan, double* h_ms, long* h_launches);

/* Number of kernels this plan has launched since it was created (for bench.py's gpu_launches). */
int cpra_launch_count(cpra_plan_t plan, long* count);

/* Free the plan (host memory only; the workspace stays the caller's). */
int cpra_destroy(cpra_plan_t plan);

/* Static, never NULL. */
const char* cpra_status_string(int status);

#ifdef __cplusplus
}
#endif
#endif /* CPRA_H */
