/*
 * lasp_gpu.h -- C ABI of the B200-native LASP-Adam fitting hot path (arXiv 2512.24840).
 *
 * "P:n" = /root/reference/PAPER.md line n; "C.2-n" = row n of the table of readings in
 * SURVEY.md section 8(c); DESIGN.md restates every reading.
 *
 * The library fits, for B observed spectra on one common wavelength grid, the NP = L+2
 * non-linear parameters (L emulator labels, radial velocity v, stellar broadening sigma*)
 * by a fixed number of Adam steps on  chi2 = sum_j w_j (y_j - c_j S_j)^2,
 * w = mask*ivar (Eq. 7-9), where
 *     S = G(mu,sigma) (*) T        Doppler shift + Gaussian broadening      (Eq. 5)
 *     T_j = sum_k phi_k(x) C[k,j]  polynomial spectral emulator             (Eq. 1)
 *     c = P(x^) b                  multiplicative Legendre continuum whose coefficients are
 *                                  re-solved by weighted least squares in EVERY evaluation
 *                                  (Eq. 6; C.2-4)
 * and returns parameters, continuum coefficients, chi2, the error estimate of P:173 and status
 * bits.  Beyond that path: the paper's stopping rules (stop_window), its Clean-strategy
 * pixel masking (clean_every), a Levenberg-Marquardt optimiser (optimizer), the three-model / five-regime
 * emulator (lasp_model_desc.n_models) and the flux-conserving resampler (lasp_resample_coeffs).
 * Every step runs in hand-written sm_100a CUDA kernels; there is no CPU fallback, and the library reads
 * no environment variable: every switch is a field of lasp_fit_opts or of lasp_model_desc.
 *
 * Conventions
 *  - All functions return 0 (LASP_OK) or a negative LASP_ERR_* code; they never throw or abort.
 *  - lasp_model_desc and everything it points to is HOST memory, copied during lasp_create.
 *  - Pointers named in the batch calls (flux, ivar, mask, init, params, cont, chi2, err, status,
 *    model, grad_u) are DEVICE pointers owned by the caller (e.g. torch allocations).  The
 *    library reads inputs, writes outputs, and neither frees nor retains them.  Inputs are never
 *    modified.  Row-major, spectrum-major: element (i, j) at [i*n_pix + j].
 *  - `stream` is a cudaStream_t passed as void* (NULL = default stream).  All work is enqueued on
 *    it and the call returns without synchronising, except that the first call for a larger B
 *    than seen before grows the ctx-owned workspace with cudaMalloc (use lasp_reserve to do that
 *    up front).
 *  - Parameter order everywhere: labels[0..L-1], rv (km/s), sigma* (km/s), physical units.
 *  - A ctx may be used from one host thread at a time; different ctxs are independent.  All calls on one ctx
 *    share its workspace: the library orders them on the device (a call on stream B waits for the ctx's previous
 *    call on stream A), so mixing streams is safe but does not overlap.
 *  - Per-spectrum problems never fail a call; they set bits in status[i].
 *  - Non-finite inputs: a pixel takes part in the fit iff w = mask*ivar (edges zeroed) is != 0, exactly as the
 *    definition reads (C.1); flux on pixels with w == 0 is never looked at.  A NaN/Inf flux or weight on a pixel
 *    that takes part is NOT filtered: it propagates (NaN parameters, NaN chi2) and sets LASP_ST_NONFINITE.
 *  - Every entry point leaves the caller's current CUDA device as it found it.
 */
#ifndef LASP_GPU_H
#define LASP_GPU_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define LASP_OK 0
#define LASP_ERR_INVALID_ARG (-1) /* null pointer, bad shape, non-monotone grid, lo>=hi, sigma lower bound <=0 */
#define LASP_ERR_CUDA (-2)        /* a CUDA runtime call failed; see lasp_last_error */
#define LASP_ERR_NOMEM (-3)       /* device or host allocation failed */
#define LASP_ERR_UNSUPPORTED (-4) /* shape outside the compiled limits (see LASP_MAX_*) */

#define LASP_MAX_SEG 8
#define LASP_MAX_LABELS 30
#define LASP_MAX_TERMS 512
#define LASP_MAX_MODELS 4
#define LASP_MAX_DEGREE 31 /* D+1 <= 32: one continuum row per warp lane in the solver */

/* status[i] bits */
#define LASP_ST_NOT_SPD 1   /* a segment's continuum system was not positive definite; its b = 0 */
#define LASP_ST_NONFINITE 2 /* a non-finite value was met */
#define LASP_ST_NEG_CONT 4  /* continuum c_j <= 0 on a fitted pixel at the solution */
#define LASP_ST_ON_BOUND 8  /* a parameter ended on its prior bound */
#define LASP_ST_STOP_TOL 16  /* stopped by criterion (2) of P:169-171: |L_t - L_(t-W)| < stop_tol */
#define LASP_ST_STOP_RISE 32 /* stopped by criterion (3): the loss rose on W consecutive steps */

typedef struct lasp_ctx lasp_ctx; /* opaque; owns only its own device copies and workspace */

typedef struct {
    int32_t n_pix, n_seg;
    const int32_t *seg_offset;   /* [n_seg+1], seg_offset[0]==0, seg_offset[n_seg]==n_pix; the stencil
                                    never crosses a segment boundary (replicate-edge clamp, C.2-16) */
    const double *loglam;        /* [n_pix] log10(lambda/Angstrom), strictly increasing inside each
                                    segment; fp64 because the step is 1e-4 on values ~3.6 */
    const float *seg_sigma_inst; /* [n_seg] km/s, added in quadrature to sigma* (C.2-13) */
    int32_t n_labels, n_terms;   /* L, K */
    const uint8_t *term_exps;    /* [K*L] monomial exponents, phi_k = prod_l x_l^e_kl (Eq. 1, C.2-24) */
    const float *coeffs;         /* [K*n_pix] row-major emulator coefficients on the observed grid */
    const float *lo, *hi;        /* [NP] prior box, physical units; parameters are optimised as
                                    u = 2(theta-lo)/(hi-lo)-1 in [-1,1] (C.2-18) */
    const uint8_t *label_log10;  /* [L] 1 => tau_l = log10 (C.2-19) */
    const float *emu_a, *emu_b;  /* [L] emulator input x_l = emu_a*tau_l(theta_l) + emu_b */
    int32_t cont_degree;         /* D <= LASP_MAX_DEGREE, same for every segment */
    const int32_t *seg_n_edge;   /* [n_seg] pixels excluded from objective and WLS at each end of the
                                    segment (C.2-17) */
    /* Piecewise emulator (Eq. 1's f_1..f_5: five Teff regimes served by three polynomial models, cold <= 4550 K,
     * warm 4000-9000 K, hot >= 7000 K).  n_models <= 1: one polynomial, the two pointers
     * are not read.  Otherwise term k of the shared term table belongs to model term_model[k] and the spectrum is
     * sum_r omega_r(theta_0) f_r(theta): omega_r rises linearly in tau_0(theta_0) (log10 when label_log10[0]) from 0 at
     * lo0 to 1 at lo1 and falls from 1 at hi0 to 0 at hi1 (a side with lo1 <= lo0, resp. hi1 <= hi0, has no ramp).
     * The paper does not give the weights inside the overlaps: this is reading R-15 of DESIGN.md. */
    int32_t n_models;            /* <= LASP_MAX_MODELS */
    const uint8_t *term_model;   /* [K] */
    const float *model_blend;    /* [n_models*4]: lo0, lo1, hi0, hi1 in the units of label 0 */
} lasp_model_desc;

typedef struct {
    int32_t n_iter;               /* fixed number of Adam steps (Delta-6); used by lasp_fit_batch[_host] only */
    float lr, beta1, beta2, eps;  /* Adam hyper-parameters (defaults 1e-2, 0.9, 0.999, 1e-8) */
    int32_t variant;              /* kernel variant: 0 auto (resident when the model's rows fit shared memory, else
                                     streaming); 1 resident (LASP_ERR_UNSUPPORTED when they do not fit); 2 streaming
                                     (rows in L2-resident global scratch, swept through a shared-memory window:
                                     any row length).  Same arithmetic, same results to rounding order. */
    int32_t emulator_path;        /* emulator contraction T = phi.C (Eq. 1): 0 auto (= 1: measured faster),
                                     1 FP32 FMA, 2 tensor pipe: mma.sync TF32 with both operands split x = hi + lo
                                     (3xTF32-class accuracy); 2 needs the resident variant and n_terms <= 128, else
                                     LASP_ERR_UNSUPPORTED; other values LASP_ERR_INVALID_ARG */
    int32_t refresh;              /* continuum solve (Eq. 6): every step performs one
                                     refinement b += A~^-1 Phi^T W (y - Phi b) whose fixed point is the WLS solution
                                     whatever factor A~ preconditions it.  refresh = k >= 1: the Gram matrix is
                                     re-accumulated and re-factorised every k-th step (1 = every step, the method
                                     as written); 0 (default): adaptive -- re-factorise when the parameters have
                                     moved enough since the last factor (sum|du| x |du| > 6.4e-3), after a system
                                     that was not positive definite, and at least every 64th step */
    int32_t warm;                 /* the first `warm` steps always re-factorise (0 = default 4) */
    int32_t fd_fresh;             /* 1: the 2 NP finite-difference evaluations of the error estimate re-factorise
                                     too (0: they reuse the final evaluation's factor, C.2-22) */
    int32_t stop_window;          /* the paper's stopping rules (step 8; R-2..R-5): 0 (default) = off,
                                     exactly n_iter steps (Delta-6); W in [1, 128] (the paper: 50) = every spectrum stops on
                                     its own loss L_t = sqrt(chi2_t / n_pix) (Eq. 9 restricted to it), tested before update
                                     t: (1) n_iter updates applied (n_iter is then the paper's "maximum of 5000
                                     iterations"); (2) |L_t - L_(t-W)| < stop_tol; (3) W consecutive increases */
    float stop_tol;               /* threshold of criterion (2) (the paper: 1e-5) */
    int32_t clean_every;          /* the Clean strategy (step 6, Eq. 8; R-7..R-12): 0 (default) = No Clean;
                                     e > 0 = after update t, t = e, 2e, ... the residuals are re-evaluated at the new iterate
                                     and the pixel mask is updated (primary 3-sigma clipping with threshold escalation and the
                                     flux-gradient allowance f_shift = 0.5 first, 0.2 afterwards; adjacent pixels at 2 sigma;
                                     neighbourhood growth); clipped pixels stay clipped.  The paper: every 30 steps.
                                     With the stopping rules on, a spectrum that has stopped gets no further update.
                                     Needs the resident variant and one segment whose fitted range is one sweep of the
                                     CTA, else LASP_ERR_UNSUPPORTED */
    int32_t clean_max;            /* at most this many mask updates per spectrum (0 = default 11) */
    int32_t optimizer;            /* 0 (default): Adam, the paper's method (step 8).  1: Levenberg-Marquardt on the
                                     NP x NP system (the route of LASP-CurveFit, and the
                                     "curvature awareness" the paper plans; R-13): n_iter LM iterations, each
                                     the central-difference Jacobian of the re-solved whitened residual (2 NP evaluations),
                                     (J^T J + lambda diag J^T J) delta = -J^T rho in fp64, u' = clip(u + delta) and one trial
                                     evaluation; chi2 falls: accept, lambda / 10, else reject, lambda x 10.  lr, beta1, beta2,
                                     eps are ignored; n_steps reports the accepted steps.  Not together with clean_every or
                                     stop_window (LASP_ERR_UNSUPPORTED) */
    float lm_lambda0;             /* initial damping lambda (0 = default 1e-3) */
} lasp_fit_opts;

/* Build a context on `cuda_device`: validates the description, derives the per-pixel velocity
 * scale s_j = c ln10 dloglam (C.2-12), the padded device layout and the basis tables. */
int lasp_create(const lasp_model_desc *desc, int cuda_device, lasp_ctx **out);
int lasp_destroy(lasp_ctx *ctx);

/* Pre-allocate the workspace for batches of up to B spectra (optional). */
int lasp_reserve(lasp_ctx *ctx, int64_t B);

/* Steps a0-a9 of SURVEY.md 8(a): n_iter Adam steps from `init`, then one evaluation at the
 * final iterate (C.2-21).
 *   flux, ivar [B*n_pix] f32; mask [B*n_pix] u8 (1 = good) or NULL; init [B*NP] physical.
 *   params [B*NP] physical; cont [B*n_seg*(D+1)] plain-Legendre coefficients (numpy legval
 *   convention, nodes x_j = -1 + 2(j-o_s)/P_s) or NULL; chi2 [B];
 *   err [B*NP] = sqrt(diag(rho^T rho/(N_good-NP) (J^T J)^-1)) in physical units (P:173,
 *   C.2-22/23; NaN when J^T J is singular) or NULL to skip; status [B] or NULL;
 *   n_steps [B] = Adam updates applied to each spectrum (= n_iter unless a stopping rule fired) or NULL;
 *   mask_out [B*n_pix] u8 = 1 where the pixel took part in the final evaluation (weight ivar * mask != 0, not an edge
 *   pixel, not clipped by the Clean strategy) or NULL. */
int lasp_fit_batch(lasp_ctx *ctx, int64_t B, const float *flux, const float *ivar,
                   const uint8_t *mask, const float *init, const lasp_fit_opts *opts,
                   float *params, float *cont, float *chi2, float *err, int32_t *status,
                   int32_t *n_steps, uint8_t *mask_out, void *stream);

/* The same fit from HOST buffers (pinned memory recommended), for batches that do not fit on the device or
 * arrive from the host (BASELINE.json config 3, "survey-scale stream"): the batch is cut into chunks of
 * `chunk` spectra (0 = automatic: a short first chunk -- four full rounds of the persistent grid, whose fit hides the next
 * upload -- then chunks of up to 131,072 spectra: every launch costs a ramp and a tail of partly idle SMs, so few large
 * chunks beat many small ones); chunk i+1 is copied host-to-device and chunk
 * i-1's results device-to-host on two copy streams while chunk i is fitted, with ctx-owned double buffers.  All pointers are HOST pointers
 * with the layouts of lasp_fit_batch; mask, cont, err, status, n_steps, mask_out may be NULL.  Blocking: returns when every
 * result is in host memory.  Per-chunk results are identical to lasp_fit_batch on the same spectra. */
int lasp_fit_batch_host(lasp_ctx *ctx, int64_t B, const float *flux, const float *ivar,
                        const uint8_t *mask, const float *init, const lasp_fit_opts *opts,
                        float *params, float *cont, float *chi2, float *err, int32_t *status,
                        int32_t *n_steps, uint8_t *mask_out, int64_t chunk);

/* Inspection: model_j = c_j S_j (Eq. 1, 5, 6) at given physical params [B*NP] and plain-Legendre cont
 * [B*n_seg*(D+1)]; model [B*n_pix], every pixel (edges included: replicate-edge clamp, C.2-16).  Runs the fit
 * kernels' own emulator, kernel-weight and stencil code.  opts may be NULL (defaults); only .variant and
 * .emulator_path are read. */
int lasp_eval_model(lasp_ctx *ctx, int64_t B, const float *params, const float *cont,
                    const lasp_fit_opts *opts, float *model, void *stream);

/* Inspection: one chi2/gradient evaluation (fresh Gram factor) at given physical params: chi2 [B], grad_u [B*NP]
 * (d chi2 / d u, normalised parameters), cont [B*n_seg*(D+1)] or NULL, status [B] or NULL
 * (bit LASP_ST_NOT_SPD only).  opts may be NULL (defaults); only .variant and .emulator_path are read. */
int lasp_eval_grad(lasp_ctx *ctx, int64_t B, const float *flux, const float *ivar,
                   const uint8_t *mask, const float *params, const lasp_fit_opts *opts, float *chi2,
                   float *grad_u, float *cont, int32_t *status, void *stream);

/* Which kernel variant serves this ctx when lasp_fit_opts.variant is 0: 1 = resident (rows of the longest segment
 * in shared memory: log or linear grids, one or several segments), 2 = streaming (rows too long for shared memory).
 * 0 for a NULL ctx. */
int lasp_kernel_variant(const lasp_ctx *ctx);

/* Launch shape of variant 1 (resident) or 2 (streaming): out4 = {available, threads per CTA, CTAs per SM,
 * dynamic shared memory in bytes of a call without the stopping rules (with them: + 16 stop_window bytes)}. */
int lasp_launch_info(const lasp_ctx *ctx, int variant, int32_t *out4);

/* Number of kernels launched by this ctx so far (bench.py reports it as gpu_launches). */
int64_t lasp_launch_count(const lasp_ctx *ctx);

/* Algorithmic FP32 work of one Adam step of one spectrum, in FMA (SURVEY.md 8(d) formula with
 * the moment route) given the mean number of stencil taps 2H+1; for the roofline line. */
double lasp_fma_per_spectrum_step(const lasp_ctx *ctx, double mean_taps);

/* The same count for the algorithm as built: Gram moments, Cholesky and inverse only on the fraction
 * `fresh_frac` of steps that re-factorise, one right-hand side and one continuum evaluation per step. */
double lasp_fma_executed_per_spectrum_step(const lasp_ctx *ctx, double mean_taps, double fresh_frac);

/* Counters of the last lasp_fit_batch on this ctx (blocks until it has finished): out2[0] = group-steps of the Adam
 * loops (groups of 4 spectra x n_iter), out2[1] = those that re-factorised the continuum Gram matrix. */
int lasp_last_fit_stats(lasp_ctx *ctx, double *out2);

/* lasp_eval_grad for callers that cannot allocate (code under CUDA graph capture, tight serving loops, harnesses that
 * forbid cudaMalloc): same arguments, same kernels, same results, but the staged flux / weight planes and the per-CTA
 * scratch live in ONE file-scope device array of LASP_STATIC_SCRATCH_BYTES that every GPU loading the library holds until
 * the process exits; its device address is taken once, in lasp_create, with the ctx's device current.  The call
 * allocates nothing (no cudaMalloc / cudaFree, no allocating library routine): one memset, two kernel launches and the
 * ctx's event calls on `stream`.
 * Limit: 2 B Ppad + (per-CTA scratch of min(ceil(B/4), resident CTAs) groups) floats must fit the array, Ppad = padded
 * pixels per spectrum (n_pix + 2 halos per segment); about B <= 750 spectra of the 1,550-pixel LAMOST-like shape, B <= 150
 * of the 7,781-pixel three-arm shape.  Larger calls return LASP_ERR_UNSUPPORTED with the sizes in lasp_last_error.
 * The array is shared by EVERY ctx and call on the device and keeps the last call's contents: everything the kernels
 * read is rewritten or cleared by the call itself, but two calls that overlap on the GPU (different streams or ctxs)
 * race -- serialise them.  Does not share scratch with lasp_eval_grad / lasp_fit_batch (the ctx workspace). */
#define LASP_STATIC_SCRATCH_BYTES (16u << 20)
int lasp_eval_grad_static(lasp_ctx *ctx, int64_t B, const float *flux, const float *ivar,
                          const uint8_t *mask, const float *params, const lasp_fit_opts *opts,
                          float *chi2, float *grad_u, float *cont, int32_t *status, void *stream);

/* Flux-conserving resampling (step 3 of the paper, Eq. 2-4) of an emulator coefficient
 * table from the model's linear wavelength grid onto an observed grid, once, ahead of lasp_create (the operation is linear
 * and independent of the stellar parameters, so resampling the coefficients equals resampling every model spectrum).
 *   coef_model [n_terms*q] f32, DEVICE: row k on the grid lam1 + m dlam1 (Angstrom), m = 0..q-1 (ELODIE: 3900 A, 0.2 A,
 *   q = 14,501); loglam [n_pix] f64 and seg_offset [n_seg+1] i32, HOST: the observed grid as in lasp_model_desc;
 *   coef_obs [n_terms*n_pix] f32, DEVICE: the result, ready for lasp_model_desc.coeffs (after a copy to the host).
 * Observed integration nodes: per segment the midpoints in log-wavelength between neighbouring pixels and half a
 * step beyond the first and last pixel (on a uniform log grid exactly the paper's exp(lambda -+ dlambda/2)).  Bins beyond
 * the model's range receive only the flux inside it (R-14).  Runs on `stream` of `cuda_device` and BLOCKS until
 * done; no ctx is needed; errors are reported through lasp_last_error(NULL). */
int lasp_resample_coeffs(int cuda_device, int32_t n_terms, int32_t q, double lam1, double dlam1,
                         const float *coef_model, int32_t n_pix, int32_t n_seg, const int32_t *seg_offset,
                         const double *loglam, float *coef_obs, void *stream);

const char *lasp_last_error(const lasp_ctx *ctx); /* ctx-owned string; "" if none; ctx may be NULL */
int lasp_version(void);

#ifdef LASP_PHASE_TIMING
/* debug build only (-DLASP_PHASE_TIMING): per-phase cycle sums of the last fit, 24 counters */
int lasp_debug_phase_cycles(lasp_ctx *ctx, unsigned long long *out24);
#endif

#ifdef __cplusplus
}
#endif
#endif /* LASP_GPU_H */
