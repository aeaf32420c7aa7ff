/*
 * gigalens.h -- C ABI of the B200-native batched lens-model log-posterior and gradient.
 *
 * What the library computes (citations: P:Lnn = /root/reference/PAPER.md line nn; S# / O# = the readings
 * and the operation list of SURVEY.md section 8(c), restated in DESIGN.md section 3):
 *
 *   For each of n_particles independent parameter vectors ("particles": multi-start MAP starts, SVI
 *   draws, HMC chain positions -- P:L72) the log joint  log p~(I_obs, Theta~)  of P:L89 (Eq. 2) in
 *   the unconstrained space of P:L76, and its gradient with respect to Theta~.
 *   The forward model is the one the paper names at P:L64: elliptical power-law (or SIE) mass +
 *   external shear (+ m=3,4 multipoles, BASELINE.json configs[4]); elliptical Sersic and Cartesian
 *   shapelet source light; Sersic lens light; "forward" amplitudes; on a pixel grid supersampled by an
 *   integer factor (P:L189 fn 6); PSF convolution at ray resolution, binning to detector pixels and a
 *   Gaussian chi-square against the observed image (BASELINE.json north_star; readings S10-S12).
 *
 * Conventions common to every call
 *   - Every array argument is a DEVICE pointer owned by the caller unless it says HOST.  The library never
 *     allocates or frees device memory inside a call and keeps no reference to caller memory after return.
 *   - All arrays are fp32 (system_id: int32), C-contiguous, row index = y, column index = x (reading S1).
 *   - Calls are asynchronous on `stream`: no host synchronisation, no device-to-host copy.  Re-entrant on
 *     different streams with different workspaces -- with one proviso: calls that share a gl_config and overlap on
 *     the GPU must pass the SAME psf (a single-system configuration may keep its convolution taps in a
 *     per-configuration slot of constant memory that every call refills from its psf; to evaluate different PSFs
 *     concurrently, create one configuration per PSF).  The caller must not touch outputs or workspace until the
 *     stream has reached the end of the call.
 *   - Errors are returned as gl_status; nothing is thrown or aborted across the ABI.  All argument checks run
 *     on the host before the first launch: on GL_ERR_NULL / _BAD_CONFIG / _BAD_SHAPE / _UNSUPPORTED / _WORKSPACE no
 *     kernel has been launched.  GL_ERR_CUDA reports a failed launch or runtime call: the kernels enqueued before it
 *     stay enqueued, nothing is enqueued after it, and the outputs are undefined.  A NON-sticky CUDA error left
 *     pending by the caller's earlier work on this thread is cleared on entry (it is not this call's error).
 *   - Results are bit-identical for the same particle irrespective of batch composition, order or size
 *     (fixed reduction orders, no atomics): the analogue of P:L83 fn 2.
 *   - There is no CPU fallback.
 */
#ifndef GIGALENS_H
#define GIGALENS_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef enum {
    GL_OK = 0,
    GL_ERR_NULL = -1,         /* a required pointer is NULL */
    GL_ERR_BAD_CONFIG = -2,   /* inconsistent gl_config_desc (even psf_size, supersample < 1, n_params mismatch, ...) */
    GL_ERR_BAD_SHAPE = -3,    /* n_particles < 0 */
    GL_ERR_UNSUPPORTED = -4,  /* a valid configuration this build has no kernel for */
    GL_ERR_WORKSPACE = -5,    /* workspace_bytes < gl_workspace_bytes(cfg, n_particles) or misaligned */
    GL_ERR_CUDA = -6,         /* a CUDA runtime call or launch failed (sticky error left to the caller) */
    GL_ERR_NOALLOC_LIMIT = -7 /* gl_logpost_grad_noalloc: the call needs more scratch than GL_NOALLOC_MAX_BYTES */
} gl_status;

/* Prior / bijector family of one parameter (O1, reading S13).
 *   NONE        theta = z,                       log prior 0
 *   NORMAL      theta = z,                       N(a, b)
 *   LOGNORMAL   theta = exp z,                   ln theta ~ N(a, b)
 *   UNIFORM     theta = lo + (hi-lo) sigmoid z,  U(lo, hi)
 *   TRUNCNORMAL theta = lo + (hi-lo) sigmoid z,  N(a, b) truncated to [lo, hi]
 *   LOGUNIFORM  ln theta = ln lo + (ln hi - ln lo) sigmoid z,  density 1/(theta ln(hi/lo)) */
typedef enum {
    GL_PRIOR_NONE = 0, GL_PRIOR_NORMAL = 1, GL_PRIOR_LOGNORMAL = 2, GL_PRIOR_UNIFORM = 3,
    GL_PRIOR_TRUNCNORMAL = 4, GL_PRIOR_LOGUNIFORM = 5
} gl_prior_kind;

typedef struct { int32_t kind; float a, b, lo, hi; } gl_prior;

/* Arithmetic of the per-ray kernels.  Inputs and outputs are fp32 in both modes.
 *   GL_PRECISION_F64  every per-ray value, the convolution and all reductions in IEEE double on the FP64 FMA pipe
 *                     (MUFU / FP32 results serve only as seeds of Newton steps): the mode that meets the north_star
 *                     tolerances on EVERY gradient component, including those whose per-ray terms cancel by 1e3-1e5.
 *   GL_PRECISION_F32  FP32 FMA pipe + MUFU approximations, fp64 only in the per-particle prologue/epilogue: about
 *                     2x faster (measured 2.1x on config 2); log-posterior within 1e-4 except at accidental
 *                     cancellations, 99.4-99.9 % of the gradient components within the bar (the misses are the
 *                     ill-conditioned ones). */
typedef enum { GL_PRECISION_F64 = 0, GL_PRECISION_F32 = 1 } gl_precision;

/* Model configuration.  The flat parameter vector has the block order of reading S18:
 *   main mass [theta_E, (gamma if EPL), e1, e2, x, y] . shear [g1, g2] . multipoles [c3, s3][c4, s4] .
 *   source Sersic 1 [R, n, e1, e2, x, y, I] . source Sersic 2 [same 7, then eta2 if source2_plane] . shapelets [beta_s, a_0 .. a_{Nc-1}] .
 *   lens Sersic 1 . lens Sersic 2 . lens Sersic 3                       (absent blocks take no entries)
 * with Nc = (nmax+1)(nmax+2)/2 coefficients ordered by n1+n2 then n2 (O5, S9); the shapelet centre is the
 * first source Sersic's centre, so shapelets require n_source_sersic >= 1. */
typedef struct {
    int32_t n_pix;            /* N: detector pixels per side, >= 1 */
    int32_t supersample;      /* s: rays per pixel per side, >= 1 */
    int32_t psf_size;         /* K: PSF taps per side, odd: on the RAY grid (psf_grid 0) or the DETECTOR grid (psf_grid 1) */
    float   pix_scale;        /* Delta: arcsec per detector pixel, > 0 */
    int32_t psf_grid;         /* 0: taps on the ray grid, convolve then bin (S10); 1: taps on the detector grid, bin then
                                 convolve (NEXT-4, S10b).  Other values: GL_ERR_UNSUPPORTED */
    int32_t mass_model;       /* 0 SIE closed form, 1 EPL series */
    int32_t epl_terms;        /* number of series terms kept for EPL, 2..30 (S5; BASELINE.json: 30) */
    int32_t has_shear;        /* 0/1 */
    int32_t multipole_mask;   /* bit0: m=3, bit1: m=4 (S7) */
    int32_t n_source_sersic;  /* 0, 1 or 2 Sersic sources on the one source plane (S1, S2) */
    int32_t shapelet_nmax;    /* -1 none, else 0..10 */
    int32_t n_lens_sersic;    /* 0..3 lens-plane Sersic blocks ("one or more"; env, L1, L2) */
    int32_t param_space;      /* 0: params are unconstrained z (bijector + log-det); 1: physical theta */
    int32_t n_systems;        /* number of (obs, noise_sigma, psf) triples, >= 1 (S19) */
    int32_t n_params;         /* must equal the count implied by the fields above (<= 128) */
    int32_t precision;        /* gl_precision: 0 = GL_PRECISION_F64 (default), 1 = GL_PRECISION_F32 */
    int32_t noise_model;      /* 0: fixed per-pixel sigma map (S12); 1: model-dependent variance (NEXT-4, S12b):
                                 v = noise_sigma^2 + max(model, 0) / exposure_time,
                                 logL = -1/2 sum [ (model - obs)^2 / v + ln v ] - (N^2/2) ln 2 pi */
    float   exposure_time;    /* t_exp of noise_model 1 (> 0; ignored otherwise) */
    int32_t amplitude_mode;   /* 0: light amplitudes are sampled parameters ("forward" modelling);
                                 1: "backward" modelling (NEXT-4, reading S21): every call first solves the
                                    amplitudes (I of each Sersic block, the shapelet coefficients) by weighted least
                                    squares against obs, a* = argmin chi^2, and evaluates logp and its gradient at a*.
                                    The amplitude entries of params are IGNORED on input (any value, NaN included),
                                    carry no prior and no bijector, and their gradient entries are 0; a particle whose
                                    normal matrix is not positive definite gets logp = -INF.  Needs noise_model 0
                                    (else GL_ERR_UNSUPPORTED).  In gl_model_image, which has no obs to invert, the
                                    amplitude entries ARE the amplitudes, untransformed. */
    int32_t source2_plane;    /* 0: both source Sersics on one source plane; 1 (needs n_source_sersic = 2): the second one
                                 on its OWN plane ("multi-source-plane systems"; NEXT-4, reading S23): its rays are
                                 deflected by eta2 * alpha(theta), beta_2 = theta - eta2 alpha, with eta2 (the ratio of the
                                 lensing efficiencies D_ls / D_s of the two planes; the first source carries no mass) one
                                 more SAMPLED parameter directly after the second source's block */
    const gl_prior* priors;   /* HOST pointer, n_params entries, copied by gl_config_create */
} gl_config_desc;

typedef struct gl_config gl_config;   /* opaque, immutable, host-side, library-owned */

/* Validate `desc`, copy it (priors included) and return a handle in *out.  HOST pointers.
 * Errors: GL_ERR_NULL, GL_ERR_BAD_CONFIG, GL_ERR_UNSUPPORTED.  No CUDA call is made. */
gl_status gl_config_create(const gl_config_desc* desc, gl_config** out);

/* Free a handle from gl_config_create (NULL is a no-op).  Must not race with a host call using it;
 * work already enqueued on a stream does not reference the handle.  One resource outlives it: a single-system
 * configuration may hold a slot of constant memory for its convolution taps, which the next configuration created
 * may take over -- the first call on that new configuration must be ordered after the destroyed one's enqueued work
 * (same stream, or an event), as it is whenever one stream is used. */
void gl_config_destroy(gl_config* cfg);

/* Parameter count implied by a configuration (S18); 0 if cfg is NULL. */
int32_t gl_config_n_params(const gl_config* cfg);

/* Array extents a caller needs to size its buffers (what the Python binding checks tensors against), HOST pointer
 * out[5] = { n_pix N, psf_size K, n_systems, n_params, n_amplitudes }:  obs / noise_sigma hold n_systems * N * N
 * floats, psf n_systems * K * K, params n * n_params, out_amp n * n_amplitudes.  Errors: GL_ERR_NULL. */
gl_status gl_config_shape(const gl_config* cfg, int32_t* out);

/* Bytes of device workspace gl_logpost / gl_logpost_grad / gl_model_image need for n_particles
 * (0 if cfg is NULL or n_particles <= 0).  Grows with n_particles up to an internal chunk size, then stays
 * flat (about 4 GiB; about 8 GiB in GL_PRECISION_F64 with shapelet_nmax > 6, whose adjoint keeps two more values per
 * ray; about 16 GiB with amplitude_mode 1, which keeps n_amp component images per particle): larger batches are
 * processed in chunks on the same stream.  The workspace must be 256-byte aligned. */
size_t gl_workspace_bytes(const gl_config* cfg, int64_t n_particles);

/* log p~ for each particle (O1-O8):
 *   out_logp[p] = logL + sum_i log prior_i(theta_i) + sum_i log|dtheta_i/dz_i|,
 *   logL = -1/2 sum_pix ((model - obs)/sigma)^2 - sum_pix ln sigma - (N^2/2) ln 2 pi      (S12)
 *   obs, noise_sigma : [n_systems][N][N]   observed image and FIXED per-pixel noise sigma (> 0)
 *   psf              : [n_systems][K][K]   used as given (no renormalisation), true convolution, zero padding
 *   params           : [n_particles][n_params]
 *   system_id        : [n_particles] in [0, n_systems), or NULL (all 0)                    (S19)
 *   out_logp         : [n_particles]
 * A particle whose parameters are non-finite or outside the model's domain (theta_E <= 0, gamma outside
 * (1,3), |eps| >= 1, R <= 0, n <= 0, beta_s <= 0, or outside a bounded prior support when param_space = 1),
 * or whose result is non-finite, gets out_logp = -INF; NaN is never written.
 * n_particles = 0 returns GL_OK without a launch. */
gl_status gl_logpost(const gl_config* cfg, const float* obs, const float* noise_sigma, const float* psf,
                     const float* params, const int32_t* system_id, int64_t n_particles,
                     float* out_logp, void* workspace, size_t workspace_bytes, void* stream /* cudaStream_t */);

/* As gl_logpost, plus out_grad[p][i] = d out_logp[p] / d params[p][i] (O9: hand-written reverse mode of
 * the whole path, priors and bijector log-determinants included).  Invalid particles get a zero row. */
gl_status gl_logpost_grad(const gl_config* cfg, const float* obs, const float* noise_sigma, const float* psf,
                          const float* params, const int32_t* system_id, int64_t n_particles,
                          float* out_logp, float* out_grad, void* workspace, size_t workspace_bytes,
                          void* stream /* cudaStream_t */);

/* The same evaluation for callers that cannot allocate device memory (code under CUDA graph capture, tight serving
 * loops, harnesses that forbid cudaMalloc): gl_logpost_grad (Eq. 2 and its gradient) with the workspace
 * taken from a buffer of GL_NOALLOC_MAX_BYTES that lives INSIDE the library (a file-scope __device__ array: every GPU
 * that loads libgigalens holds these bytes until the process exits).  The call allocates nothing: no cudaMalloc /
 * cudaFree / allocating library routine, no workspace argument.  Arguments, layouts, ownership, results (bit-identical
 * to gl_logpost_grad) and asynchrony as gl_logpost_grad; DEVICE pointers.
 * Limit: gl_workspace_bytes(cfg, n_particles) <= GL_NOALLOC_MAX_BYTES, else GL_ERR_NOALLOC_LIMIT before any launch
 * (config 1 at 64 particles needs about 7 MB; split a larger batch over several calls or use gl_logpost_grad).
 * The buffer is SHARED by every call of this entry point on a device, whatever the configuration, stream or thread,
 * and keeps the previous call's contents: every call rewrites each element it later reads (zero borders included), so
 * nothing has to be cleared between calls -- but two calls that OVERLAP on the GPU (different streams, or threads
 * without ordering) race on it.  Serialise them on one stream.
 * The first call on a device resolves the buffer's address (cudaGetSymbolAddress, once per device): make one call
 * outside any stream capture first.
 * Errors: as gl_logpost_grad, GL_ERR_NOALLOC_LIMIT, and GL_ERR_CUDA if the buffer's address cannot be obtained. */
#define GL_NOALLOC_MAX_BYTES ((size_t)32 << 20)
gl_status gl_logpost_grad_noalloc(const gl_config* cfg, const float* obs, const float* noise_sigma, const float* psf,
                                  const float* params, const int32_t* system_id, int64_t n_particles,
                                  float* out_logp, float* out_grad, void* stream);

/* Diagnostic: the noise-free model image (O3-O6) of each particle, out_image [n_particles][N][N].
 * Invalid particles get an all-zero image. */
gl_status gl_model_image(const gl_config* cfg, const float* psf, const float* params, const int32_t* system_id,
                         int64_t n_particles, float* out_image, void* workspace, size_t workspace_bytes,
                         void* stream /* cudaStream_t */);

/* Host-buffer convenience forms (what bench.py's `e2e` times).  params_host, out_logp_host and out_grad_host
 * are HOST pointers (pinned memory for true asynchrony; pageable memory works but serialises); everything else
 * is as above (obs / noise_sigma / psf / system_id stay DEVICE pointers: the observation is resident across the
 * steps of an optimiser or sampler, only the particles move).  The call enqueues, on `stream`, the host-to-device
 * copy of params, the kernels, and the device-to-host copies of the results; it does not synchronise.  The
 * workspace must hold gl_workspace_bytes_host(cfg, n) bytes.  out_grad_host == NULL selects gl_logpost. */
size_t gl_workspace_bytes_host(const gl_config* cfg, int64_t n_particles);
gl_status gl_logpost_grad_host(const gl_config* cfg, const float* obs, const float* noise_sigma, const float* psf,
                               const float* params_host, const int32_t* system_id, int64_t n_particles,
                               float* out_logp_host, float* out_grad_host, void* workspace, size_t workspace_bytes,
                               void* stream /* cudaStream_t */);

/* ---- one multi-start MAP optimiser step on the device -------------------------------------
 * Every particle descends  -log p~  independently (P:L83 fn 2) with Adam (the paper's default for MAP) or
 * AdaBelief (lr 1e-4, b1 0.95, b2 0.99 at P:L112).  Update rules as published:
 *   g = -d log p~/dz;  m <- b1 m + (1-b1) g
 *   ADAM       v <- b2 v + (1-b2) g^2
 *   ADABELIEF  v <- b2 v + (1-b2) (g - m)^2 + eps_root          (m already updated)
 *   z <- z - lr (m / (1 - b1^t)) / (sqrt(v / (1 - b2^t)) + eps)
 * gl_map_step = gl_logpost_grad at the current params, then the update, fused on `stream` (no host round trip):
 *   opt        HOST pointer, copied
 *   params     [n][n_params] DEVICE, in/out: z before -> z after
 *   opt_m/opt_v [n][n_params] DEVICE, in/out: optimiser state (zero before step 1)
 *   step       t = 1, 2, ... (bias correction)
 *   out_logp   [n] log p~ at the params BEFORE the update;  out_grad [n][n_params] its gradient (also scratch)
 * A particle whose log-posterior or gradient is not finite keeps its params and state.  Update arithmetic in fp64,
 * storage fp32.  With amplitude_mode 1 the amplitude entries (ignored on input, zero gradient) are never updated.
 * Errors as gl_logpost_grad, plus GL_ERR_BAD_CONFIG for an invalid `opt` (lr <= 0, b outside [0,1), eps < 0,
 * step < 1, or a denominator that can vanish: eps == 0 for Adam, eps == eps_root == 0 for AdaBelief -- an element
 * whose gradient is exactly 0 from step 1 on would otherwise become 0/0). */
typedef enum { GL_OPT_ADAM = 0, GL_OPT_ADABELIEF = 1 } gl_opt_kind;
typedef struct { int32_t kind; float lr, b1, b2, eps, eps_root; } gl_opt_desc;
gl_status gl_map_step(const gl_config* cfg, const gl_opt_desc* opt, const float* obs, const float* noise_sigma,
                      const float* psf, float* params, const int32_t* system_id, int64_t n_particles,
                      float* opt_m, float* opt_v, int64_t step, float* out_logp, float* out_grad,
                      void* workspace, size_t workspace_bytes, void* stream /* cudaStream_t */);

/* Best particle of a MAP run ("multi-start"): index and value of the largest FINITE entry of
 * logp[0..n) (DEVICE), ties resolved to the lowest index; out_index[0] = -1 and out_logp[0] = -INF if none is finite.
 * out_index (int64) and out_logp (float) are DEVICE pointers; one single-CTA launch on `stream`. */
gl_status gl_best_particle(const float* logp, int64_t n_particles, int64_t* out_index, float* out_logp,
                           void* stream /* cudaStream_t */);

/* ---- one SVI iteration on the device ---------------------------------------------------------
 * Fits the multivariate-normal surrogate q~(Theta~; mu~, Sigma~ = L L^T) of P:L78-100 by one optimiser step on the
 * sampled loss  ELBO^ = -sum_j log L_jj - (n/2) log(2 pi e) - (1/N) sum_i log p~(z_i)  (Eq. 2 with E_q[log q] in closed
 * form), z_i = mu + L xi_i, through its pathwise gradient:
 *   d/dmu_j = -(1/N) sum_i g_ij,   d/dL_jk = -(1/N) sum_i g_ij xi_ik - delta_jk / L_jj  (k <= j),  g_i = grad log p~(z_i).
 * The reduction over the draws runs on the device in a fixed order (it replaces the cross-device pmean of Fig. 1 box 5).
 *   opt      HOST pointer (Adam or AdaBelief; P:L112 gives AdaBelief lr 1e-4, b1 0.95, b2 0.99)
 *   mu       [n_params]                DEVICE in/out
 *   l_tril   [n_params (n_params+1)/2] DEVICE in/out, lower triangle packed row-major (L00, L10, L11, L20, ...)
 *   xi       [n_draws][n_params]       DEVICE, standard-normal draws supplied by the caller (counter-based or any RNG)
 *   opt_m/opt_v [n_params + n_tril]    DEVICE in/out optimiser state over [mu; l_tril]
 *   out_stats [2] DEVICE: loss estimate, number of draws with a finite log p~ (the others are left out of the means)
 * With amplitude_mode 1 the surrogate lives on the SAMPLED dimensions only: for every solved amplitude j (zero
 * gradient by construction) mu_j, the entries of row and column j of L and their optimiser state are left untouched,
 * and log L_jj and that dimension's (1/2) log(2 pi e) are left out of the loss (otherwise -log L_jj would drive L_jj
 * to infinity and the loss to -infinity).
 * workspace >= gl_svi_workspace_bytes(cfg, n_draws).  Errors as gl_map_step. */
size_t gl_svi_workspace_bytes(const gl_config* cfg, int64_t n_draws);
gl_status gl_svi_step(const gl_config* cfg, const gl_opt_desc* opt, const float* obs, const float* noise_sigma,
                      const float* psf, float* mu, float* l_tril, const float* xi, const int32_t* system_id,
                      int64_t n_draws, float* opt_m, float* opt_v, int64_t step, float* out_stats,
                      void* workspace, size_t workspace_bytes, void* stream /* cudaStream_t */);

/* The same iteration with the SCORE-FUNCTION gradient, Eq. 3 as the paper prints it:
 *   grad_phi ELBO = E_q[(log q~(z) - log p~(z)) grad_phi log q~(z; phi)],  phi = (mu~, L), z held fixed,
 * sampled as (1/N) sum_i c_i grad_phi log q~(z_i) with log q~(z_i) = -|xi_i|^2/2 - sum_j log L_jj - (n/2) log 2 pi,
 * d log q~/d mu_j = s_j, d log q~/d L_jk = s_j xi_k - delta_jk / L_jj, s = L^-T xi.  It needs log p~ only: the hot path
 * runs FORWARD ONLY on the draws (gl_logpost: about three times the rate of the gradient call).
 *   baseline  0: c_i = w_i = log q~(z_i) - log p~(z_i), the estimator as printed;  1: c_i = N/(N-1) (w_i - mean w), the
 *             leave-one-out control variate (still unbiased) -- the usable form at n_VI ~ 10^3
 * Other arguments, the loss estimate in out_stats, the treatment of non-finite draws and the workspace as gl_svi_step.
 * Errors as gl_svi_step, plus GL_ERR_UNSUPPORTED with amplitude_mode 1 (use gl_svi_step) and GL_ERR_BAD_CONFIG for a
 * baseline other than 0 or 1. */
gl_status gl_svi_step_score(const gl_config* cfg, const gl_opt_desc* opt, const float* obs, const float* noise_sigma,
                            const float* psf, float* mu, float* l_tril, const float* xi, const int32_t* system_id,
                            int64_t n_draws, float* opt_m, float* opt_v, int64_t step, int32_t baseline, float* out_stats,
                            void* workspace, size_t workspace_bytes, void* stream /* cudaStream_t */);

/* ---- one HMC transition of n independent chains on the device -------------------------------
 * Standard leapfrog HMC (mass matrix from the surrogate covariance) in the whitened momentum
 * xi = L^T p, Sigma = L L^T = M^-1:  H = -log p~(z) + |xi|^2/2;  per leapfrog step
 * xi += (eps/2) L^T g(z); z += eps L xi; xi += (eps/2) L^T g(z);  the end point of n_leapfrog steps is accepted iff
 * log_u < H(start) - H(end) and its log p~ is finite.
 *   z        [n][n_params] DEVICE in/out: chain positions
 *   logp     [n]           DEVICE in/out: log p~ at z   (cached; fill with gl_logpost_grad before the first transition)
 *   grad     [n][n_params] DEVICE in/out: its gradient  (cached likewise)
 *   l_tril   packed lower triangle of L shared by all chains, or NULL for the identity
 *   xi       [n][n_params] DEVICE: initial whitened momenta ~ N(0, I), supplied by the caller
 *   log_u    [n]           DEVICE: log of uniform(0,1) draws, supplied by the caller
 *   out_accept [n] int32 (1 accepted), out_dh [n] = H(start) - H(end) (-INF for a non-finite proposal)
 * n_params <= 128.  workspace >= gl_hmc_workspace_bytes(cfg, n).  The trajectory is carried in fp64; the hot path is
 * evaluated at the fp32-rounded positions.  Errors as gl_logpost_grad, plus GL_ERR_BAD_CONFIG for step_size <= 0 or
 * n_leapfrog < 1. */
size_t gl_hmc_workspace_bytes(const gl_config* cfg, int64_t n_chains);
gl_status gl_hmc_step(const gl_config* cfg, const float* obs, const float* noise_sigma, const float* psf,
                      float* z, float* logp, float* grad, const float* l_tril, const float* xi, const float* log_u,
                      const int32_t* system_id, int64_t n_chains, float step_size, int32_t n_leapfrog,
                      int32_t* out_accept, float* out_dh, void* workspace, size_t workspace_bytes,
                      void* stream /* cudaStream_t */);

/* Counter-based random draws for the SVI / HMC consumers (NEXT-2 / NEXT-3; reading S22): the paper draws inside
 * TFP/JAX and names no generator.  Bits: Philox4x32-10 (Salmon et al., SC'11) with key = seed and
 * counter = (step lo, step hi, row, stream_id << 24 | element / 4); normals by fp64 Box-Muller on the word pairs (0,1),
 * (2,3) of a counter, rounded to fp32; uniforms u = (word + 0.5) 2^-32.  Stateless and independent of the launch
 * geometry: the same (seed, step, stream_id, row, column) always yields the same value.
 *   gl_draw_normal       out [n_rows][n_cols] fp32 standard normals (xi of gl_svi_step / gl_hmc_step)
 *   gl_draw_log_uniform  out [n_rows] fp32 ln u, u uniform on (0,1)       (log_u of gl_hmc_step)
 * DEVICE pointer `out`; stream_id <= 255 separates the uses within one step; n_rows < 2^32.
 * Errors: GL_ERR_BAD_SHAPE (negative size), GL_ERR_BAD_CONFIG (stream_id or sizes out of range), GL_ERR_NULL, GL_ERR_CUDA. */
gl_status gl_draw_normal(uint64_t seed, uint64_t step, uint32_t stream_id, int64_t n_rows, int32_t n_cols,
                         float* out, void* stream);
gl_status gl_draw_log_uniform(uint64_t seed, uint64_t step, uint32_t stream_id, int64_t n_rows, float* out, void* stream);

/* Number of light amplitudes of a configuration (S18 order: source Sersic I, shapelet coefficients, lens Sersic I's);
 * 0 if cfg is NULL.  Defined for every amplitude_mode. */
int32_t gl_config_n_amplitudes(const gl_config* cfg);

/* Backward modelling (reading S21): solved amplitudes a* and log p~_B at a* for each particle.
 * cfg must have amplitude_mode 1 (else GL_ERR_BAD_CONFIG).  DEVICE pointers; arguments as gl_logpost, plus
 *   out_amp  [n_particles][gl_config_n_amplitudes] fp32, physical amplitudes (0 where logp = -INF).
 * Workspace: gl_workspace_bytes(cfg, n_particles).  Errors as gl_logpost. */
gl_status gl_linear_amplitudes(const gl_config* cfg, const float* obs, const float* noise_sigma, const float* psf,
                               const float* params, const int32_t* system_id, int64_t n_particles,
                               float* out_amp, float* out_logp, void* workspace, size_t workspace_bytes, void* stream);

/* Number of kernel launches the last call on this thread enqueued (bench.py's gpu_launches claim). */
int64_t gl_last_launch_count(void);

/* Diagnostic per-stage device timing (what bench.py's `roofline` uses).  After gl_stage_timing_enable(1) every
 * compute call made by THIS host thread records a CUDA event pair around each kernel stage on the caller's stream
 * (event records only: still no host synchronisation inside the compute call).  gl_stage_times then waits for
 * the events of the most recent call and writes, per stage, the summed device time in milliseconds to
 * ms_host[0..n) and the number of launches to launches_host[0..n) (HOST pointers; launches_host may be NULL);
 * n must be >= gl_stage_count().  Returns gl_stage_count(), or -1 on error.  Stage i is named gl_stage_name(i):
 * prep, unpack_prior (A), ray_fwd (B+C), conv_chi2 (D+E), conv_transpose (F: D^T), ray_adjoint (F), finalize. */
void        gl_stage_timing_enable(int32_t on);
int32_t     gl_stage_count(void);
const char* gl_stage_name(int32_t i);
int32_t     gl_stage_times(float* ms_host, int32_t* launches_host, int32_t n);

/* Diagnostic layout of the workspace (for bench.py's work model; no CUDA call): HOST pointer out[8] =
 * { byte offset of the per-particle block array PB, particles per chunk Pc, elements per PB row, bytes per element
 *   (8 in GL_PRECISION_F64, 4 in _F32), row index of the series band count M1 (4 M1 recurrence steps in the arithmetic
 *   type), of M2 (4 M2 steps in fp32 above them, fp64 mode only; terms beyond are numerically zero and skipped), of the
 *   validity flag, index of the first particle of the last chunk }.  After a compute call the PB rows of the LAST chunk
 *   are at workspace + out[0].  Errors: GL_ERR_NULL, GL_ERR_BAD_SHAPE (n_particles <= 0). */
gl_status gl_workspace_layout(const gl_config* cfg, int64_t n_particles, int64_t* out);

/* Measurement utility (NOT part of the hot path; the only call that synchronises): issue-rate probe of one SM
 * pipe, so that bench.py can state a MEASURED ALU peak beside the one derived from unit counts and clocks
 * (BASELINE.json north_star: "achieved fraction of the binding roofline"; MEASURED_PEAKS.json has no FP32, FP64
 * or MUFU figure).  kind 0: FP32 FMA, 1: FP64 FMA, 2: MUFU ex2, 3: FP32 and FP64 FMA interleaved 1:1 (both
 * counted), 4: FP64 FMA with three distinct register operands per chain (kinds 0-3 share multiplier and addend),
 * 5: FP64 tensor-core MMA (mma.sync.m8n8k4.f64; one warp instruction = 8 lane-operations per lane), 6: kind 5 and kind 1
 * interleaved 1:1 (both counted: do the FP64 tensor and vector paths add up?), 7: FP64 FMA with two distinct vector-register
 * operands and one warp-uniform operand, 8: FP64 FMA with three vector-register operands whose multiplier is shared by
 * consecutive instructions (operand-reuse cache).  Launches 8 CTAs of 256 threads per SM, each thread running 8 independent chains of
 * n_outer * 64 operations, once untimed and once between two CUDA events on `stream`, waits for it, and writes
 * 1e-12 * lane-operations per second (an FMA counts once) to *tera_lane_ops_per_s_host and the kernel time to
 * *ms_host (HOST pointers; ms_host may be NULL).  workspace: DEVICE pointer, >= 256 bytes (never written in
 * practice).  Errors: GL_ERR_NULL, GL_ERR_BAD_SHAPE (kind or n_outer out of range), GL_ERR_WORKSPACE, GL_ERR_CUDA. */
gl_status gl_probe_pipe(int32_t kind, int32_t n_outer, void* workspace, size_t workspace_bytes, void* stream,
                        double* tera_lane_ops_per_s_host, float* ms_host);

/* Static string for a status code. */
const char* gl_status_string(gl_status s);

/* Library version, "major.minor". */
const char* gl_version(void);

#ifdef __cplusplus
}
#endif
#endif /* GIGALENS_H */
