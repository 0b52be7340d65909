/*
 * jt.h -- C ABI of libjt: lensed-image simulation on one NVIDIA B200 (sm_100a).
 *
 * The hot path is the three-step image simulation of PAPER.md:55 (section "Improvements over
 * lenstronomy in image simulation"): (1) a coordinate grid in the observer's angles is ray-traced
 * through every deflector back to the source plane, (2) the source surface brightness is evaluated
 * on the traced grid, (3) the lensed image is convolved with the PSF.  Where the time goes:
 * PAPER.md:47 ("ray-tracing through tens of thousands of dark matter substructures").  Profile
 * names: NIE/SIE PAPER.md:80, SHEAR :85, TNFW :87, SERSIC_ELLIPSE :103; FFT convolution :110-114.
 * The paper prints no formula; the definitions used (G, E, S, H, T, R, B, P) are the readings
 * listed in DESIGN.md "Readings of the paper".
 *
 * Conventions for EVERY function:
 *   - extern "C", returns jt_status (0 = JT_OK), never throws, never exits.
 *   - All work is enqueued on `stream` (a cudaStream_t passed as void*; NULL = legacy default
 *     stream).  No function synchronises the device; host structs are read before the call
 *     returns, so the caller may free them immediately.
 *   - The caller owns every buffer, workspace included.  The library allocates no device memory.
 *     State it keeps between calls, all of it listed here: per host thread the last CUDA error code, the
 *     launch counter and -- only while jt_profile_enable(1) is in force -- four CUDA events and a 48-byte
 *     pinned host buffer; per process one 60 KB __constant__ buffer per device (the taps of the direct
 *     convolution) with the event that orders its users (see jt_psf_convolve), the 32 MiB scratch array of
 *     jt_ray_shoot_noalloc per device, one bit per kernel and device ("shared-memory attribute set") and, per host
 *     thread, the last four convolution plans.
 *   - "device [n]" = pointer to device memory holding n elements of the call's dtype
 *     (float for JT_F32, double for JT_F64), aligned to the element size.  "host" = ordinary
 *     host memory.  Arrays are row-major, x (column) fastest.
 *   - In/out aliasing is not allowed.  Outputs are unspecified after an error.
 *   - JT_F32 mode: storage and the O(rays x subhalos) loop are float; the O(rays) per-ray work
 *     (grid angle, SIE, shear, lens equation) is done in double because beta = theta - alpha
 *     cancels near the Einstein ring.  JT_F64: everything double.
 *   - There is no CPU fallback: on a machine without an sm_100 device every compute call returns
 *     JT_ERR_UNSUPPORTED or JT_ERR_CUDA.
 *
 * Error codes: JT_ERR_INVALID_VALUE  null pointer where data is required, negative count,
 *              nx/ny < 1, supersample < 1 or > JT_MAX_SUPERSAMPLE, pixel_scale <= 0,
 *              even or < 1 kernel size, n_src < 0 or > JT_MAX_SOURCES, in == out, a workspace that is not
 *              16-byte aligned;
 *              JT_ERR_UNSUPPORTED    unknown dtype / method, device is not compute capability 10.x;
 *              JT_ERR_WORKSPACE      workspace_bytes smaller than the matching *_workspace_bytes query
 *                                    (or workspace NULL when the query is non-zero);
 *              JT_ERR_CUDA           a CUDA call failed; jt_last_cuda_error() returns its cudaError_t.
 * Parameter VALUES held in device arrays (Rs <= 0, r_trunc <= 0, NaN) are not validated:
 * IEEE garbage in, garbage out, never a fault.  Zero-sized problems (n_rays = 0, B = 0) are no-ops.
 * |e| >= 1 ellipticities are clamped to 0.9999 (definition E), not rejected.
 */
#ifndef JT_H
#define JT_H

#include <stddef.h>
#include <stdint.h>

#if defined(__GNUC__)
#define JT_API __attribute__((visibility("default")))
#else
#define JT_API
#endif

#ifdef __cplusplus
extern "C" {
#endif

#define JT_VERSION 200           /* 0.2.0 */
#define JT_MAX_SUPERSAMPLE 16    /* s x s sub-rays per pixel, binned with warp shuffles */
#define JT_MAX_SOURCES 16        /* Sersic components per system (host arrays, passed by value to kernels) */

typedef enum { JT_OK = 0, JT_ERR_INVALID_VALUE = 1, JT_ERR_UNSUPPORTED = 2, JT_ERR_WORKSPACE = 3, JT_ERR_CUDA = 4 } jt_status;
typedef enum { JT_F32 = 0, JT_F64 = 1 } jt_dtype;
typedef enum { JT_CONV_AUTO = 0, JT_CONV_DIRECT = 1, JT_CONV_FFT = 2 } jt_conv_method;

/* Definition G (observer grid).  Host struct.  Pixel (j,i), j = row (y), i = column (x); sub-ray
 * (J,I), J in [0,ny*s), I in [0,nx*s): theta_x = cx + (I - (nx*s-1)/2) h, theta_y = cy + (J - (ny*s-1)/2) h,
 * h = pixel_scale/s.  Sub-ray (J,I) belongs to pixel (J/s, I/s). */
typedef struct {
    int32_t nx, ny;          /* pixels */
    double  pixel_scale;     /* arcsec per pixel, > 0 */
    double  cx, cy;          /* grid centre, arcsec */
    int32_t supersample;     /* s >= 1 */
} jt_grid;

/* Deflectors (host struct).  Definitions S (SIE), H (external shear about the origin,
 * PAPER.md:85), T (truncated NFW).  The five TNFW arrays are DEVICE pointers of the
 * call's dtype, each [n_tnfw]; they may be NULL iff n_tnfw == 0. */
typedef struct {
    int32_t has_sie;   double sie_theta_E, sie_e1, sie_e2, sie_cx, sie_cy;
    int32_t has_shear; double shear_gamma1, shear_gamma2;
    int64_t n_tnfw;
    const void *tnfw_cx, *tnfw_cy, *tnfw_Rs, *tnfw_alpha_Rs, *tnfw_r_trunc;
} jt_lens;

/* Elliptical Sersic components (definition R).  HOST arrays of doubles, each [n]. */
typedef struct {
    int32_t n;
    const double *amp, *R_sersic, *n_sersic, *e1, *e2, *cx, *cy;
} jt_sources;

/* Step 1 ("ray-traced through the deflectors back to the source plane"):
 * beta = theta - alpha_SIE - alpha_shear - sum_j alpha_TNFW,j on caller-supplied ray positions.
 * theta_x, theta_y: device [n_rays] (in).  beta_x, beta_y: device [n_rays] (out).
 * workspace: device scratch of at least jt_ray_shoot_workspace_bytes(dtype, n_rays, n_tnfw) bytes, 16-byte aligned
 * (the derived subhalo records, written at the start of every call, and partial sums when the subhalo list is split
 * over thread blocks; may be NULL when that is 0, i.e. when n_tnfw = 0). */
JT_API size_t    jt_ray_shoot_workspace_bytes(jt_dtype dtype, int64_t n_rays, int64_t n_tnfw);
JT_API jt_status jt_ray_shoot(jt_dtype dtype, int64_t n_rays, const void *theta_x, const void *theta_y,
                       const jt_lens *lens, void *workspace, size_t workspace_bytes,
                       void *beta_x, void *beta_y, void *stream);

/* jt_ray_shoot for callers that cannot supply a workspace because they cannot allocate device memory where they call
 * this library: a callback inside a host framework that passes finished input / output buffers and forbids allocation
 * (an XLA / JAX custom call, a serving-runtime plug-in, a fixed-budget acquisition loop), or a process whose memory
 * pool already owns the device so that a cudaMalloc beside it fails, fragments or stalls every stream.  Same operation,
 * same kernels and same results as jt_ray_shoot; the scratch is a fixed array of JT_NOALLOC_SCRATCH_BYTES that is part
 * of the library image, so EVERY GPU on which the process uses libjt holds that much memory from the moment the
 * library's code is loaded there until the process exits, called or not.  The entry point and everything below it call
 * no cudaMalloc / cudaFree and no allocating library routine.
 *   - Limit: the call is accepted iff jt_ray_shoot_workspace_bytes(dtype, n_rays, n_tnfw) <= JT_NOALLOC_SCRATCH_BYTES
 *     (also returned by jt_ray_shoot_noalloc_capacity()); otherwise JT_ERR_WORKSPACE, nothing is enqueued and the
 *     outputs are untouched.  The derived records cost 224 bytes (JT_F64) / 96 bytes (JT_F32) per subhalo, and a subhalo
 *     list that is split over thread blocks adds 16 bytes per ray and chunk: BASELINE.json config 2 as a ray list
 *     (160,000 rays, 10,000 subhalos: 30.5 MB in JT_F64, 29.4 MB in JT_F32) fits, the same rays through 50,000 subhalos
 *     (49.8 MB in JT_F64) do not.  Ask the query rather than guessing.
 *   - First call on each device: looks up the array's device address (cudaGetSymbolAddress, with that device current;
 *     a failure is reported as JT_ERR_CUDA).  Make that first call outside any stream capture; later calls on the same
 *     device do no set-up.
 *   - All calls on a device share the one array.  Nothing needs to be cleared by the caller (each call rewrites what
 *     it reads and zeroes its own counters first), but two calls whose kernels can overlap on the GPU -- different
 *     streams without an ordering between them, or host threads on different streams -- race on it and both results
 *     are garbage.  Keep calls on one stream, or order them with events.  jt_ray_shoot has no such restriction.
 * theta_x, theta_y: device [n_rays] (in); beta_x, beta_y: device [n_rays] (out); lens as for jt_ray_shoot. */
#define JT_NOALLOC_SCRATCH_BYTES (32u << 20)     /* 32 MiB per GPU */
JT_API size_t    jt_ray_shoot_noalloc_capacity(void);
JT_API jt_status jt_ray_shoot_noalloc(jt_dtype dtype, int64_t n_rays, const void *theta_x, const void *theta_y,
                               const jt_lens *lens, void *beta_x, void *beta_y, void *stream);

/* Step 2 ("surface brightness of the source is calculated on the ray-traced grid"):
 * flux[i] = sum_k Sersic_k(beta_x[i], beta_y[i]) -- surface brightness, no pixel-area factor.
 * beta_x, beta_y: device [n] (in).  flux: device [n] (out). */
JT_API jt_status jt_source_brightness(jt_dtype dtype, int64_t n, const void *beta_x, const void *beta_y,
                               const jt_sources *sources, void *flux, void *stream);

/* Step 3 ("convolved by the point spread function"), definition P:
 * out[j][i] = sum_{u<ky} sum_{v<kx} K[u][v] img[j-(u-ky/2)][i-(v-kx/2)], out-of-range terms dropped
 * (zero padding, 'same' size, true convolution -- kernel flipped relative to correlation).
 * image: device [ny][nx] (in).  kernel: device [ky][kx], ky and kx odd (in); used as given, never
 * renormalised.  out: device [ny][nx].  method: DIRECT = register-blocked sum over a TMA-loaded shared-memory halo tile,
 * taps fed from the constant bank through uniform registers; when the tiles alone cannot fill the SMs, pairs of kernel
 * columns are dealt to independent thread blocks whose partial images are added through L2 in a fixed order; FFT =
 * zero-pad to P >= n+K-1, hand-written shared-memory FFTs; AUTO picks the path a time model calibrated on B200 expects
 * to be faster.  workspace: device scratch >= jt_psf_convolve_workspace_bytes(...) for the same arguments, 16-byte
 * aligned.  Non-finite pixels may reach outputs up to one pixel beyond the kernel's support (0 x inf).
 * DIRECT stages its taps in the library's one __constant__ buffer per device: calls on different streams are ordered
 * by an event the library keeps for that purpose (not while a stream is being captured into a CUDA graph: graphs
 * that contain DIRECT convolutions must not be replayed concurrently with other DIRECT calls). */
JT_API size_t    jt_psf_convolve_workspace_bytes(jt_dtype dtype, int32_t ny, int32_t nx, int32_t ky, int32_t kx,
                                          jt_conv_method method);
JT_API jt_status jt_psf_convolve(jt_dtype dtype, int32_t ny, int32_t nx, const void *image,
                          int32_t ky, int32_t kx, const void *kernel, jt_conv_method method,
                          void *workspace, size_t workspace_bytes, void *out, void *stream);

/* The same on B images with ONE kernel in one call (the batched form of the paper's convolution benchmark,
 * PAPER.md:112-114; SURVEY.md section 8(d) D4 "batch B in {1, 1024} images").  images, out: device [B][ny][nx].
 * DIRECT runs all images in one launch (B x tiles x row bands CTAs); FFT transforms the kernel once and the images
 * in groups whose spectra fit 2 GiB of workspace (four launches per group). */
JT_API size_t    jt_psf_convolve_batch_workspace_bytes(jt_dtype dtype, int64_t B, int32_t ny, int32_t nx, int32_t ky, int32_t kx,
                                                jt_conv_method method);
JT_API jt_status jt_psf_convolve_batch(jt_dtype dtype, int64_t B, int32_t ny, int32_t nx, const void *images,
                                int32_t ky, int32_t kx, const void *kernel, jt_conv_method method,
                                void *workspace, size_t workspace_bytes, void *out, void *stream);

/* Steps 1-3 fused on one system: grid G generated in registers, ray-shoot, Sersic,
 * binning B (image[j][i] = pixel_scale^2/s^2 * sum of the pixel's s*s sub-ray brightnesses, reduced
 * with warp shuffles), then PSF convolution.  Traced coordinates never leave the chip.
 * kernel: device [ky][kx] or NULL with ky = kx = 0 to skip the convolution (out = pre-PSF image).
 * out: device [ny][nx].  workspace >= jt_simulate_image_workspace_bytes(...). */
JT_API size_t    jt_simulate_image_workspace_bytes(jt_dtype dtype, const jt_grid *grid, int64_t n_tnfw,
                                            int32_t ky, int32_t kx, jt_conv_method method);
JT_API jt_status jt_simulate_image(jt_dtype dtype, const jt_grid *grid, const jt_lens *lens, const jt_sources *sources,
                            int32_t ky, int32_t kx, const void *kernel, jt_conv_method method,
                            void *workspace, size_t workspace_bytes, void *out, void *stream);

/* B independent systems sharing one grid (PAPER.md:47 training-set generation; BASELINE.json configs[3]).
 * All pointers are DEVICE arrays of the call's dtype with leading dimension B. */
typedef struct {
    const void *sie;                      /* [B][5]  theta_E, e1, e2, cx, cy */
    const void *shear;                    /* [B][2]  gamma1, gamma2 */
    int32_t n_tnfw;  const void *tnfw;    /* [B][5][n_tnfw]  rows cx, cy, Rs, alpha_Rs, r_trunc */
    int32_t n_src;   const void *sersic;  /* [B][n_src][7]   amp, R_sersic, n_sersic, e1, e2, cx, cy */
    int32_t ky, kx;  const void *psf;     /* [B][ky][kx], odd sizes; ky = kx = 0 and NULL skips the convolution */
} jt_batch_params;

/* One launch; one thread block per system keeps the pre-PSF image in shared memory and convolves it
 * in place (direct sum).  out: device [B][ny][nx].  Limits: ny*nx*sizeof(dtype) + tables must fit
 * 227 KB of shared memory (JT_ERR_UNSUPPORTED otherwise); no workspace. */
JT_API jt_status jt_simulate_batch(jt_dtype dtype, int64_t B, const jt_grid *grid, const jt_batch_params *params,
                            void *out, void *stream);

/* ---------------------------------------------------------------------------------------------------------------
 * SURVEY.md section 8(f) rows beside the hot path.  Correct-first kernels: parity with the oracle and a measured rate,
 * not tier-tuned like the subhalo sum.
 * --------------------------------------------------------------------------------------------------------------- */

/* NEXT-3 (the particle-swarm benchmark evaluates every particle's simulated image against the same
 * data).  Reading Q24: chi2[b] = sum over pixels of ((model[b] - data) / sigma)^2, log-likelihood = -chi2 / 2.
 * models: device [B][ny][nx]; data, sigma (noise rms, > 0): device [ny][nx], all of the call's dtype.
 * chi2: device [B], ALWAYS double.  One thread block per image, fixed summation order (deterministic). */
JT_API jt_status jt_chi2_batch(jt_dtype dtype, int64_t B, int32_t ny, int32_t nx, const void *models, const void *data,
                        const void *sigma, double *chi2, void *stream);
/* jt_simulate_batch with the chi^2 against (data, sigma) accumulated by the same thread block that forms the image,
 * so a swarm step returns B doubles instead of B images.  images: device [B][ny][nx] or NULL (images not wanted).
 * chi2: device [B] double.  Same limits as jt_simulate_batch. */
JT_API jt_status jt_simulate_batch_chi2(jt_dtype dtype, int64_t B, const jt_grid *grid, const jt_batch_params *params,
                                 const void *data, const void *sigma, void *images, double *chi2, void *stream);

/* NEXT-2 (the paper differentiates by autodiff; reading Q25 writes the derivatives out).  Jacobian of
 * the lens equation A = d beta / d theta = I - H at caller-supplied points, for the hot path's deflectors:
 * kappa = (H_xx + H_yy)/2, gamma1 = (H_xx - H_yy)/2, gamma2 = H_xy, mu = 1/((1 - kappa)^2 - gamma1^2 - gamma2^2).
 * theta_x, theta_y: device [n] (in); kappa, gamma1, gamma2, mu: device [n] (out), any of them may be NULL.
 * A point exactly on a deflector's centre gets no contribution from that deflector. */
JT_API jt_status jt_lensing_maps(jt_dtype dtype, int64_t n, const void *theta_x, const void *theta_y, const jt_lens *lens,
                          void *kappa, void *gamma1, void *gamma2, void *mu, void *stream);

/* NEXT-1 (PAPER.md:63-87 deflector table, :95-108 light table): typed profile lists.  A record is a type and up to
 * eight double parameters; the lists are DEVICE arrays of jt_profile (72 bytes each), whatever the call's dtype.
 *   deflectors                          p[]
 *   JT_DEFL_CONVERGENCE   kappa, cx, cy                 alpha = kappa (theta - c)
 *   JT_DEFL_SIS         (:86)           theta_E, cx, cy
 *   JT_DEFL_NFW         (:81)           Rs, alpha_Rs, cx, cy          alpha_Rs = deflection at Rs
 *   JT_DEFL_HERNQUIST   (:71)           Rs, sigma0, cx, cy            sigma0 = rho0 Rs
 *   JT_DEFL_PJAFFE      (:83)           sigma0, Ra, Rs, cx, cy
 *   JT_DEFL_SIE         (:80)           theta_E, e1, e2, cx, cy       definition S
 *   JT_DEFL_SHEAR       (:85)           gamma1, gamma2                definition H
 *   JT_DEFL_TNFW        (:87)           Rs, alpha_Rs, r_trunc, cx, cy definition T
 *   JT_DEFL_NIE         (:80)           theta_E, e1, e2, s_scale, cx, cy   definition S with a core (reading Q31)
 *   JT_DEFL_EPL         (:66-70)        theta_E, gamma, e1, e2, cx, cy     elliptical power law, 1 < gamma < 3 (Q32)
 *   JT_DEFL_MULTIPOLE   (:78)           m, a_m, phi_m, cx, cy              multipole of integer order m >= 2 (Q36)
 *   JT_DEFL_CSE         (:66)           A, s, e1, e2, cx, cy               cored steep ellipsoid, s > 0 (Q37)
 *   JT_DEFL_PJAFFE_ELLIPSE_POTENTIAL (:84)  sigma0, Ra, Rs, e1, e2, cx, cy     PJAFFE potential made elliptical (Q38)
 *   light
 *   JT_LIGHT_SERSIC_ELLIPSE   (:103)    amp, R_sersic, n_sersic, e1, e2, cx, cy      definition R
 *   JT_LIGHT_GAUSSIAN_ELLIPSE (:98-101) amp (total flux), sigma, e1, e2, cx, cy; GAUSSIAN is e1 = e2 = 0,
 *                                       MULTI_GAUSSIAN(_ELLIPSE) is several records
 * NIE (s_scale > 0), CSE and PJAFFE_ELLIPSE_POTENTIAL with q != 1: how the core / scale radii are spread over the two axes
 * is THIS library's reading (Q31, Q37, Q38) and may differ from the lenstronomy / JAXtronomy profile of the same name --
 * upstream could not be consulted; parity with upstream is unpinned for them.  DESIGN.md section 3 ("Conventions for
 * q != 1") gives the remembered differences and the parameter mapping.  At q = 1 there is no difference.
 * Formulas: DESIGN.md readings Q26-Q38.  Unknown types contribute nothing (deflector and light lists alike; a
 * zero-filled light record is type 0 = SERSIC_ELLIPSE, not "unknown").
 * Parameter domains (NOT checked on the device -- outside them the record yields IEEE inf / NaN, which then poisons every
 * ray's sum, never a fault): Rs, Ra, R_sersic, n_sersic, sigma, s (CSE) > 0; PJAFFE Ra != Rs; theta_E >= 0; s_scale >= 0;
 * 1 < gamma < 3; integer m >= 2; |e| < 1 (clamped to 0.9999 like everywhere else). */
typedef enum { JT_DEFL_CONVERGENCE = 0, JT_DEFL_SIS = 1, JT_DEFL_NFW = 2, JT_DEFL_HERNQUIST = 3, JT_DEFL_PJAFFE = 4,
               JT_DEFL_SIE = 5, JT_DEFL_SHEAR = 6, JT_DEFL_TNFW = 7, JT_DEFL_NIE = 8, JT_DEFL_EPL = 9,
               JT_DEFL_MULTIPOLE = 10, JT_DEFL_CSE = 11,
               JT_DEFL_PJAFFE_ELLIPSE_POTENTIAL = 12 } jt_deflector_type;
typedef enum { JT_LIGHT_SERSIC_ELLIPSE = 0, JT_LIGHT_GAUSSIAN_ELLIPSE = 1 } jt_light_type;
typedef struct { int32_t type; int32_t reserved; double p[8]; } jt_profile;
/* beta = theta - sum of the n_def deflectors.  theta, beta: device [n]; deflectors: device [n_def]. */
JT_API jt_status jt_ray_shoot_profiles(jt_dtype dtype, int64_t n, const void *theta_x, const void *theta_y, int64_t n_def,
                                const jt_profile *deflectors, void *beta_x, void *beta_y, void *stream);
/* flux[i] = sum of the n_comp light components at (beta_x[i], beta_y[i]) (surface brightness). */
JT_API jt_status jt_light_profiles(jt_dtype dtype, int64_t n, const void *beta_x, const void *beta_y, int64_t n_comp,
                            const jt_profile *components, void *flux, void *stream);

/* CORE_SERSIC (reading Q33): params (HOST, 10 doubles) = amp, R_sersic, n_sersic, Rb, gamma, alpha, e1, e2,
 * cx, cy;  I = amp (1 + (Rb/R)^alpha)^(gamma/alpha) exp(-b_n [((R^alpha + Rb^alpha)/R_sersic^alpha)^(1/(alpha n)) - 1]),
 * R the product-averaged radius of definition R.  beta_x, beta_y, flux: device [n]. */
JT_API jt_status jt_light_core_sersic(jt_dtype dtype, int64_t n, const void *beta_x, const void *beta_y, const double *params,
                               void *flux, void *stream);
/* SHAPELETS (n_max = 6 and 10; reading Q34): Cartesian Gauss-Hermite basis of scale beta about
 * (cx, cy); coef: device [(n_max+1)(n_max+2)/2] of the call's dtype, ordered by N = n1 + n2 ascending and, within N, by
 * n2 = 0 ... N;  flux[i] = sum_k coef[k] B_n1(u) B_n2(v) / beta.  n_max <= JT_MAX_SHAPELET_ORDER. */
#define JT_MAX_SHAPELET_ORDER 12
JT_API jt_status jt_light_shapelets(jt_dtype dtype, int64_t n, const void *beta_x, const void *beta_y, int32_t n_max, double beta,
                             double cx, double cy, const void *coef, void *flux, void *stream);

/* NEXT-4 (not in the paper): jt_simulate_image with the convolution done at RAY resolution --
 * the unbinned ray image [ny s][nx s] (each ray carrying pixel_scale^2/s^2 of surface brightness) is convolved with a
 * PSF sampled on the ray grid, kernel_fine: device [ky][kx] (odd sizes, in rays), and binned s x s afterwards.
 * out: device [ny][nx].  workspace >= jt_simulate_image_supersampled_psf_workspace_bytes(...). */
JT_API size_t    jt_simulate_image_supersampled_psf_workspace_bytes(jt_dtype dtype, const jt_grid *grid, int64_t n_tnfw, int32_t ky,
                                                             int32_t kx, jt_conv_method method);
JT_API jt_status jt_simulate_image_supersampled_psf(jt_dtype dtype, const jt_grid *grid, const jt_lens *lens,
                                             const jt_sources *sources, int32_t ky, int32_t kx, const void *kernel_fine,
                                             jt_conv_method method, void *workspace, size_t workspace_bytes, void *out,
                                             void *stream);

/* Read-only launch plans (host only: no device is touched, nothing is enqueued).  The library picks among several launch
 * shapes per call from time models; these queries say which one a call with the same arguments takes, so that a test can
 * assert the path it is named after and a user can see what AUTO resolves to.
 * jt_psf_convolve_plan: `image` may be NULL (then its address is taken to be 16-byte aligned).
 *   method    JT_CONV_DIRECT / JT_CONV_FFT -- what the call runs (AUTO resolved)
 *   path      JT_PATH_CONV_SMALL  one launch, taps + halo tile staged by the CTA (tiny kernels on small single images)
 *             JT_PATH_CONV_TILE   tap kernel + constant-bank sweep kernel (k_conv_ur); then: tma = 1 halo tile by TMA,
 *                                 0 plain loads (image address or row pitch not 16-byte aligned, tile side > 256);
 *                                 z_split > 1 = kernel-column pairs dealt to z_split CTAs per tile, partial images added
 *                                 through L2; row_bands > 1 = the 60 KB constant bank holds only a band of kernel rows,
 *                                 one sweep launch per band
 *             JT_PATH_CONV_FFT    hand-written FFT (pad_y x pad_x padded transform)
 *   oy, warps rows per thread and warps per CTA of the tile kernel; est_us the time model's estimate. */
typedef enum { JT_PATH_CONV_SMALL = 0, JT_PATH_CONV_TILE = 1, JT_PATH_CONV_FFT = 2 } jt_conv_path;
typedef struct {
    int32_t method, path, tma, z_split, row_bands, oy, warps, pad_y, pad_x, reserved;
    double  est_us;
} jt_conv_plan;
JT_API jt_status jt_psf_convolve_plan(jt_dtype dtype, int64_t B, int32_t ny, int32_t nx, int32_t ky, int32_t kx,
                               jt_conv_method method, const void *image, jt_conv_plan *plan);
/* Ray-tracing kernel (k_trace) of jt_simulate_image (grid != NULL) or jt_ray_shoot (grid == NULL, n_rays used):
 *   rays_per_thread  R (grid mode: R = s means one pixel row per thread, the launch-latency shape for next to no subhalos)
 *   threads          per CTA;  wide = 1: CTA-wide ray tiles binned through shared memory (s does not divide 32)
 *   n_chunks         > 1: the subhalo list is split over CTAs, partial sums meet in the workspace;  chunk_len subhalos each
 *   n_ctas           ray tiles x chunks;  tile_recs = subhalo records per shared-memory stage of the TMA ring */
typedef struct {
    int32_t rays_per_thread, threads, wide, n_chunks, tile_recs, reserved;
    int64_t chunk_len, n_ctas;
} jt_trace_plan;
JT_API jt_status jt_trace_plan_query(jt_dtype dtype, const jt_grid *grid, int64_t n_rays, int64_t n_tnfw, jt_trace_plan *plan);

/* Measurement aid (bench.py's roofline leg).  jt_profile_enable(1) makes every following
 * jt_simulate_image call on this host thread record CUDA events on its stream before the ray-tracing kernel, between it
 * and the convolution, and after the convolution, and copy the kernel's JT_N_TIERS tier counters (48 bytes) to a pinned host
 * buffer the library owns (event records and one cudaMemcpyAsync: no synchronisation, nothing keeps pointing into the
 * caller's workspace).  jt_profile_read waits for the events of the LAST such call and returns the two intervals in
 * milliseconds (conv_ms = 0 when the call had no PSF).  JT_ERR_INVALID_VALUE when profiling is off or no call has been
 * recorded.  jt_profile_enable(0) destroys the events and frees the buffer. */
JT_API jt_status jt_profile_enable(int on);
JT_API jt_status jt_profile_read(float *trace_ms, float *conv_ms);
/* counts[JT_N_TIERS] (host) receives, for the LAST profiled jt_simulate_image call, the number of (warp, subhalo-record)
 * pairs evaluated by each form of definition T: the far-far series at its three lengths (longest first), the far form,
 * the mid form and the per-ray cold path.  Waits for that call's counter copy (an event), not
 * for the device. */
#define JT_N_TIERS 6
JT_API jt_status jt_profile_tiers(uint64_t *counts);

/* Number of CUDA kernels this library has launched from the calling host thread since it was loaded
 * (bench.py's "gpu_launches" claim; memsets and event records are not counted). */
JT_API uint64_t jt_kernel_launches(void);

JT_API const char *jt_status_string(jt_status s);
JT_API int         jt_last_cuda_error(void);     /* cudaError_t of the last JT_ERR_CUDA on this thread, else 0 */
JT_API int         jt_version(void);             /* JT_VERSION */

#ifdef __cplusplus
}
#endif
#endif /* JT_H */
