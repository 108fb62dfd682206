/* bang.h -- C ABI of libbang: the batched likelihood of Rigamonti et al. 2022 (arXiv 2205.06819) on one B200.
 *
 * The two calls of the paper's problem statement:
 *     bang_model_maps(theta[B], grid, psf) -> B / v_los / sigma_los / M/L maps
 *     bang_loglike   (theta[B], data, err, mask) -> logL[B]
 * plus context management.  No torch types cross this boundary: plain pointers and sizes.  Every pointer
 * argument says whether it is HOST or DEVICE memory.  All device work is enqueued on the CUDA stream given
 * at bang_create(); calls are asynchronous with respect to the host unless stated otherwise, and results
 * are valid once the caller has synchronised that stream.  There is no CPU fallback: without a CUDA device
 * every call that needs one returns BANG_ECUDA.
 *
 * Citations are PAPER.md:<line> (section / equation); "reading X" refers to DESIGN.md, "Readings".
 *
 * The model (sec. 2.1-2.4, lines 58-193; Table 1 at 168-183):
 *   sky grid -> translate by (x0,y0), rotate by P.A., deproject by the inclination i   (sec. 2.1, :60-70)
 *   Hernquist bulge:  Sigma_b(R) eq. 4-5 (:96-101);  Sigma_b sigma_b^2 (R) = l.o.s. integral of rho_b v_r^2,
 *                     eq. 6 first form (:105), by an N_J-node quadrature (readings B, C)
 *   exponential discs j=1,2:  Sigma_d,j eq. 7-8 (:117-123)
 *   circular speed:   v_c^2 = bulge eq. 2 (:84) + discs eq. 9 (:127, reading D) + halo (eq. 2 form or NFW,
 *                     reading H), eq. 10 (:136-139)
 *   disc kinematics:  v_d,j = -k_j sin i cos(phi) v_c  eq. 11;  sigma_d,j^2 = (1-k_j^2) v_c^2 / 3  eq. 12 (:141-147)
 *   observables:      B_tot eq. 13, v_los eq. 14, sigma_los eq. 15 (:159-189), <L/M> eq. 19 (:233)
 *   PSF:              normalised Gaussian, eq. 21 (:265-270, :296), on the x s supersampled grid (App. A, :528),
 *                     applied to B_tot, v_los, sigma_los and <L/M> separately (reading G); then the mean over the
 *                     s x s sub-cells of each data pixel, and M/L = 1/<L/M> (fn 10, :259)
 *   likelihood:       eq. 18 (:225-229): sum over the four observables and the unmasked pixels of
 *                     -1/2 [ (d-m)^2/e^2 + ln(2 pi e^2) ]   (reading L)
 */
#ifndef BANG_H
#define BANG_H

#ifdef __cplusplus
extern "C" {
#endif

#define BANG_NTHETA 17

/* theta layout, Table 1 order; units as in the BASELINE.json prior boxes:
 *  0 x0 [arcsec]   1 y0 [arcsec]   2 P.A. [deg, counter-clockwise from +x]   3 i [deg]
 *  4 log10 M_b [Msun]   5 R_b [kpc]   6 log10 M_d1   7 R_d1 [kpc]   8 log10 M_d2   9 R_d2 [kpc]
 * 10 log10 M_h (HERNQUIST halo) or log10 M200 (NFW)   11 R_h [kpc] (HERNQUIST) or concentration c (NFW)
 * 12 (M/L)_b   13 (M/L)_d1   14 (M/L)_d2   15 k_1   16 k_2
 * Entries of components absent from bang_model.components are ignored. */

/* error codes (0 = success) */
#define BANG_OK        0
#define BANG_EINVAL   (-1)  /* bad argument, unsupported configuration, or invalid data (err <= 0 on a used pixel) */
#define BANG_ENOMEM   (-2)  /* host or device allocation failed */
#define BANG_ECUDA    (-3)  /* CUDA runtime error (no device, launch failure, ...) */
#define BANG_ENODATA  (-4)  /* bang_loglike before bang_set_data */

/* bang_model.components bits */
#define BANG_BULGE 1u
#define BANG_DISC1 2u
#define BANG_DISC2 4u
#define BANG_HALO  8u

#define BANG_BULGE_HERNQUIST 0   /* the paper's default, eq. 1-6 */
#define BANG_BULGE_JAFFE     1   /* Appendix B: eq. B1, B2, B4; Sigma_b sigma_b^2 = the N_J-node l.o.s.
                                    integral of eq. B1 x B3 (B3 as corrected by reading J), which eq. B5 pins */
#define BANG_HALO_HERNQUIST  0   /* the paper's halo: eq. 2 with (M_h, R_h) */
#define BANG_HALO_NFW        1   /* BASELINE.json configs 2-5: (log10 M200, c), H0 = 70 km/s/Mpc (reading H) */
#define BANG_PSF_FIELDS 0        /* the paper: eq. 21 applied to B, v_los, sigma_los, <L/M> separately (reading G) */
#define BANG_PSF_FLUX   1        /* variant (reading G'): PSF + rebin applied to the light moments B, B v, B (sigma^2 + v^2)
                                    and to the mass surface density; v = M1/M0, sigma^2 = M2/M0 - v^2, M/L = M3/M0.
                                    bang_model_fine then returns those four moment fields.  Runs in the fused kernel (its
                                    own instantiation: the four moments of a pixel meet by warp shuffle when its row
                                    completes) */
#define BANG_POTENTIAL_SELF  0    /* the paper: the bulge's dispersion in its own potential, eq. 6 */
#define BANG_POTENTIAL_TOTAL 1    /* variant (reading U'; PAPER.md:417-419 names the approximation above as the model's first
                                    limitation): Sigma_b sigma_b^2 gains I_ext(R) = 2 int_R^inf rho_b v_ext^2 sqrt(x^2-R^2)/x dx,
                                    v_ext^2 = discs (eq. 9) + halo, by the same N_J-node rule -- the isotropic Jeans
                                    equation in the total potential of eq. 10.  Tabulated per theta inside the fused kernel */
#define BANG_FP32 0              /* fp32 model arithmetic; residuals and logL accumulation in fp64 */
#define BANG_FP64 1              /* everything in fp64 */

typedef struct bang_ctx bang_ctx;   /* opaque, library-owned */

typedef struct {
    int    nx, ny;         /* data pixels along x (fast axis) and y; maps are row-major [ny][nx], row index grows with +y */
    double pix_arcsec;     /* pixel scale [arcsec] */
    int    supersample;    /* s >= 1: the model is evaluated on an s x s sub-grid of every pixel (App. A) */
    double dist_mpc;       /* distance [Mpc]; kpc per arcsec = dist_mpc * 4.84813681109536e-3 */
} bang_grid;

typedef struct {
    double sigma_pix;      /* Gaussian PSF sigma in DATA pixels (>= 0; 0 = no PSF) */
    double trunc_nsigma;   /* support half-width in sigma (the paper's 3); r_k = ceil(trunc*sigma*s) fine cells */
} bang_psf;

typedef struct {
    unsigned components;   /* BANG_BULGE | BANG_DISC1 | BANG_DISC2 | BANG_HALO; at least one luminous component */
    int bulge_profile;     /* BANG_BULGE_HERNQUIST or BANG_BULGE_JAFFE */
    int halo_profile;      /* BANG_HALO_HERNQUIST or BANG_HALO_NFW */
    int jeans_nodes;       /* N_J >= 1: nodes of the Gauss-Legendre rule for the bulge Jeans l.o.s. integral (reading B) */
    int precision;         /* BANG_FP32 or BANG_FP64 */
    int psf_weighting;     /* BANG_PSF_FIELDS (the paper) or BANG_PSF_FLUX */
    int bulge_potential;   /* BANG_POTENTIAL_SELF (the paper) or BANG_POTENTIAL_TOTAL */
} bang_model;

/* Create a context on CUDA device `device`.  `cuda_stream` is a cudaStream_t (NULL = the legacy default stream) on
 * which every later call enqueues its work.  Builds the scale-free radial tables (Hernquist Sigma~(s), the N_J-node
 * Jeans integral I~(s), the Freeman-disc function F(y)) once, on the device.  Synchronises the
 * stream before returning.  grid/psf/model are HOST pointers, copied.  On failure *out is NULL.
 * BANG_EINVAL: nx,ny < 1, s < 1 or s > 4, pix/dist <= 0, sigma < 0, no luminous component, unknown profile or
 * precision, a PSF whose footprint (2 r_k + s)/s exceeds 13 data pixels, or a row too wide for one CTA (nx > 512 in
 * fp32 mode, nx > 256 in fp64 mode) or for shared memory.
 * The calling thread's current CUDA device is left as it was found, here and in every other call.
 * The launch shape is derived from the grid alone; a development build (-DBANG_TUNING) can override it from the
 * environment (BANG_P, BANG_THREADS, BANG_CTAS, BANG_VERBOSE) -- the default build reads no environment variable. */
int bang_create(bang_ctx **out, const bang_grid *grid, const bang_psf *psf, const bang_model *model,
                int device, void *cuda_stream);

/* Load the observed maps ("allocated and loaded once").  DEVICE pointers, each [4][ny][nx], map order
 * 0 B [Lsun/pc^2]  1 v_los [km/s]  2 sigma_los [km/s]  3 M/L [Msun/Lsun]; mask 1 = use the pixel, 0 = ignore it (one
 * mask per observable, reading M).  The library copies what it needs into the context (the caller keeps ownership and
 * may free the buffers after the call, which synchronises the stream).  Values at masked pixels are never read into
 * the likelihood (they may be NaN).  BANG_EINVAL if any used pixel has err <= 0 or a non-finite data/err value; the
 * context then keeps its previous data, if any. */
int bang_set_data(bang_ctx *ctx, const double *data_dev, const double *err_dev, const unsigned char *mask_dev);

/* Model maps for a batch: theta_dev DEVICE [B][17] doubles; maps_dev DEVICE [B][4][ny][nx], float if the context is
 * BANG_FP32, double if BANG_FP64 (map order as above; B in linear units).  theta outside the model's domain (R <= 0,
 * M/L <= 0, |k| > 1, |i| >= 90 deg, non-finite entries of a present component) is not an error: its maps are NaN.
 * The library's domain is the model's, not its tables': a theta whose radii leave the tabulated ranges of the fused
 * kernel (more than 32 octaves of r^2 on the grid, R/R_b outside [2^-22, 2^18), or i > 89.1 deg in BANG_FP32 mode, where
 * fp32 coordinates no longer carry r) is evaluated by a second, direct kernel (eq. 4-5 in closed form, eq. 6 by the
 * N_J-node rule, eq. 10 term by term, fp64 geometry; ~1e3 times slower per theta), launched after the fused one in every
 * call and empty for any theta of a sensible prior box.  Only on a grid whose row does not fit that kernel's shared
 * memory (4 (nx s + 2 r_k) + 4 NACC nx values) are such theta reported as out of domain.  B = 0 is a no-op.
 * Asynchronous. */
int bang_model_maps(bang_ctx *ctx, const double *theta_dev, int B, void *maps_dev);

/* Un-convolved model on the supersampled grid, the intermediate of the path before the PSF (App. A Alg. 1 line 3,
 * PAPER.md:537): fine_dev DEVICE [B][4][ny*s + 2 r_k][nx*s + 2 r_k] (float or double as above) = B_tot, v_los, sigma_los,
 * <L/M> at the fine-cell centres, including the PSF halo of r_k cells.  For parity checks of steps a0-a3.  Asynchronous. */
int bang_model_fine(bang_ctx *ctx, const double *theta_dev, int B, void *fine_dev);

/* log-likelihood (eq. 18) for a batch: theta_dev DEVICE [B][17]; logL_dev DEVICE [B] doubles.  Out-of-domain theta
 * gives -inf (a nested sampler treats it as zero likelihood).  BANG_ENODATA before bang_set_data.
 * Asynchronous. */
int bang_loglike(bang_ctx *ctx, const double *theta_dev, int B, double *logL_dev);

/* bang_loglike for callers that cannot allocate (code under CUDA graph capture, tight serving loops, harnesses that forbid
 * cudaMalloc): same arguments, same kernels, same results, but NO allocation on its path -- no cudaMalloc, cudaFree or
 * allocating library routine.  bang_loglike keeps the list through which the fused kernel hands theta outside its tabulated
 * ranges to the direct-path kernel in a buffer that grows with B; here that list lives in a file-scope static __device__
 * array of BANG_NOALLOC_MAX_B entries (256 KiB + 256 B, held by every GPU that loads the library until the process exits;
 * its device address is taken with cudaGetSymbolAddress at bang_create, once per device).  B > BANG_NOALLOC_MAX_B returns
 * BANG_EINVAL with a message in bang_last_error (split the batch, or call bang_loglike).  theta_dev, logL_dev: DEVICE, as
 * for bang_loglike; asynchronous on the context's stream.  The array is ONE per device, shared by every call and every
 * context, and keeps the last call's contents (the call clears the counters it needs at zero): calls that overlap on the
 * GPU -- two streams, two contexts on one device -- race on it; calls ordered on one stream do not. */
#define BANG_NOALLOC_MAX_B 65536
int bang_loglike_noalloc(bang_ctx *ctx, const double *theta_dev, int B, double *logL_dev);

/* The replacement step of nested sampling on the device (the worst live point is
 * replaced by one of higher likelihood found by MCMC): K constrained random walks of `steps` Metropolis steps in lock-step,
 * each step = proposal kernel -> bang_loglike on the K proposals -> accept kernel, with walkers, proposals and their
 * parameter vectors resident in device memory throughout (one small host<->device exchange per CALL, none per step).
 * Walkers live in the unit cube u in [0,1]^d (uniform prior); theta = theta0 with theta[free_idx[j]] = lo[j] + (hi[j] -
 * lo[j]) u[j].  Walker k belongs to group[k] in [0, n_groups) -- one group per independent run or retire batch, so that
 * several of them share one call and fill the GPU: a proposal is u + scale[g] (2.38/sqrt d) chol[g] z, z ~ N(0, 1)^d
 * (Philox4x32-10, counter = (walker, step, draw), key = seed), accepted iff it stays in the cube and its logL exceeds
 * Lstar[k] (out-of-domain theta: logL = -inf, never accepted).
 * HOST: free_idx[d], lo[d], hi[d], theta0[17], chol[n_groups][d][d] (lower triangular, row-major), scale[n_groups],
 * n_accept[n_groups] (out: accepted proposals per group).  DEVICE: u [K][d] and logL [K] (in/out: the walkers and their
 * likelihoods), Lstar [K], group [K].  d <= 17.  Synchronises the stream before returning.  BANG_ENODATA before
 * bang_set_data; BANG_EINVAL on bad sizes or NULL pointers. */
int bang_ns_walk(bang_ctx *ctx, int K, int d, const int *free_idx_host, const double *lo_host, const double *hi_host,
                 const double *theta0_host, double *u_dev, double *logL_dev, const double *Lstar_dev, const int *group_dev,
                 int n_groups, const double *chol_host, const double *scale_host, int steps, unsigned long long seed,
                 int *n_accept_host);

/* Same calls with HOST buffers: the library stages theta in pinned memory, copies it to the device, runs, and copies
 * the result back; synchronises the stream before returning.  logL_host [B] doubles; maps_host as maps_dev above. */
int bang_loglike_host(bang_ctx *ctx, const double *theta_host, int B, double *logL_host);
int bang_model_maps_host(bang_ctx *ctx, const double *theta_host, int B, void *maps_host);

/* Geometry the context derived: r_k (PSF half-width in fine cells), fine grid size n*s + 2 r_k.  HOST out pointers, any may be NULL. */
int bang_get_geometry(const bang_ctx *ctx, int *r_k, int *nfx, int *nfy);

/* How many kernels the library has launched on this context since creation (for bench.py's gpu_launches). */
long long bang_launch_count(const bang_ctx *ctx);

/* Measurement aid, not part of the path: times dependency-free chains of FFMA,
 * MUFU.EX2 and DFMA that fill the whole device and writes the sustained thread-level instruction rates [instr/s] to the
 * HOST array out[3] = {fp32 FMA, MUFU, fp64 FMA}.  These are the measured counterparts of the roofline denominators
 * that DESIGN.md derives from unit counts and clocks (128 / 16 / 64 lanes per SM per clock).  Uses the context's device
 * and stream; synchronises.  BANG_EINVAL on NULL arguments, BANG_ECUDA on a CUDA failure. */
int bang_probe_peaks(bang_ctx *ctx, double *out_host);

/* Pre-step: resolved M/L maps from two photometric bands through a colour-M/L relation,
 * eq. 20 with the error model of App. C:
 *   log10 (M/L) = a + b (m_beta - m_gamma),   d log10(M/L) = sqrt(b^2 (dm_beta^2 + dm_gamma^2) + sigma_alpha^2),
 *   d(M/L) = ln 10 (M/L) d log10(M/L).   (The paper's test case: a = -0.70, b = 0.89, sigma_alpha = 0.07.)
 * All arrays are DEVICE pointers of n doubles (magnitudes and their errors in, M/L and its error out; out may alias
 * nothing).  Non-finite inputs give non-finite outputs for that pixel.  No context: runs on `device`, enqueued on
 * `cuda_stream` (asynchronous).  BANG_EINVAL on NULL pointers, BANG_ECUDA on a CUDA failure. */
int bang_ml_from_colour(const double *m_beta_dev, const double *m_gamma_dev, const double *dm_beta_dev,
                        const double *dm_gamma_dev, long long n, double a, double b, double sigma_alpha,
                        double *ml_dev, double *ml_err_dev, int device, void *cuda_stream);

void bang_destroy(bang_ctx *ctx);   /* NULL is allowed; synchronises the stream, frees everything the context owns */

const char *bang_strerror(int code);               /* static string */
const char *bang_last_error(const bang_ctx *ctx);  /* detail of the last failure on this context ("" if none); owned by ctx */

#ifdef __cplusplus
}
#endif
#endif /* BANG_H */
