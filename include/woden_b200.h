/* woden_b200.h -- C ABI of libwoden_b200.so: direct measurement-equation visibility
 * prediction (the WODEN hot path of Line et al. 2020, arXiv:2005.09316) on one B200.
 *
 * Citations are PAPER.md line numbers (text of the paper) and DESIGN.md readings (G1-G14).
 *
 * What every predict call computes, for each baseline b, time step t and channel f
 * (Eq 9 / Eq 11, primary beam B == 1, :125):
 *
 *   V(b,t,f) = sum_j  S_j(nu_f) * xi_j(u,v) * exp(-2 pi i (u l_j + v m_j + w (n_j - 1)))
 *
 *   (u,v,w)  = (u_m,v_m,w_m)[t][b] * nu_f / c      wavelengths; "u,v,w only differ in
 *                                                  frequency by a scaling factor" (:161)
 *   n_j      = sqrt(1 - l_j^2 - m_j^2)             (:115)
 *   S_j(nu)  = s0_j * (nu / ref_freq)^alpha_j      single spectral index per source (:169, :365)
 *   xi_j     = 1                                                         point source
 *            = exp(-pi^2/(4 ln 2) (kx^2 maj^2 + ky^2 min^2)),
 *              kx = cos(pa) v + sin(pa) u,  ky = -sin(pa) v + cos(pa) u   Gaussian, Eq 12-14 (:141-146)
 *            = sum_q coeff_q i^(n1_q+n2_q) h_{n1_q}(beta1 K kx') h_{n2_q}(beta2 K ky'),
 *              K = pi / sqrt(2 ln 2), kx', ky' as above from (u',v')     shapelet, Eq 15-17 (:150-157)
 *              h_p(x) = H_p(x) exp(-x^2/2) / sqrt(2^p p!)                 Eq 1/3 (:51, :60), reading G2
 *              (u',v') = M_j (u,v,w)^T, or (u,v) when uv_basis == NULL    (:157), reading G4
 *
 * Conventions (G6, G7): l, m direction cosines; angles in radians; maj/min are FWHM;
 * pa is measured from North through East; c = 299792458 m/s; flux in Jy.  A shapelet with the
 * single coefficient (0,0) = 1 and beta1 = maj, beta2 = min IS the Gaussian (:159).
 *
 * Memory: pointers marked DEVICE must be device memory on the context's GPU (e.g. a torch
 * tensor's data_ptr()); pointers marked HOST are ordinary host memory read before the call
 * returns.  The library never frees or keeps caller pointers after the call's work has run.
 * Device calls only enqueue work on `cuda_stream` (a cudaStream_t, NULL = legacy default
 * stream) and return without synchronising; internal scratch belongs to the context, so one
 * context serves one stream at a time (a context's next call may go to another stream only after
 * its previous call's work has finished).  Different contexts on one GPU are independent and may be
 * driven from different host threads and streams: the one resource they share, the constant bank the
 * channel-walking kernels read their component blocks from, is handed from call to call by the
 * library (walking calls on one device run one after another on the GPU, whatever their streams).
 *
 * Output layout: complex64 interleaved (re, im), vis[((t * n_freqs) + f) * n_baselines + b].
 *
 * Phase range: the phase u l + v m + w (n - 1) is formed in FP64 and reduced to its fraction to
 * 2^-23 turn before the FP32 sin/cos, on every path (general, channel-walking, shapelets), as
 * long as sqrt(2) |b| nu / c < 2^28 wavelengths for every baseline b = (u_m, v_m, w_m) and channel
 * (a bound on the phase for l^2 + m^2 < 1).  The point / Gaussian kernels count baselines beyond
 * that range for woden_check() (WODEN_ERR_DATA); their output is then undefined.
 *
 * There is no CPU fallback anywhere: without a CUDA device every entry point that needs one
 * returns WODEN_ERR_CUDA.
 */
#ifndef WODEN_B200_H
#define WODEN_B200_H

#ifdef __cplusplus
extern "C" {
#endif

#define WODEN_OK                 0
#define WODEN_ERR_NULL          -1   /* a required pointer is NULL                              */
#define WODEN_ERR_DIM           -2   /* a size is non-positive / inconsistent / too large       */
#define WODEN_ERR_ORDER         -3   /* p_max outside 0..WODEN_MAX_ORDER                        */
#define WODEN_ERR_CUDA          -4   /* CUDA allocation / launch / copy failed (woden_last_error) */
#define WODEN_ERR_UNIMPLEMENTED -5
#define WODEN_ERR_DATA          -6   /* woden_check(): a device-side precondition was violated  */
#define WODEN_ERR_STATIC_LIMIT  -7   /* woden_truncate_select_static(): n beyond the built-in scratch */

#define WODEN_MAX_ORDER 100          /* largest shapelet order n1 + n2 (paper uses <= 86, :183) */

typedef struct woden_ctx woden_ctx;  /* owns internal device scratch only */

/* Create / destroy a context bound to CUDA device `cuda_device`. */
int woden_create(woden_ctx **ctx, int cuda_device);
int woden_destroy(woden_ctx *ctx);

/* Static description of a status code; woden_last_error() adds the CUDA error string of the
 * last WODEN_ERR_CUDA on this context ("" if none).  Both return pointers owned by the library. */
const char *woden_strerror(int status);
const char *woden_last_error(const woden_ctx *ctx);

/* Number of CUDA kernels this library has launched since it was loaded (all contexts; copies and
 * memsets are not counted).  Host-side counter, not thread-safe against concurrent callers. */
unsigned long long woden_kernel_launches(void);

/* Synchronises the context's last stream and reports device-side precondition violations
 * counted since the last check (l^2+m^2 >= 1, non-finite parameters, a flux s0 (nu/ref)^alpha that
 * is not finite in FP32 at any channel, negative widths, beta <= 0, shapelet orders above p_max,
 * baselines beyond the phase range above): WODEN_OK or WODEN_ERR_DATA.  Not on the hot path. */
int woden_check(woden_ctx *ctx);

/* Algorithm selection (measurement / testing).  Default WODEN_PATH_AUTO.
 *   AUTO    : channel-walking fast path when freqs_hz is an arithmetic progression (to 1e-9 of
 *             the step) of >= 8 channels whose step is at most 1/64 of the lowest frequency of
 *             the list continued to a multiple of 32 channels (so that a 16-channel chain spans
 *             at most +-12.5 % in frequency); otherwise the general path
 *   GENERAL : always one sin/cos (and one exp2 for Gaussians) per component x visibility
 * Both meet the same parity tolerance and the same phase range. */
#define WODEN_PATH_AUTO    0
#define WODEN_PATH_GENERAL 1
int woden_set_path(woden_ctx *ctx, int path);
/* Which point / Gaussian kernel family the last woden_predict_points / _gaussians call on this
 * context launched: WODEN_PATH_GENERAL, WODEN_PATH_WALKING, or WODEN_PATH_NONE (n == 0 / no call
 * yet).  For tests and reports; never changes behaviour. */
#define WODEN_PATH_NONE    -1
#define WODEN_PATH_WALKING 2
int woden_last_path(const woden_ctx *ctx);

/* Shapelet engine selection (measurement / testing).  Default WODEN_SHAPELET_AUTO.
 *   REGISTER : FP32 register path, one FFMA per coefficient (predict_shapelets.cu)
 *   TENSOR   : the coefficient sum of each shapelet as a batched matrix product on the tensor cores
 *              (tcgen05, FP16 hi + lo operands, FP32 accumulation in TMEM; predict_shapelets_mma.cu)
 *   AUTO     : whichever measured faster for the order
 * All meet the same parity tolerance. */
#define WODEN_SHAPELET_AUTO     0
#define WODEN_SHAPELET_REGISTER 1
#define WODEN_SHAPELET_TENSOR   2
int woden_set_shapelet_path(woden_ctx *ctx, int path);
/* Which shapelet engine the last woden_predict_shapelets call on this context launched, and at which
 * compile-time order bucket (the kernels are instantiated for orders 4, 8, 12, 16, 20, 24, 32, 40, 48, 60, 72,
 * 86, 100; a call runs the smallest bucket >= p_max): WODEN_SHAPELET_REGISTER, WODEN_SHAPELET_REGISTER_SPARSE
 * (the register engine's variant that skips empty 4-coefficient chunks of truncated models,
 * PAPER.md:271-284), WODEN_SHAPELET_TENSOR, or WODEN_PATH_NONE (n == 0 / no call yet; bucket -1).
 * For tests and reports; never changes behaviour. */
#define WODEN_SHAPELET_REGISTER_SPARSE 3
int woden_last_shapelet_path(const woden_ctx *ctx);
int woden_last_shapelet_bucket(const woden_ctx *ctx);

/* Baseline coordinates and channels ("array layout and observation parameters"). */
typedef struct {
    int n_baselines, n_times, n_freqs;
    const double *u_m, *v_m, *w_m;  /* DEVICE [n_times][n_baselines], metres, phase-centre frame */
    const double *freqs_hz;         /* HOST   [n_freqs], any spacing, each > 0                    */
} woden_uvw;

/* Eq 9.  n components; l, m, s0_jy, alpha: DEVICE [n].
 * vis: DEVICE complex64 [n_times][n_freqs][n_baselines].  accumulate = 0 overwrites vis,
 * 1 adds into it.  n == 0: zero-fill (accumulate = 0) or no-op (accumulate = 1). */
int woden_predict_points(woden_ctx *ctx, const woden_uvw *uvw, int n,
                         const double *l, const double *m,
                         const double *s0_jy, const double *alpha, double ref_freq_hz,
                         float *vis, int accumulate, void *cuda_stream);

/* Eq 11 with the Gaussian envelope of Eq 12-14.
 * maj_fwhm_rad, min_fwhm_rad (>= 0; both 0 is a point source, reading G13), pa_rad: DEVICE [n]. */
int woden_predict_gaussians(woden_ctx *ctx, const woden_uvw *uvw, int n,
                            const double *l, const double *m,
                            const double *s0_jy, const double *alpha, double ref_freq_hz,
                            const double *maj_fwhm_rad, const double *min_fwhm_rad,
                            const double *pa_rad,
                            float *vis, int accumulate, void *cuda_stream);

/* Eq 11 with the shapelet envelope of Eq 15-17.
 * beta1_rad, beta2_rad (> 0), pa_rad: DEVICE [n].
 * uv_basis: DEVICE [n][6] row-major 2x3 M_j, or NULL for (u',v') = (u,v) (reading G4).
 * coeff_offset: DEVICE int [n+1], CSR offsets into n1/n2/coeff, non-decreasing from 0;
 * n_coeff = coeff_offset[n] is passed explicitly so the call never reads device memory.
 * n1, n2: DEVICE int [n_coeff], n1, n2 >= 0 and n1 + n2 <= p_max (the paper's p_max, Eq 6 /
 * Eq 15; reading G5); coeff: DEVICE [n_coeff], already divided by the
 * component's integrated flux (:157).  Repeated (n1,n2) pairs add; missing pairs are zero
 * (truncated models).  0 <= p_max <= WODEN_MAX_ORDER. */
int woden_predict_shapelets(woden_ctx *ctx, const woden_uvw *uvw, int n,
                            const double *l, const double *m,
                            const double *s0_jy, const double *alpha, double ref_freq_hz,
                            const double *beta1_rad, const double *beta2_rad, const double *pa_rad,
                            const double *uv_basis,
                            const int *coeff_offset, int n_coeff, int p_max,
                            const int *n1, const int *n2, const double *coeff,
                            float *vis, int accumulate, void *cuda_stream);

/* Whole-sky convenience call on HOST buffers (the call a user with a sky model in host memory
 * makes; bench.py's end-to-end number).  Every pointer inside the structs and `vis_host` is
 * HOST memory (pinned or pageable).  Copies inputs to the GPU, runs the three predictors above in the order
 * shapelets, points, Gaussians (the first non-empty type overwrites, the others accumulate) and copies the result
 * back on an internal second stream while the LAST predictor is still running (pinned `vis_host` makes that overlap
 * real): on the channel-walking path, into a page-locked buffer, that predictor finishes the output one 32-channel
 * tile at a time and every finished tile is copied back (a strided 2-D copy) under the tiles that follow; otherwise
 * (general path, shapelet-only sky, pageable `vis_host`) it runs in up to 8 chunks
 * of time steps (of at least 64 MB of output each) and every finished chunk is copied back under the next one.  Both
 * streams are synchronised before returning.  The values are bit-identical to the three device calls in that order.
 * A type with n == 0 may have NULL arrays. */
typedef struct {
    int n;
    const double *l, *m, *s0_jy, *alpha;
} woden_points_host;
typedef struct {
    int n;
    const double *l, *m, *s0_jy, *alpha, *maj_fwhm_rad, *min_fwhm_rad, *pa_rad;
} woden_gaussians_host;
typedef struct {
    int n, n_coeff, p_max;
    const double *l, *m, *s0_jy, *alpha, *beta1_rad, *beta2_rad, *pa_rad;
    const double *uv_basis;        /* [n][6] or NULL */
    const int *coeff_offset, *n1, *n2;
    const double *coeff;
} woden_shapelets_host;

int woden_simulate_host(woden_ctx *ctx,
                        int n_baselines, int n_times, int n_freqs,
                        const double *u_m, const double *v_m, const double *w_m, /* HOST [T][B] */
                        const double *freqs_hz, double ref_freq_hz,
                        const woden_points_host *points,        /* may be NULL */
                        const woden_gaussians_host *gaussians,  /* may be NULL */
                        const woden_shapelets_host *shapelets,  /* may be NULL */
                        float *vis_host, void *cuda_stream);

/* The step before the hot path (u,v,w are computed once per time step and only
 * scaled per channel).  Baseline coordinates in metres from antenna positions by the textbook
 * rotation (Thompson, Moran & Swenson, cited at PAPER.md:110; reading G14):
 *   u =  sin H X + cos H Y
 *   v = -sin d0 cos H X + sin d0 sin H Y + cos d0 Z
 *   w =  cos d0 cos H X - cos d0 sin H Y + sin d0 Z
 * with (X,Y,Z) = antenna p - antenna q in the local equatorial frame (X towards the meridian on
 * the equator, Y east, Z the pole), H the hour angle of the phase centre and d0 its declination.
 * x_m, y_m, z_m: DEVICE [n_antennas].  hour_angle_rad: HOST [n_times].  u_m, v_m, w_m: DEVICE
 * [n_times][n_antennas (n_antennas - 1) / 2], pairs p < q in p-major order: exactly what
 * woden_uvw takes. */
int woden_uvw_from_antennas(woden_ctx *ctx, int n_antennas,
                            const double *x_m, const double *y_m, const double *z_m,
                            int n_times, const double *hour_angle_rad, double dec0_rad,
                            double *u_m, double *v_m, double *w_m, void *cuda_stream);

/* The time-independent 2x3 matrices M_j of reading G4: rows are the local East
 * and North unit vectors at direction (l_j, m_j, n_j) in the phase-centre (u,v,w) frame,
 * e = (p x s)/|p x s|, n = s x e, p = (0, cos d0, sin d0).  l, m: DEVICE [n]; uv_basis: DEVICE
 * [n][6], the `uv_basis` argument of woden_predict_shapelets.  A component with l^2+m^2 >= 1 or
 * on the celestial pole gets the identity rows and is counted for woden_check. */
int woden_shapelet_uv_basis(woden_ctx *ctx, int n, const double *l, const double *m, double dec0_rad,
                            double *uv_basis, void *cuda_stream);

/* The consumer of the predicted visibilities in the paper (section 5.1, Eq 18-22): one
 * complex gain per antenna, fitted independently for every (time, frequency) cell by n_iter
 * (the paper: 10) passes of  x = [A^T A]^-1 A^T b  on the linearised residual
 *   R_ij = V_ij - g_i g_j^* I_ij ~ e_i g_j^* I_ij + g_i e_j^* I_ij,   g <- g + e,  from g = 1
 * (readings G15, G16: Eq 18's g_i g_i^* is read g_i g_j^*; the overall phase is unconstrained, so
 * each step is the minimum-norm least-squares solution).  vis_data (V) and vis_model (I): DEVICE
 * complex64 [n_cells][n_antennas (n_antennas - 1) / 2], i.e. a woden_predict_* buffer viewed as
 * n_cells = n_times * n_freqs cells of all pairs i < j in i-major order.  gains: DEVICE complex128
 * [n_cells][n_antennas], written.  n_antennas is limited by shared memory (the strict upper
 * triangle of |I_ij|^2 in FP64 plus 12 vectors: <= 200).
 * The spline smoothing of the gains across the band (:237) is not implemented. */
int woden_calibrate_gains(woden_ctx *ctx, int n_antennas, long long n_cells,
                          const float *vis_data, const float *vis_model, int n_iter,
                          double *gains, void *cuda_stream);

/* vis_out = V_ij - g_i g_j^* I_ij (Eq 20 with the fitted gains), same layouts; vis_out may alias
 * vis_data. */
int woden_peel(woden_ctx *ctx, int n_antennas, long long n_cells,
               const float *vis_data, const float *vis_model, const double *gains,
               float *vis_out, void *cuda_stream);

/* Image-space shapelet fit (SHAMFI, section 2.1, :89-102): the step
 * that produces the coefficients woden_predict_shapelets consumes.  Eq 7 (:93): one linear equation
 * per pixel, one unknown per basis function B_{p1,p2}, p1 + p2 <= p_max (all (p_max+1)(p_max+2)/2 of
 * them, Eq 6, in p1-major order: (0,0), (0,1), ... (0,p_max), (1,0), ...), each basis function imaged
 * on the pixel grid and convolved with the restoring beam (:98-100); the coefficients minimise
 * ||b - A x||^2 (:96).  It is done for each of n_beta pairs (beta1_rad[k], beta2_rad[k]); `best`
 * receives the index of the pair with the smallest residual (:102).  Readings (G17-G19):
 *   basis    Bimg_{n1,n2}(l, m) = 4 ln2 / (pi beta1 beta2) h_{n1}(-a x / beta1) h_{n2}(-a y / beta2),
 *            a = 2 sqrt(2 ln 2), x = sin(pa) (l - l0) + cos(pa) (m - m0), y = cos(pa) (l - l0) - sin(pa) (m - m0):
 *            the function whose transform is what woden_predict_shapelets evaluates for coefficient 1,
 *            so coeff[k] can be passed to it unchanged (s0_jy = 1, l = l0, m = m0, pa, beta1, beta2);
 *            a pixel holds Bimg dl dm (Jy/pixel for coefficients in Jy)
 *   beam     Eq 10's Gaussian (FWHM bmaj_rad, bmin_rad, position angle bpa_rad) sampled on a
 *            (2 half_width + 1)^2 pixel stencil and divided by its sum; zero padding outside the image;
 *            beam == NULL or bmaj_rad == 0: no convolution
 *   residual sum over pixels of (P - A x)^2
 *   weights  Eq 25 (:279): |C_{p1,p2}| sum over pixels |(G * B_{p1,p2})(x_s, y_t)|
 * grid: pixel (s, t) is at l = l_c + (s - (n_l-1)/2) dl, m = m_c + (t - (n_m-1)/2) dm (dl, dm signed,
 * non-zero); image: DEVICE [n_m][n_l] (index t * n_l + s).  beta1_rad, beta2_rad: HOST [n_beta], > 0.
 * coeff: DEVICE [n_beta][P]; residual: DEVICE [n_beta]; weights: DEVICE [n_beta][P] or NULL; best:
 * DEVICE int[1] or NULL.  n_refine: refinement passes of the normal equations with the exact FP64
 * operator (the tensor-core Gram matrix only preconditions them); 0 selects the default (6), which
 * reaches the FP64 least-squares solution when the scaled design matrix has a condition number
 * below ~10^3 and otherwise still reduces the residual monotonically.  0 <= p_max <= 86 (the paper's
 * orders, :183; WODEN_ERR_ORDER), half_width <= 24, n_l n_m <= 2^22 and P n_l n_m <= 2^32 (the FP64 design
 * matrix is kept in device memory: WODEN_ERR_DIM).  A Gram matrix that is not
 * positive definite even after diagonal loading is counted for woden_check(). */
typedef struct {
    int n_l, n_m;
    double dl, dm, l_c, m_c;
} woden_image_grid;
typedef struct {
    double bmaj_rad, bmin_rad, bpa_rad;
    int half_width;
} woden_restoring_beam;
#define WODEN_FIT_MAX_ORDER 86
int woden_fit_shapelets(woden_ctx *ctx, const woden_image_grid *grid, const double *image,
                        double l0, double m0, double pa_rad, int p_max,
                        int n_beta, const double *beta1_rad, const double *beta2_rad,
                        const woden_restoring_beam *beam, int n_refine,
                        double *coeff, double *residual, double *weights, int *best, void *cuda_stream);

/* Eq 25 without the coefficient: abs_sums[q] = sum over the grid's pixels of
 * |(G * B_q)(x_s, y_t)| for every basis function q of order <= p_max (same order, basis, beam and grid
 * conventions as woden_fit_shapelets); the truncation weight of a basis function is |C_q| abs_sums[q]
 * (what woden_fit_shapelets returns in `weights` for the coefficients it fitted).  abs_sums: DEVICE [P].
 * 0 <= p_max <= WODEN_MAX_ORDER (no solve is involved). */
int woden_shapelet_basis_sums(woden_ctx *ctx, const woden_image_grid *grid, double l0, double m0, double pa_rad,
                              int p_max, double beta1_rad, double beta2_rad, const woden_restoring_beam *beam,
                              double *abs_sums, void *cuda_stream);

/* Eq 25 for a whole shapelet model that was NOT fitted by woden_fit_shapelets (which returns
 * these weights itself): weights[i] = |coeff[i] s0_jy[j]| x sum over pixels of |(G * B_{n1[i], n2[i]})| for every
 * listed basis function i of every component j, the sums being woden_shapelet_basis_sums of component j (order =
 * the highest n1 + n2 in its list, its beta1 / beta2 / pa) on the grid and beam below.  The paper sums over "the
 * pixels used during the model fit" with the restoring beam G; a model whose coefficients were not fitted to an
 * image has neither, so a grid and a beam are part of the call (reading G20): n_pix x n_pix pixels centred
 * on the component, spanning +-1.5 sqrt(2 p + 1) max(beta1, beta2) / (2 sqrt(2 ln 2)) per axis (1.5 x the highest
 * order's turning point), and a circular Gaussian beam of FWHM beam_fwhm_rad sampled to +-min(24, ceil(1.5 FWHM /
 * pixel)) pixels.  n_pix <= 0 selects WODEN_EQ25_PIXELS, beam_fwhm_rad < 0 selects WODEN_EQ25_BEAM_FWHM_RAD (about
 * the resolution of a 3 km array at 180 MHz), beam_fwhm_rad == 0 means no beam.
 * s0_jy, beta1_rad, beta2_rad, pa_rad: HOST [n]; coeff_offset: HOST [n + 1] (CSR, coeff_offset[0] = 0); n1, n2,
 * coeff: HOST [coeff_offset[n]]; weights: DEVICE [coeff_offset[n]] (ready for woden_truncate_select).  Orders above
 * WODEN_MAX_ORDER: WODEN_ERR_ORDER; 3 <= n_pix <= 2048. */
#define WODEN_EQ25_PIXELS        257
#define WODEN_EQ25_BEAM_FWHM_RAD (2.0 * 3.14159265358979323846 / 10800.0)   /* 2 arcmin */
int woden_shapelet_truncation_weights(woden_ctx *ctx, int n, const double *s0_jy, const double *beta1_rad,
                                      const double *beta2_rad, const double *pa_rad, const int *coeff_offset,
                                      const int *n1, const int *n2, const double *coeff, int n_pix,
                                      double beam_fwhm_rad, double *weights, void *cuda_stream);

/* Model truncation, section 5.3 (Eq 23-24, :273-275): with the n
 * components ranked by |weights[j]|, largest first (equal values in their original order), keep the
 * largest N_comp whose summed absolute weight does not exceed f_comp times the total,
 *     sum_{j <= N_comp} |I_j| <= f_comp sum_{j <= N_tot} |I_j|     (Eq 23),  |I_j| >= |I_{j+1}|   (Eq 24).
 * weights: DEVICE [n] (the integrated flux density of a point source or Gaussian; Eq 25's weight of a
 * shapelet basis function).  keep: DEVICE int [n], 1 for a kept component, else 0; n_keep: DEVICE
 * int [1] = N_comp.  f_comp >= 1 keeps everything; the running sum is formed in ranked order in FP64 and
 * compared with f_comp * total * (1 + 1e-15).  0 <= n <= 2^17 (ranking is by counting, O(n^2): 0.1 s at the
 * limit; the paper's models have 7656 components).  A non-finite weight ranks as 0 (last) and is
 * counted for woden_check() (WODEN_ERR_DATA); woden_truncate_select_static ranks it the same way but has no
 * context to report it through. */
int woden_truncate_select(woden_ctx *ctx, int n, const double *weights, double f_comp, int *keep, int *n_keep,
                          void *cuda_stream);

/* The same selection (Eq 23-24; same arguments, same results bit for bit) for callers
 * that must not allocate device memory: a stage running inside a host framework's fixed device arena, a
 * plug-in called while the allocator is locked, a process under a hard GPU memory quota, a real-time
 * loop that cannot take the device-wide stall cudaMalloc / cudaFree may cause.  It needs no woden_ctx
 * and calls no cudaMalloc, cudaFree or other allocating routine: the ranked list is kept in a fixed
 * array inside the library image, WODEN_STATIC_TRUNCATE_MAX entries (192 KiB).  Every GPU that loads
 * the library holds that array until the process exits, used or not.
 *   - n > WODEN_STATIC_TRUNCATE_MAX returns WODEN_ERR_STATIC_LIMIT and does nothing (use
 *     woden_truncate_select for longer lists); other argument errors as for woden_truncate_select.
 *   - weights, keep, n_keep: DEVICE pointers on the CURRENT device, owned by the caller; the call is
 *     asynchronous on cuda_stream.
 *   - The first call on each device looks up that device's address of the array (cudaGetSymbolAddress,
 *     with that device current).  Make that first call outside any stream capture.
 *   - All calls on a device share the one array, which keeps the last call's contents (each call clears
 *     the part it uses first).  Two calls that overlap on the GPU -- different streams with no ordering
 *     between them, or two host threads -- race on it and return garbage: keep calls on one stream or
 *     order them with events.
 * woden_static_last_error(): text of this thread's last failure in woden_truncate_select_static ("" if
 * the last call succeeded); pointer owned by the library. */
#define WODEN_STATIC_TRUNCATE_MAX 16384
int woden_truncate_select_static(int n, const double *weights, double f_comp, int *keep, int *n_keep,
                                 void *cuda_stream);
const char *woden_static_last_error(void);

/* Measurement aid: device time in milliseconds of the Gram-matrix kernel (the tcgen05 contraction) of
 * the LAST (beta1, beta2) pair of the last woden_fit_shapelets call on this context, from CUDA events
 * recorded around it on the call's stream.  Synchronises on that kernel.  WODEN_ERR_DIM before any fit. */
int woden_fit_gram_ms(woden_ctx *ctx, float *ms);

/* Basis-evaluation experiment: the 1-D shapelet series
 *   out[i] = sum_{p <= p_max} coeff[p] h_p(x[i]),   h_p(x) = H_p(x) exp(-x^2/2)/sqrt(2^p p!)
 * by the FP32 three-term recurrence of the predict kernels (WODEN_BASIS_RECURRENCE) or by the
 * paper's mechanism: linear interpolation in one-dimensional look-up tables of
 * h_p on the grid ix * lut_dx, 0 <= x < lut_x_max, built on the device in FP64 and cached in the
 * context (WODEN_BASIS_LUT; error <= lut_dx^2 (2p+1) 1.09 / 8 per basis value; |x| beyond the
 * table gives 0).  x, coeff ([p_max + 1]) and out: DEVICE float arrays, n values. */
#define WODEN_BASIS_RECURRENCE 0
#define WODEN_BASIS_LUT        1
int woden_shapelet_series(woden_ctx *ctx, int method, int p_max, long long n, const float *x,
                          const float *coeff, double lut_dx, double lut_x_max, float *out,
                          void *cuda_stream);

/* Pipe microbenchmarks used to MEASURE the roofline denominators.
 * Runs pattern `which` (WODEN_PIPE_*) for `iters` loop iterations of 16 independent register
 * chains per thread on every SM (2 CTAs of 512 threads each) and returns, for the whole GPU, the
 * rate of the counted operation in THREAD-operations per second in *thread_ops_per_s (one FFMA2
 * counts as two FMAs; warp-instructions/s = that / 32) and the SM clock in Hz observed by
 * clock64 against the global timer in *sm_clock_hz.  Synchronous (default stream). */
#define WODEN_PIPE_FFMA         0   /* FFMA, a = a b + c with b, c fixed (operand-reuse cache hits)  */
#define WODEN_PIPE_MUFU         1   /* sin.approx + cos.approx mix on the XU pipe                    */
#define WODEN_PIPE_DFMA         2
#define WODEN_PIPE_I2F          3
#define WODEN_PIPE_LOP3         4
#define WODEN_PIPE_FFMA2        5   /* packed fma.rn.f32x2, operands as in FFMA; counts 2 FMAs each  */
#define WODEN_PIPE_FFMA_IMM     6   /* FFMA with immediate multiplier and addend                     */
#define WODEN_PIPE_F2F          7   /* F2F.F32.F64 conversions                                       */
#define WODEN_PIPE_MUFU_EX2     8   /* ex2.approx only                                               */
#define WODEN_PIPE_MUFU_FFMA    9   /* 2 MUFU + 12 FFMA interleaved; counts the MUFUs                */
#define WODEN_PIPE_FFMA_3REG   10   /* FFMA with three distinct, changing register operands          */
#define WODEN_PIPE_FFMA2_3REG  11   /* FFMA2 with three distinct, changing register pairs            */
#define WODEN_PIPE_FFMA2_BCAST 12   /* FFMA2 with one fixed pair and two changing pairs              */
#define WODEN_PIPE_FFMA2_UR    13   /* FFMA2 with two changing pairs and one uniform-register pair   */
#define WODEN_PIPE_WALK        14   /* the channel-walking kernel's 4-FFMA2 pattern per channel pair */
#define WODEN_PIPE_COUNT       15
int woden_pipe_rate(woden_ctx *ctx, int which, int iters, double *thread_ops_per_s,
                    double *sm_clock_hz);

#ifdef __cplusplus
}
#endif
#endif /* WODEN_B200_H */
