// kernels.h -- internal launch interface between api.cu and the kernel translation units.
#pragma once
#include <cuda_fp16.h>
#include <cuda_runtime.h>

#include "layout.h"

namespace woden {

// every kernel launch of the library is counted (woden_kernel_launches; bench.py's gpu_launches)
extern unsigned long long g_kernel_launches;
inline void note_launch() { ++g_kernel_launches; }

struct UvwDev {
    const double *u_m, *v_m, *w_m;
    int B, T, F;
};

// ---- staging (pack.cu) ------------------------------------------------------------------
void launch_pack_points(const double *l, const double *m, int n, int n_pad, GeoP *geo,
                        unsigned int *err, cudaStream_t st);
void launch_pack_gaussians(const double *l, const double *m, const double *maj, const double *mnr,
                           const double *pa, int n, int n_pad, GeoG *geo, unsigned int *err,
                           cudaStream_t st);
// flux table [n_ftiles][n_pad][FT] = s0 (nu_f/ref)^alpha, zero outside n x F; `interleave` stores
// channel pairs (j, j + FT/2) in adjacent floats (channel-walking kernel)
void launch_pack_flux(const double *s0, const double *alpha, double ref_freq, int n, int n_pad,
                      const ChanTable &ch, int FT, bool interleave, float *flux, unsigned int *err,
                      cudaStream_t st);
void launch_pack_shapelets(const double *l, const double *m, const double *beta1, const double *beta2,
                           const double *pa, const double *uv_basis, int n, int PM, GeoS *geo,
                           unsigned int *err, cudaStream_t st);
// zero `tri` (n * tri_size(PM) floats) then scatter-add sign- and scale-folded coefficients
void launch_pack_coeffs(const int *coeff_offset, const int *n1, const int *n2, const double *coeff,
                        int n, int n_coeff, int p_max, int PM, float *tri, unsigned int *err,
                        cudaStream_t st);

// ---- predict kernels ---------------------------------------------------------------------
// general path (predict_pg.cu): any channel list, one sin/cos (+ one exp2) per eval
constexpr int PG_FT = 16;        // channels per thread
cudaError_t launch_predict_points(const UvwDev &uvw, const ChanTable &ch, const GeoP *geo, const float *flux,
                                  int n_pad, float2 *vis, int accumulate, unsigned int *err, cudaStream_t st);
cudaError_t launch_predict_gaussians(const UvwDev &uvw, const ChanTable &ch, const GeoG *geo,
                                     const float *flux, int n_pad, float2 *vis, int accumulate,
                                     unsigned int *err, cudaStream_t st);
// channel-walking path (predict_walk.cu): equally spaced channels only.  Component data reaches the
// kernel through the constant bank, one block of WALK_CB_BYTES per launch (half of the 64 KB bank):
// launch_pack_walk_* fills blocks[(ftile * n_chunks + chunk)] in device memory from the packed
// geometry records, launch_walk_* copies block after block into the bank and launches.
constexpr int WALK_FT = 32;      // channels per thread: two chains of 16
constexpr int WALK_CB_BYTES = 32768;
constexpr int WALK_KC_POINTS = WALK_CB_BYTES / (32 + WALK_FT * 4);     // 204 components per launch
constexpr int WALK_KC_GAUSS = WALK_CB_BYTES / (48 + WALK_FT * 4);      // 186
struct WalkStreams {
    cudaStream_t main, aux;      // the caller's stream and the context's second lane
    cudaEvent_t fork, join;
    // Optional host hook, called right after the last launch of channel tile `ftile` has been enqueued on `st`
    // (calls with >= 2 channel tiles only): woden_simulate_host starts the copy-back of the finished tile from it.
    void (*tile_done)(void *user, int ftile, cudaStream_t st) = nullptr;
    void *user = nullptr;
};
size_t walk_blocks_bytes(int n, int n_ftiles, bool gauss);
void launch_pack_walk_points(const GeoP *geo, const double *s0, const double *alpha, double ref_freq, int n,
                             const ChanTable &ch, unsigned char *blocks, unsigned int *err, cudaStream_t st);
void launch_pack_walk_gaussians(const GeoG *geo, const double *s0, const double *alpha, double ref_freq, int n,
                                const ChanTable &ch, unsigned char *blocks, unsigned int *err, cudaStream_t st);
cudaError_t launch_walk_points(const UvwDev &uvw, const ChanTable &ch, const unsigned char *blocks, int n,
                               float2 *vis, int accumulate, unsigned int *err, const WalkStreams &ws);
cudaError_t launch_walk_gaussians(const UvwDev &uvw, const ChanTable &ch, const unsigned char *blocks, int n,
                                  float2 *vis, int accumulate, unsigned int *err, const WalkStreams &ws);

constexpr int SH_FT = 1;         // flux table tile for shapelets: [F][n] layout
int shapelet_order_bucket(int p_max);     // compile-time order PM >= p_max, or -1
cudaError_t launch_predict_shapelets(const UvwDev &uvw, const ChanTable &ch, const GeoS *geo, const float *tri,
                                     const float *flux, int n, int PM, bool sparse, float2 *vis, int accumulate,
                                     cudaStream_t st);

// tensor-core variant (predict_shapelets_mma.cu): T = G_y F'^T on tcgen05, operands FP16 hi + lo
size_t mma_bmat_halves(int PM, int n);
cudaError_t launch_predict_shapelets_mma(const UvwDev &uvw, const ChanTable &ch, const GeoS *geo, const float *tri,
                                         const float *flux, int n, int PM, __half *bmat, float *bscale, float2 *vis,
                                         int accumulate, cudaStream_t st);

// ---- geometry before the hot path (geometry.cu) ---------------------
cudaError_t launch_uvw(const double *X, const double *Y, const double *Z, int n_ant, int T, const double *hour_angle_dev,
                       double dec0, double *u, double *v, double *w, cudaStream_t st);
cudaError_t launch_uv_basis(const double *l, const double *m, int n, double dec0, double *M, unsigned int *err,
                            cudaStream_t st);

// ---- gain calibration and peel (calibrate.cu) -------------------------
size_t calibrate_smem_bytes(int N);
cudaError_t launch_calibrate(const float2 *data, const float2 *model, double2 *gains, int N, long long cells,
                             int n_iter, cudaStream_t st);
cudaError_t launch_peel(const float2 *data, const float2 *model, const double2 *gains, float2 *out, int N,
                        long long cells, cudaStream_t st);

// ---- basis evaluation experiment: look-up table vs recurrence (basis_lut.cu)
cudaError_t launch_lut_build(float2 *T, int n_x, int PM, double dx, cudaStream_t st);
cudaError_t launch_series(int method, const float *x, const float *c, int PM, long long n, const float2 *T, int n_x,
                          double dx, float *out, cudaStream_t st);

// ---- image-space shapelet fit (fit.cu) ------------------
constexpr int FIT_MAX_N = 3840;          // padded unknowns (p_max <= 86: 3828): the substitution kernel's shared vector
struct FitSizes {
    int P, n_rt, n_pad, n_kt, n_pairs, n_split, kt_per_split;
    size_t hermite_doubles, at_doubles, ops_halves, partial_floats, gram_doubles;
};
FitSizes fit_sizes(int n_pix, int p_max);
struct FitProblem {                      // one (beta1, beta2) pair
    int n_l, n_m, p_max, half_width, n_refine;
    double dl, dm, l_c, m_c, l0, m0, pa, beta1, beta2, bmaj, bmin, bpa;
    const double *image;                 // [n_m][n_l]
    double *coeff, *weights, *residual;  // [P], [P] or NULL, [1]
};
struct FitScratch {
    double *hx, *a0, *at, *stencil, *scale, *abssum, *gram, *z, *g, *r;
    __half *ops;
    float *partial;
    unsigned int *err;
    cudaEvent_t gram_t0, gram_t1;        // recorded around the Gram kernel when not NULL (bench.py --fit)
};
cudaError_t launch_fit_one(const FitProblem &f, const FitScratch &w, cudaStream_t st);
cudaError_t launch_fit_argmin(const double *residual, int n, int *best, cudaStream_t st);

// Eq 25 without |C|: abs_sums[q] = sum over pixels of |(G * B_q)| (steps 1-3 of the fit for one beta pair)
cudaError_t launch_fit_basis_sums(const FitProblem &f, const FitScratch &w, double *abs_sums, cudaStream_t st);

// ---- model truncation (truncate.cu, Eq 23-24) ---------------------
cudaError_t launch_eq25_weights(const double *coeff, const int *n1, const int *n2, int count, int pm, double s0,
                                const double *abs_sums, double *weights, unsigned int *err, cudaStream_t st);
cudaError_t launch_truncate_select(const double *weights, int n, double f_comp, int *rank, double *sorted, int *keep,
                                   int *n_keep, unsigned int *err, cudaStream_t st);

// ---- pipe microbenchmarks (pipes.cu) -----------------------------------------------------
cudaError_t run_pipe_rate(int which, int iters, double *thread_ops_per_s, double *sm_clock_hz);

}  // namespace woden
