// fit.cu -- image-space shapelet fit (SHAMFI, section 2.1, :89-102).
//
// Eq 7 (:93): one linear equation per pixel, one unknown per basis function B_{p1,p2}, p1 + p2 <= p_max,
// each basis function imaged on the pixel grid and convolved with the restoring beam (:98-100); the
// coefficients minimise ||b - A x||^2 (:96); a list of (beta1, beta2) pairs is searched by the residual
// of each fit (:102).  Eq 25 (:279): truncation weight of a basis function = sum over pixels of
// |C (G * B)|.  Image basis, beam stencil and residual follow DESIGN.md readings G17-G19.
//
// How it is computed here (the oracle calls numpy.linalg.lstsq on the explicit matrix; this is a
// different route to the same least-squares solution):
//   1. basis:   h_p(-a x/beta1), h_p(-a y/beta2) for every pixel by the normalised three-term recurrence
//               in FP64; At[q][i] = norm h_{n1}(x_i) h_{n2}(y_i) (basis-major, pixel contiguous).
//   2. beam:    direct 2-D convolution of every basis image with the unit-sum stencil, FP64.
//   3. scaling: every row of At is scaled by a power of two to max |.| in [1/2, 1) (the unknowns become
//               z = x / scale); row sums of |At| give the Eq 25 weights.
//   4. Gram:    G = At At^T, the one dense contraction of the path (pixels are the K dimension,
//               tens of thousands x ~10^3 basis functions), on the tensor cores: tcgen05.mma kind::f16,
//               operands split FP16 hi + lo (three products, ~22 bits), FP32 accumulation in TMEM over a
//               K range per CTA, K-split partials summed in FP64 in a fixed order.  Operand tiles are
//               staged through a 3-stage ring of bulk async copies (TMA engine) on mbarriers; one thread
//               issues the MMAs and releases stages with tcgen05.commit.
//   5. solve:   Cholesky of G + ridge (FP64, one CTA), then iterative refinement on the normal
//               equations with the EXACT FP64 operator: z += (L L^T)^-1 At (b - At^T z).  The Gram matrix
//               only preconditions; the fixed point is the least-squares solution of the FP64 system.
//   6. outputs: x = scale z, residual = ||b - At^T z||^2, weights, arg-min over the beta list.
#include <cuda_fp16.h>

#include <cmath>

#include "kernels.h"
#include "ptx.cuh"

namespace woden {
namespace {

constexpr double LN2 = 0.693147180559945309417232121458176568;
constexpr double PI = 3.14159265358979323846264338327950288;

// ---------------------------------------------------------------------------------- 1. basis
struct BasisParams {
    int n_l, n_m, p_max;
    double dl, dm, l_c, m_c, l0, m0, sp, cp;      // sin / cos of the position angle
    double ax, ay;                                 // -a / beta1, -a / beta2 (reading G17: reflected)
};

// hx[p][i], hy[p][i]: h_p at the pixel's scaled, rotated coordinates (h_p = H_p exp(-t^2/2)/sqrt(2^p p!))
__global__ void fit_hermite_kernel(const BasisParams b, double *__restrict__ hx, double *__restrict__ hy)
{
    const int n_pix = b.n_l * b.n_m;
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n_pix) return;
    const int s = i % b.n_l, t = i / b.n_l;
    const double l = b.l_c + (s - 0.5 * (b.n_l - 1)) * b.dl - b.l0;
    const double m = b.m_c + (t - 0.5 * (b.n_m - 1)) * b.dm - b.m0;
    const double tx = b.ax * (b.sp * l + b.cp * m);       // along the major axis (reading G7)
    const double ty = b.ay * (b.cp * l - b.sp * m);
#pragma unroll
    for (int which = 0; which < 2; ++which) {
        const double x = which ? ty : tx;
        double *out = which ? hy : hx;
        double hm = 0.0, hc = exp(-0.5 * x * x);
        out[i] = hc;
        for (int p = 0; p < b.p_max; ++p) {
            const double hn = sqrt(2.0 / (p + 1.0)) * x * hc - sqrt(p / (p + 1.0)) * hm;
            hm = hc; hc = hn;
            out[(size_t)(p + 1) * n_pix + i] = hn;
        }
    }
}

// At[q][i] = norm hx[n1_q][i] hy[n2_q][i], q in full-triangle (n1-major) order
__global__ void fit_product_kernel(const double *__restrict__ hx, const double *__restrict__ hy, int n_pix, int p_max,
                                   int P, double norm, double *__restrict__ At)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    const int q = blockIdx.y;
    if (i >= n_pix || q >= P) return;
    // invert q -> (n1, n2): rows n1 = 0.. hold p_max + 1 - n1 entries
    int n1 = 0, off = 0;
    while (off + (p_max + 1 - n1) <= q) { off += p_max + 1 - n1; ++n1; }
    const int n2 = q - off;
    At[(size_t)q * n_pix + i] = norm * hx[(size_t)n1 * n_pix + i] * hy[(size_t)n2 * n_pix + i];
}

// ---------------------------------------------------------------------------------- 2. beam
// stencil[(dt + hw) * (2hw+1) + (ds + hw)] = Eq 10 at the pixel offset, divided by the sum (one CTA)
__global__ void fit_stencil_kernel(double dl, double dm, double bmaj, double bmin, double sb, double cb, int hw,
                                   double *__restrict__ stencil)
{
    __shared__ double red[256];
    const int w = 2 * hw + 1, n = w * w;
    double part = 0.0;
    for (int k = threadIdx.x; k < n; k += blockDim.x) {
        const double ol = (k % w - hw) * dl, om = (k / w - hw) * dm;
        const double xb = sb * ol + cb * om, yb = cb * ol - sb * om;
        const double ex = bmaj > 0.0 ? xb * xb / (bmaj * bmaj) : (xb == 0.0 ? 0.0 : INFINITY);
        const double ey = bmin > 0.0 ? yb * yb / (bmin * bmin) : (yb == 0.0 ? 0.0 : INFINITY);
        const double v = exp(-4.0 * LN2 * (ex + ey));
        stencil[k] = v;
        part += v;
    }
    red[threadIdx.x] = part;
    __syncthreads();
    for (int o = blockDim.x / 2; o > 0; o >>= 1) {
        if ((int)threadIdx.x < o) red[threadIdx.x] += red[threadIdx.x + o];
        __syncthreads();
    }
    const double inv = 1.0 / red[0];
    for (int k = threadIdx.x; k < n; k += blockDim.x) stencil[k] *= inv;
}

// out[q][t][s] = sum_{dt, ds} stencil[dt][ds] in[q][t - (dt - hw)][s - (ds - hw)], zero outside the image.
// One CTA = 64 x 16 output pixels of one basis image; a thread owns 4 consecutive pixels along s and
// slides a 4-value register window over the shared-memory patch (one patch load per 4 FMAs).
constexpr int CV_W = 64, CV_H = 16;
__global__ void __launch_bounds__(256) fit_convolve_kernel(const double *__restrict__ in, const double *__restrict__ stencil,
                                                           int n_l, int n_m, int hw, double *__restrict__ out)
{
    extern __shared__ double sm[];
    const int w = 2 * hw + 1, tw = CV_W + 2 * hw, th = CV_H + 2 * hw;
    double *st = sm, *patch = sm + w * w;
    const int q = blockIdx.z, s0 = blockIdx.x * CV_W, t0 = blockIdx.y * CV_H;
    const double *img = in + (size_t)q * n_l * n_m;
    const int tx = threadIdx.x, ty = threadIdx.y, tid = ty * 16 + tx;
    for (int k = tid; k < w * w; k += 256) st[k] = stencil[k];
    for (int k = tid; k < tw * th; k += 256) {
        const int s = s0 - hw + k % tw, t = t0 - hw + k / tw;
        patch[k] = (s >= 0 && s < n_l && t >= 0 && t < n_m) ? img[(size_t)t * n_l + s] : 0.0;
    }
    __syncthreads();
    double acc[4] = {0.0, 0.0, 0.0, 0.0};
    for (int dt = 0; dt < w; ++dt) {
        const double *row = patch + (ty + 2 * hw - dt) * tw + 4 * tx + 2 * hw;      // ds = 0 position of output 0
        double v1 = row[1], v2 = row[2], v3 = row[3];
        for (int ds = 0; ds < w; ++ds) {
            const double v0 = row[-ds], c = st[dt * w + ds];
            acc[0] = fma(c, v0, acc[0]); acc[1] = fma(c, v1, acc[1]);
            acc[2] = fma(c, v2, acc[2]); acc[3] = fma(c, v3, acc[3]);
            v3 = v2; v2 = v1; v1 = v0;
        }
    }
    const int t = t0 + ty;
    if (t >= n_m) return;
#pragma unroll
    for (int i = 0; i < 4; ++i) {
        const int s = s0 + 4 * tx + i;
        if (s < n_l) out[(size_t)q * n_l * n_m + (size_t)t * n_l + s] = acc[i];
    }
}

// ---------------------------------------------------------------------------------- 3. scaling
// per row q: scale[q] = 2^-e with max|At[q]| = f 2^e, f in [1/2, 1) (1 for an all-zero row);
// abssum[q] = sum_i |At[q][i]| (Eq 25); the row is scaled in place.
__global__ void fit_scale_rows_kernel(double *__restrict__ At, int n_pix, double *__restrict__ scale,
                                      double *__restrict__ abssum)
{
    __shared__ double red_m[256], red_s[256];
    double *row = At + (size_t)blockIdx.x * n_pix;
    double mx = 0.0, sum = 0.0;
    for (int i = threadIdx.x; i < n_pix; i += blockDim.x) { const double a = fabs(row[i]); mx = fmax(mx, a); sum += a; }
    red_m[threadIdx.x] = mx; red_s[threadIdx.x] = sum;
    __syncthreads();
    for (int o = blockDim.x / 2; o > 0; o >>= 1) {
        if ((int)threadIdx.x < o) {
            red_m[threadIdx.x] = fmax(red_m[threadIdx.x], red_m[threadIdx.x + o]);
            red_s[threadIdx.x] += red_s[threadIdx.x + o];
        }
        __syncthreads();
    }
    int e = 0;
    if (red_m[0] > 0.0 && isfinite(red_m[0])) frexp(red_m[0], &e);
    const double sc = ldexp(1.0, -e);
    if (threadIdx.x == 0) { scale[blockIdx.x] = sc; abssum[blockIdx.x] = red_s[0]; }
    for (int i = threadIdx.x; i < n_pix; i += blockDim.x) row[i] *= sc;
}

// ---------------------------------------------------------------------------------- 4. Gram on tcgen05
constexpr int GT = 128;                  // tile rows (UMMA M = N = 128)
constexpr int GK = 64;                   // pixels per pipeline stage (4 UMMA K steps of 16)
constexpr int GSTAGES = 3;
constexpr int G_BLOCK_BYTES = GT * GK * 2;            // one operand tile of one stage: 16 KB
constexpr int G_STAGE_BYTES = 4 * G_BLOCK_BYTES;      // A hi, A lo, B hi, B lo

// FP16 hi + lo of the scaled rows in the tcgen05 no-swizzle K-major core-matrix layout, blocked so that
// one (k tile, row tile) operand block is 16 KB contiguous: halves[part][kt][rt][k8][row][8].
__global__ void fit_split_kernel(const double *__restrict__ At, int P, int n_pix, int n_rt, int n_kt,
                                 __half *__restrict__ ops)
{
    const long long g = (long long)blockIdx.x * blockDim.x + threadIdx.x;      // (row, 8-pixel group)
    const int n_k8 = n_kt * (GK / 8);
    if (g >= (long long)n_rt * GT * n_k8) return;
    const int row = (int)(g / n_k8), k8g = (int)(g % n_k8);
    __align__(16) __half hi[8], lo[8];
#pragma unroll
    for (int j = 0; j < 8; ++j) {
        const int i = k8g * 8 + j;
        const double v = (row < P && i < n_pix) ? At[(size_t)row * n_pix + i] : 0.0;
        const float f = (float)v;
        hi[j] = __float2half_rn(f);
        lo[j] = __float2half_rn((float)(v - (double)__half2float(hi[j])));
    }
    const int kt = k8g / (GK / 8), k8 = k8g % (GK / 8), rt = row / GT, r = row % GT;
    const size_t blk = ((size_t)kt * n_rt + rt) * (GK / 8) + k8;
    const size_t part = (size_t)n_kt * n_rt * GT * GK;
    *reinterpret_cast<uint4 *>(ops + (blk * GT + r) * 8) = *reinterpret_cast<const uint4 *>(hi);
    *reinterpret_cast<uint4 *>(ops + part + (blk * GT + r) * 8) = *reinterpret_cast<const uint4 *>(lo);
}

struct GramParams {
    const __half *ops;       // [2][n_kt][n_rt][8][128][8]
    float *partial;          // [n_split][n_pairs][128][128]
    int n_rt, n_kt, n_pairs, kt_per_split;
};

// One CTA = one tile pair (ti <= tj) x one K split: D[128 x 128] = sum over its k tiles of A_ti B_tj^T.
__global__ void __launch_bounds__(128) fit_gram_kernel(const GramParams p)
{
    extern __shared__ __align__(128) unsigned char smem[];
    __shared__ __align__(8) uint64_t full_bar[GSTAGES], empty_bar[GSTAGES], done_bar;
    __shared__ uint32_t tmem_holder;

    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    // tile pair index -> (ti, tj), ti <= tj
    int ti = 0, rem = blockIdx.x;
    while (rem >= p.n_rt - ti) { rem -= p.n_rt - ti; ++ti; }
    const int tj = ti + rem;
    const int kt0 = blockIdx.y * p.kt_per_split;
    const int kt1 = min(p.n_kt, kt0 + p.kt_per_split);
    const int n_it = kt1 - kt0;

    if (warp == 0) tmem_alloc(&tmem_holder, 128);
    if (tid == 0) {
        for (int s = 0; s < GSTAGES; ++s) { mbar_init(&full_bar[s], 1); mbar_init(&empty_bar[s], 1); }
        mbar_init(&done_bar, 1);
        fence_mbar_init();
    }
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    const uint32_t tmem = tmem_holder;
    const size_t part = (size_t)p.n_kt * p.n_rt * GT * GK;        // halves per hi / lo part

    if (warp == 0 && lane == 0) {
        // producer: four 16 KB bulk copies per stage
        for (int it = 0; it < n_it; ++it) {
            const int s = it % GSTAGES;
            if (it >= GSTAGES) mbar_wait(&empty_bar[s], ((it / GSTAGES) - 1) & 1);
            unsigned char *dst = smem + (size_t)s * G_STAGE_BYTES;
            const size_t a_off = ((size_t)(kt0 + it) * p.n_rt + ti) * GT * GK, b_off = ((size_t)(kt0 + it) * p.n_rt + tj) * GT * GK;
            mbar_arrive_expect_tx(&full_bar[s], G_STAGE_BYTES);
            bulk_g2s(dst, p.ops + a_off, G_BLOCK_BYTES, &full_bar[s]);
            bulk_g2s(dst + G_BLOCK_BYTES, p.ops + part + a_off, G_BLOCK_BYTES, &full_bar[s]);
            bulk_g2s(dst + 2 * G_BLOCK_BYTES, p.ops + b_off, G_BLOCK_BYTES, &full_bar[s]);
            bulk_g2s(dst + 3 * G_BLOCK_BYTES, p.ops + part + b_off, G_BLOCK_BYTES, &full_bar[s]);
        }
    } else if (warp == 1 && lane == 0) {
        // MMA issuer: 4 K steps x (hi hi + hi lo + lo hi) per stage, then release the stage
        const uint32_t idesc = umma_idesc_f16(GT, GT);
        const uint32_t lbo = GT * 16, sbo = 128;                   // K-chunk stride, 8-row group stride
        for (int it = 0; it < n_it; ++it) {
            const int s = it % GSTAGES;
            mbar_wait(&full_bar[s], (it / GSTAGES) & 1);
            tc_fence_after();
            const uint32_t base = smem_u32(smem + (size_t)s * G_STAGE_BYTES);
#pragma unroll
            for (int ks = 0; ks < GK / 16; ++ks) {
                const uint32_t ko = (uint32_t)ks * 2u * lbo;       // two 16-byte K chunks per step
                const uint64_t aH = umma_desc_kmajor(base + ko, lbo, sbo);
                const uint64_t aL = umma_desc_kmajor(base + G_BLOCK_BYTES + ko, lbo, sbo);
                const uint64_t bH = umma_desc_kmajor(base + 2 * G_BLOCK_BYTES + ko, lbo, sbo);
                const uint64_t bL = umma_desc_kmajor(base + 3 * G_BLOCK_BYTES + ko, lbo, sbo);
                umma_f16(tmem, aH, bH, idesc, (it > 0 || ks > 0) ? 1u : 0u);
                umma_f16(tmem, aH, bL, idesc, 1u);
                umma_f16(tmem, aL, bH, idesc, 1u);
            }
            umma_commit(&empty_bar[s]);                            // arrives when these MMAs have read smem
        }
        umma_commit(&done_bar);
    }
    __syncwarp();
    // epilogue: every thread reads its TMEM lane (= tile row) and writes the FP32 partial
    if (n_it > 0) {
        mbar_wait(&done_bar, 0);
        tc_fence_after();
    }
    float *dst = p.partial + (((size_t)blockIdx.y * p.n_pairs + blockIdx.x) * GT + tid) * GT;
    const uint32_t lane_base = tmem + ((uint32_t)(warp * 32) << 16);
#pragma unroll 1
    for (int c = 0; c < GT; c += 16) {
        uint32_t v[16];
        if (n_it > 0) { tmem_ld16_issue(lane_base + (uint32_t)c, v); tmem_ld_wait(); }
        else {
#pragma unroll
            for (int j = 0; j < 16; ++j) v[j] = 0u;
        }
#pragma unroll
        for (int j = 0; j < 16; j += 4)
            *reinterpret_cast<uint4 *>(dst + c + j) = make_uint4(v[j], v[j + 1], v[j + 2], v[j + 3]);
    }
    tc_fence_before();
    __syncthreads();
    if (warp == 0) tmem_dealloc(tmem, 128);
}

// G[r][c] = sum over splits (fixed order, FP64) of the tile partials, mirrored to the full matrix;
// + ridge on the diagonal; rows >= P (padding) become identity rows.
__global__ void fit_gram_reduce_kernel(const float *__restrict__ partial, int n_split, int n_pairs, int n_rt, int P,
                                       double ridge, double *__restrict__ G)
{
    const int n = n_rt * GT;
    const int c = blockIdx.x * blockDim.x + threadIdx.x, r = blockIdx.y;
    if (c >= n || c < r) return;                                 // upper triangle incl. diagonal: r <= c
    const int ti = r / GT, tj = c / GT;
    int pair = 0;
    for (int t = 0; t < ti; ++t) pair += n_rt - t;
    pair += tj - ti;
    double s = 0.0;
    for (int k = 0; k < n_split; ++k)
        s += (double)partial[(((size_t)k * n_pairs + pair) * GT + (r % GT)) * GT + (c % GT)];
    if (r >= P || c >= P) s = (r == c) ? 1.0 : 0.0;
    else if (r == c) s += ridge * s;
    G[(size_t)r * n + c] = s;
    G[(size_t)c * n + r] = s;
}

// ---------------------------------------------------------------------------------- 5. solve
// In-place blocked Cholesky G = L L^T (right-looking, panels of CB = 64 columns; n is a multiple of
// 128): per panel three kernels -- the 64 x 64 diagonal block in shared memory by one CTA, the rows
// below it by triangular solves (one CTA per 64 rows), then the rank-64 update of the trailing lower
// triangle (one CTA per 64 x 64 tile).  On return the lower triangle holds L and the upper triangle
// L^T, so that both triangular solves of the refinement read rows.
constexpr int CB = 64;

__global__ void __launch_bounds__(256) chol_diag_kernel(double *__restrict__ G, int n, int j0, unsigned int *__restrict__ err)
{
    __shared__ double D[CB][CB + 1];
    const int tid = threadIdx.x;
    for (int e = tid; e < CB * CB; e += 256) {
        const int r = e / CB, c = e % CB;
        D[r][c] = c <= r ? G[(size_t)(j0 + r) * n + j0 + c] : 0.0;
    }
    __syncthreads();
    for (int c = 0; c < CB; ++c) {
        if (tid == 0) {
            double d = D[c][c];
            if (!(d > 0.0)) { atomicAdd(err, 1u); d = 1.0; }      // not positive definite: counted (woden_check)
            D[c][c] = sqrt(d);
        }
        __syncthreads();
        if (tid > c && tid < CB) D[tid][c] /= D[c][c];
        __syncthreads();
        // trailing update of the block's lower triangle: D[r][k] -= D[r][c] D[k][c], c < k <= r
        for (int e = tid; e < CB * CB; e += 256) {
            const int r = e / CB, k = e % CB;
            if (k > c && k <= r) D[r][k] = fma(-D[r][c], D[k][c], D[r][k]);
        }
        __syncthreads();
    }
    for (int e = tid; e < CB * CB; e += 256) {
        const int r = e / CB, c = e % CB;
        if (c <= r) {
            G[(size_t)(j0 + r) * n + j0 + c] = D[r][c];
            G[(size_t)(j0 + c) * n + j0 + r] = D[r][c];
        }
    }
}

// rows below the diagonal block: X L_d^T = A  (thread = one row, forward substitution over 64 columns)
__global__ void __launch_bounds__(CB) chol_trsm_kernel(double *__restrict__ G, int n, int j0)
{
    extern __shared__ double chol_sm[];
    double (*Ld)[CB + 1] = reinterpret_cast<double (*)[CB + 1]>(chol_sm);
    double (*X)[CB + 1] = reinterpret_cast<double (*)[CB + 1]>(chol_sm + CB * (CB + 1));
    const int tid = threadIdx.x, r0 = j0 + CB + blockIdx.x * CB;
    for (int e = tid; e < CB * CB; e += CB) {
        const int r = e / CB, c = e % CB;
        Ld[r][c] = G[(size_t)(j0 + r) * n + j0 + c];
        X[r][c] = G[(size_t)(r0 + r) * n + j0 + c];               // coalesced over c
    }
    __syncthreads();
    for (int c = 0; c < CB; ++c) {
        double s = X[tid][c];
        for (int k = 0; k < c; ++k) s = fma(-X[tid][k], Ld[c][k], s);
        X[tid][c] = s / Ld[c][c];
    }
    __syncthreads();
    for (int e = tid; e < CB * CB; e += CB) {
        const int r = e / CB, c = e % CB;
        G[(size_t)(r0 + r) * n + j0 + c] = X[r][c];
    }
    for (int e = tid; e < CB * CB; e += CB) {
        const int c = e / CB, r = e % CB;                         // coalesced over r: the mirrored copy
        G[(size_t)(j0 + c) * n + r0 + r] = X[r][c];
    }
}

// trailing lower triangle: G[bi][bj] -= X_bi X_bj^T for the 64 x 64 tiles bj <= bi below the panel
__global__ void __launch_bounds__(256) chol_syrk_kernel(double *__restrict__ G, int n, int j0)
{
    extern __shared__ double chol_sm[];
    double (*Xi)[CB + 1] = reinterpret_cast<double (*)[CB + 1]>(chol_sm);
    double (*Xj)[CB + 1] = reinterpret_cast<double (*)[CB + 1]>(chol_sm + CB * (CB + 1));
    int bi = 0, rem = blockIdx.x;
    while (rem > bi) { rem -= bi + 1; ++bi; }
    const int bj = rem;
    const int ri = j0 + CB + bi * CB, rj = j0 + CB + bj * CB;
    const int tid = threadIdx.x;
    for (int e = tid; e < CB * CB; e += 256) {
        const int r = e / CB, c = e % CB;
        Xi[r][c] = G[(size_t)(ri + r) * n + j0 + c];
        Xj[r][c] = G[(size_t)(rj + r) * n + j0 + c];
    }
    __syncthreads();
    const int tr = (tid / 16) * 4, tc = (tid % 16) * 4;
    double acc[4][4] = {};
    for (int k = 0; k < CB; ++k) {
        double a[4], b[4];
#pragma unroll
        for (int i = 0; i < 4; ++i) { a[i] = Xi[tr + i][k]; b[i] = Xj[tc + i][k]; }
#pragma unroll
        for (int i = 0; i < 4; ++i)
#pragma unroll
            for (int j = 0; j < 4; ++j) acc[i][j] = fma(a[i], b[j], acc[i][j]);
    }
#pragma unroll
    for (int i = 0; i < 4; ++i)
#pragma unroll
        for (int j = 0; j < 4; ++j) G[(size_t)(ri + tr + i) * n + rj + tc + j] -= acc[i][j];
}

void launch_cholesky(double *G, int n, unsigned int *err, cudaStream_t st)
{
    constexpr int SM2 = 2 * CB * (CB + 1) * (int)sizeof(double);
    cudaFuncSetAttribute(chol_trsm_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, SM2);
    cudaFuncSetAttribute(chol_syrk_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, SM2);
    for (int j0 = 0; j0 < n; j0 += CB) {
        chol_diag_kernel<<<1, 256, 0, st>>>(G, n, j0, err); note_launch();
        const int below = (n - j0 - CB) / CB;
        if (below > 0) {
            chol_trsm_kernel<<<below, CB, SM2, st>>>(G, n, j0); note_launch();
            chol_syrk_kernel<<<below * (below + 1) / 2, 256, SM2, st>>>(G, n, j0); note_launch();
        }
    }
}

// z += (L L^T)^-1 g by one CTA (n <= FIT_MAX_N): forward then backward substitution, 32 rows per step:
// the rows' dots over the already solved part run one warp per row, the 32 x 32 diagonal block is
// finished by warp 0.
__global__ void __launch_bounds__(1024) fit_solve_kernel(const double *__restrict__ G, int n, const double *__restrict__ g,
                                                         double *__restrict__ z)
{
    __shared__ double y[FIT_MAX_N], part[32], Dg[32][33];
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    for (int i = threadIdx.x; i < n; i += blockDim.x) y[i] = g[i];
    __syncthreads();
    // forward: L y = g (lower triangle, rows)
    for (int r0 = 0; r0 < n; r0 += 32) {
        const int i = r0 + warp;
        if (i < n) {
            const double *Li = G + (size_t)i * n;
            double s = 0.0;
            double s1 = 0.0, s2 = 0.0, s3 = 0.0;
            int k = lane;
            for (; k + 96 < r0; k += 128) {                       // four loads in flight per lane
                s = fma(Li[k], y[k], s); s1 = fma(Li[k + 32], y[k + 32], s1);
                s2 = fma(Li[k + 64], y[k + 64], s2); s3 = fma(Li[k + 96], y[k + 96], s3);
            }
            for (; k < r0; k += 32) s = fma(Li[k], y[k], s);
            s = (s + s1) + (s2 + s3);
            for (int o = 16; o > 0; o >>= 1) s += __shfl_xor_sync(0xffffffffu, s, o);
            if (lane == 0) part[warp] = y[i] - s;
            if (r0 + lane < n) Dg[warp][lane] = Li[r0 + lane];      // the 32 x 32 diagonal block (lower part used)
        }
        __syncthreads();
        if (warp == 0) {
            const int rows = min(32, n - r0);
            double v = lane < rows ? part[lane] : 0.0;
            for (int c = 0; c < rows; ++c) {
                const double yc = __shfl_sync(0xffffffffu, v, c) / Dg[c][c];
                if (lane == c) v = yc;
                else if (lane > c && lane < rows) v -= Dg[lane][c] * yc;
            }
            if (lane < rows) y[r0 + lane] = v;
        }
        __syncthreads();
    }
    // backward: L^T x = y (upper triangle holds L^T, rows), blocks from the bottom
    const int n_blocks = (n + 31) / 32;
    for (int b = n_blocks - 1; b >= 0; --b) {
        const int r0 = b * 32, r1 = min(n, r0 + 32);
        const int i = r0 + warp;
        if (i < r1) {
            const double *Ui = G + (size_t)i * n;
            double s = 0.0;
            double s1 = 0.0, s2 = 0.0, s3 = 0.0;
            int k = r1 + lane;
            for (; k + 96 < n; k += 128) {
                s = fma(Ui[k], y[k], s); s1 = fma(Ui[k + 32], y[k + 32], s1);
                s2 = fma(Ui[k + 64], y[k + 64], s2); s3 = fma(Ui[k + 96], y[k + 96], s3);
            }
            for (; k < n; k += 32) s = fma(Ui[k], y[k], s);
            s = (s + s1) + (s2 + s3);
            for (int o = 16; o > 0; o >>= 1) s += __shfl_xor_sync(0xffffffffu, s, o);
            if (lane == 0) part[warp] = y[i] - s;
            if (r0 + lane < n) Dg[warp][lane] = Ui[r0 + lane];      // diagonal block of L^T (upper part used)
        }
        __syncthreads();
        if (warp == 0) {
            const int rows = r1 - r0;
            double v = lane < rows ? part[lane] : 0.0;
            for (int c = rows - 1; c >= 0; --c) {
                const double xc = __shfl_sync(0xffffffffu, v, c) / Dg[c][c];
                if (lane == c) v = xc;
                else if (lane < c) v -= Dg[lane][c] * xc;
            }
            if (lane < rows) y[r0 + lane] = v;
        }
        __syncthreads();
    }
    for (int i = threadIdx.x; i < n; i += blockDim.x) z[i] += y[i];
}

// r[i] = b[i] - sum_q At[q][i] z[q]   (FP64; coalesced over pixels)
__global__ void fit_residual_kernel(const double *__restrict__ At, const double *__restrict__ z, const double *__restrict__ b,
                                    int P, int n_pix, double *__restrict__ r)
{
    extern __shared__ double zs[];
    for (int q = threadIdx.x; q < P; q += blockDim.x) zs[q] = z[q];
    __syncthreads();
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n_pix) return;
    double s0 = 0.0, s1 = 0.0;
    int q = 0;
    for (; q + 1 < P; q += 2) {
        s0 = fma(At[(size_t)q * n_pix + i], zs[q], s0);
        s1 = fma(At[(size_t)(q + 1) * n_pix + i], zs[q + 1], s1);
    }
    if (q < P) s0 = fma(At[(size_t)q * n_pix + i], zs[q], s0);
    r[i] = b[i] - (s0 + s1);
}

// g[q] = sum_i At[q][i] r[i] (one CTA per row, fixed-order tree); rows >= P of g are zero
__global__ void fit_atr_kernel(const double *__restrict__ At, const double *__restrict__ r, int P, int n_pix,
                               double *__restrict__ g)
{
    __shared__ double red[256];
    const int q = blockIdx.x;
    double s = 0.0;
    if (q < P) {
        const double *row = At + (size_t)q * n_pix;
        for (int i = threadIdx.x; i < n_pix; i += blockDim.x) s = fma(row[i], r[i], s);
    }
    red[threadIdx.x] = s;
    __syncthreads();
    for (int o = blockDim.x / 2; o > 0; o >>= 1) {
        if ((int)threadIdx.x < o) red[threadIdx.x] += red[threadIdx.x + o];
        __syncthreads();
    }
    if (threadIdx.x == 0) g[q] = red[0];
}

// ---------------------------------------------------------------------------------- 6. outputs
// coeff[q] = scale[q] z[q]; weights[q] = |z[q]| abssum_scaled[q]... (abssum was taken before scaling:
// |x_q| sum_i |A[q][i]| = |z_q scale_q| abssum[q]); residual = sum r^2 (one CTA, fixed order)
__global__ void fit_finish_kernel(const double *__restrict__ z, const double *__restrict__ scale,
                                  const double *__restrict__ abssum, const double *__restrict__ r, int P, int n_pix,
                                  double *__restrict__ coeff, double *__restrict__ weights, double *__restrict__ residual)
{
    __shared__ double red[1024];
    for (int q = threadIdx.x; q < P; q += blockDim.x) {
        const double x = scale[q] * z[q];
        coeff[q] = x;
        if (weights) weights[q] = fabs(x) * abssum[q];
    }
    double s = 0.0;
    for (int i = threadIdx.x; i < n_pix; i += blockDim.x) s = fma(r[i], r[i], s);
    red[threadIdx.x] = s;
    __syncthreads();
    for (int o = blockDim.x / 2; o > 0; o >>= 1) {
        if ((int)threadIdx.x < o) red[threadIdx.x] += red[threadIdx.x + o];
        __syncthreads();
    }
    if (threadIdx.x == 0) *residual = red[0];
}

__global__ void fit_argmin_kernel(const double *__restrict__ residual, int n, int *__restrict__ best)
{
    if (threadIdx.x || blockIdx.x) return;
    int b = 0;
    for (int k = 1; k < n; ++k)
        if (residual[k] < residual[b]) b = k;                    // first minimum, like numpy.argmin
    *best = b;
}

__global__ void fit_zero_kernel(double *__restrict__ p, long long n)
{
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n) p[i] = 0.0;
}

}  // namespace

FitSizes fit_sizes(int n_pix, int p_max)
{
    FitSizes s;
    s.P = (p_max + 1) * (p_max + 2) / 2;
    s.n_rt = (s.P + GT - 1) / GT;
    s.n_pad = s.n_rt * GT;
    s.n_kt = (n_pix + GK - 1) / GK;
    s.n_pairs = s.n_rt * (s.n_rt + 1) / 2;
    // K splits: enough CTAs for two waves of the 148 SMs, at least 4 stages each
    int split = (2 * 148 + s.n_pairs - 1) / s.n_pairs;
    const int max_split = (s.n_kt + 3) / 4;
    if (split > max_split) split = max_split;
    if (split < 1) split = 1;
    s.kt_per_split = (s.n_kt + split - 1) / split;
    s.n_split = (s.n_kt + s.kt_per_split - 1) / s.kt_per_split;
    s.hermite_doubles = (size_t)2 * (p_max + 1) * n_pix;
    s.at_doubles = (size_t)s.P * n_pix;
    s.ops_halves = (size_t)2 * s.n_kt * s.n_rt * GT * GK;
    s.partial_floats = (size_t)s.n_split * s.n_pairs * GT * GT;
    s.gram_doubles = (size_t)s.n_pad * s.n_pad;
    return s;
}

// steps 1-3: basis images, beam convolution, row scaling (+ Eq 25 row sums) into w.at / w.scale / w.abssum
static cudaError_t fit_build_rows(const FitProblem &f, const FitScratch &w, cudaStream_t st)
{
    const int n_pix = f.n_l * f.n_m;
    const int P = (f.p_max + 1) * (f.p_max + 2) / 2;
    const double a = 2.0 * sqrt(2.0 * LN2);
    BasisParams b;
    b.n_l = f.n_l; b.n_m = f.n_m; b.p_max = f.p_max;
    b.dl = f.dl; b.dm = f.dm; b.l_c = f.l_c; b.m_c = f.m_c; b.l0 = f.l0; b.m0 = f.m0;
    b.sp = sin(f.pa); b.cp = cos(f.pa);
    b.ax = -a / f.beta1; b.ay = -a / f.beta2;
    fit_hermite_kernel<<<(n_pix + 127) / 128, 128, 0, st>>>(b, w.hx, w.hx + (size_t)(f.p_max + 1) * n_pix); note_launch();
    const double norm = 4.0 * LN2 / (PI * f.beta1 * f.beta2) * fabs(f.dl * f.dm);
    const bool beam = f.bmaj > 0.0;
    double *unconv = beam ? w.a0 : w.at;
    fit_product_kernel<<<dim3((n_pix + 255) / 256, P), 256, 0, st>>>(w.hx, w.hx + (size_t)(f.p_max + 1) * n_pix, n_pix,
                                                                      f.p_max, P, norm, unconv); note_launch();
    if (beam) {
        const int hw = f.half_width, wd = 2 * hw + 1;
        const size_t smem = ((size_t)wd * wd + (size_t)(CV_W + 2 * hw) * (CV_H + 2 * hw)) * sizeof(double);
        cudaError_t e = cudaFuncSetAttribute(fit_convolve_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e != cudaSuccess) return e;
        fit_stencil_kernel<<<1, 256, 0, st>>>(f.dl, f.dm, f.bmaj, f.bmin, sin(f.bpa), cos(f.bpa), hw, w.stencil); note_launch();
        fit_convolve_kernel<<<dim3((f.n_l + CV_W - 1) / CV_W, (f.n_m + CV_H - 1) / CV_H, P), dim3(16, 16), smem, st>>>(
            w.a0, w.stencil, f.n_l, f.n_m, hw, w.at); note_launch();
    }
    fit_scale_rows_kernel<<<P, 256, 0, st>>>(w.at, n_pix, w.scale, w.abssum); note_launch();
    return cudaGetLastError();
}

cudaError_t launch_fit_basis_sums(const FitProblem &f, const FitScratch &w, double *abs_sums, cudaStream_t st)
{
    cudaError_t e = fit_build_rows(f, w, st);
    if (e != cudaSuccess) return e;
    const int P = (f.p_max + 1) * (f.p_max + 2) / 2;
    return cudaMemcpyAsync(abs_sums, w.abssum, (size_t)P * sizeof(double), cudaMemcpyDeviceToDevice, st);
}

cudaError_t launch_fit_one(const FitProblem &f, const FitScratch &w, cudaStream_t st)
{
    const int n_pix = f.n_l * f.n_m;
    const FitSizes sz = fit_sizes(n_pix, f.p_max);
    const int P = sz.P;
    cudaError_t e0 = fit_build_rows(f, w, st);
    if (e0 != cudaSuccess) return e0;
    {
        const long long groups = (long long)sz.n_pad * sz.n_kt * (GK / 8);
        fit_split_kernel<<<(unsigned)((groups + 255) / 256), 256, 0, st>>>(w.at, P, n_pix, sz.n_rt, sz.n_kt, w.ops); note_launch();
    }
    GramParams gp;
    gp.ops = w.ops; gp.partial = w.partial; gp.n_rt = sz.n_rt; gp.n_kt = sz.n_kt; gp.n_pairs = sz.n_pairs;
    gp.kt_per_split = sz.kt_per_split;
    const int gsmem = GSTAGES * G_STAGE_BYTES;
    cudaError_t e = cudaFuncSetAttribute(fit_gram_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, gsmem);
    if (e != cudaSuccess) return e;
    if (w.gram_t0) cudaEventRecord(w.gram_t0, st);
    fit_gram_kernel<<<dim3(sz.n_pairs, sz.n_split), 128, gsmem, st>>>(gp); note_launch();
    if (w.gram_t1) cudaEventRecord(w.gram_t1, st);
    // relative diagonal loading: the split-FP16 Gram matrix carries ~2^-21 sqrt(G_rr G_cc) of error per
    // entry; loading the diagonal by 2^-14 keeps the preconditioner positive definite for ~10^3 unknowns
    const double ridge = ldexp(1.0, -14);
    fit_gram_reduce_kernel<<<dim3((sz.n_pad + 127) / 128, sz.n_pad), 128, 0, st>>>(w.partial, sz.n_split, sz.n_pairs, sz.n_rt,
                                                                                  P, ridge, w.gram); note_launch();
    launch_cholesky(w.gram, sz.n_pad, w.err, st);
    fit_zero_kernel<<<(sz.n_pad + 255) / 256, 256, 0, st>>>(w.z, sz.n_pad); note_launch();
    for (int it = 0; it <= f.n_refine; ++it) {
        fit_residual_kernel<<<(n_pix + 127) / 128, 128, P * sizeof(double), st>>>(w.at, w.z, f.image, P, n_pix, w.r); note_launch();
        if (it == f.n_refine) break;
        fit_atr_kernel<<<sz.n_pad, 256, 0, st>>>(w.at, w.r, P, n_pix, w.g); note_launch();
        fit_solve_kernel<<<1, 1024, 0, st>>>(w.gram, sz.n_pad, w.g, w.z); note_launch();
    }
    fit_finish_kernel<<<1, 1024, 0, st>>>(w.z, w.scale, w.abssum, w.r, P, n_pix, f.coeff, f.weights, f.residual); note_launch();
    return cudaGetLastError();
}

cudaError_t launch_fit_argmin(const double *residual, int n, int *best, cudaStream_t st)
{
    fit_argmin_kernel<<<1, 32, 0, st>>>(residual, n, best); note_launch();
    return cudaGetLastError();
}

}  // namespace woden
