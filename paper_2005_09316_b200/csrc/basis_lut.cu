// basis_lut.cu -- SURVEY.md §8(f) NEXT-5: the paper's own way of evaluating the shapelet basis,
// "interpolating from one dimensional look-up tables of B~(k_x; 1) ... and scaling by the
// appropriate beta", measured against the three-term recurrence the predict
// kernels use.  Both evaluate the 1-D shapelet series  s(x) = sum_{p <= PM} c_p h_p(x)
// (h_p(x) = H_p(x) exp(-x^2/2)/sqrt(2^p p!), reading G2) for a batch of arguments x, one per thread.
//   method 0: FP32 recurrence h_{p+1} = sqrt(2/(p+1)) x h_p - sqrt(p/(p+1)) h_{p-1} started from
//             2^64 exp(-x^2/2) (hard part H4), the arithmetic of predict_shapelets*.cu
//   method 1: linear interpolation in a table T[ix][p] = (h_p(x_ix), h_p(x_{ix+1}) - h_p(x_ix)) on
//             the grid x_ix = ix * dx, 0 <= x < x_max, with h_p(-x) = (-1)^p h_p(x); the table is
//             built on the device in FP64.  Interpolation error <= dx^2 max|h_p''| / 8 <= dx^2 (2p+1) 1.09 / 8.
#include <cmath>

#include "hermite_rec.cuh"
#include "kernels.h"
#include "phase.cuh"

namespace woden {
namespace {

// sqrt(2/(p+1)) and sqrt(p/(p+1)) of the normalised recurrence, as the predict kernels keep theirs
struct NormRec {
    float a[MAX_ORDER + 1], b[MAX_ORDER + 1];
};
constexpr NormRec make_norm_rec()
{
    NormRec t{};
    for (int p = 0; p <= MAX_ORDER; ++p) {
        t.a[p] = (float)csqrt(2.0 / (p + 1.0));
        t.b[p] = p == 0 ? 0.f : (float)csqrt((double)p / (p + 1.0));
    }
    return t;
}
__constant__ NormRec NREC = make_norm_rec();

// table of h_p on the grid, FP64 recurrence in the log-free scaled form (start 2^512 exp(-x^2/2))
__global__ void lut_build_kernel(float2 *__restrict__ T, int n_x, int PM, double dx)
{
    const int ix = blockIdx.x * blockDim.x + threadIdx.x;
    if (ix >= n_x) return;
    for (int side = 0; side < 2; ++side) {
        const double x = (ix + side) * dx;
        double hm = 0.0, h = exp(-0.5 * x * x + 354.0);           // scaled by e^354: no underflow for x <= 37
        const double unscale = exp(-354.0);
        for (int p = 0; p <= PM; ++p) {
            const float val = (float)(h * unscale);
            float2 &e = T[(size_t)ix * (PM + 1) + p];
            if (side == 0) e.x = val; else e.y = val - e.x;
            const double hn = sqrt(2.0 / (p + 1.0)) * x * h - sqrt(p / (p + 1.0)) * hm;
            hm = h; h = hn;
        }
    }
}

__global__ void series_recurrence_kernel(const float *__restrict__ x_in, const float *__restrict__ c, int PM,
                                         long long n, float *__restrict__ out)
{
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    const float x = x_in[i];
    float hm = 0.f, h = ex2_approx(fmaf(x * x, -0.7213475204444817f, 64.f)), acc = 0.f;
    for (int p = 0; p <= PM; ++p) {
        acc = fmaf(c[p], h, acc);
        const float hn = fmaf(NREC.a[p] * x, h, -NREC.b[p] * hm);
        hm = h; h = hn;
    }
    out[i] = acc * 5.421010862427522e-20f;      // 2^-64
}

__global__ void series_lut_kernel(const float *__restrict__ x_in, const float *__restrict__ c, int PM, long long n,
                                  const float2 *__restrict__ T, int n_x, float inv_dx, float *__restrict__ out)
{
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    const float x = x_in[i], ax = fabsf(x) * inv_dx;
    const int ix = (int)ax;
    float acc = 0.f;
    if (ix < n_x) {                                           // beyond the table every h_p has underflowed
        const float fr = ax - (float)ix;
        const float2 *row = T + (size_t)ix * (PM + 1);
        float even = 0.f, odd = 0.f;
        for (int p = 0; p <= PM; ++p) {
            const float2 e = row[p];
            const float h = fmaf(fr, e.y, e.x);
            if (p & 1) odd = fmaf(c[p], h, odd); else even = fmaf(c[p], h, even);
        }
        acc = x < 0.f ? even - odd : even + odd;             // h_p(-x) = (-1)^p h_p(x)
    }
    out[i] = acc;
}

}  // namespace

cudaError_t launch_lut_build(float2 *T, int n_x, int PM, double dx, cudaStream_t st)
{
    lut_build_kernel<<<(n_x + 127) / 128, 128, 0, st>>>(T, n_x, PM, dx); note_launch();
    return cudaGetLastError();
}

cudaError_t launch_series(int method, const float *x, const float *c, int PM, long long n, const float2 *T, int n_x,
                          double dx, float *out, cudaStream_t st)
{
    const unsigned grid = (unsigned)((n + 255) / 256);
    if (method == 0) { series_recurrence_kernel<<<grid, 256, 0, st>>>(x, c, PM, n, out); note_launch(); }
    else { series_lut_kernel<<<grid, 256, 0, st>>>(x, c, PM, n, T, n_x, (float)(1.0 / dx), out); note_launch(); }
    return cudaGetLastError();
}

}  // namespace woden
