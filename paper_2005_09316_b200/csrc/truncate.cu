// truncate.cu -- model truncation of PAPER.md section 5.3 (Eq 23-24, :273-275):
// rank the components (or shapelet basis functions) by |I_j|, largest first, and keep the largest N_comp
// with  sum_{j <= N_comp} |I_j| <= f_comp sum_{j <= N_tot} |I_j|.
//
// Three small kernels: ranks by counting (rank_j = number of components with a larger |I|, ties in
// original order: a stable descending sort without a sort), the running sum over the ranked list by ONE
// thread in list order (the same association as a sequential cumulative sum, so N_comp is decided on
// exactly the same FP64 numbers as the oracle's), and the keep flags.
#include "kernels.h"

namespace woden {
namespace {

// |I_j| as ranked: a non-finite weight (NaN would make the order partial and leave slots of the ranked list
// unwritten) counts as 0 -- it ranks last -- and is reported through the context's error counter
__device__ __forceinline__ double trunc_abs(double w) { return isfinite(w) ? fabs(w) : 0.0; }

__global__ void trunc_rank_kernel(const double *__restrict__ w, int n, int *__restrict__ rank, double *__restrict__ sorted,
                                  unsigned int *__restrict__ err)
{
    const int j = blockIdx.x * blockDim.x + threadIdx.x;
    if (j >= n) return;
    if (!isfinite(w[j])) atomicAdd(err, 1u);
    const double a = trunc_abs(w[j]);
    int r = 0;
    for (int i = 0; i < n; ++i) {
        const double b = trunc_abs(w[i]);
        r += (b > a) || (b == a && i < j);
    }
    rank[j] = r;
    sorted[r] = a;
}

__global__ void trunc_count_kernel(const double *__restrict__ sorted, int n, double f_comp, int *__restrict__ n_keep)
{
    if (threadIdx.x || blockIdx.x) return;
    if (f_comp >= 1.0) { *n_keep = n; return; }
    double total = 0.0;
    for (int k = 0; k < n; ++k) total += sorted[k];
    const double limit = f_comp * total * (1.0 + 1e-15);       // Eq 23 with one rounding of slack
    double run = 0.0;
    int keep = 0;
    for (int k = 0; k < n; ++k) {
        run += sorted[k];
        if (run <= limit) keep = k + 1; else break;
    }
    *n_keep = keep;
}

__global__ void trunc_flag_kernel(const int *__restrict__ rank, int n, const int *__restrict__ n_keep, int *__restrict__ keep)
{
    const int j = blockIdx.x * blockDim.x + threadIdx.x;
    if (j < n) keep[j] = rank[j] < *n_keep ? 1 : 0;
}

// Eq 25 for the listed basis functions of ONE shapelet component: weight_i = |C_i S0| x the
// beam-convolved basis image's absolute pixel sum of (n1_i, n2_i) (abs_sums over the full triangle of order pm,
// n1-major: q = n1 (pm + 1) - n1 (n1 - 1) / 2 + n2).  An order pair outside the triangle gets weight 0 and is counted.
__global__ void eq25_weight_kernel(const double *__restrict__ coeff, const int *__restrict__ n1, const int *__restrict__ n2,
                                   int count, int pm, double s0, const double *__restrict__ abs_sums,
                                   double *__restrict__ weights, unsigned int *__restrict__ err)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= count) return;
    const int a = n1[i], b = n2[i];
    if (a < 0 || b < 0 || a + b > pm) { weights[i] = 0.0; atomicAdd(err, 1u); return; }
    const int q = a * (pm + 1) - a * (a - 1) / 2 + b;
    weights[i] = fabs(coeff[i] * s0) * abs_sums[q];
}

}  // namespace

cudaError_t launch_eq25_weights(const double *coeff, const int *n1, const int *n2, int count, int pm, double s0,
                                const double *abs_sums, double *weights, unsigned int *err, cudaStream_t st)
{
    if (count <= 0) return cudaSuccess;
    eq25_weight_kernel<<<(count + 255) / 256, 256, 0, st>>>(coeff, n1, n2, count, pm, s0, abs_sums, weights, err); note_launch();
    return cudaGetLastError();
}

cudaError_t launch_truncate_select(const double *weights, int n, double f_comp, int *rank, double *sorted, int *keep,
                                   int *n_keep, unsigned int *err, cudaStream_t st)
{
    trunc_rank_kernel<<<(n + 127) / 128, 128, 0, st>>>(weights, n, rank, sorted, err); note_launch();
    trunc_count_kernel<<<1, 32, 0, st>>>(sorted, n, f_comp, n_keep); note_launch();
    trunc_flag_kernel<<<(n + 255) / 256, 256, 0, st>>>(rank, n, n_keep, keep); note_launch();
    return cudaGetLastError();
}

}  // namespace woden
