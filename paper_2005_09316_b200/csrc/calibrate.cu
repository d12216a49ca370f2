// calibrate.cu -- SURVEY.md §8(f) NEXT-3: the consumer of the hot path in the paper, per-antenna
// complex gain fit and peel (section 5.1, Eq 18-22).
//
// Per (time, frequency) cell and iteration the paper solves x = [A^T A]^-1 A^T b (Eq 22) for the
// additive gain errors e, with A the 2B x 2N real design matrix of the linearised residual
//   R_ij = V_ij - g_i g_j^* I_ij  ~  e_i g_j^* I_ij + g_i e_j^* I_ij        (Eq 18-21; reading G15)
// and updates g <- g + e, 10 times from g = 1.  Written in the relative error eps_i = e_i / g_i the
// normal equations of that least-squares problem decouple into two REAL N x N systems that need
// only the N x N matrix W_ij = |I_ij|^2 (W_ii = 0):
//   q_i = |g_i|^2,  d_i = sum_j W_ij q_j,  rho_i = [ sum_j g_j conj(I_ij) V_ij  -  g_i d_i ] / g_i
//   (Q D + Q W Q) Re eps = q o Re rho          symmetric positive definite
//   (Q D - Q W Q) Im eps = q o Im rho          symmetric, null vector (1,..,1): the overall phase
// (I_ji = conj I_ij, V_ji = conj V_ij).  One CTA per cell keeps W in shared memory (FP64, N x N) and
// solves both systems together by Jacobi-preconditioned conjugate gradients; the singular one is
// started from zero with its right-hand side projected on the range, and the result is moved to
// the minimum-norm solution in e (the one Eq 22 has as a pseudo-inverse; reading G16) by removing
// the component along the gauge direction i g.  All FP64.  Matrix-vector products read W[j][i]
// (symmetric) so that a warp's lanes touch consecutive shared-memory words.
#include <cmath>

#include "kernels.h"

namespace woden {
namespace {

constexpr int CAL_THREADS = 512;

struct CalParams {
    const float2 *data, *model;   // [cells][B] complex64
    double2 *gains;               // [cells][N] complex128
    int N, n_iter, cg_max;
    long long B;
    double cg_tol2;               // squared relative residual at which CG stops
    double cg_abs2;               // squared absolute size of the remaining correction at which CG stops
};

// index of pair (i, j), i < j, in i-major order
__device__ __forceinline__ long long pair_index(int i, int j, int N)
{
    return (long long)i * (2 * N - i - 1) / 2 + (j - i - 1);
}

__device__ __forceinline__ double warp_sum(double v)
{
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}

// sum of up to four per-thread values over the CTA; every thread gets the totals
template <int NV>
__device__ __forceinline__ void block_sum(double (&v)[NV], double *scratch /* [NV][CAL_THREADS / 32] */)
{
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
#pragma unroll
    for (int k = 0; k < NV; ++k) {
        const double s = warp_sum(v[k]);
        if (lane == 0) scratch[k * (CAL_THREADS / 32) + wid] = s;
    }
    __syncthreads();
#pragma unroll
    for (int k = 0; k < NV; ++k) {
        double s = 0.0;
#pragma unroll
        for (int w = 0; w < CAL_THREADS / 32; ++w) s += scratch[k * (CAL_THREADS / 32) + w];
        v[k] = s;
    }
    __syncthreads();
}

__global__ void __launch_bounds__(CAL_THREADS) calibrate_kernel(const CalParams p)
{
    extern __shared__ __align__(16) double sm[];
    const int N = p.N, tid = threadIdx.x;
    double *W = sm;                              // [N][N]
    double *q = W + (size_t)N * N;               // |g|^2
    double *d = q + N;                           // sum_j W_ij q_j
    double *gre = d + N, *gim = gre + N;         // gains
    double *rhs0 = gim + N, *rhs1 = rhs0 + N;    // q o Re rho, q o Im rho
    double *x0 = rhs1 + N, *x1 = x0 + N;         // CG iterates (Re eps, Im eps)
    double *r0 = x1 + N, *r1 = r0 + N;           // CG residuals
    double *p0 = r1 + N, *p1 = p0 + N;           // CG directions (pre-multiplied by q for the product)
    double *a0 = p1 + N, *a1 = a0 + N;           // M p
    double *scratch = a1 + N;                    // [4][CAL_THREADS / 32]
    double *part = scratch + 4 * (CAL_THREADS / 32);   // [split][2][N] partial products, split N <= CAL_THREADS
    double *invd = part + 2 * (size_t)(N > CAL_THREADS ? N : CAL_THREADS);    // Jacobi preconditioner 1 / (q d)
    double2 *qp = reinterpret_cast<double2 *>(invd + N);   // q o (p0, p1); offset N (N + 15) + 4 (CAL_THREADS / 32) + 2 max(N, CAL_THREADS) doubles is even: 16-byte aligned
    const int split = N >= CAL_THREADS ? 1 : CAL_THREADS / N;
    const int jchunk = (N + split - 1) / split;

    const float2 *V = p.data + (size_t)blockIdx.x * p.B;
    const float2 *I = p.model + (size_t)blockIdx.x * p.B;

    // W_ij = |I_ij|^2 (FP64 from the complex64 model), symmetric, zero diagonal
    for (int idx = tid; idx < N * N; idx += CAL_THREADS) {
        const int i = idx / N, j = idx - i * N;
        double w = 0.0;
        if (i != j) {
            const float2 m = I[i < j ? pair_index(i, j, N) : pair_index(j, i, N)];
            w = (double)m.x * m.x + (double)m.y * m.y;
        }
        W[idx] = w;
    }
    for (int i = tid; i < N; i += CAL_THREADS) { gre[i] = 1.0; gim[i] = 0.0; }
    __syncthreads();

    for (int it = 0; it < p.n_iter; ++it) {
        for (int i = tid; i < N; i += CAL_THREADS) q[i] = gre[i] * gre[i] + gim[i] * gim[i];
        __syncthreads();
        // d_i and rho_i: one warp per antenna i, lanes over the partners j (coalesced rows of I, V)
        for (int i = tid >> 5; i < N; i += CAL_THREADS / 32) {
            double di = 0.0, sr = 0.0, si = 0.0;
#pragma unroll 4
            for (int j = tid & 31; j < N; j += 32) {
                if (j == i) continue;
                di = fma(W[(size_t)i * N + j], q[j], di);
                const long long b = i < j ? pair_index(i, j, N) : pair_index(j, i, N);
                const float2 m = I[b], v = V[b];
                // C_ij = conj(I_ij) V_ij for the ordered pair (i, j); the stored pair is (min, max)
                double cr = (double)m.x * v.x + (double)m.y * v.y;
                double ci = (double)m.x * v.y - (double)m.y * v.x;
                if (i > j) ci = -ci;
                sr += gre[j] * cr - gim[j] * ci;             // g_j C_ij
                si += gre[j] * ci + gim[j] * cr;
            }
            di = warp_sum(di); sr = warp_sum(sr); si = warp_sum(si);
            if ((tid & 31) == 0) {
                d[i] = di;
                const double rr = sr - gre[i] * di, ri = si - gim[i] * di;       // r_i = sum - g_i d_i
                // rho = r / g, then scaled by q = |g|^2:  q rho = r conj(g)
                rhs0[i] = rr * gre[i] + ri * gim[i];
                rhs1[i] = ri * gre[i] - rr * gim[i];
            }
        }
        __syncthreads();
        // range projection of the singular system's right-hand side (null vector: all ones)
        {
            double s[1] = {0.0};
            for (int i = tid; i < N; i += CAL_THREADS) s[0] += rhs1[i];
            block_sum<1>(s, scratch);
            const double mean = s[0] / N;
            for (int i = tid; i < N; i += CAL_THREADS) rhs1[i] -= mean;
        }
        // Jacobi-preconditioned CG on both systems, x = 0 start.  qp[j] = q_j (p0_j, p1_j) is formed
        // once per iteration so the product loop reads one W word and one 16-byte broadcast per j.
        double rz[3] = {0.0, 0.0, 0.0};
        for (int i = tid; i < N; i += CAL_THREADS) {
            const double dg = q[i] * d[i], inv = dg > 0.0 ? 1.0 / dg : 0.0;
            invd[i] = inv;
            rz[2] += dg;
            x0[i] = 0.0; x1[i] = 0.0;
            r0[i] = rhs0[i]; r1[i] = rhs1[i];
            p0[i] = r0[i] * inv; p1[i] = r1[i] * inv;
            qp[i] = make_double2(q[i] * p0[i], q[i] * p1[i]);
            rz[0] += r0[i] * p0[i]; rz[1] += r1[i] * p1[i];
        }
        block_sum<3>(rz, scratch);
        // stop at a residual reduced by sqrt(cg_tol2), or once the correction it stands for is below
        // cg_abs in the (q d)-weighted rms of eps (late outer iterations start almost converged)
        const double floor0 = fmax(p.cg_tol2 * rz[0], p.cg_abs2 * rz[2]);
        const double floor1 = fmax(p.cg_tol2 * rz[1], p.cg_abs2 * rz[2]);
        for (int cg = 0; cg < p.cg_max; ++cg) {
            const bool live0 = rz[0] > floor0;
            const bool live1 = rz[1] > floor1;
            if (!live0 && !live1) break;
            // t = W (q o p): `split` thread groups each take a slice of the partners j of antenna i
            if (tid < split * N) {
                const int i = tid % N, h = tid / N;
                const int j0 = h * jchunk, j1 = min(N, j0 + jchunk);
                const double *Wc = W + i;
                double t0 = 0.0, t1 = 0.0, u0 = 0.0, u1 = 0.0;
                int j = j0;
#pragma unroll 4
                for (; j + 1 < j1; j += 2) {
                    const double wa = Wc[(size_t)j * N], wb = Wc[(size_t)(j + 1) * N];
                    const double2 a = qp[j], b = qp[j + 1];
                    t0 = fma(wa, a.x, t0); t1 = fma(wa, a.y, t1);
                    u0 = fma(wb, b.x, u0); u1 = fma(wb, b.y, u1);
                }
                if (j < j1) { const double wa = Wc[(size_t)j * N]; const double2 a = qp[j]; t0 = fma(wa, a.x, t0); t1 = fma(wa, a.y, t1); }
                part[(2 * h) * N + i] = t0 + u0;
                part[(2 * h + 1) * N + i] = t1 + u1;
            }
            __syncthreads();
            double pa[2] = {0.0, 0.0};
            for (int i = tid; i < N; i += CAL_THREADS) {
                double t0 = 0.0, t1 = 0.0;
                for (int h = 0; h < split; ++h) { t0 += part[(2 * h) * N + i]; t1 += part[(2 * h + 1) * N + i]; }
                a0[i] = q[i] * (d[i] * p0[i] + t0);
                a1[i] = q[i] * (d[i] * p1[i] - t1);
                pa[0] += p0[i] * a0[i]; pa[1] += p1[i] * a1[i];
            }
            block_sum<2>(pa, scratch);
            const double al0 = live0 && pa[0] > 0.0 ? rz[0] / pa[0] : 0.0;
            const double al1 = live1 && pa[1] > 0.0 ? rz[1] / pa[1] : 0.0;
            double rzn[2] = {0.0, 0.0};
            for (int i = tid; i < N; i += CAL_THREADS) {
                x0[i] += al0 * p0[i]; x1[i] += al1 * p1[i];
                r0[i] -= al0 * a0[i]; r1[i] -= al1 * a1[i];
                rzn[0] += r0[i] * r0[i] * invd[i]; rzn[1] += r1[i] * r1[i] * invd[i];
            }
            block_sum<2>(rzn, scratch);
            const double be0 = live0 ? rzn[0] / rz[0] : 0.0;
            const double be1 = live1 ? rzn[1] / rz[1] : 0.0;
            for (int i = tid; i < N; i += CAL_THREADS) {
                if (live0) p0[i] = r0[i] * invd[i] + be0 * p0[i];
                if (live1) p1[i] = r1[i] * invd[i] + be1 * p1[i];
                qp[i] = make_double2(live0 ? q[i] * p0[i] : 0.0, live1 ? q[i] * p1[i] : 0.0);
            }
            if (live0) rz[0] = rzn[0];
            if (live1) rz[1] = rzn[1];
            __syncthreads();
        }
        // gauge: minimum norm in e = g eps  <=>  sum_i q_i Im eps_i = 0
        {
            double s[2] = {0.0, 0.0};
            for (int i = tid; i < N; i += CAL_THREADS) { s[0] += q[i] * x1[i]; s[1] += q[i]; }
            block_sum<2>(s, scratch);
            const double phi = s[1] > 0.0 ? s[0] / s[1] : 0.0;
            // g <- g + e = g (1 + eps)
            for (int i = tid; i < N; i += CAL_THREADS) {
                const double er = x0[i], ei = x1[i] - phi;
                const double nr = gre[i] + gre[i] * er - gim[i] * ei;
                const double ni = gim[i] + gre[i] * ei + gim[i] * er;
                gre[i] = nr; gim[i] = ni;
            }
        }
        __syncthreads();
    }
    for (int i = tid; i < N; i += CAL_THREADS)
        p.gains[(size_t)blockIdx.x * N + i] = make_double2(gre[i], gim[i]);
}

// out = V - g_i g_j^* I (Eq 20 with the fitted gains).  One CTA per cell: gains in shared memory,
// one warp per baseline row i, lanes over j > i (consecutive visibilities).  HBM-bound: 24 B per
// visibility.
__global__ void __launch_bounds__(CAL_THREADS) peel_kernel(const float2 *__restrict__ data,
                                                           const float2 *__restrict__ model,
                                                           const double2 *__restrict__ gains, float2 *__restrict__ out,
                                                           int N, long long B)
{
    extern __shared__ __align__(16) double2 gs[];
    const size_t cell = blockIdx.x;
    for (int i = threadIdx.x; i < N; i += CAL_THREADS) gs[i] = gains[cell * N + i];
    __syncthreads();
    const float2 *v = data + cell * B, *m = model + cell * B;
    float2 *o = out + cell * B;
    for (int i = threadIdx.x >> 5; i < N - 1; i += CAL_THREADS / 32) {
        const double2 gi = gs[i];
        const long long row = pair_index(i, i + 1, N);
        for (int j = i + 1 + (threadIdx.x & 31); j < N; j += 32) {
            const double2 gj = gs[j];
            const double pr = gi.x * gj.x + gi.y * gj.y, pi = gi.y * gj.x - gi.x * gj.y;      // g_i conj(g_j)
            const long long b = row + (j - i - 1);
            const float2 mm = m[b], vv = v[b];
            o[b] = make_float2((float)((double)vv.x - (pr * mm.x - pi * mm.y)),
                               (float)((double)vv.y - (pr * mm.y + pi * mm.x)));
        }
    }
}

}  // namespace

size_t calibrate_smem_bytes(int N)
{
    return ((size_t)N * N + 20 * (size_t)N + 2 + 4 * (CAL_THREADS / 32) + 2 * (size_t)(N > CAL_THREADS ? N : CAL_THREADS)) * sizeof(double);
}

cudaError_t launch_calibrate(const float2 *data, const float2 *model, double2 *gains, int N, long long cells, int n_iter,
                             cudaStream_t st)
{
    CalParams p;
    p.data = data; p.model = model; p.gains = gains; p.N = N; p.n_iter = n_iter;
    p.B = (long long)N * (N - 1) / 2;
    p.cg_max = 2 * N + 10;
    p.cg_tol2 = 1e-26;             // residual reduced by 1e-13
    p.cg_abs2 = 1e-28;             // or the remaining relative gain correction below 1e-14
    const size_t smem = calibrate_smem_bytes(N);
    cudaError_t e = cudaFuncSetAttribute(calibrate_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    calibrate_kernel<<<(unsigned)cells, CAL_THREADS, smem, st>>>(p); note_launch();
    return cudaGetLastError();
}

cudaError_t launch_peel(const float2 *data, const float2 *model, const double2 *gains, float2 *out, int N,
                        long long cells, cudaStream_t st)
{
    const long long B = (long long)N * (N - 1) / 2;
    peel_kernel<<<(unsigned)cells, CAL_THREADS, (size_t)N * sizeof(double2), st>>>(data, model, gains, out, N, B); note_launch();
    return cudaGetLastError();
}

}  // namespace woden
