// predict_shapelets.cu -- step S6 (+S1, S3, S4, S7) of the hot path for shapelet components
// (Eq 11 with the envelope of Eq 15-17; basis FT Eq 3, :60).
//
// Register engine (the tensor-core engine is predict_shapelets_mma.cu): one
// thread owns NV visibilities, one (baseline, time) pair at NV consecutive channels.  Per shapelet
// and visibility it evaluates the scaled Hermite functions g_p(y) = h_p(y)/lam_p, p = 0..PM, into
// registers by the two-operation recurrence g_{p+1} = (c_p y) g_p - g_{p-1}, walks g_{n1}(x) on
// the fly, and contracts the dense coefficient triangle, one FFMA per coefficient, with the
// coefficients broadcast from shared memory (LDS.128 = 4 coefficients).  The triangle of each
// shapelet is fetched by one bulk async copy (TMA engine) into shared memory.  The order PM is a
// compile-time bucket so that every register index and shared-memory offset is static.  The
// SPARSE variant (truncated models) skips the 4-coefficient chunks whose staged
// mask bit is clear.
//
// i^(n1+n2) (reading G3): the sign part (-1)^floor(p/2) of each factor i^p is folded into the
// stored coefficient by pack.cu, so even n2 add to E, odd n2 to O, and row n1 contributes
// g_{n1}(x) (E + iO) for even n1, g_{n1}(x) (-O + iE) for odd n1.
//
// Underflow (hard part H4): both recurrences start from 2^64 exp(-x^2/2), formed by one ex2, so
// orders up to 100 stay accurate where h_0 underflows; g(x) is scaled back by 2^-64 per row and
// the row sums (which carry g(y)'s 2^64) once per shapelet.
#include <type_traits>

#include "hermite_rec.cuh"
#include "kernels.h"
#include "phase.cuh"
#include "ptx.cuh"

namespace woden {
namespace {

constexpr int SH_THREADS = 128;

struct SParams {
    const double *u_m, *v_m, *w_m;
    const GeoS *geo;
    const float *tri;
    const float *flux;     // [F][n]
    const double *chan_s;  // [F_pad]
    float2 *vis;
    long long n_bt;
    int B, F, n, accumulate;
};

// g_{Q+1}(y) = (c_Q y) g_Q - g_{Q-1}, Q = 1..PM-1, with compile-time constants
template <int PM, int Q>
struct HermY {
    static __device__ __forceinline__ void run(float (&gy)[PM + 1], float y)
    {
        if constexpr (Q < PM) {
            constexpr float cq = REC.c[Q];
            gy[Q + 1] = fmaf(cq * y, gy[Q], -gy[Q - 1]);
            HermY<PM, Q + 1>::run(gy, y);
        }
    }
};

template <int PM, int NV, bool SPARSE, int N1>
struct Rows {
    // process rows N1..PM of the triangle for NV visibilities; gx0[v] = g_{N1}(x_v) * 2^64,
    // gxm[v] = g_{N1-1}(x_v) * 2^64.  One LDS.128 (4 coefficients) feeds 4 NV FFMAs.
    static __device__ __forceinline__ void run(const float *__restrict__ tri, const float (&gy)[NV][PM + 1],
                                               const float (&x)[NV], float (&gx0)[NV], float (&gxm)[NV],
                                               float (&re)[NV], float (&im)[NV], unsigned &mw)
    {
        constexpr int LEN = PM - N1 + 1;
        constexpr int OFF = tri_row_off(PM, N1);
        (void)mw;
        // NV >= 2 already gives 2 NV independent FFMA chains; NV == 1 splits each into two
        constexpr int NS = NV >= 2 ? 1 : 2;
        float aE[NV][NS], aO[NV][NS];
#pragma unroll
        for (int v = 0; v < NV; ++v)
#pragma unroll
            for (int h = 0; h < NS; ++h) { aE[v][h] = 0.f; aO[v][h] = 0.f; }
        const float4 *row = reinterpret_cast<const float4 *>(tri + OFF);
#pragma unroll
        for (int q = 0; q < (LEN + 3) / 4; ++q) {
            if constexpr (SPARSE) {
                // truncated model: chunk bit (warp-uniform) says whether any of the 4 coefficients is set
                const int ch = OFF / 4 + q;
                if (ch % 32 == 0) mw = reinterpret_cast<const unsigned *>(tri + tri_size(PM))[ch / 32];
                if (!((mw >> (ch % 32)) & 1u)) continue;
            }
            const float4 c = row[q];
#pragma unroll
            for (int v = 0; v < NV; ++v) {
                if (4 * q + 0 < LEN) aE[v][0] = fmaf(c.x, gy[v][4 * q + 0], aE[v][0]);
                if (4 * q + 1 < LEN) aO[v][0] = fmaf(c.y, gy[v][4 * q + 1], aO[v][0]);
                if (4 * q + 2 < LEN) aE[v][NS - 1] = fmaf(c.z, gy[v][4 * q + 2], aE[v][NS - 1]);
                if (4 * q + 3 < LEN) aO[v][NS - 1] = fmaf(c.w, gy[v][4 * q + 3], aO[v][NS - 1]);
            }
        }
#pragma unroll
        for (int v = 0; v < NV; ++v) {
            const float E = NS == 2 ? aE[v][0] + aE[v][NS - 1] : aE[v][0];
            const float O = NS == 2 ? aO[v][0] + aO[v][NS - 1] : aO[v][0];
            // gx0 carries 2^64 (hard part H4); gy's 2^64 is undone once per shapelet by the caller
            const float gx = gx0[v] * 5.421010862427522e-20f;     // 2^-64
            if ((N1 & 1) == 0) { re[v] = fmaf(gx, E, re[v]); im[v] = fmaf(gx, O, im[v]); }
            else               { re[v] = fmaf(-gx, O, re[v]); im[v] = fmaf(gx, E, im[v]); }
        }
        if constexpr (N1 < PM) {
            constexpr float cn = REC.c[N1];
#pragma unroll
            for (int v = 0; v < NV; ++v) {
                const float g1 = fmaf(cn * x[v], gx0[v], -gxm[v]);
                gxm[v] = gx0[v]; gx0[v] = g1;
            }
            Rows<PM, NV, SPARSE, N1 + 1>::run(tri, gy, x, gx0, gxm, re, im, mw);
        }
    }
};

// One thread owns NV visibilities: one (baseline, time) pair at NV consecutive channels.  The
// coefficient triangle is broadcast from shared memory; a broadcast LDS.128 occupies the shared
// memory return path for ~2 cycles per SM (profiles/ncu_r1_*.md), i.e. it can feed at most
// 2 x 4 warp-FFMAs per NV = 1, half of the FMA pipe's rate: NV = 2 lifts that bound.
template <int PM, int NV, bool SPARSE>
__global__ void __launch_bounds__(SH_THREADS) predict_shapelets_kernel(const SParams p)
{
    constexpr int TRI = tri_stride(PM);             // triangle + chunk mask
    __shared__ __align__(128) float tri_s[TRI];
    __shared__ __align__(8) uint64_t bar;

    const int tid = threadIdx.x;
    const long long bt = (long long)blockIdx.x * SH_THREADS + tid;
    const bool valid = bt < p.n_bt;
    const int f0 = blockIdx.y * NV;

    if (tid == 0) { mbar_init(&bar, 1); fence_mbar_init(); }

    double u = 0.0, v = 0.0, w = 0.0;
    if (valid) { u = p.u_m[bt]; v = p.v_m[bt]; w = p.w_m[bt]; }
    double s[NV];                                   // S1: nu_f / c (zero past F: chan_s is padded)
#pragma unroll
    for (int i = 0; i < NV; ++i) s[i] = p.chan_s[f0 + i];
    float acc_re[NV], acc_im[NV];
#pragma unroll
    for (int i = 0; i < NV; ++i) { acc_re[i] = 0.f; acc_im[i] = 0.f; }

    for (int j = 0; j < p.n; ++j) {
        __syncthreads();                            // previous triangle fully consumed; barrier init visible
        if (tid == 0) {
            mbar_arrive_expect_tx(&bar, TRI * 4);
            bulk_g2s(tri_s, p.tri + (size_t)j * TRI, TRI * 4, &bar);
        }
        const GeoS &g = p.geo[j];
        // S3: phase in metres; S6 (i)-(ii): x = beta1 K kx', y = beta2 K ky' (Eq 16-17) in metres
        const double D = fma(u, g.l, fma(v, g.m, w * g.n1));
        const double xm = fma(u, g.X[0], fma(v, g.X[1], w * g.X[2]));
        const double ym = fma(u, g.Y[0], fma(v, g.Y[1], w * g.Y[2]));
        float cs[NV], sn[NV], x[NV], S[NV], gx0[NV], gxm[NV];
        float gy[NV][PM + 1];
#pragma unroll
        for (int i = 0; i < NV; ++i) {
            // S4: phasor e^{-2 pi i phi} = cs + i sn
            const float th = theta_from_magic(fma(D, s[i], MAGIC23));
            cs[i] = -__cosf(th); sn[i] = __sinf(th);
            x[i] = (float)(xm * s[i]);              // FP64 product, one rounding to FP32
            const float y = (float)(ym * s[i]);
            S[i] = (f0 + i < p.F) ? p.flux[(size_t)(f0 + i) * p.n + j] : 0.f;
            // S6 (iii): g_p(y), p = 0..PM, scaled by 2^64 during the recurrence (hard part H4)
            gy[i][0] = ex2_approx(fmaf(y * y, -0.7213475204444817f, 64.f));      // 2^64 exp(-y^2/2)
            if constexpr (PM >= 1) {
                constexpr float c0 = REC.c[0];
                gy[i][1] = (c0 * y) * gy[i][0];
                HermY<PM, 1>::run(gy[i], y);
            }
            gx0[i] = ex2_approx(fmaf(x[i] * x[i], -0.7213475204444817f, 64.f));
            gxm[i] = 0.f;
        }

        mbar_wait(&bar, j & 1);
        // S6 (iv): xi = sum_{n1} i^{n1} g_{n1}(x) sum_{n2} i^{n2} f'_{n1 n2} g_{n2}(y)
        float xr[NV], xi[NV];
#pragma unroll
        for (int i = 0; i < NV; ++i) { xr[i] = 0.f; xi[i] = 0.f; }
        unsigned mw = 0u;
        Rows<PM, NV, SPARSE, 0>::run(tri_s, gy, x, gx0, gxm, xr, xi, mw);
        // S7: V += S xi e^{-2 pi i phi}
#pragma unroll
        for (int i = 0; i < NV; ++i) {
            xr[i] *= 5.421010862427522e-20f; xi[i] *= 5.421010862427522e-20f;      // gy's 2^64
            const float zr = xr[i] * cs[i] - xi[i] * sn[i], zi = xr[i] * sn[i] + xi[i] * cs[i];
            acc_re[i] = fmaf(S[i], zr, acc_re[i]);
            acc_im[i] = fmaf(S[i], zi, acc_im[i]);
        }
    }

    if (valid) {
        const long long t = bt / p.B;
        const int b = (int)(bt - t * p.B);
#pragma unroll
        for (int i = 0; i < NV; ++i) {
            if (f0 + i < p.F) {
                float2 *dst = p.vis + ((size_t)t * p.F + f0 + i) * p.B + b;
                float2 val = make_float2(acc_re[i], acc_im[i]);
                if (p.accumulate) { const float2 old = *dst; val.x += old.x; val.y += old.y; }
                *dst = val;
            }
        }
    }
}

// visibilities per thread: registers hold NV (PM + 1) Hermite values
constexpr int nv_for(int PM) { return PM <= 16 ? 4 : (PM <= 40 ? 2 : 1); }

template <int PM>
cudaError_t launch_pm(const SParams &p, int F, bool sparse, cudaStream_t st)
{
    constexpr int NV = nv_for(PM);
    dim3 grid((unsigned)((p.n_bt + SH_THREADS - 1) / SH_THREADS), (unsigned)((F + NV - 1) / NV));
    if (sparse) { predict_shapelets_kernel<PM, NV, true><<<grid, SH_THREADS, 0, st>>>(p); note_launch(); }
    else { predict_shapelets_kernel<PM, NV, false><<<grid, SH_THREADS, 0, st>>>(p); note_launch(); }
    return cudaGetLastError();
}

constexpr int BUCKETS[] = {4, 8, 12, 16, 20, 24, 32, 40, 48, 60, 72, 86, 100};

}  // namespace

int shapelet_order_bucket(int p_max)
{
    if (p_max < 0) return -1;
    for (int b : BUCKETS)
        if (p_max <= b) return b;
    return -1;
}

cudaError_t launch_predict_shapelets(const UvwDev &uvw, const ChanTable &ch, const GeoS *geo, const float *tri,
                                     const float *flux, int n, int PM, bool sparse, float2 *vis, int accumulate,
                                     cudaStream_t st)
{
    SParams p;
    p.u_m = uvw.u_m; p.v_m = uvw.v_m; p.w_m = uvw.w_m;
    p.geo = geo; p.tri = tri; p.flux = flux; p.chan_s = ch.s; p.vis = vis;
    p.n_bt = (long long)uvw.T * uvw.B;
    p.B = uvw.B; p.F = uvw.F; p.n = n; p.accumulate = accumulate;
    switch (PM) {
    case 4: return launch_pm<4>(p, uvw.F, sparse, st);
    case 8: return launch_pm<8>(p, uvw.F, sparse, st);
    case 12: return launch_pm<12>(p, uvw.F, sparse, st);
    case 16: return launch_pm<16>(p, uvw.F, sparse, st);
    case 20: return launch_pm<20>(p, uvw.F, sparse, st);
    case 24: return launch_pm<24>(p, uvw.F, sparse, st);
    case 32: return launch_pm<32>(p, uvw.F, sparse, st);
    case 40: return launch_pm<40>(p, uvw.F, sparse, st);
    case 48: return launch_pm<48>(p, uvw.F, sparse, st);
    case 60: return launch_pm<60>(p, uvw.F, sparse, st);
    case 72: return launch_pm<72>(p, uvw.F, sparse, st);
    case 86: return launch_pm<86>(p, uvw.F, sparse, st);
    case 100: return launch_pm<100>(p, uvw.F, sparse, st);
    }
    return cudaErrorInvalidValue;
}

}  // namespace woden
