// predict_pg.cu -- general path of steps S1, S3, S4, S5, S7 for point sources (Eq 9,
// PAPER.md:117) and Gaussians (Eq 11-14): any channel list, one true sin/cos
// (and one exp2 for Gaussians) per component x visibility.  (Equally spaced channels take the
// channel-walking kernel of predict_walk.cu instead.)
//
// Mapping: one thread owns one (baseline, time) pair and FT = 16 consecutive channels; the complex
// accumulators for those visibilities live in registers for the whole sum over components (no
// atomics -- the paper's atomicAdd, is prior art for a GTX 1080 Ti).  A CTA of 256
// threads streams every component through shared memory in blocks of KB: a 32/48-byte geometry
// record and the FT precomputed fluxes S_k(nu_f) per component, fetched by 1-D bulk async copies
// (TMA engine, SASS UBLKCP) into a 3-stage mbarrier ring and read back as warp-wide broadcasts.
//
// Phase (hard part H1/H2): D = u_m l + v_m m + w_m (n-1) in FP64 metres, once per (thread,
// component).  Per channel one DFMA forms D * (nu_f/c) + 1.5*2^29, whose low mantissa word holds
// frac(phase) to 2^-23 turn; a LOP3 turns it into a float in [1,2) and one FFMA into an angle
// in [-pi, pi) for MUFU.SIN / MUFU.COS.  No FP64->FP32 conversion instruction is issued.
// The kernel accumulates sum S q with q = exp(+i theta), theta = 2 pi (frac(phi) - 1/2);
// exp(-2 pi i phi) = -conj(q), so the epilogue stores (-re, im).
#include <type_traits>

#include "kernels.h"
#include "phase.cuh"
#include "ptx.cuh"

namespace woden {
namespace {

template <typename Geo>
struct PGParams {
    const double *u_m, *v_m, *w_m;   // [T][B]
    const Geo *geo;                  // [n_pad]
    const float *flux;               // [n_ftiles][n_pad][FT]
    const double *chan_s;            // [F_pad]
    const float *chan_ns2;           // [F_pad]
    float2 *vis;                     // [T][F][B]
    long long n_bt;                  // T * B
    int B, F, n_pad, accumulate;
    unsigned int *err;               // device-side precondition counter (woden_check)
};

template <int FT, bool GAUSS>
__global__ void __launch_bounds__(PG_THREADS, 2)
predict_pg_kernel(const PGParams<typename std::conditional<GAUSS, GeoG, GeoP>::type> p)
{
    using Geo = typename std::conditional<GAUSS, GeoG, GeoP>::type;
    constexpr int GEO_BYTES = KB * (int)sizeof(Geo);
    constexpr int FLUX_BYTES = KB * FT * 4;
    constexpr int STAGE_BYTES = GEO_BYTES + FLUX_BYTES;
    static_assert(FT % 4 == 0, "flux rows are read as 128-bit words");

    extern __shared__ __align__(128) unsigned char smem[];
    __shared__ __align__(8) uint64_t full_bar[NSTAGE];

    const int tid = threadIdx.x;
    const long long bt = (long long)blockIdx.x * PG_THREADS + tid;
    const bool valid = bt < p.n_bt;
    const int ftile = blockIdx.y;
    const int n_blk = p.n_pad / KB;

    const char *geo_src = reinterpret_cast<const char *>(p.geo);
    const char *flux_src = reinterpret_cast<const char *>(p.flux + (size_t)ftile * p.n_pad * FT);

    if (tid == 0) {
#pragma unroll
        for (int s = 0; s < NSTAGE; ++s) mbar_init(&full_bar[s], 1);
        fence_mbar_init();
    }
    __syncthreads();
    if (tid == 0) {
        const int pre = n_blk < NSTAGE ? n_blk : NSTAGE;
        for (int s = 0; s < pre; ++s) {
            mbar_arrive_expect_tx(&full_bar[s], STAGE_BYTES);
            bulk_g2s(smem + s * STAGE_BYTES, geo_src + (size_t)s * GEO_BYTES, GEO_BYTES, &full_bar[s]);
            bulk_g2s(smem + s * STAGE_BYTES + GEO_BYTES, flux_src + (size_t)s * FLUX_BYTES, FLUX_BYTES,
                     &full_bar[s]);
        }
    }

    // S1: this thread's baseline in metres; channel scales nu_f / c for its tile
    double u = 0.0, v = 0.0, w = 0.0;
    if (valid) { u = p.u_m[bt]; v = p.v_m[bt]; w = p.w_m[bt]; }
    const float uf = (float)u, vf = (float)v;
    (void)uf; (void)vf;

    double sf[FT];
    float ns2[GAUSS ? FT : 1];
#pragma unroll
    for (int j = 0; j < FT; ++j) sf[j] = p.chan_s[ftile * FT + j];
    if (GAUSS) {
#pragma unroll
        for (int j = 0; j < FT; ++j) ns2[j] = p.chan_ns2[ftile * FT + j];
    }
    (void)ns2;
    {
        // the MAGIC23 hand-off holds while |phase| < 2^28 turns; |D nu/c| <= sqrt(2) |b| max(nu)/c
        double smax = 0.0;
#pragma unroll
        for (int j = 0; j < FT; ++j) smax = fmax(smax, sf[j]);
        const double bound = sqrt(fma(u, u, fma(v, v, w * w))) * 1.4142135623730951 * smax;
        if (valid && !(bound < 268435456.0)) atomicAdd(p.err, 1u);
    }

    float acc_re[FT], acc_im[FT];
#pragma unroll
    for (int j = 0; j < FT; ++j) { acc_re[j] = 0.f; acc_im[j] = 0.f; }

    for (int blk = 0; blk < n_blk; ++blk) {
        const int s = blk % NSTAGE;
        mbar_wait(&full_bar[s], (blk / NSTAGE) & 1);
        const Geo *g = reinterpret_cast<const Geo *>(smem + s * STAGE_BYTES);
        const unsigned char *fl = smem + s * STAGE_BYTES + GEO_BYTES;

#pragma unroll 2
        for (int k = 0; k < KB; ++k) {
            // S3: D = u l + v m + w (n-1), FP64 metres
            const double D = fma(u, g[k].l, fma(v, g[k].m, w * g[k].n1));
            float Q = 0.f;
            if (GAUSS) {
                const GeoG &gg = *reinterpret_cast<const GeoG *>(&g[k]);
                const float gx = fmaf(gg.as, uf, gg.ac * vf);
                const float gy = fmaf(gg.bc, uf, -gg.bs * vf);
                Q = fminf(fmaf(gx, gx, gy * gy), 1.0e30f);
            }
            (void)Q;
            float S[FT];
            const float4 *fl4 = reinterpret_cast<const float4 *>(fl + (size_t)k * FT * 4);
#pragma unroll
            for (int j4 = 0; j4 < FT / 4; ++j4) {
                const float4 t = fl4[j4];
                S[4 * j4 + 0] = t.x; S[4 * j4 + 1] = t.y; S[4 * j4 + 2] = t.z; S[4 * j4 + 3] = t.w;
            }
#pragma unroll
            for (int j = 0; j < FT; ++j) {
                const float th = theta_from_magic(fma(D, sf[j], MAGIC23));
                const float sn = __sinf(th), cs = __cosf(th);       // S4: 2 MUFU
                float Sj = S[j];
                if (GAUSS) Sj *= ex2_approx(Q * ns2[j]);            // S5: 1 MUFU
                acc_re[j] = fmaf(Sj, cs, acc_re[j]);                // S7 (sign fixed in the epilogue)
                acc_im[j] = fmaf(Sj, sn, acc_im[j]);
            }
        }
        __syncthreads();      // every thread is done reading stage s
        if (tid == 0 && blk + NSTAGE < n_blk) {
            const int nb = blk + NSTAGE;
            mbar_arrive_expect_tx(&full_bar[s], STAGE_BYTES);
            bulk_g2s(smem + s * STAGE_BYTES, geo_src + (size_t)nb * GEO_BYTES, GEO_BYTES, &full_bar[s]);
            bulk_g2s(smem + s * STAGE_BYTES + GEO_BYTES, flux_src + (size_t)nb * FLUX_BYTES, FLUX_BYTES,
                     &full_bar[s]);
        }
    }

    // S7: exp(-2 pi i phi) = -conj(q): V = (-re, im); coalesced float2 stores along b
    if (valid) {
        const long long t = bt / p.B;
        const int b = (int)(bt - t * p.B);
#pragma unroll
        for (int j = 0; j < FT; ++j) {
            const int f = ftile * FT + j;
            if (f < p.F) {
                float2 *dst = p.vis + ((size_t)t * p.F + f) * p.B + b;
                float2 val = make_float2(-acc_re[j], acc_im[j]);
                if (p.accumulate) { const float2 old = *dst; val.x += old.x; val.y += old.y; }
                *dst = val;
            }
        }
    }
}

template <bool GAUSS, typename Geo>
cudaError_t launch(const UvwDev &uvw, const ChanTable &ch, const Geo *geo, const float *flux, int n_pad,
                   float2 *vis, int accumulate, unsigned int *err, cudaStream_t st)
{
    constexpr int FT = PG_FT;
    PGParams<Geo> p;
    p.u_m = uvw.u_m; p.v_m = uvw.v_m; p.w_m = uvw.w_m;
    p.geo = geo; p.flux = flux; p.chan_s = ch.s; p.chan_ns2 = ch.ns2; p.vis = vis;
    p.n_bt = (long long)uvw.T * uvw.B;
    p.B = uvw.B; p.F = uvw.F; p.n_pad = n_pad; p.accumulate = accumulate; p.err = err;
    const int smem = NSTAGE * KB * ((int)sizeof(Geo) + FT * 4);
    auto kern = predict_pg_kernel<FT, GAUSS>;
    cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, smem);
    if (e != cudaSuccess) return e;
    dim3 grid((unsigned)((p.n_bt + PG_THREADS - 1) / PG_THREADS), (unsigned)(ch.F_pad / FT));
    kern<<<grid, PG_THREADS, smem, st>>>(p); note_launch();
    return cudaGetLastError();
}

}  // namespace

cudaError_t launch_predict_points(const UvwDev &uvw, const ChanTable &ch, const GeoP *geo, const float *flux,
                                  int n_pad, float2 *vis, int accumulate, unsigned int *err, cudaStream_t st)
{
    return launch<false>(uvw, ch, geo, flux, n_pad, vis, accumulate, err, st);
}

cudaError_t launch_predict_gaussians(const UvwDev &uvw, const ChanTable &ch, const GeoG *geo, const float *flux,
                                     int n_pad, float2 *vis, int accumulate, unsigned int *err, cudaStream_t st)
{
    return launch<true>(uvw, ch, geo, flux, n_pad, vis, accumulate, err, st);
}

}  // namespace woden
