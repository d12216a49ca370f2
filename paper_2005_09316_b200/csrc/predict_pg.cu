// predict_pg.cu -- steps S1, S3, S4, S5, S7 of the hot path for point sources (Eq 9,
// PAPER.md:117) and Gaussians (Eq 11-14).
//
// Mapping: one thread owns one (baseline, time) pair and FT consecutive channels; the complex
// accumulators for those FT visibilities live in registers for the whole sum over components
// (no atomics -- the paper's atomicAdd, is prior art for a GTX 1080 Ti).  A CTA
// of 256 threads streams every component through shared memory in blocks of KB: a 32/48-byte
// geometry record and the FT precomputed fluxes S_k(nu_f) per component, fetched by 1-D bulk
// async copies (TMA engine, SASS UBLKCP) into a 3-stage mbarrier ring and read back as
// warp-wide broadcasts.
//
// Phase (hard part H1/H2): D = u_m l + v_m m + w_m (n-1) in FP64 metres, once per (thread,
// component).  Per channel one DFMA forms D * (nu_f/c) + 1.5*2^29, whose low mantissa word holds
// frac(phase) to 2^-23 turn; a LOP3 turns it into a float in [1,2) and one FFMA into an angle
// in [-pi, pi) for MUFU.SIN / MUFU.COS.  No FP64->FP32 conversion instruction is issued.
//
// WALK variant (uniformly spaced channels only).  With
// channels nu_0 + j dnu the phasor q_j = exp(i theta_j) advances by a fixed angle
// delta = 2 pi D dnu/c per channel, so its real and imaginary parts each obey the three-term
// recurrence  x_{j+1} = 2 cos(delta) x_j - x_{j-1}  -- ONE FMA per real part per channel instead
// of 2 MUFU.  The FT channels of a thread form two chains of H = FT/2 (channels j and j + H),
// each seeded in its middle: q at position H/2-1 by a true sincos (MUFU), q at H/2 by one complex
// rotation with w = exp(i delta) (MUFU sincos of delta, shared by both chains); the recurrence
// then runs at most H/2 steps outwards in both directions, which bounds the growth of the
// rounding error of c = 2 cos(delta) to ~ (H/2)^3/12 ulp-of-MUFU (~1e-5 for H = 8).
// The two chains ride in the two lanes of the packed FP32x2 instructions of sm_100
// (fma/mul.rn.f32x2, SASS FFMA2/FMUL2): same FMA-pipe work, half the issue slots.
// PTX has no negate for f32x2, so the recurrence runs on u_j = s_j x_j with the sign pattern
// s = (+,-,-,+,+,-,-,+): then u_{j+1} = (s_{j+1} s_j) c u_j + u_{j-1} needs only +c / -c scalars,
// and s_j is applied once per visibility in the epilogue.
// The Gaussian envelope exp2(-Q s^2) is advanced by a second-order multiplicative recurrence.
// The kernel accumulates Q = sum S q with q = exp(+i theta), theta = 2 pi (frac(phi) - 1/2);
// exp(-2 pi i phi) = -conj(q), so the epilogue stores (-Q_re, Q_im).
#include <type_traits>

#include "kernels.h"
#include "ptx.cuh"

namespace woden {
namespace {

constexpr double MAGIC23 = 805306368.0;  // 1.5 * 2^29 : ulp = 2^-23 turn
constexpr double MAGIC32 = 1572864.0;    // 1.5 * 2^20 : low word = frac as Q0.32
constexpr float TWO_PI_F = 6.283185307179586f;
constexpr float THREE_PI_F = 9.42477796076938f;
constexpr float Q32_TO_RAD = 1.4629180792671596e-09f;   // 2 pi / 2^32

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
    double ds;                       // channel step / c (WALK)
};

// angle in [-pi, pi) equal to 2 pi (frac(phi) - 1/2), from r = phi + MAGIC23
__device__ __forceinline__ float theta_from_magic(double r)
{
    const unsigned lo = (unsigned)__double2loint(r);
    const float x = __uint_as_float((lo & 0x007fffffu) | 0x3f800000u);   // 1 + frac(phi)
    return fmaf(x, TWO_PI_F, -THREE_PI_F);
}

__device__ __forceinline__ float ex2_approx(float x)
{
    float y;
    asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}

// ---- packed FP32x2 (sm_100+): one instruction, two independent lanes ----------------------
typedef unsigned long long f32x2;
__device__ __forceinline__ f32x2 pack2(float lo, float hi)
{
    f32x2 r;
    asm("mov.b64 %0, {%1, %2};" : "=l"(r) : "f"(lo), "f"(hi));
    return r;
}
__device__ __forceinline__ void unpack2(f32x2 v, float &lo, float &hi)
{
    asm("mov.b64 {%0, %1}, %2;" : "=f"(lo), "=f"(hi) : "l"(v));
}
__device__ __forceinline__ f32x2 fma2(f32x2 a, f32x2 b, f32x2 c)
{
    f32x2 d;
    asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(d) : "l"(a), "l"(b), "l"(c));
    return d;
}
__device__ __forceinline__ f32x2 mul2(f32x2 a, f32x2 b)
{
    f32x2 d;
    asm("mul.rn.f32x2 %0, %1, %2;" : "=l"(d) : "l"(a), "l"(b));
    return d;
}

// position of channel j (0..FT-1) inside a flux-table tile: chains interleaved, so that one
// 64-bit shared-memory word holds (S[j], S[j + FT/2])
template <int FT>
__host__ __device__ constexpr int flux_pos(int j) { return FT >= 2 ? ((j % (FT / 2)) * 2 + j / (FT / 2)) : 0; }

// sign pattern of the WALK recurrence: s_j = +1 for (j - J0) mod 4 in {0, 1}, else -1
__host__ __device__ constexpr bool walk_neg(int j, int J0) { return (((j - J0) % 4 + 4) % 4) >= 2; }

template <int FT, bool GAUSS, bool WALK>
__global__ void __launch_bounds__(PG_THREADS, 2)
predict_pg_kernel(const PGParams<typename std::conditional<GAUSS, GeoG, GeoP>::type> p)
{
    using Geo = typename std::conditional<GAUSS, GeoG, GeoP>::type;
    constexpr int H = FT / 2;                       // chain length (WALK), pair stride
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

    // general path: every channel's scale; WALK: the two chains' seed channels only
    constexpr int J0 = H / 2 - 1;
    double sf[WALK ? 2 : FT];
    float ns2[(GAUSS && !WALK) ? FT : 1];
    if (WALK) {
        sf[0] = p.chan_s[ftile * FT + J0];
        sf[1] = p.chan_s[ftile * FT + H + J0];
    } else {
#pragma unroll
        for (int j = 0; j < FT; ++j) sf[j] = p.chan_s[ftile * FT + j];
        if (GAUSS) {
#pragma unroll
            for (int j = 0; j < FT; ++j) ns2[j] = p.chan_ns2[ftile * FT + j];
        }
    }
    (void)ns2;
    // WALK Gaussian: exponent(s) = -Q s^2 with s_j = s_head + j ds, from each chain's first channel:
    //   xi_0 = exp2(Q e0), rho_0 = exp2(Q e1), qq = exp2(Q e2), xi_{j+1} = xi_j rho_j, rho_{j+1} = rho_j qq
    float g_e0[2] = {0.f, 0.f}, g_e1[2] = {0.f, 0.f}, g_e2 = 0.f;
    if (GAUSS && WALK) {
#pragma unroll
        for (int c = 0; c < 2; ++c) {
            const double s0 = p.chan_s[ftile * FT + c * H];
            g_e0[c] = (float)(-s0 * s0);
            g_e1[c] = (float)(-(2.0 * s0 * p.ds + p.ds * p.ds));
        }
        g_e2 = (float)(-2.0 * p.ds * p.ds);
    }
    (void)g_e0; (void)g_e1; (void)g_e2;

    // accumulators: general path scalar per channel; WALK packed (channel j, channel j + H)
    float acc_re[WALK ? 1 : FT], acc_im[WALK ? 1 : FT];
    f32x2 acc_re2[WALK ? H : 1], acc_im2[WALK ? H : 1];
    if (WALK) {
#pragma unroll
        for (int j = 0; j < H; ++j) { acc_re2[j] = 0ull; acc_im2[j] = 0ull; }
    } else {
#pragma unroll
        for (int j = 0; j < FT; ++j) { acc_re[j] = 0.f; acc_im[j] = 0.f; }
    }
    (void)acc_re; (void)acc_im; (void)acc_re2; (void)acc_im2;

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
                Q = fmaf(gx, gx, gy * gy);
            }
            (void)Q;
            if (!WALK) {
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
                    float Sj = S[flux_pos<FT>(j)];
                    if (GAUSS) Sj *= ex2_approx(Q * ns2[j]);            // S5: 1 MUFU
                    acc_re[j] = fmaf(Sj, cs, acc_re[j]);                // S7 (sign fixed in the epilogue)
                    acc_im[j] = fmaf(Sj, sn, acc_im[j]);
                }
            } else {
                // seeds: q = exp(i theta) at position J0 of both chains (4 MUFU)
                const float thA = theta_from_magic(fma(D, sf[0], MAGIC23));
                const float thB = theta_from_magic(fma(D, sf[1], MAGIC23));
                f32x2 ur[H], ui[H];
                ur[J0] = pack2(__cosf(thA), __cosf(thB));
                ui[J0] = pack2(__sinf(thA), __sinf(thB));
                // w = exp(+2 pi i D ds) (2 MUFU), the same for both chains; c = 2 cos(delta)
                const int qd = __double2loint(fma(D, p.ds, MAGIC32));   // frac(D ds) as signed Q0.32
                const float thd = (float)qd * Q32_TO_RAD;
                const float wrf = __cosf(thd), wif = __sinf(thd);
                const f32x2 wr = pack2(wrf, wrf), wi = pack2(wif, wif), nwi = pack2(-wif, -wif);
                const float cf = wrf + wrf;
                const f32x2 c2 = pack2(cf, cf), nc2 = pack2(-cf, -cf);
                // position J0+1 by one complex rotation (s_{J0} = s_{J0+1} = +1)
                ur[J0 + 1] = fma2(ui[J0], nwi, mul2(ur[J0], wr));
                ui[J0 + 1] = fma2(ur[J0], wi, mul2(ui[J0], wr));
                // outwards: u_{j+1} = (s_{j+1} s_j) c u_j + u_{j-1};  u_{j-1} = (s_{j-1} s_j) c u_j + u_{j+1}
#pragma unroll
                for (int j = J0 + 1; j + 1 < H; ++j) {
                    const f32x2 cc = (walk_neg(j + 1, J0) != walk_neg(j, J0)) ? nc2 : c2;
                    ur[j + 1] = fma2(cc, ur[j], ur[j - 1]);
                    ui[j + 1] = fma2(cc, ui[j], ui[j - 1]);
                }
#pragma unroll
                for (int j = J0; j >= 1; --j) {
                    const f32x2 cc = (walk_neg(j - 1, J0) != walk_neg(j, J0)) ? nc2 : c2;
                    ur[j - 1] = fma2(cc, ur[j], ur[j + 1]);
                    ui[j - 1] = fma2(cc, ui[j], ui[j + 1]);
                }
                f32x2 xi = 0ull, rho = 0ull, qq = 0ull;
                if (GAUSS) {
                    xi = pack2(ex2_approx(Q * g_e0[0]), ex2_approx(Q * g_e0[1]));
                    rho = pack2(ex2_approx(Q * g_e1[0]), ex2_approx(Q * g_e1[1]));
                    const float qf = ex2_approx(Q * g_e2);
                    qq = pack2(qf, qf);
                }
                (void)xi; (void)rho; (void)qq;
                const ulonglong2 *fl2 = reinterpret_cast<const ulonglong2 *>(fl + (size_t)k * FT * 4);
#pragma unroll
                for (int j2 = 0; j2 < H / 2; ++j2) {
                    const ulonglong2 t = fl2[j2];                       // (S[j],S[j+H]), (S[j+1],S[j+1+H])
#pragma unroll
                    for (int e = 0; e < 2; ++e) {
                        const int j = 2 * j2 + e;
                        f32x2 Sj = e ? t.y : t.x;
                        if (GAUSS) {
                            Sj = mul2(Sj, xi);
                            if (j + 1 < H) { xi = mul2(xi, rho); rho = mul2(rho, qq); }
                        }
                        acc_re2[j] = fma2(Sj, ur[j], acc_re2[j]);
                        acc_im2[j] = fma2(Sj, ui[j], acc_im2[j]);
                    }
                }
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

    // S7: exp(-2 pi i phi) = -conj(q): V = (-Q_re, Q_im); coalesced float2 stores along b
    if (valid) {
        const long long t = bt / p.B;
        const int b = (int)(bt - t * p.B);
#pragma unroll
        for (int j = 0; j < FT; ++j) {
            const int f = ftile * FT + j;
            float re, im;
            if (WALK) {
                float a0, a1, b0, b1;
                unpack2(acc_re2[j % H], a0, a1);
                unpack2(acc_im2[j % H], b0, b1);
                re = j < H ? a0 : a1;
                im = j < H ? b0 : b1;
            } else {
                re = acc_re[j]; im = acc_im[j];
            }
            if (WALK && walk_neg(j % H, J0)) { re = -re; im = -im; }     // s_j of the recurrence
            if (f < p.F) {
                float2 *dst = p.vis + ((size_t)t * p.F + f) * p.B + b;
                float2 val = make_float2(-re, im);
                if (p.accumulate) { const float2 old = *dst; val.x += old.x; val.y += old.y; }
                *dst = val;
            }
        }
    }
}

template <bool GAUSS, bool WALK, typename Geo>
cudaError_t launch(const UvwDev &uvw, const ChanTable &ch, const Geo *geo, const float *flux, int n_pad,
                   float2 *vis, int accumulate, cudaStream_t st)
{
    constexpr int FT = PG_FT;
    PGParams<Geo> p;
    p.u_m = uvw.u_m; p.v_m = uvw.v_m; p.w_m = uvw.w_m;
    p.geo = geo; p.flux = flux; p.chan_s = ch.s; p.chan_ns2 = ch.ns2; p.vis = vis;
    p.n_bt = (long long)uvw.T * uvw.B;
    p.B = uvw.B; p.F = uvw.F; p.n_pad = n_pad; p.accumulate = accumulate; p.ds = ch.ds;
    const int smem = NSTAGE * KB * ((int)sizeof(Geo) + FT * 4);
    auto kern = predict_pg_kernel<FT, GAUSS, WALK>;
    cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, smem);
    if (e != cudaSuccess) return e;
    dim3 grid((unsigned)((p.n_bt + PG_THREADS - 1) / PG_THREADS), (unsigned)(ch.F_pad / FT));
    kern<<<grid, PG_THREADS, smem, st>>>(p);
    return cudaGetLastError();
}

}  // namespace

int pg_smem_bytes(bool gauss) { return NSTAGE * KB * ((gauss ? (int)sizeof(GeoG) : (int)sizeof(GeoP)) + PG_FT * 4); }

cudaError_t launch_predict_points(const UvwDev &uvw, const ChanTable &ch, const GeoP *geo, const float *flux,
                                  int n_pad, float2 *vis, int accumulate, bool walk, cudaStream_t st)
{
    return walk ? launch<false, true>(uvw, ch, geo, flux, n_pad, vis, accumulate, st)
                : launch<false, false>(uvw, ch, geo, flux, n_pad, vis, accumulate, st);
}

cudaError_t launch_predict_gaussians(const UvwDev &uvw, const ChanTable &ch, const GeoG *geo, const float *flux,
                                     int n_pad, float2 *vis, int accumulate, bool walk, cudaStream_t st)
{
    return walk ? launch<true, true>(uvw, ch, geo, flux, n_pad, vis, accumulate, st)
                : launch<true, false>(uvw, ch, geo, flux, n_pad, vis, accumulate, st);
}

}  // namespace woden
