// predict_walk.cu -- channel-walking variant of steps S3, S4, S5, S7 for point sources (Eq 9,
// PAPER.md:117) and Gaussians (Eq 11-14), used when the channels are equally
// spaced (all BASELINE.json configs: 80 kHz).  The general path (predict_pg.cu) spends 2 MUFU
// (+1 for Gaussians) per component x visibility; this one spends 4 FP32 lane-operations.
//
// Mapping: one thread owns one (baseline, time) pair and WFT = 32 consecutive channels, held as
// two chains of WH = 16 (channels j and j + 16) that ride in the two lanes of the packed FP32x2
// instructions of sm_100 (SASS FFMA2 / FMUL2).  All 2 x 32 accumulators stay in registers for
// the whole sum over components (no atomics; the paper's atomicAdd, is prior art).
//
// Per (thread, component):
//   D = u_m l + v_m m + w_m (n-1)                       FP64 metres (3 FP64 ops, hard part H1)
//   seeds: q = exp(i theta) at chain position J0 = 7 of both chains by true sin/cos of the FP64
//          phase reduced to its fraction as Q0.32 (4 MUFU), w = exp(i delta), delta = 2 pi D dnu/c (2 MUFU);
//          position J0 + 1 by one complex rotation with w.
//   walk : with channels nu_0 + j dnu the real and imaginary parts of q_j each obey
//          x_{j+1} = 2 cos(delta) x_j - x_{j-1}: ONE FMA per real number per channel.  The chain
//          is walked from the middle outwards (7 steps each way), which bounds the growth of
//          rounding error (~ steps^2 / 2 ulp); every new value is
//          accumulated at once, so only two chain values per direction are live.
//   PTX has no negate for f32x2, so the recurrence runs on y_j = s_j x_j with the sign pattern
//   s = (+,+,-,-) repeating from J0: y_{j+1} = (s_{j+1} s_j) c y_j + y_{j-1} needs only the
//   scalars +c / -c, and s_j is applied once per visibility in the epilogue.
//   Gaussians: xi_j = exp2(-Q s_j^2), s_j = nu_j / c, is walked both ways by the second-order
//   multiplicative recurrence xi_{j+1} = xi_j rho_j, rho_{j+1} = rho_j qq (7 MUFU seeds).
//   The kernel accumulates sum S q with q = exp(+i theta), theta = 2 pi frac(phi);
//   exp(-2 pi i phi) = conj(q), so the epilogue stores (re, -im).
//
// Staging: component geometry (32 / 48 B) and the 32 precomputed fluxes S_k(nu_f) of the tile are
// fetched in blocks of KB = 64 components by 1-D bulk async copies (TMA engine, SASS UBLKCP) into a
// 4-stage ring with full/empty mbarriers: warps release a stage when done and only the producer
// thread waits, so the warps of a CTA drift freely within two blocks (no __syncthreads in the loop).
#include <type_traits>

#include "kernels.h"
#include "phase.cuh"
#include "ptx.cuh"

namespace woden {
namespace {

constexpr int WH = WALK_FT / 2;      // chain length
constexpr int WJ0 = WH / 2 - 1;      // seed position (and WJ0 + 1)
constexpr int WSTAGES = 4;
constexpr int WLAG = 2;              // the producer refills the stage consumed WLAG blocks ago
constexpr int WWARPS = PG_THREADS / 32;

template <typename Geo>
struct WParams {
    const double *u_m, *v_m, *w_m;   // [T][B]
    const Geo *geo;                  // [n_pad]
    const float *flux;               // [n_ftiles][n_pad][WALK_FT], chains interleaved
    const double *chan_s;            // [F_pad], extrapolated past F
    float2 *vis;                     // [T][F][B]
    long long n_bt;                  // T * B
    int B, F, n_pad, accumulate;
    double ds;                       // channel step / c
    unsigned int *err;               // device-side precondition counter (woden_check)
};

// sign pattern of the recurrence: s_j = +1 for (j - J0) mod 4 in {0, 1}, else -1
__host__ __device__ constexpr bool walk_neg(int j) { return (((j - WJ0) % 4 + 4) % 4) >= 2; }

template <bool GAUSS>
struct Seed {
    float cA, sA, cB, sB;     // q at position J0 of chain A (lane 0) and chain B (lane 1)
    float wr, wi;             // exp(i delta)
    float Q;                  // Gaussian: metres-domain quadratic form
};

template <bool GAUSS, typename Geo>
__device__ __forceinline__ void make_seed(const Geo &g, double u, double v, double w, float uf, float vf,
                                          double sfA, double ds, double magic, int kshift, Seed<GAUSS> &sd)
{
    // S3: D = u l + v m + w (n-1), FP64 metres
    const double D = fma(u, g.l, fma(v, g.m, w * g.n1));
    // frac(phase) as signed Q0.32: the low word of phase + 1.5*2^(20+k) holds the phase modulo 2^k
    // turns in units of 2^(k-32) turn, so a left shift by k leaves the fraction (k = 0 while the
    // thread's phases stay below 2^19 turns; see phase_shift_for).  Chain A's seed and the channel
    // step by one DFMA each; chain B's seed, WH channels up, by integer arithmetic (wraps mod 1 turn)
    const unsigned qA = (unsigned)__double2loint(fma(D, sfA, magic)) << kshift;
    const unsigned qd = (unsigned)__double2loint(fma(D, ds, magic)) << kshift;
    const unsigned qB = qA + (unsigned)WH * qd;
    const float thA = (float)(int)qA * Q32_TO_RAD;
    const float thB = (float)(int)qB * Q32_TO_RAD;
    const float thd = (float)(int)qd * Q32_TO_RAD;
    sd.cA = __cosf(thA); sd.sA = __sinf(thA);
    sd.cB = __cosf(thB); sd.sB = __sinf(thB);
    sd.wr = __cosf(thd); sd.wi = __sinf(thd);
    if constexpr (GAUSS) {
        // Eq 13-14 in metres: gx = cg maj (sin pa u + cos pa v), gy = cg min (cos pa u - sin pa v)
        const float gx = fmaf(g.as, uf, g.ac * vf);
        const float gy = fmaf(g.bc, uf, -g.bs * vf);
        sd.Q = fminf(fmaf(gx, gx, gy * gy), 1.0e30f);     // finite: 0 x inf cannot arise below
    } else {
        sd.Q = 0.f;
    }
}

// Gaussian envelope constants of a thread (per chain lane): exponents in units of Q
struct EnvConst {
    f32x2 e0, ef, eb;   // xi at J0; forward ratio J0 -> J0+1; backward ratio J0 -> J0-1
    float e2;           // second difference
};

template <bool GAUSS>
__global__ void __launch_bounds__(PG_THREADS, 2)
predict_walk_kernel(const WParams<typename std::conditional<GAUSS, GeoG, GeoP>::type> p)
{
    using Geo = typename std::conditional<GAUSS, GeoG, GeoP>::type;
    constexpr int FT = WALK_FT, H = WH, J0 = WJ0;
    constexpr int GEO_BYTES = KB * (int)sizeof(Geo);
    constexpr int FLUX_BYTES = KB * FT * 4;
    constexpr int STAGE_BYTES = GEO_BYTES + FLUX_BYTES;

    extern __shared__ __align__(128) unsigned char smem[];
    __shared__ __align__(8) uint64_t full_bar[WSTAGES];
    __shared__ __align__(8) uint64_t empty_bar[WSTAGES];

    const int tid = threadIdx.x;
    const long long bt = (long long)blockIdx.x * PG_THREADS + tid;
    const bool valid = bt < p.n_bt;
    const int ftile = blockIdx.y;
    const int n_blk = p.n_pad / KB;

    const char *geo_src = reinterpret_cast<const char *>(p.geo);
    const char *flux_src = reinterpret_cast<const char *>(p.flux + (size_t)ftile * p.n_pad * FT);

    auto issue = [&](int blk) {
        const int s = blk % WSTAGES;
        mbar_arrive_expect_tx(&full_bar[s], STAGE_BYTES);
        bulk_g2s(smem + s * STAGE_BYTES, geo_src + (size_t)blk * GEO_BYTES, GEO_BYTES, &full_bar[s]);
        bulk_g2s(smem + s * STAGE_BYTES + GEO_BYTES, flux_src + (size_t)blk * FLUX_BYTES, FLUX_BYTES,
                 &full_bar[s]);
    };

    if (tid == 0) {
#pragma unroll
        for (int s = 0; s < WSTAGES; ++s) { mbar_init(&full_bar[s], 1); mbar_init(&empty_bar[s], WWARPS); }
        fence_mbar_init();
    }
    __syncthreads();
    if (tid == 0) {
        const int pre = n_blk < WSTAGES ? n_blk : WSTAGES;
        for (int b = 0; b < pre; ++b) issue(b);
    }

    // S1: this thread's baseline in metres; nu/c at the two chains' seed channels
    double u = 0.0, v = 0.0, w = 0.0;
    if (valid) { u = p.u_m[bt]; v = p.v_m[bt]; w = p.w_m[bt]; }
    const float uf = (float)u, vf = (float)v;
    const double sfA = p.chan_s[ftile * FT + J0];
    const double sfB = p.chan_s[ftile * FT + H + J0];
    const double ds = p.ds;
    // phase range of this thread: |D nu/c| <= sqrt(2) |b| max(nu)/c turns (l^2 + m^2 < 1)
    const double smax = fmax(fabs(p.chan_s[ftile * FT]), fabs(p.chan_s[ftile * FT + FT - 1]));
    int kshift = phase_shift_for(sqrt(fma(u, u, fma(v, v, w * w))) * 1.4142135623730951 * smax);
    if (kshift > PHASE_MAX_SHIFT) {              // beyond 2^28 turns: counted for woden_check
        if (valid) atomicAdd(p.err, 1u);
        kshift = PHASE_MAX_SHIFT;
    }
    const double magic = magic32_shifted(kshift);

    EnvConst ec;
    ec.e0 = ec.ef = ec.eb = 0ull; ec.e2 = 0.f;
    if constexpr (GAUSS) {
        // exponent(s) = -Q s^2, s_j = s_J0 + (j - J0) ds
        const float e0A = (float)(-sfA * sfA), e0B = (float)(-sfB * sfB);
        const float efA = (float)(-(2.0 * sfA * ds + ds * ds)), efB = (float)(-(2.0 * sfB * ds + ds * ds));
        const float ebA = (float)(2.0 * sfA * ds - ds * ds), ebB = (float)(2.0 * sfB * ds - ds * ds);
        ec.e0 = pack2(e0A, e0B); ec.ef = pack2(efA, efB); ec.eb = pack2(ebA, ebB);
        ec.e2 = (float)(-2.0 * ds * ds);
    }

    f32x2 acc_re[H], acc_im[H];
#pragma unroll
    for (int j = 0; j < H; ++j) { acc_re[j] = 0ull; acc_im[j] = 0ull; }

    for (int blk = 0; blk < n_blk; ++blk) {
        const int s = blk % WSTAGES;
        // producer: refill the stage every warp released WLAG blocks ago
        if (tid == 0 && blk >= WLAG && blk - WLAG + WSTAGES < n_blk) {
            const int ob = blk - WLAG;
            mbar_wait(&empty_bar[ob % WSTAGES], (ob / WSTAGES) & 1);
            issue(ob + WSTAGES);
        }
        mbar_wait(&full_bar[s], (blk / WSTAGES) & 1);
        const Geo *g = reinterpret_cast<const Geo *>(smem + s * STAGE_BYTES);
        const unsigned char *fl = smem + s * STAGE_BYTES + GEO_BYTES;

        Seed<GAUSS> sd;
        make_seed<GAUSS>(g[0], u, v, w, uf, vf, sfA, ds, magic, kshift, sd);
#pragma unroll (GAUSS ? 2 : 1)
        for (int k = 0; k < KB; ++k) {
            // software pipeline: the seed (FP64 + MUFU) of component k+1 overlaps the FP32 walk of k
            Seed<GAUSS> nx;
            make_seed<GAUSS>(g[k + 1 < KB ? k + 1 : k], u, v, w, uf, vf, sfA, ds, magic, kshift, nx);

            const ulonglong2 *fl2 = reinterpret_cast<const ulonglong2 *>(fl + (size_t)k * FT * 4);
            const float cf = sd.wr + sd.wr;                    // c = 2 cos(delta)
            const f32x2 c2 = pack2(cf, cf), nc2 = pack2(-cf, -cf);
            const f32x2 wr = pack2(sd.wr, sd.wr), wi = pack2(sd.wi, sd.wi), nwi = pack2(-sd.wi, -sd.wi);
            // positions J0 (MUFU) and J0 + 1 (one complex rotation); s_J0 = s_{J0+1} = +1
            const f32x2 r0 = pack2(sd.cA, sd.cB), i0 = pack2(sd.sA, sd.sB);
            const f32x2 r1 = fma2(i0, nwi, mul2(r0, wr));
            const f32x2 i1 = fma2(r0, wi, mul2(i0, wr));

            f32x2 xf = 0ull, rf = 0ull, xb = 0ull, rb = 0ull, qq = 0ull;
            if constexpr (GAUSS) {
                float a, b;
                const f32x2 Q2 = pack2(sd.Q, sd.Q);
                unpack2(mul2(Q2, ec.e0), a, b);
                xb = pack2(ex2_approx(a), ex2_approx(b));                 // xi at J0
                // The step ratios are clamped to finite values: where xi at J0 has flushed to zero
                // (Q s^2 > 126) a ratio 2^(+big) would give 0 x inf = NaN; clamped, the chain is an
                // exact 0, which it is to 2^-90 because the walking path is only taken when a chain
                // spans at most +-12.5 % in frequency (api.cu).  Where xi at J0 is normal the ratio
                // exponents are <= 2 x 126 x 1/64 and the clamp is idle.
                unpack2(mul2(Q2, ec.ef), a, b);
                rf = pack2(ex2_approx(fminf(a, 126.f)), ex2_approx(fminf(b, 126.f)));   // xi_{J0+1} / xi_{J0}
                unpack2(mul2(Q2, ec.eb), a, b);
                rb = pack2(ex2_approx(fminf(a, 126.f)), ex2_approx(fminf(b, 126.f)));   // xi_{J0-1} / xi_{J0}
                const float qf = ex2_approx(sd.Q * ec.e2);
                qq = pack2(qf, qf);
                xf = mul2(xb, rf);                                        // xi at J0 + 1
                rf = mul2(rf, qq);                                        // ratio J0+1 -> J0+2
            }

            // flux words: 64-bit word j holds (S[j], S[j + H]); one LDS.128 = words 2q, 2q + 1.
            // Each value is accumulated right AFTER the recurrence step that consumes it as its
            // multiplicand, so both instructions read it in the same operand slot (register reuse
            // cache: the register file delivers only two 32-bit operands per cycle, which makes an
            // FFMA2 with three fresh register pairs cost 3 cycles instead of 2; profiles/pipes_r1.txt).
            static_assert(J0 % 2 == 1, "seed position must be the high word of a 128-bit flux granule");
            // ---- forward: y_{j+1} = (s_{j+1} s_j) c y_j + y_{j-1}; accumulates positions J0+1 .. H-1
            {
                f32x2 ra = r0, ia = i0, rc = r1, ic = i1, Skeep = 0ull;
#pragma unroll
                for (int j = J0 + 1; j < H; ++j) {
                    f32x2 rn = 0ull, in = 0ull;
                    if (j + 1 < H) {
                        const f32x2 cc = (walk_neg(j + 1) != walk_neg(j)) ? nc2 : c2;
                        rn = fma2(cc, rc, ra); in = fma2(cc, ic, ia);
                    }
                    f32x2 Sj;
                    if (j % 2 == 1) { Sj = Skeep; }                            // high word of the granule in hand
                    else { const ulonglong2 q = fl2[j / 2]; Sj = q.x; Skeep = q.y; }
                    if constexpr (GAUSS) { Sj = mul2(Sj, xf); if (j + 1 < H) { xf = mul2(xf, rf); rf = mul2(rf, qq); } }
                    acc_re[j] = fma2(Sj, rc, acc_re[j]);
                    acc_im[j] = fma2(Sj, ic, acc_im[j]);
                    ra = rc; ia = ic; rc = rn; ic = in;
                }
            }
            // ---- backward: y_{j-1} = (s_{j-1} s_j) c y_j + y_{j+1}; accumulates positions J0 .. 0
            {
                f32x2 ra = r1, ia = i1, rc = r0, ic = i0, Skeep = 0ull;
#pragma unroll
                for (int j = J0; j >= 0; --j) {
                    f32x2 rn = 0ull, in = 0ull;
                    if (j >= 1) {
                        const f32x2 cc = (walk_neg(j - 1) != walk_neg(j)) ? nc2 : c2;
                        rn = fma2(cc, rc, ra); in = fma2(cc, ic, ia);
                    }
                    f32x2 Sj;
                    if (j % 2 == 0) { Sj = Skeep; }                            // low word of the granule in hand
                    else { const ulonglong2 q = fl2[j / 2]; Sj = q.y; Skeep = q.x; }
                    if constexpr (GAUSS) { Sj = mul2(Sj, xb); if (j >= 1) { xb = mul2(xb, rb); rb = mul2(rb, qq); } }
                    acc_re[j] = fma2(Sj, rc, acc_re[j]);
                    acc_im[j] = fma2(Sj, ic, acc_im[j]);
                    ra = rc; ia = ic; rc = rn; ic = in;
                }
            }
            sd = nx;
        }
        // consumer release: this warp is done reading stage s
        __syncwarp();
        if ((tid & 31) == 0) mbar_arrive(&empty_bar[s]);
    }

    // S7: exp(-2 pi i phi) = conj(q): V = (re, -im); coalesced float2 stores along b
    if (valid) {
        const long long t = bt / p.B;
        const int b = (int)(bt - t * p.B);
#pragma unroll
        for (int j = 0; j < FT; ++j) {
            const int f = ftile * FT + j;
            float a0, a1, b0, b1;
            unpack2(acc_re[j % H], a0, a1);
            unpack2(acc_im[j % H], b0, b1);
            float re = j < H ? a0 : a1;
            float im = j < H ? b0 : b1;
            if (walk_neg(j % H)) { re = -re; im = -im; }      // s_j of the recurrence
            if (f < p.F) {
                float2 *dst = p.vis + ((size_t)t * p.F + f) * p.B + b;
                float2 val = make_float2(re, -im);
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
    WParams<Geo> p;
    p.u_m = uvw.u_m; p.v_m = uvw.v_m; p.w_m = uvw.w_m;
    p.geo = geo; p.flux = flux; p.chan_s = ch.s; p.vis = vis;
    p.n_bt = (long long)uvw.T * uvw.B;
    p.B = uvw.B; p.F = uvw.F; p.n_pad = n_pad; p.accumulate = accumulate; p.ds = ch.ds; p.err = err;
    const int smem = WSTAGES * KB * ((int)sizeof(Geo) + WALK_FT * 4);
    auto kern = predict_walk_kernel<GAUSS>;
    cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, smem);
    if (e != cudaSuccess) return e;
    dim3 grid((unsigned)((p.n_bt + PG_THREADS - 1) / PG_THREADS), (unsigned)(ch.F_pad / WALK_FT));
    kern<<<grid, PG_THREADS, smem, st>>>(p);
    return cudaGetLastError();
}

}  // namespace

cudaError_t launch_walk_points(const UvwDev &uvw, const ChanTable &ch, const GeoP *geo, const float *flux,
                               int n_pad, float2 *vis, int accumulate, unsigned int *err, cudaStream_t st)
{
    return launch<false>(uvw, ch, geo, flux, n_pad, vis, accumulate, err, st);
}

cudaError_t launch_walk_gaussians(const UvwDev &uvw, const ChanTable &ch, const GeoG *geo, const float *flux,
                                  int n_pad, float2 *vis, int accumulate, unsigned int *err, cudaStream_t st)
{
    return launch<true>(uvw, ch, geo, flux, n_pad, vis, accumulate, err, st);
}

}  // namespace woden
