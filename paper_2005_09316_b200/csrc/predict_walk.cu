// predict_walk.cu -- channel-walking variant of steps S3, S4, S5, S7 for point sources (Eq 9,
// PAPER.md:117) and Gaussians (Eq 11-14), used when the channels are equally
// spaced (all BASELINE.json configs: 80 kHz).  The general path (predict_pg.cu) spends 2 MUFU
// (+1 for Gaussians) per component x visibility; this one spends 4 FP32 lane-operations.
//
// Mapping: one thread owns one (baseline, time) pair and WFT = 32 consecutive channels, held as
// ONE chain that is walked from its middle outwards: the two lanes of the packed FP32x2
// instructions of sm_100 (SASS FFMA2 / FMUL2) carry the two DIRECTIONS (lane 0: channel J0+1+t,
// lane 1: channel J0-t at step t = 0..15, J0 = 15).  All 2 x 32 accumulators stay in registers for
// the sum over the components of one launch (no atomics; the paper's atomicAdd, is
// prior art).
//
// Per (thread, component):
//   D = u_m l + v_m m + w_m (n-1)                       FP64 metres (3 FP64 ops, hard part H1)
//   seeds: q = exp(i theta) at chain position J0 = 15 by true sin/cos of the FP64 phase reduced to
//          its fraction as Q0.32 (2 MUFU), w = exp(i delta), delta = 2 pi D dnu/c (2 MUFU);
//          position J0 + 1 by one complex rotation with w.  ONE seed serves all 32 channels (the
//          round-2 kernel seeded two chains of 16 with 6 MUFU).
//   walk : with channels nu_0 + j dnu the real and imaginary parts of q_j each obey
//          x_{j+1} = 2 cos(delta) x_j - x_{j-1}: ONE FMA per real number per channel.  The chain
//          is walked from the middle outwards (15 steps each way, both directions in one packed
//          instruction), which bounds the growth of rounding error (~ steps^2 / 2 ulp, DESIGN.md
//          "Tolerance"); every new value is accumulated at once, so only two chain values are live.
//   PTX has no negate for f32x2, so the recurrence runs on y_j = s_j x_j with the sign pattern
//   s = (+,+,-,-) repeating from J0: y_{j+1} = (s_{j+1} s_j) c y_j + y_{j-1} needs only the
//   scalars +c / -c, and s_j is applied once per visibility in the epilogue.  The pattern is
//   symmetric about J0 + 1/2, so both lanes of a step carry the same sign: s(t) = - for t mod 4 in {1, 2}.
//   Gaussians: xi_j = exp2(-Q s_j^2), s_j = nu_j / c, is walked both ways (one lane each) by the
//   second-order multiplicative recurrence xi_{t+1} = xi_t rho_t, rho_{t+1} = rho_t qq (5 MUFU seeds).
//   The kernel accumulates sum S q with q = exp(+i theta), theta = 2 pi frac(phi);
//   exp(-2 pi i phi) = conj(q), so the epilogue stores (re, -im).
//
// Operand delivery.  The register file of an SM sub-partition has an even
// and an odd bank, each feeding one 32-bit operand per lane per clock, and every instruction holds
// the read stage for max(#even, #odd) distinct registers it reads (operands served by the
// operand-reuse cache -- same register, same slot, previous instruction -- are free).  Measured on
// the B200, the kernel's time is 1.05 x the sum of those read cycles over ALL its instructions
// (profiles/walk_rf_r2.md), not the FMA pipe's 2 cycles per FFMA2.  Hence:
//   * everything a component contributes besides the thread's own baseline -- its direction
//     (l, m, n-1), its envelope scales and its 32 fluxes S_k(nu_f) of the channel tile -- is the same
//     for every thread of the launch and is served from the CONSTANT BANK: ptxas loads it into
//     uniform registers (SASS LDCU) and the accumulate becomes FFMA2 R, R, UR, R;
//   * the recurrence is written fma2(y_j, c, y_{j-1}) with the chain value FIRST: ptxas then keeps
//     y_j in operand slot A of the recurrence (flagged .reuse) and of the accumulate that follows
//     it, so a (recurrence, accumulate) pair reads 3 + 1 register pairs instead of 3 + 2.
// There is no shared-memory staging, no barrier and no divergent branch in the kernel.  The price
// is that the constant bank is fixed per launch: one launch covers one channel tile and one block
// of <= 204 (186) components (32 KB of the 64 KB bank); the accumulators are carried from launch
// to launch through the output buffer (a read-modify-write of 8 B per visibility per launch,
// < 10 % of the launch's duration on HBM and overlapped by the other CTAs).  Launches alternate
// between the two halves of the bank and between two streams that own disjoint parts of the
// output, so the copy into one half and the tail of one launch hide behind the launch running
// from the other half.
#include <mutex>
#include <type_traits>

#include "kernels.h"
#include "phase.cuh"

namespace woden {
namespace {

#ifndef WALK_THREADS
#define WALK_THREADS 128
#define WALK_CTAS 4
#endif
constexpr int WTHREADS = WALK_THREADS;   // (baseline, time) pairs per CTA
constexpr int WH = WALK_FT / 2;      // steps each way = packed accumulator pairs per thread
constexpr int WJ0 = WH - 1;          // seed position (and WJ0 + 1): the middle of the 32-channel chain
// step t of the walk: lane 0 is at channel WJ0 + 1 + t (forward), lane 1 at channel WJ0 - t (backward)
__host__ __device__ constexpr int walk_chan(int t, int lane) { return lane ? WJ0 - t : WJ0 + 1 + t; }

// one launch's constants: per component its geometry record and 16 flux words (S[j], S[j + WH]),
// interleaved so that every constant-bank offset in the loop body is a small immediate
template <typename Geo>
struct WalkRec {
    Geo geo;
    ulonglong2 flux[WH / 2];          // 128-bit granule q = words 2q, 2q + 1; word t = (S[J0+1+t], S[J0-t])
};
template <typename Geo>
struct WalkBlock {
    static constexpr int KC = WALK_CB_BYTES / (int)sizeof(WalkRec<Geo>);
    WalkRec<Geo> rec[KC];
};
static_assert(sizeof(WalkBlock<GeoP>) <= WALK_CB_BYTES && sizeof(WalkBlock<GeoG>) <= WALK_CB_BYTES, "constant block");
static_assert(WalkBlock<GeoP>::KC == WALK_KC_POINTS && WalkBlock<GeoG>::KC == WALK_KC_GAUSS, "kernels.h constants");

__constant__ __align__(16) unsigned char CBANK[2 * WALK_CB_BYTES];

struct WParams {
    const double *u_m, *v_m, *w_m;   // [T][B]
    float2 *vis;                     // [T][F][B]
    long long bt0, bt1;              // (baseline, time) pairs of this launch: [bt0, bt1)
    int B, F, ftile;
    int k0, n_k;                     // first record of this launch's block in the bank; components in it
    int load_acc;                    // 1: continue from the values in vis, 0: start from zero
    int first;                       // first block of the call: range violations are counted once
    double sf0, ds, smax;            // nu/c at the seed channel J0, channel step / c, max |nu/c| of the tile
    unsigned int *err;               // device-side precondition counter (woden_check)
};

// sign pattern of the recurrence: s_j = +1 for (j - J0) mod 4 in {0, 1}, else -1; at step t both lanes
// (j - J0 = 1 + t and -t) carry the same sign
__host__ __device__ constexpr bool walk_neg(int t) { return (t & 3) == 1 || (t & 3) == 2; }
static_assert(!walk_neg(0) && walk_neg(1) && walk_neg(2) && !walk_neg(3), "sign pattern");

template <bool GAUSS>
struct Seed {
    float r0, i0, r1, i1;     // q at positions J0 and J0 + 1
    float wr;                 // cos(delta)
    float Q;                  // Gaussian: metres-domain quadratic form
};

template <bool GAUSS, typename Geo>
__device__ __forceinline__ void make_seed(const Geo &g, double u, double v, double w, float uf, float vf,
                                          double sf0, double ds, double magic, int kshift, float qmax, Seed<GAUSS> &sd)
{
    // S3: D = u l + v m + w (n-1), FP64 metres
    const double D = fma(u, g.l, fma(v, g.m, w * g.n1));
    // frac(phase) as signed Q0.32: the low word of phase + 1.5*2^(20+k) holds the phase modulo 2^k
    // turns in units of 2^(k-32) turn, so a left shift by k leaves the fraction (k = 0 while the
    // thread's phases stay below 2^19 turns; see phase_shift_for).  The seed and the channel step by
    // one DFMA each.
    const unsigned q0 = (unsigned)__double2loint(fma(D, sf0, magic)) << kshift;
    const unsigned qd = (unsigned)__double2loint(fma(D, ds, magic)) << kshift;
    const float th0 = (float)(int)q0 * Q32_TO_RAD;
    const float thd = (float)(int)qd * Q32_TO_RAD;
    sd.r0 = __cosf(th0); sd.i0 = __sinf(th0);
    const float wi = __sinf(thd);
    sd.wr = __cosf(thd);
    // position J0 + 1 by one complex rotation with w = exp(i delta)
    sd.r1 = fmaf(-sd.i0, wi, sd.r0 * sd.wr);
    sd.i1 = fmaf(sd.r0, wi, sd.i0 * sd.wr);
    if constexpr (GAUSS) {
        // Eq 13-14 in metres: gx = cg maj (sin pa u + cos pa v), gy = cg min (cos pa u - sin pa v)
        const float gx = fmaf(g.as, uf, g.ac * vf);
        const float gy = fmaf(g.bc, uf, -g.bs * vf);
        sd.Q = fminf(fmaf(gx, gx, gy * gy), qmax);        // see EnvConst::qmax: 0 x inf cannot arise below
    } else {
        sd.Q = 0.f;
    }
}

// Gaussian envelope constants of a thread (per chain lane): exponents in units of Q
struct EnvConst {
    f32x2 e0, er;       // lanes (forward, backward): xi at (J0+1, J0); first ratio (J0+1 -> J0+2, J0 -> J0-1)
    float e2;           // second difference (the same in both directions)
    // Largest Q this thread walks with: Q |er| <= 126 in both lanes, so the first step ratios 2^(Q e) are
    // finite; the ratio that is > 1 (towards lower |nu|) only shrinks along the walk, the other one only
    // underflows.  Where the clamp bites, xi at the seeds is 2^(-126 |e0| / |er|) with |e0| / |er| ~
    // s / (2 ds) >= 32 (the walking path is only taken when the channel step is at most 1/64 of the lowest
    // frequency, api.cu): it has flushed to zero, as has the true envelope at every channel of the chain
    // (at its far end |nu| is still >= 0.75 of the seed's: < 2^-2000), and the chain is an exact 0 instead
    // of 0 x inf = NaN.  Otherwise the clamp is idle.
    float qmax;
};

template <bool GAUSS>
__global__ void __launch_bounds__(WTHREADS, WALK_CTAS) predict_walk_kernel(const WParams p)
{
    using Geo = typename std::conditional<GAUSS, GeoG, GeoP>::type;
    constexpr int FT = WALK_FT, H = WH;
    // the bank as one array of records; k0 is a run-time value on purpose: the record index then
    // carries the half's base and every constant-bank offset below is a small immediate
    const WalkRec<Geo> *const rec = reinterpret_cast<const WalkRec<Geo> *>(CBANK);
    const int k0 = p.k0, k1 = p.k0 + p.n_k;

    const long long bt = p.bt0 + (long long)blockIdx.x * WTHREADS + threadIdx.x;
    const bool valid = bt < p.bt1;

    // S1: this thread's baseline in metres; nu/c at the two chains' seed channels
    double u = 0.0, v = 0.0, w = 0.0;
    if (valid) { u = p.u_m[bt]; v = p.v_m[bt]; w = p.w_m[bt]; }
    const float uf = (float)u, vf = (float)v;
    const double sf0 = p.sf0, ds = p.ds;
    // phase range of this thread: |D nu/c| <= sqrt(2) |b| max(nu)/c turns (l^2 + m^2 < 1)
    int kshift = phase_shift_for(sqrt(fma(u, u, fma(v, v, w * w))) * 1.4142135623730951 * p.smax);
    if (kshift > PHASE_MAX_SHIFT) {              // beyond 2^28 turns: counted for woden_check
        if (valid && p.first) atomicAdd(p.err, 1u);
        kshift = PHASE_MAX_SHIFT;
    }
    const double magic = magic32_shifted(kshift);

    EnvConst ec;
    ec.e0 = ec.er = 0ull; ec.e2 = 0.f; ec.qmax = 0.f;
    if constexpr (GAUSS) {
        // exponent(s) = -Q s^2, s_j = s_J0 + (j - J0) ds
        const double s1 = sf0 + ds;
        const float e0f = (float)(-s1 * s1), e0b = (float)(-sf0 * sf0);
        const float erf = (float)(-(2.0 * s1 * ds + ds * ds)), erb = (float)(2.0 * sf0 * ds - ds * ds);
        ec.e0 = pack2(e0f, e0b); ec.er = pack2(erf, erb);
        ec.e2 = (float)(-2.0 * ds * ds);
        ec.qmax = fminf(126.f / fmaxf(fabsf(erf), fabsf(erb)), 1.0e30f);
    }

    // accumulators: y_j = s_j x_j of q = conj(exp(-2 pi i phi)); the output holds V = (s re, -s im),
    // a transformation that is its own inverse, so a later launch reloads them the same way
    const long long t = valid ? bt / p.B : 0;
    const int b = valid ? (int)(bt - t * p.B) : 0;
    float2 *const row = p.vis + ((size_t)t * p.F + (size_t)p.ftile * FT) * p.B + b;
    f32x2 acc_re[H], acc_im[H];
    if (p.load_acc) {
#pragma unroll
        for (int j = 0; j < H; ++j) {
            const int jf = walk_chan(j, 0), jb = walk_chan(j, 1);
            float2 a = make_float2(0.f, 0.f), c = make_float2(0.f, 0.f);
            if (valid && p.ftile * FT + jf < p.F) a = row[(size_t)jf * p.B];
            if (valid && p.ftile * FT + jb < p.F) c = row[(size_t)jb * p.B];
            const float sg = walk_neg(j) ? -1.f : 1.f;
            acc_re[j] = pack2(sg * a.x, sg * c.x);
            acc_im[j] = pack2(-sg * a.y, -sg * c.y);
        }
    } else {
#pragma unroll
        for (int j = 0; j < H; ++j) { acc_re[j] = 0ull; acc_im[j] = 0ull; }
    }

    Seed<GAUSS> sd;
    make_seed<GAUSS>(rec[k0].geo, u, v, w, uf, vf, sf0, ds, magic, kshift, ec.qmax, sd);
    constexpr int UNROLL_K = GAUSS ? 4 : 2;      // measured: points 205.6 ms at 2 (206.9 at 4), Gaussians 89.4 at 4 (91.0 at 2)
#pragma unroll UNROLL_K
    for (int k = k0; k < k1; ++k) {
        // software pipeline: the seed (FP64 + MUFU) of component k+1 overlaps the FP32 walk of k
        Seed<GAUSS> nx;
        make_seed<GAUSS>(rec[k + 1 < k1 ? k + 1 : k].geo, u, v, w, uf, vf, sf0, ds, magic, kshift, ec.qmax, nx);

        // word t = (S[J0+1+t], S[J0-t]), read as 128-bit granules into uniform registers
        const ulonglong2 *fl = rec[k].flux;
        const float cf = sd.wr + sd.wr;                    // c = 2 cos(delta)
        const f32x2 c2 = pack2(cf, cf), nc2 = pack2(-cf, -cf);

        f32x2 x = 0ull, r = 0ull, qq = 0ull;
        if constexpr (GAUSS) {
            float a, b2;
            const f32x2 Q2 = pack2(sd.Q, sd.Q);
            unpack2(mul2(Q2, ec.e0), a, b2);
            x = pack2(ex2_approx(a), ex2_approx(b2));                 // xi at (J0+1, J0)
            // first step ratios: finite because Q <= ec.qmax (see EnvConst)
            unpack2(mul2(Q2, ec.er), a, b2);
            r = pack2(ex2_approx(a), ex2_approx(b2));                 // xi_{J0+2} / xi_{J0+1}, xi_{J0-1} / xi_{J0}
            const float qf = ex2_approx(sd.Q * ec.e2);
            qq = pack2(qf, qf);
        }

        // ---- both directions in the two lanes: y_{t+1} = (s_{t+1} s_t) c y_t + y_{t-1}, forward over channels
        // J0+1 .. 31 in lane 0 and backward over J0 .. 0 in lane 1; at t = 0 the "previous" value of each
        // lane is the other lane's seed.
        {
            f32x2 ra = pack2(sd.r0, sd.r1), rc = pack2(sd.r1, sd.r0);      // previous, current
            f32x2 ia = pack2(sd.i0, sd.i1), ic = pack2(sd.i1, sd.i0);
#pragma unroll
            for (int t = 0; t < H; ++t) {
                f32x2 rn = 0ull, in = 0ull;
                const bool more = t + 1 < H;
                const bool flip = walk_neg(t + 1) != walk_neg(t);
                const f32x2 cc = flip ? nc2 : c2;
                f32x2 S = (t & 1) ? fl[t >> 1].y : fl[t >> 1].x;
                if constexpr (GAUSS) {
                    S = mul2(S, x);
                    if (more) { x = mul2(x, r); r = mul2(r, qq); }
                }
                // source order measured best (profiles/walk_rf_r3.md): ptxas keeps each chain's recurrence and
                // accumulate adjacent (shared slot-A operand) and pairs slightly better from this order
                if (more) rn = fma2(rc, cc, ra);
                if (more) in = fma2(ic, cc, ia);
                acc_im[t] = fma2(ic, S, acc_im[t]);
                acc_re[t] = fma2(rc, S, acc_re[t]);
                ra = rc; ia = ic; rc = rn; ic = in;
            }
        }
        sd = nx;
    }

    // S7: exp(-2 pi i phi) = conj(q): V = (s re, -s im); coalesced float2 stores along b
    if (valid) {
#pragma unroll
        for (int j = 0; j < H; ++j) {
            float a0, a1, b0, b1;
            unpack2(acc_re[j], a0, a1);
            unpack2(acc_im[j], b0, b1);
            const float sg = walk_neg(j) ? -1.f : 1.f;
            const int jf = walk_chan(j, 0), jb = walk_chan(j, 1);
            if (p.ftile * FT + jf < p.F) row[(size_t)jf * p.B] = make_float2(sg * a0, -sg * b0);
            if (p.ftile * FT + jb < p.F) row[(size_t)jb * p.B] = make_float2(sg * a1, -sg * b1);
        }
    }
}

// Fills the per-launch constant blocks: blocks[(ftile * n_chunks + chunk)] = WalkBlock<Geo>.
// One thread per (ftile, component, flux slot); slot 0 also copies the geometry record.
template <typename Geo>
__global__ void pack_walk_blocks_kernel(const Geo *__restrict__ geo, const double *__restrict__ s0,
                                        const double *__restrict__ alpha, double inv_ref, int n,
                                        const double *__restrict__ nu, int F, int n_ftiles, int n_chunks,
                                        unsigned char *__restrict__ blocks, unsigned int *err)
{
    constexpr int KC = WalkBlock<Geo>::KC;
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= (long long)n_ftiles * n * WALK_FT) return;
    const int pos = (int)(i % WALK_FT);
    const long long r = i / WALK_FT;
    const int k = (int)(r % n), ftile = (int)(r / n);
    const int j = walk_chan(pos >> 1, pos & 1);              // word t = pos / 2: lane 0 forward, lane 1 backward
    const int f = ftile * WALK_FT + j;
    WalkBlock<Geo> *blk = reinterpret_cast<WalkBlock<Geo> *>(blocks + ((size_t)ftile * n_chunks + k / KC) * WALK_CB_BYTES);
    float val = 0.f;
    if (f < F) {
        // step S2: S_k(nu_f) = s0 (nu_f / ref)^alpha in FP64, stored FP32; not finite in FP32: 0 and counted
        const double sv = s0[k] * pow(nu[f] * inv_ref, alpha[k]);
        if (isfinite(sv) && fabs(sv) <= 3.4028234663852886e38) val = (float)sv;
        else atomicAdd(err, 1u);
    }
    reinterpret_cast<float *>(blk->rec[k % KC].flux)[pos] = val;
    if (pos == 0) blk->rec[k % KC].geo = geo[k];
}

// Per-device ordering of the calls that refill CBANK (see launch()).
constexpr int BANK_MAX_DEVICES = 64;
std::mutex g_bank_mu[BANK_MAX_DEVICES];
cudaEvent_t g_bank_done[BANK_MAX_DEVICES] = {};      // "the last walking call on this device has finished"

struct BankOrder {
    int dev = -1;
    cudaError_t begin(cudaStream_t main)
    {
        int d = -1;
        cudaError_t e = cudaGetDevice(&d);
        if (e != cudaSuccess) return e;
        if (d < 0 || d >= BANK_MAX_DEVICES) return cudaErrorInvalidDevice;
        g_bank_mu[d].lock();
        dev = d;
        if (!g_bank_done[d]) {
            e = cudaEventCreateWithFlags(&g_bank_done[d], cudaEventDisableTiming);
            if (e != cudaSuccess) { g_bank_done[d] = nullptr; return e; }
        }
        return cudaStreamWaitEvent(main, g_bank_done[d], 0);      // the aux lane follows through the fork event
    }
    cudaError_t end(cudaStream_t main) { return dev >= 0 && g_bank_done[dev] ? cudaEventRecord(g_bank_done[dev], main) : cudaSuccess; }
    ~BankOrder() { if (dev >= 0) g_bank_mu[dev].unlock(); }
};

template <bool GAUSS, typename Geo>
cudaError_t launch(const UvwDev &uvw, const ChanTable &ch, const unsigned char *blocks, int n, float2 *vis,
                   int accumulate, unsigned int *err, const WalkStreams &ws)
{
    constexpr int KC = WalkBlock<Geo>::KC;
    const int n_ftiles = ch.F_pad / WALK_FT, n_chunks = (n + KC - 1) / KC;
    const long long n_bt = (long long)uvw.T * uvw.B;
    WParams p;
    p.u_m = uvw.u_m; p.v_m = uvw.v_m; p.w_m = uvw.w_m; p.vis = vis;
    p.B = uvw.B; p.F = uvw.F; p.ds = ch.ds; p.err = err;

    // CBANK is one symbol per device, shared by every context and stream of the process: walking calls on
    // a device are ordered one after another.  The host lock keeps two threads' enqueue loops apart; the
    // per-device event (recorded when a call's last launch has been enqueued, waited on by the next
    // call's streams before its first bank copy) keeps their GPU work apart.  Successive calls on one
    // stream wait on an event of their own stream: no cost on the usual path.
    BankOrder order;
    cudaError_t e = order.begin(ws.main);
    // Two lanes (bank half + stream each) that own disjoint outputs: whole channel tiles dealt
    // alternately, or the two halves of the (baseline, time) range when there is one tile.
    if (e == cudaSuccess) e = cudaEventRecord(ws.fork, ws.main);
    if (e == cudaSuccess) e = cudaStreamWaitEvent(ws.aux, ws.fork, 0);
    const int n_units = n_ftiles >= 2 ? n_ftiles : 2;
    const long long half_bt = (n_bt / 2 + WTHREADS - 1) / WTHREADS * WTHREADS;
    for (int unit = 0; unit < n_units && e == cudaSuccess; ++unit) {
        const int lane = unit & 1;
        const cudaStream_t st = lane ? ws.aux : ws.main;
        const int ftile = n_ftiles >= 2 ? unit : 0;
        p.bt0 = n_ftiles >= 2 ? 0 : (unit == 0 ? 0 : half_bt);
        p.bt1 = n_ftiles >= 2 ? n_bt : (unit == 0 ? (half_bt < n_bt ? half_bt : n_bt) : n_bt);
        if (p.bt1 <= p.bt0) continue;
        p.ftile = ftile;
        p.sf0 = ch.s_host[ftile * WALK_FT + WJ0];
        const double sa = ch.s_host[ftile * WALK_FT], sb = ch.s_host[ftile * WALK_FT + WALK_FT - 1];
        p.smax = sa > sb ? sa : sb;
        const unsigned grid = (unsigned)((p.bt1 - p.bt0 + WTHREADS - 1) / WTHREADS);
        for (int c = 0; c < n_chunks && e == cudaSuccess; ++c) {
            p.n_k = n - c * KC < KC ? n - c * KC : KC;
            p.load_acc = (accumulate || c > 0) ? 1 : 0;
            p.first = c == 0;
            p.k0 = lane * KC;
            const size_t bytes = sizeof(WalkRec<Geo>) * (size_t)p.n_k;
            e = cudaMemcpyToSymbolAsync(CBANK, blocks + ((size_t)ftile * n_chunks + c) * WALK_CB_BYTES, bytes,
                                        (size_t)lane * KC * sizeof(WalkRec<Geo>), cudaMemcpyDeviceToDevice, st);
            if (e != cudaSuccess) break;
            predict_walk_kernel<GAUSS><<<grid, WTHREADS, 0, st>>>(p); note_launch();
            e = cudaGetLastError();
        }
        if (e == cudaSuccess && n_ftiles >= 2 && ws.tile_done) ws.tile_done(ws.user, ftile, st);
    }
    // join even after an error so that the caller's stream stays ordered after the aux work
    cudaError_t e2 = cudaEventRecord(ws.join, ws.aux);
    if (e2 == cudaSuccess) e2 = cudaStreamWaitEvent(ws.main, ws.join, 0);
    if (e2 == cudaSuccess) e2 = order.end(ws.main);
    return e != cudaSuccess ? e : e2;
}

template <typename Geo>
void pack_blocks(const Geo *geo, const double *s0, const double *alpha, double ref_freq, int n, const ChanTable &ch,
                 unsigned char *blocks, unsigned int *err, cudaStream_t st)
{
    constexpr int KC = WalkBlock<Geo>::KC;
    const int n_ftiles = ch.F_pad / WALK_FT, n_chunks = (n + KC - 1) / KC;
    const long long total = (long long)n_ftiles * n * WALK_FT;
    pack_walk_blocks_kernel<Geo><<<(unsigned)((total + 255) / 256), 256, 0, st>>>(geo, s0, alpha, 1.0 / ref_freq, n, ch.nu,
                                                                                   ch.F, n_ftiles, n_chunks, blocks, err); note_launch();
}

}  // namespace

size_t walk_blocks_bytes(int n, int n_ftiles, bool gauss)
{
    const int KC = gauss ? WALK_KC_GAUSS : WALK_KC_POINTS;
    return (size_t)n_ftiles * ((n + KC - 1) / KC) * WALK_CB_BYTES;
}

void launch_pack_walk_points(const GeoP *geo, const double *s0, const double *alpha, double ref_freq, int n,
                             const ChanTable &ch, unsigned char *blocks, unsigned int *err, cudaStream_t st)
{
    pack_blocks<GeoP>(geo, s0, alpha, ref_freq, n, ch, blocks, err, st);
}

void launch_pack_walk_gaussians(const GeoG *geo, const double *s0, const double *alpha, double ref_freq, int n,
                                const ChanTable &ch, unsigned char *blocks, unsigned int *err, cudaStream_t st)
{
    pack_blocks<GeoG>(geo, s0, alpha, ref_freq, n, ch, blocks, err, st);
}

cudaError_t launch_walk_points(const UvwDev &uvw, const ChanTable &ch, const unsigned char *blocks, int n,
                               float2 *vis, int accumulate, unsigned int *err, const WalkStreams &ws)
{
    return launch<false, GeoP>(uvw, ch, blocks, n, vis, accumulate, err, ws);
}

cudaError_t launch_walk_gaussians(const UvwDev &uvw, const ChanTable &ch, const unsigned char *blocks, int n,
                                  float2 *vis, int accumulate, unsigned int *err, const WalkStreams &ws)
{
    return launch<true, GeoG>(uvw, ch, blocks, n, vis, accumulate, err, ws);
}

}  // namespace woden
