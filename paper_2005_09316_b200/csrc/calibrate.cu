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
// (I_ji = conj I_ij, V_ji = conj V_ij).  One CTA per cell keeps W in shared memory (FP64, upper triangle)
// and solves both systems together by Jacobi-preconditioned conjugate gradients; the singular one is
// started from zero with its right-hand side projected on the range, and the result is moved to
// the minimum-norm solution in e (the one Eq 22 has as a pseudo-inverse; reading G16) by removing
// the component along the gauge direction i g.  All FP64.
#include <cmath>

#include "kernels.h"

namespace woden {
namespace {

constexpr int CAL_THREADS = 256;

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

// sum of up to NV per-thread values over the CTA; every thread gets the totals.  One barrier per call:
// consecutive calls alternate between two scratch areas (`flip`), so a slow thread still reading the
// totals of call n cannot be overtaken by the partial sums of call n + 1.
template <int NV>
__device__ __forceinline__ void block_sum(double (&v)[NV], double *scratch /* [2][NV_MAX][CAL_THREADS / 32] */, int &flip)
{
    constexpr int NW = CAL_THREADS / 32, NV_MAX = 5;
    static_assert(NV <= NV_MAX, "scratch size");
    double *sc = scratch + flip * NV_MAX * NW;
    flip ^= 1;
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
#pragma unroll
    for (int k = 0; k < NV; ++k) {
        const double s = warp_sum(v[k]);
        if (lane == 0) sc[k * NW + wid] = s;
    }
    __syncthreads();
#pragma unroll
    for (int k = 0; k < NV; ++k) {
        double s = 0.0;
#pragma unroll
        for (int w = 0; w < NW; ++w) s += sc[k * NW + w];
        v[k] = s;
    }
}

// One CTA per (time, frequency) cell.  W_ij = |I_ij|^2 is kept in shared memory as its strict upper
// triangle in the visibilities' own pair order (FP64, N (N - 1) / 2 words: 65 KB for 128 antennas, so two
// cells are resident per SM and one cell's barrier waits are covered by the other's arithmetic).
// Both systems are solved together by Jacobi-preconditioned conjugate gradients in the
// single-reduction form (Chronopoulos & Gear): per iteration one matrix-vector product and ONE fused
// reduction (gamma = (r, u), delta = (A u, u)), three barriers in all.
__global__ void __launch_bounds__(CAL_THREADS, 2) calibrate_kernel(const CalParams p)
{
    extern __shared__ __align__(16) double sm[];
    const int N = p.N, tid = threadIdx.x;
    double *Wt = sm;                             // [N (N - 1) / 2] strict upper triangle, pair order
    double2 *qu = reinterpret_cast<double2 *>(Wt + p.B + (p.B & 1));   // q o (u0, u1); even offset: 16-byte aligned
    double *q = reinterpret_cast<double *>(qu + N);  // |g|^2
    double *d = q + N;                           // sum_j W_ij q_j
    double *gre = d + N, *gim = gre + N;         // gains
    double *rhs0 = gim + N, *rhs1 = rhs0 + N;    // q o Re rho, q o Im rho
    double *x1s = rhs1 + N;                      // Im eps (for the gauge step)
    double *scratch = x1s + N;                   // [2][5][CAL_THREADS / 32]
    double *part = scratch + 10 * (CAL_THREADS / 32);   // [split][2][N] partial products, split N <= CAL_THREADS
    int *rowoff = reinterpret_cast<int *>(part + 2 * (size_t)(N > CAL_THREADS ? N : CAL_THREADS));   // pair(i, j) = rowoff[i] + j, i < j
    const int split = N >= CAL_THREADS ? 1 : CAL_THREADS / N;
    const int jchunk = (N + split - 1) / split;
    int flip = 0;

    const float2 *V = p.data + (size_t)blockIdx.x * p.B;
    const float2 *I = p.model + (size_t)blockIdx.x * p.B;

    // W = |I|^2 (FP64 from the complex64 model), coalesced over the pair list
    for (long long b = tid; b < p.B; b += CAL_THREADS) {
        const float2 m = I[b];
        Wt[b] = (double)m.x * m.x + (double)m.y * m.y;
    }
    for (int i = tid; i < N; i += CAL_THREADS) {
        gre[i] = 1.0; gim[i] = 0.0;
        rowoff[i] = (int)((long long)i * (2 * N - i - 1) / 2) - i - 1;
    }
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
                const long long b = i < j ? rowoff[i] + j : rowoff[j] + i;
                di = fma(Wt[b], q[j], di);
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
        double mean1;
        {
            double s[1] = {0.0};
            for (int i = tid; i < N; i += CAL_THREADS) s[0] += rhs1[i];
            block_sum<1>(s, scratch, flip);
            mean1 = s[0] / N;
        }

        // ---- CG state of antenna i lives in the registers of thread i (N <= CAL_THREADS is enforced)
        const bool own = tid < N;
        const int i = own ? tid : 0;
        const double qi = q[i], di = d[i];
        const double dg = qi * di, inv = dg > 0.0 ? 1.0 / dg : 0.0;       // Jacobi preconditioner 1 / (q d)
        double x0 = 0.0, x1 = 0.0, r0 = own ? rhs0[i] : 0.0, r1 = own ? rhs1[i] - mean1 : 0.0;
        double u0 = r0 * inv, u1 = r1 * inv, w0 = 0.0, w1 = 0.0;
        double p0 = 0.0, p1 = 0.0, s0 = 0.0, s1 = 0.0;
        double gam0 = 0.0, gam1 = 0.0, al0 = 0.0, al1 = 0.0, floor0 = 0.0, floor1 = 0.0;
        bool live0 = true, live1 = true;

        // w = A u for both systems: t = W (q o u) by `split` thread groups over slices of the partners j,
        // then w0 = q (d u0 + t0), w1 = q (d u1 - t1); fused with the reduction of (r, u) and (w, u)
        auto product_and_dots = [&](double (&red)[5]) {
            if (own) qu[i] = make_double2(live0 ? qi * u0 : 0.0, live1 ? qi * u1 : 0.0);
            __syncthreads();
            if (tid < split * N) {
                const int ii = tid % N, h = tid / N;
                const int j0 = h * jchunk, j1 = min(N, j0 + jchunk);
                double t0 = 0.0, t1 = 0.0, v0 = 0.0, v1 = 0.0;
                // partners j < ii: element (j, ii) at rowoff[j] + ii (consecutive over ii: conflict-free)
                const int ja = min(ii, j1);
                int j = j0;
                // column walk: rowoff[j + 1] - rowoff[j] = N - j - 2, so the offset is carried, not loaded
                const double *col = Wt + rowoff[j0 < N ? j0 : 0] + ii;
#pragma unroll 4
                for (; j + 1 < ja; j += 2) {
                    const double wa = col[0], wb = col[N - j - 2];
                    col += 2 * N - 2 * j - 5;
                    const double2 a = qu[j], b = qu[j + 1];
                    t0 = fma(wa, a.x, t0); t1 = fma(wa, a.y, t1);
                    v0 = fma(wb, b.x, v0); v1 = fma(wb, b.y, v1);
                }
                if (j < ja) { const double wa = col[0]; const double2 a = qu[j]; t0 = fma(wa, a.x, t0); t1 = fma(wa, a.y, t1); }
                // partners j > ii: element (ii, j) at rowoff[ii] + j (a row of the triangle)
                const double *row = Wt + rowoff[ii];
                j = max(ii + 1, j0);
#pragma unroll 4
                for (; j + 1 < j1; j += 2) {
                    const double wa = row[j], wb = row[j + 1];
                    const double2 a = qu[j], b = qu[j + 1];
                    t0 = fma(wa, a.x, t0); t1 = fma(wa, a.y, t1);
                    v0 = fma(wb, b.x, v0); v1 = fma(wb, b.y, v1);
                }
                if (j < j1) { const double wa = row[j]; const double2 a = qu[j]; t0 = fma(wa, a.x, t0); t1 = fma(wa, a.y, t1); }
                part[(2 * h) * N + ii] = t0 + v0;
                part[(2 * h + 1) * N + ii] = t1 + v1;
            }
            __syncthreads();
            if (own) {
                double t0 = 0.0, t1 = 0.0;
                for (int h = 0; h < split; ++h) { t0 += part[(2 * h) * N + i]; t1 += part[(2 * h + 1) * N + i]; }
                w0 = qi * (di * u0 + t0);
                w1 = qi * (di * u1 - t1);
                red[0] = r0 * u0; red[1] = r1 * u1; red[2] = w0 * u0; red[3] = w1 * u1; red[4] = dg;
            } else {
                red[0] = red[1] = red[2] = red[3] = red[4] = 0.0;
            }
            block_sum<5>(red, scratch, flip);
        };

        {
            double red[5];
            product_and_dots(red);
            gam0 = red[0]; gam1 = red[1];
            // stop at a preconditioned residual reduced by cg_tol2, or once the correction it stands for is
            // below cg_abs in the (q d)-weighted rms of eps (late outer iterations start almost converged)
            floor0 = fmax(p.cg_tol2 * gam0, p.cg_abs2 * red[4]);
            floor1 = fmax(p.cg_tol2 * gam1, p.cg_abs2 * red[4]);
            live0 = gam0 > floor0 && red[2] > 0.0;
            live1 = gam1 > floor1 && red[3] > 0.0;
            al0 = live0 ? gam0 / red[2] : 0.0;
            al1 = live1 ? gam1 / red[3] : 0.0;
            p0 = u0; p1 = u1; s0 = w0; s1 = w1;
        }
        for (int cg = 0; cg < p.cg_max && (live0 || live1); ++cg) {
            if (live0) { x0 = fma(al0, p0, x0); r0 = fma(-al0, s0, r0); u0 = r0 * inv; }
            if (live1) { x1 = fma(al1, p1, x1); r1 = fma(-al1, s1, r1); u1 = r1 * inv; }
            double red[5];
            product_and_dots(red);
            if (live0) {
                const double gn = red[0], be = gn / gam0, den = red[2] - be * gn / al0;
                live0 = gn > floor0 && den > 0.0;
                al0 = live0 ? gn / den : 0.0;
                p0 = fma(be, p0, u0); s0 = fma(be, s0, w0); gam0 = gn;
            }
            if (live1) {
                const double gn = red[1], be = gn / gam1, den = red[3] - be * gn / al1;
                live1 = gn > floor1 && den > 0.0;
                al1 = live1 ? gn / den : 0.0;
                p1 = fma(be, p1, u1); s1 = fma(be, s1, w1); gam1 = gn;
            }
        }
        // gauge: minimum norm in e = g eps  <=>  sum_i q_i Im eps_i = 0
        {
            double s[2] = {own ? qi * x1 : 0.0, own ? qi : 0.0};
            block_sum<2>(s, scratch, flip);
            const double phi = s[1] > 0.0 ? s[0] / s[1] : 0.0;
            // g <- g + e = g (1 + eps)
            if (own) {
                const double er = x0, ei = x1 - phi;
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

// ---------------------------------------------------------------------------------------------------
// Register-resident variant for 64 < N <= 128 antennas.  The kernel above reads W from shared memory for
// every product (two wavefronts per warp and element + one for q o u): measured shared-memory-bound, 23 %
// of the FP64 pipe.  Here the FULL symmetric W lives in registers: thread (i = tid % 128, h = tid / 128)
// holds W[i][32 h .. 32 h + 31] (32 doubles), so a product is 32 broadcast loads of q o u and 64 DFMA per
// thread, and the four partial sums of a row meet in shared memory.  Shared memory instead holds
// C_ij = conj(I_ij) V_ij in FP64 for the right-hand-side pass of every outer iteration (130 KB at 128 antennas),
// which the kernel above re-reads from global memory ten times.  One 512-thread cell per SM.  The CG is the
// same single-reduction Jacobi-PCG, stopping rules and gauge step included.
constexpr int CR_THREADS = 512, CR_ROWS = 128, CR_SEG = 32;

__global__ void __launch_bounds__(CR_THREADS, 1) calibrate_reg_kernel(const CalParams p)
{
    extern __shared__ __align__(16) double sm[];
    const int N = p.N, tid = threadIdx.x;
    const int i = tid % CR_ROWS, h = tid / CR_ROWS;       // row, partner segment (warp-uniform)
    const int j0 = h * CR_SEG;
    // the small arrays sit at FIXED offsets from the base (no pointer registers: they are needed for W), C last
    double2 *const qu = reinterpret_cast<double2 *>(sm);              // [128] q o (u0, u1), zero past N
    double *const q = sm + 2 * CR_ROWS;                               // [128] |g|^2, zero past N
    double *const gre = sm + 3 * CR_ROWS, *const gim = sm + 4 * CR_ROWS;   // [128] gains
    double *const part = sm + 5 * CR_ROWS;                            // [4][3][128] partial sums of the four segments
    double *const scratch = sm + 17 * CR_ROWS;                        // [2][5][16]
    double *const cgv = sm + 17 * CR_ROWS + 2 * 5 * (CR_THREADS / 32);     // [14][128] CG vectors and scalars of row i
    int *const rowoff = reinterpret_cast<int *>(sm + 31 * CR_ROWS + 2 * 5 * (CR_THREADS / 32));   // [128] pair(a, b) = rowoff[a] + b, a < b
    double *const ctl = sm + 31 * CR_ROWS + 2 * 5 * (CR_THREADS / 32) + CR_ROWS / 2;   // [16] ctl[0]: "another product follows" flag
    double2 *const Cc = reinterpret_cast<double2 *>(sm + 31 * CR_ROWS + 2 * 5 * (CR_THREADS / 32) + CR_ROWS / 2 + 16);   // [B] conj(I) V
    int flip = 0;

    const float2 *V = p.data + (size_t)blockIdx.x * p.B;
    const float2 *I = p.model + (size_t)blockIdx.x * p.B;
    const bool own = tid < N;                                         // h == 0 and a real antenna: holds the CG state
    if (tid < CR_ROWS) rowoff[tid] = (int)((long long)tid * (2 * N - tid - 1) / 2) - tid - 1;
    __syncthreads();
    // pair (min, max) of (i, j): the row offset of the smaller index comes from the shared table at the point of
    // use (kept out of registers on purpose: 32 hoisted indices per thread would cost the registers W needs)
    const int ro_i = rowoff[i];
    auto pair_ij = [&](int j) { return i < j ? ro_i + j : rowoff[j] + i; };

    // C = conj(I) V in FP64 from the complex64 inputs (exact products), coalesced over the pair list
    for (long long b = tid; b < p.B; b += CR_THREADS) {
        const float2 m = I[b], v = V[b];
        Cc[b] = make_double2((double)m.x * v.x + (double)m.y * v.y, (double)m.x * v.y - (double)m.y * v.x);
    }
    // this thread's 32 entries of W = |I|^2 (zero on the diagonal and past N)
    double W[CR_SEG];
#pragma unroll
    for (int k = 0; k < CR_SEG; ++k) {
        if (k % 8 == 0 && k > 0) asm volatile("" ::: "memory");
        const int j = j0 + k;
        double wv = 0.0;
        if (i < N && j < N && j != i) {
            const float2 m = I[pair_ij(j)];
            wv = (double)m.x * m.x + (double)m.y * m.y;
        }
        W[k] = wv;
    }
    if (tid < CR_ROWS) { gre[tid] = 1.0; gim[tid] = 0.0; q[tid] = 0.0; qu[tid] = make_double2(0.0, 0.0); }
    __syncthreads();

    // Only the four OWNER warps (tid < 128: h == 0) run the scalar side of the CG (dot products, step lengths,
    // stopping rules): the other twelve only multiply.  Sums over rows therefore involve four warps.
    const bool owner_warp = tid < CR_ROWS;
    enum { X0, X1, R0, R1, U0, U1, P0, P1, S0, S1, QI, DI, DG, INV };
    auto cv = [&](int k) -> double & { return cgv[k * CR_ROWS + i]; };
    // sum of NV per-row values over the owner warps; every owner thread gets the totals.  One barrier (all threads).
    auto owner_sum = [&](double *v, int nv) {
        double *sc = scratch + flip * 5 * 4;
        flip ^= 1;
        if (owner_warp) {
            for (int k = 0; k < nv; ++k) {
                const double t = warp_sum(v[k]);
                if ((tid & 31) == 0) sc[k * 4 + (tid >> 5)] = t;
            }
        }
        __syncthreads();
        if (owner_warp)
            for (int k = 0; k < nv; ++k) v[k] = (sc[k * 4] + sc[k * 4 + 1]) + (sc[k * 4 + 2] + sc[k * 4 + 3]);
    };
    // t = W (q o u) for both systems from the register rows; the four partial sums of a row meet in `part`
    auto product = [&]() {
        double t0 = 0.0, t1 = 0.0, v0 = 0.0, v1 = 0.0;
#pragma unroll
        for (int k = 0; k < CR_SEG; k += 2) {
            const double2 a = qu[j0 + k], b = qu[j0 + k + 1];      // warp-uniform addresses: broadcasts
            t0 = fma(W[k], a.x, t0); t1 = fma(W[k], a.y, t1);
            v0 = fma(W[k + 1], b.x, v0); v1 = fma(W[k + 1], b.y, v1);
        }
        part[(3 * h) * CR_ROWS + i] = t0 + v0;
        part[(3 * h + 1) * CR_ROWS + i] = t1 + v1;
    };

    for (int it = 0; it < p.n_iter; ++it) {
        if (own) q[i] = gre[i] * gre[i] + gim[i] * gim[i];
        __syncthreads();
        // d_i = sum_j W_ij q_j and sum_j g_j C_ij over this thread's segment
        {
            double di = 0.0, sr = 0.0, si = 0.0;
#pragma unroll                                   // full: W[] must stay in registers (static indices)
            for (int k = 0; k < CR_SEG; ++k) di = fma(W[k], q[j0 + k], di);
            // the complex sum runs as a ROLLED loop: unrolled, its 32 pair indices are hoisted out of the outer
            // iteration and cost the registers W needs
#pragma unroll 1
            for (int k = 0; k < CR_SEG; ++k) {
                const int j = j0 + k;
                if (i < N && j < N && j != i) {
                    double2 c = Cc[pair_ij(j)];
                    if (i > j) c.y = -c.y;                       // C_ij for the ordered pair (i, j)
                    sr += gre[j] * c.x - gim[j] * c.y;           // g_j C_ij
                    si += gre[j] * c.y + gim[j] * c.x;
                }
            }
            part[(3 * h) * CR_ROWS + i] = di;
            part[(3 * h + 1) * CR_ROWS + i] = sr;
            part[(3 * h + 2) * CR_ROWS + i] = si;
        }
        __syncthreads();
        double rhs1 = 0.0;
        if (own) {
            double sr = 0.0, si = 0.0, di = 0.0;
#pragma unroll
            for (int hh = 0; hh < 4; ++hh) {
                di += part[(3 * hh) * CR_ROWS + i]; sr += part[(3 * hh + 1) * CR_ROWS + i]; si += part[(3 * hh + 2) * CR_ROWS + i];
            }
            const double qi = q[i];
            const double rr = sr - gre[i] * di, ri = si - gim[i] * di;       // r_i = sum - g_i d_i
            const double rhs0 = rr * gre[i] + ri * gim[i];                   // q rho = r conj(g)
            rhs1 = ri * gre[i] - rr * gim[i];
            const double dg = qi * di, inv = dg > 0.0 ? 1.0 / dg : 0.0;      // Jacobi preconditioner 1 / (q d)
            cv(QI) = qi; cv(DI) = di; cv(DG) = dg; cv(INV) = inv;
            cv(X0) = 0.0; cv(X1) = 0.0; cv(R0) = rhs0; cv(U0) = rhs0 * inv;
        }
        // range projection of the singular system's right-hand side (null vector: all ones)
        {
            double sv[1] = {rhs1};
            owner_sum(sv, 1);
            const double mean1 = sv[0] / N;
            if (own) { cv(R1) = rhs1 - mean1; cv(U1) = (rhs1 - mean1) * cv(INV); }
        }

        // ---- Jacobi-PCG in the single-reduction form: state of the scalar side (owner warps only)
        double gam0 = 0.0, gam1 = 0.0, al0 = 0.0, al1 = 0.0, floor0 = 0.0, floor1 = 0.0;
        bool live0 = true, live1 = true;
        for (int cg = -1; cg < p.cg_max; ++cg) {          // pass -1 sets up gamma, alpha, p = u, s = A u
            if (own) {
                if (cg >= 0) {
                    const double inv = cv(INV);
                    if (live0) { cv(X0) = fma(al0, cv(P0), cv(X0)); const double r = fma(-al0, cv(S0), cv(R0)); cv(R0) = r; cv(U0) = r * inv; }
                    if (live1) { cv(X1) = fma(al1, cv(P1), cv(X1)); const double r = fma(-al1, cv(S1), cv(R1)); cv(R1) = r; cv(U1) = r * inv; }
                }
                const double qi = cv(QI);
                qu[i] = make_double2(live0 ? qi * cv(U0) : 0.0, live1 ? qi * cv(U1) : 0.0);
            }
            if (tid == 0) ctl[0] = (live0 || live1) ? 1.0 : 0.0;       // every owner thread holds the same flags
            __syncthreads();
            if (ctl[0] == 0.0) break;                                   // uniform: read after the barrier, rewritten only after the next two
            product();
            __syncthreads();
            double red[5] = {0.0, 0.0, 0.0, 0.0, 0.0}, w0 = 0.0, w1 = 0.0;
            if (own) {
                double a0 = 0.0, a1 = 0.0;
#pragma unroll
                for (int hh = 0; hh < 4; ++hh) { a0 += part[(3 * hh) * CR_ROWS + i]; a1 += part[(3 * hh + 1) * CR_ROWS + i]; }
                const double u0 = cv(U0), u1 = cv(U1), qi = cv(QI), di = cv(DI);
                w0 = qi * (di * u0 + a0);                               // w = A u: w0 = q (d u0 + t0), w1 = q (d u1 - t1)
                w1 = qi * (di * u1 - a1);
                red[0] = cv(R0) * u0; red[1] = cv(R1) * u1; red[2] = w0 * u0; red[3] = w1 * u1; red[4] = cv(DG);
            }
            owner_sum(red, 5);
            if (owner_warp) {
                if (cg < 0) {
                    gam0 = red[0]; gam1 = red[1];
                    // stop at a preconditioned residual reduced by cg_tol2, or once the correction it stands for is
                    // below cg_abs in the (q d)-weighted rms of eps (late outer iterations start almost converged)
                    floor0 = fmax(p.cg_tol2 * gam0, p.cg_abs2 * red[4]);
                    floor1 = fmax(p.cg_tol2 * gam1, p.cg_abs2 * red[4]);
                    live0 = gam0 > floor0 && red[2] > 0.0;
                    live1 = gam1 > floor1 && red[3] > 0.0;
                    al0 = live0 ? gam0 / red[2] : 0.0;
                    al1 = live1 ? gam1 / red[3] : 0.0;
                    if (own) { cv(P0) = cv(U0); cv(P1) = cv(U1); cv(S0) = w0; cv(S1) = w1; }
                } else {
                    if (live0) {
                        const double gn = red[0], be = gn / gam0, den = red[2] - be * gn / al0;
                        live0 = gn > floor0 && den > 0.0;
                        al0 = live0 ? gn / den : 0.0;
                        if (own) { cv(P0) = fma(be, cv(P0), cv(U0)); cv(S0) = fma(be, cv(S0), w0); }
                        gam0 = gn;
                    }
                    if (live1) {
                        const double gn = red[1], be = gn / gam1, den = red[3] - be * gn / al1;
                        live1 = gn > floor1 && den > 0.0;
                        al1 = live1 ? gn / den : 0.0;
                        if (own) { cv(P1) = fma(be, cv(P1), cv(U1)); cv(S1) = fma(be, cv(S1), w1); }
                        gam1 = gn;
                    }
                }
            }
        }
        // gauge: minimum norm in e = g eps  <=>  sum_i q_i Im eps_i = 0
        {
            double sv[2] = {own ? cv(QI) * cv(X1) : 0.0, own ? cv(QI) : 0.0};
            owner_sum(sv, 2);
            const double phi = sv[1] > 0.0 ? sv[0] / sv[1] : 0.0;
            if (own) {                                                   // g <- g + e = g (1 + eps)
                const double er = cv(X0), ei = cv(X1) - phi;
                const double nr = gre[i] + gre[i] * er - gim[i] * ei;
                const double ni = gim[i] + gre[i] * ei + gim[i] * er;
                gre[i] = nr; gim[i] = ni;
            }
        }
        __syncthreads();
    }
    if (own) p.gains[(size_t)blockIdx.x * N + i] = make_double2(gre[i], gim[i]);
}

size_t calibrate_reg_smem_bytes(int N)
{
    const size_t B = (size_t)N * (N - 1) / 2;
    return B * 16 + ((size_t)31 * CR_ROWS + (size_t)2 * 5 * (CR_THREADS / 32) + CR_ROWS / 2 + 16) * 8;
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
    const size_t B = (size_t)N * (N - 1) / 2;
    return (B + (B & 1) + 7 * (size_t)N + 10 * (CAL_THREADS / 32) + 2 * (size_t)(N > CAL_THREADS ? N : CAL_THREADS) + 2 * (size_t)N + (N + 1) / 2) * sizeof(double);
}

cudaError_t launch_calibrate(const float2 *data, const float2 *model, double2 *gains, int N, long long cells, int n_iter,
                             cudaStream_t st)
{
    CalParams p;
    p.data = data; p.model = model; p.gains = gains; p.N = N; p.n_iter = n_iter;
    p.B = (long long)N * (N - 1) / 2;
    p.cg_max = 2 * N + 10;
    p.cg_tol2 = 1e-22;             // preconditioned residual reduced by 1e-11 (gains are compared at 1e-9)
    p.cg_abs2 = 1e-28;             // or the remaining relative gain correction below 1e-14
    if (N > CAL_THREADS) return cudaErrorInvalidValue;         // the CG state of antenna i lives in thread i
    if (N > 64 && N <= CR_ROWS) {                              // register-resident W: measured faster there
        const size_t smem_r = calibrate_reg_smem_bytes(N);
        cudaError_t er = cudaFuncSetAttribute(calibrate_reg_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_r);
        if (er != cudaSuccess) return er;
        calibrate_reg_kernel<<<(unsigned)cells, CR_THREADS, smem_r, st>>>(p); note_launch();
        return cudaGetLastError();
    }
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
