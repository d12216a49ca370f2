// pack.cu -- step S0 of the hot path: O(K) staging kernels that turn the caller's
// FP64 component arrays into the packed device blocks the predict kernels stream through
// shared memory.  All arithmetic here is FP64; results are stored FP64 (geometry) or FP32
// (envelope scales, fluxes, coefficients).
#include <cmath>

#include "kernels.h"

namespace woden {
namespace {

constexpr double PI = 3.14159265358979323846264338327950288;
constexpr double LN2 = 0.693147180559945309417232121458176568;

__device__ __forceinline__ bool finite3(double a, double b, double c)
{
    return isfinite(a) && isfinite(b) && isfinite(c);
}

// n - 1 = -(l^2 + m^2) / (1 + n), n = sqrt(1 - l^2 - m^2): no cancellation.
__device__ __forceinline__ bool direction(double l, double m, double *n1)
{
    const double r2 = l * l + m * m;
    if (!(r2 < 1.0)) { *n1 = 0.0; return false; }
    *n1 = -r2 / (1.0 + sqrt(1.0 - r2));
    return true;
}

__global__ void pack_points_kernel(const double *__restrict__ l, const double *__restrict__ m, int n, int n_pad,
                                   GeoP *__restrict__ geo, unsigned int *err)
{
    const int k = blockIdx.x * blockDim.x + threadIdx.x;
    if (k >= n_pad) return;
    GeoP g = {0.0, 0.0, 0.0, 0.0};
    if (k < n) {
        double n1;
        if (direction(l[k], m[k], &n1)) { g.l = l[k]; g.m = m[k]; g.n1 = n1; }
        else atomicAdd(err, 1u);
    }
    geo[k] = g;
}

__global__ void pack_gaussians_kernel(const double *__restrict__ l, const double *__restrict__ m,
                                      const double *__restrict__ maj, const double *__restrict__ mnr,
                                      const double *__restrict__ pa, int n, int n_pad, GeoG *__restrict__ geo,
                                      unsigned int *err)
{
    const int k = blockIdx.x * blockDim.x + threadIdx.x;
    if (k >= n_pad) return;
    GeoG g = {0.0, 0.0, 0.0, 0.f, 0.f, 0.f, 0.f, {0.f, 0.f}};
    if (k < n) {
        double n1;
        const bool ok = direction(l[k], m[k], &n1) && finite3(maj[k], mnr[k], pa[k]) && maj[k] >= 0.0 &&
                        mnr[k] >= 0.0;
        if (ok) {
            // Eq 12: xi = exp(-pi^2/(4 ln2) (kx^2 maj^2 + ky^2 min^2))
            //                          = exp2(-[(cg maj kx)^2 + (cg min ky)^2]),  cg = pi / (2 ln 2)
            // Eq 13-14 (:144-146): kx = cos(pa) v + sin(pa) u, ky = -sin(pa) v + cos(pa) u
            const double cg = PI / (2.0 * LN2);
            double sp, cp;
            sincos(pa[k], &sp, &cp);
            g.l = l[k]; g.m = m[k]; g.n1 = n1;
            g.as = (float)(cg * maj[k] * sp);
            g.ac = (float)(cg * maj[k] * cp);
            g.bs = (float)(cg * mnr[k] * sp);
            g.bc = (float)(cg * mnr[k] * cp);
        } else {
            atomicAdd(err, 1u);
        }
    }
    geo[k] = g;
}

// flux[(ftile * n_pad + k) * FT + pos] = s0_k (nu_f / ref)^alpha_k  (step S2).  Plain layout:
// pos = channel within the tile (FT == 1 is [F][n]).  Interleaved layout (channel-walking kernel):
// pos holds channel f = ftile*FT + (pos >> 1) + (pos & 1) * FT/2, i.e. the two half-tiles are
// interleaved so that one 64-bit word feeds both lanes of a packed FP32x2 instruction.
__global__ void pack_flux_kernel(const double *__restrict__ s0, const double *__restrict__ alpha, double inv_ref,
                                 int n, int n_pad, const double *__restrict__ nu, int F, int FT, int interleave,
                                 long long total, float *__restrict__ flux, unsigned int *err)
{
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= total) return;
    const int pos = (int)(i % FT);
    const int j = interleave ? (pos >> 1) + (pos & 1) * (FT / 2) : pos;
    const long long r = i / FT;
    const int k = (int)(r % n_pad);
    const int f = (int)(r / n_pad) * FT + j;
    float val = 0.f;
    if (k < n && f < F) {
        const double v = s0[k] * pow(nu[f] * inv_ref, alpha[k]);
        // FP32 table: a flux that is not finite (or overflows FP32) is replaced by 0 and counted
        if (isfinite(v) && fabs(v) <= 3.4028234663852886e38) val = (float)v;
        else atomicAdd(err, 1u);
    }
    flux[i] = val;
}

__global__ void pack_shapelets_kernel(const double *__restrict__ l, const double *__restrict__ m,
                                      const double *__restrict__ beta1, const double *__restrict__ beta2,
                                      const double *__restrict__ pa, const double *__restrict__ uv_basis, int n,
                                      int tri_floats, GeoS *__restrict__ geo, unsigned int *err)
{
    const int k = blockIdx.x * blockDim.x + threadIdx.x;
    if (k >= n) return;
    GeoS g;
    g.l = g.m = g.n1 = 0.0;
    for (int i = 0; i < 3; ++i) g.X[i] = g.Y[i] = 0.0;
    g.tri_offset = k * tri_floats;
    for (int i = 0; i < 5; ++i) g.pad[i] = 0;
    double n1;
    bool ok = direction(l[k], m[k], &n1) && finite3(beta1[k], beta2[k], pa[k]) && beta1[k] > 0.0 && beta2[k] > 0.0;
    if (ok) {
        double M[6] = {1.0, 0.0, 0.0, 0.0, 1.0, 0.0};      // (u',v') = (u,v) when no M_j (reading G4)
        if (uv_basis)
            for (int i = 0; i < 6; ++i) M[i] = uv_basis[6 * (size_t)k + i];
        // Eq 16-17 with the beta scaling of Eq 15's basis argument:
        //   x = beta1 K ( cos(pa) v' + sin(pa) u'),  y = beta2 K (-sin(pa) v' + cos(pa) u'),  K = pi/sqrt(2 ln2)
        const double kap = PI / sqrt(2.0 * LN2);
        double sp, cp;
        sincos(pa[k], &sp, &cp);
        g.l = l[k]; g.m = m[k]; g.n1 = n1;
        for (int i = 0; i < 3; ++i) {
            g.X[i] = beta1[k] * kap * (cp * M[3 + i] + sp * M[i]);
            g.Y[i] = beta2[k] * kap * (-sp * M[3 + i] + cp * M[i]);
            ok = ok && isfinite(g.X[i]) && isfinite(g.Y[i]);
        }
    }
    if (!ok) {
        atomicAdd(err, 1u);
        g.l = g.m = g.n1 = 0.0;
        for (int i = 0; i < 3; ++i) g.X[i] = g.Y[i] = 0.0;
    }
    geo[k] = g;
}

// The predict kernel evaluates g_p = h_p / lam_p with the two-operation recurrence
//   g_{p+1} = (c_p x) g_p - g_{p-1},   lam_0 = lam_1 = 1, lam_{p+1} = sqrt(p/(p+1)) lam_{p-1},
//   c_p = sqrt(2/(p+1)) lam_p / lam_{p+1}
// (the normalised Hermite-function recurrence h_{p+1} = sqrt(2/(p+1)) x h_p - sqrt(p/(p+1)) h_{p-1}
// with the second coefficient scaled to one).  lam_{n1} lam_{n2} and the sign part of i^(n1+n2),
// sig_p = (-1)^floor(p/2), are folded into the stored coefficient here.
__device__ double lam_of(int p)
{
    double lam = 1.0;
    for (int q = (p & 1) ? 1 : 0; q + 2 <= p; q += 2) lam *= sqrt((double)(q + 1) / (double)(q + 2));
    return lam;
}

__global__ void zero_kernel(float *__restrict__ p, long long n)
{
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n) p[i] = 0.f;
}

template <int DUMMY>
__device__ int tri_index_rt(int PM, int a, int b)
{
    int o = 0;
    for (int r = 0; r < a; ++r) o += ((PM - r + 1) + 3) & ~3;
    return o + b;
}

__global__ void pack_coeffs_kernel(const int *__restrict__ coeff_offset, const int *__restrict__ n1,
                                   const int *__restrict__ n2, const double *__restrict__ coeff, int n, int n_coeff,
                                   int p_max, int PM, int tri_floats, float *__restrict__ tri, unsigned int *err)
{
    const int q = blockIdx.x * blockDim.x + threadIdx.x;
    if (q >= n_coeff) return;
    // owning component: last j with coeff_offset[j] <= q  (binary search over n+1 offsets)
    int lo = 0, hi = n;
    while (hi - lo > 1) {
        const int mid = (lo + hi) >> 1;
        if (coeff_offset[mid] <= q) lo = mid; else hi = mid;
    }
    const int a = n1[q], b = n2[q];
    const double c = coeff[q];
    if (a < 0 || b < 0 || a + b > p_max || a + b > PM || !isfinite(c) || q >= coeff_offset[n] ||
        q < coeff_offset[lo] || q >= coeff_offset[lo + 1]) {
        atomicAdd(err, 1u);
        return;
    }
    const double sig = (((a >> 1) + (b >> 1)) & 1) ? -1.0 : 1.0;
    const float val = (float)(c * sig * lam_of(a) * lam_of(b));
    atomicAdd(&tri[(size_t)lo * tri_floats + tri_index_rt<0>(PM, a, b)], val);
}

// mask bit c of component k = chunk c (floats 4c..4c+3) of its triangle holds a non-zero coefficient
__global__ void tri_mask_kernel(float *__restrict__ tri, int n, int tri_floats, int stride)
{
    const int chunks = tri_floats / 4;
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= (long long)n * chunks) return;
    const int k = (int)(i / chunks), c = (int)(i % chunks);
    const float4 v = *reinterpret_cast<const float4 *>(tri + (size_t)k * stride + 4 * (size_t)c);
    if (v.x != 0.f || v.y != 0.f || v.z != 0.f || v.w != 0.f)
        atomicOr(reinterpret_cast<unsigned int *>(tri + (size_t)k * stride + tri_floats) + c / 32, 1u << (c % 32));
}

inline int blocks_for(long long n, int t) { return (int)((n + t - 1) / t); }

}  // namespace

void launch_pack_points(const double *l, const double *m, int n, int n_pad, GeoP *geo, unsigned int *err,
                        cudaStream_t st)
{
    pack_points_kernel<<<blocks_for(n_pad, 256), 256, 0, st>>>(l, m, n, n_pad, geo, err); note_launch();
}

void launch_pack_gaussians(const double *l, const double *m, const double *maj, const double *mnr,
                           const double *pa, int n, int n_pad, GeoG *geo, unsigned int *err, cudaStream_t st)
{
    pack_gaussians_kernel<<<blocks_for(n_pad, 256), 256, 0, st>>>(l, m, maj, mnr, pa, n, n_pad, geo, err); note_launch();
}

void launch_pack_flux(const double *s0, const double *alpha, double ref_freq, int n, int n_pad,
                      const ChanTable &ch, int FT, bool interleave, float *flux, unsigned int *err, cudaStream_t st)
{
    const long long total = (long long)(ch.F_pad / FT) * n_pad * FT;
    pack_flux_kernel<<<blocks_for(total, 256), 256, 0, st>>>(s0, alpha, 1.0 / ref_freq, n, n_pad, ch.nu, ch.F, FT,
                                                             interleave ? 1 : 0, total, flux, err); note_launch();
}

void launch_pack_shapelets(const double *l, const double *m, const double *beta1, const double *beta2,
                           const double *pa, const double *uv_basis, int n, int PM, GeoS *geo,
                           unsigned int *err, cudaStream_t st)
{
    pack_shapelets_kernel<<<blocks_for(n, 128), 128, 0, st>>>(l, m, beta1, beta2, pa, uv_basis, n, tri_stride(PM),
                                                              geo, err); note_launch();
}

void launch_pack_coeffs(const int *coeff_offset, const int *n1, const int *n2, const double *coeff, int n,
                        int n_coeff, int p_max, int PM, float *tri, unsigned int *err, cudaStream_t st)
{
    const long long tot = (long long)n * tri_stride(PM);
    zero_kernel<<<blocks_for(tot, 256), 256, 0, st>>>(tri, tot); note_launch();
    if (n_coeff > 0) {
        pack_coeffs_kernel<<<blocks_for(n_coeff, 256), 256, 0, st>>>(coeff_offset, n1, n2, coeff, n, n_coeff, p_max,
                                                                     PM, tri_stride(PM), tri, err); note_launch();
    }
    tri_mask_kernel<<<blocks_for((long long)n * (tri_size(PM) / 4), 256), 256, 0, st>>>(tri, n, tri_size(PM),
                                                                                         tri_stride(PM)); note_launch();
}

}  // namespace woden
