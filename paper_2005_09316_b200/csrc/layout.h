// layout.h -- packed device layouts shared by the staging kernels, the predict kernels and the
// API translation unit of libwoden_b200.so.  (Nothing here is used by the CPU oracle.)
#pragma once
#include <cstdint>

namespace woden {

constexpr double C_LIGHT = 299792458.0;     // m/s (reading G6)
constexpr int KB = 64;                      // components per staged shared-memory block
constexpr int NSTAGE = 3;                   // bulk-copy pipeline depth
constexpr int PG_THREADS = 256;             // (baseline,time) pairs per CTA, points/Gaussians
constexpr int MAX_ORDER = 100;

// One point component, 32 B: direction cosines and n-1 = -(l^2+m^2)/(1+n) in FP64 (hard part H1).
struct __align__(16) GeoP {
    double l, m, n1, pad;
};

// One Gaussian component, 48 B.  (as,ac,bs,bc) = pi/(2 ln 2) * (maj sin pa, maj cos pa,
// min sin pa, min cos pa), so that with metres-domain gx = as*u + ac*v, gy = bc*u - bs*v the
// envelope of Eq 12 is xi = exp2(-(gx^2 + gy^2) * (nu/c)^2).
struct __align__(16) GeoG {
    double l, m, n1;
    float as, ac, bs, bc;
    float pad[2];
};

// One shapelet component, 96 B.  x = beta1 K kx', y = beta2 K ky' (Eq 16-17) are linear in the
// metres-domain (u,v,w): x = (X . uvw) * nu/c, y = (Y . uvw) * nu/c with the 2x3 matrix M_j,
// the PA rotation and beta * pi/sqrt(2 ln 2) folded into X and Y.
struct __align__(16) GeoS {
    double l, m, n1;
    double X[3], Y[3];
    int tri_offset;          // float offset of this component's packed coefficient triangle
    int pad[5];
};

// Packed coefficient triangle for compile-time order PM: row n1 holds n2 = 0..PM-n1, padded
// to a multiple of 4 floats so every row starts 16-byte aligned.
__host__ __device__ constexpr int tri_row_len(int PM, int n1) { return ((PM - n1 + 1) + 3) & ~3; }
__host__ __device__ constexpr int tri_row_off(int PM, int n1)
{
    int o = 0;
    for (int r = 0; r < n1; ++r) o += tri_row_len(PM, r);
    return o;
}
__host__ __device__ constexpr int tri_size(int PM) { return tri_row_off(PM, PM + 1); }
// One bit per 4-float chunk of the triangle (bit = float offset / 4), set when any of its four
// coefficients is non-zero, follows the triangle: truncated models skip the
// load and the FFMAs of empty chunks.  tri_stride = triangle + mask words, padded to 16 bytes.
__host__ __device__ constexpr int tri_mask_words(int PM) { return (tri_size(PM) / 4 + 31) / 32; }
__host__ __device__ constexpr int tri_stride(int PM) { return tri_size(PM) + ((tri_mask_words(PM) + 3) & ~3); }

// Per-call channel table, device resident: one block of doubles then floats.
//   s[f]    = nu_f / c            (FP64, metres -> wavelengths)
//   nu[f]   = nu_f                (FP64, for the flux law)
//   ns2[f]  = -(nu_f / c)^2       (FP32, Gaussian exponent scale)
// padded with zeros to F_pad (a multiple of the channel tile).
struct ChanTable {
    const double *s_host;   // HOST copy of s[] (per-launch scalars of the channel-walking kernel)
    const double *s;
    const double *nu;
    const float *ns2;
    int F, F_pad;
    int uniform;        // 1 when channels are equally spaced (fast path eligible)
    double ds;          // (nu_1 - nu_0) / c when uniform
};

}  // namespace woden
