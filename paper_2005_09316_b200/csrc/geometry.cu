// geometry.cu -- SURVEY.md §8(f) NEXT-2: the step immediately before the hot path, on the device.
//   * antenna positions -> baseline (u,v,w) in metres, once per time step ("u,v,w only differ in
//     frequency by a scaling factor, we only calculate them once per time step"),
//     by the textbook rotation of local equatorial XYZ (Thompson, Moran & Swenson, cited at
//     PAPER.md:110; reading G14);
//   * the shapelet 2x3 matrices M_j of reading G4 from (l, m) and the phase-centre
//     declination.
// All FP64; O(T B) and O(K): negligible next to the predict kernels.
#include <cmath>

#include "kernels.h"

namespace woden {
namespace {

// baseline index b (pairs p < q in p-major order) -> (p, q) for n antennas
__device__ __forceinline__ void pair_of(long long b, int n, int *p_out, int *q_out)
{
    // rows before p hold p (2n - p - 1) / 2 pairs; start from the real root and correct
    const double nn = 2.0 * n - 1.0;
    int p = (int)floor((nn - sqrt(nn * nn - 8.0 * (double)b)) * 0.5);
    if (p < 0) p = 0;
    if (p > n - 2) p = n - 2;
    while (p > 0 && (long long)p * (2LL * n - p - 1) / 2 > b) --p;
    while ((long long)(p + 1) * (2LL * n - p - 2) / 2 <= b) ++p;
    *p_out = p;
    *q_out = (int)(b - (long long)p * (2LL * n - p - 1) / 2) + p + 1;
}

__global__ void uvw_kernel(const double *__restrict__ X, const double *__restrict__ Y, const double *__restrict__ Z,
                           int n_ant, long long B, int T, const double *__restrict__ hour_angle, double sd, double cd,
                           double *__restrict__ u, double *__restrict__ v, double *__restrict__ w)
{
    const long long b = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (b >= B) return;
    int p, q;
    pair_of(b, n_ant, &p, &q);
    const double bx = X[p] - X[q], by = Y[p] - Y[q], bz = Z[p] - Z[q];      // baseline = antenna p - antenna q
    for (int t = 0; t < T; ++t) {
        double sH, cH;
        sincos(hour_angle[t], &sH, &cH);
        u[(size_t)t * B + b] = sH * bx + cH * by;
        v[(size_t)t * B + b] = -sd * cH * bx + sd * sH * by + cd * bz;
        w[(size_t)t * B + b] = cd * cH * bx - cd * sH * by + sd * bz;
    }
}

// M_j rows: local East e = (p x s)/|p x s| and North n = s x e at s = (l, m, n), with
// p = (0, cos dec0, sin dec0) the celestial pole in the phase-centre (u,v,w) frame (reading G4)
__global__ void uv_basis_kernel(const double *__restrict__ l, const double *__restrict__ m, int n, double sd, double cd,
                                double *__restrict__ M, unsigned int *err)
{
    const int k = blockIdx.x * blockDim.x + threadIdx.x;
    if (k >= n) return;
    const double sx = l[k], sy = m[k], r2 = sx * sx + sy * sy;
    double out[6] = {1.0, 0.0, 0.0, 0.0, 1.0, 0.0};
    if (r2 < 1.0) {
        const double sz = sqrt(1.0 - r2);
        // p x s with p = (0, cd, sd)
        double ex = cd * sz - sd * sy, ey = sd * sx, ez = -cd * sx;
        const double en = sqrt(ex * ex + ey * ey + ez * ez);
        if (en > 0.0) {
            ex /= en; ey /= en; ez /= en;
            out[0] = ex; out[1] = ey; out[2] = ez;
            out[3] = sy * ez - sz * ey;          // s x e
            out[4] = sz * ex - sx * ez;
            out[5] = sx * ey - sy * ex;
        } else {
            atomicAdd(err, 1u);                  // the component sits on the celestial pole: East undefined
        }
    } else {
        atomicAdd(err, 1u);
    }
    for (int i = 0; i < 6; ++i) M[6 * (size_t)k + i] = out[i];
}

}  // namespace

cudaError_t launch_uvw(const double *X, const double *Y, const double *Z, int n_ant, int T, const double *hour_angle_dev,
                       double dec0, double *u, double *v, double *w, cudaStream_t st)
{
    const long long B = (long long)n_ant * (n_ant - 1) / 2;
    uvw_kernel<<<(unsigned)((B + 127) / 128), 128, 0, st>>>(X, Y, Z, n_ant, B, T, hour_angle_dev, sin(dec0), cos(dec0),
                                                            u, v, w); note_launch();
    return cudaGetLastError();
}

cudaError_t launch_uv_basis(const double *l, const double *m, int n, double dec0, double *M, unsigned int *err,
                            cudaStream_t st)
{
    uv_basis_kernel<<<(n + 127) / 128, 128, 0, st>>>(l, m, n, sin(dec0), cos(dec0), M, err); note_launch();
    return cudaGetLastError();
}

}  // namespace woden
