// hermite_rec.cuh -- constants of the two-operation Hermite-function recurrence used by the
// shapelet kernels: g_p = h_p / lam_p with lam_0 = lam_1 = 1, lam_{p+1} = sqrt(p/(p+1)) lam_{p-1},
// so that g_{p+1} = (c_p x) g_p - g_{p-1}, c_p = sqrt(2/(p+1)) lam_p / lam_{p+1}
// (h_p(x) = H_p(x) exp(-x^2/2)/sqrt(2^p p!), reading G2).  pack.cu folds lam into the
// stored coefficients.
#pragma once
#include "layout.h"

namespace woden {

constexpr double csqrt(double x)
{
    double r = x > 1.0 ? x : 1.0;
    for (int i = 0; i < 64; ++i) r = 0.5 * (r + x / r);
    return r;
}
// lam_0 = lam_1 = 1, lam_{p+1} = sqrt(p/(p+1)) lam_{p-1}
constexpr double lam_c(int p)
{
    double lam = 1.0;
    for (int q = (p & 1) ? 1 : 0; q + 2 <= p; q += 2) lam *= csqrt((double)(q + 1) / (double)(q + 2));
    return lam;
}
// g_{p+1} = (c_p x) g_p - g_{p-1}
constexpr double c_rec(int p) { return csqrt(2.0 / (double)(p + 1)) * lam_c(p) / lam_c(p + 1); }

struct RecTable {
    float c[MAX_ORDER + 1];
};
constexpr RecTable make_rec()
{
    RecTable t{};
    for (int p = 0; p <= MAX_ORDER; ++p) t.c[p] = (float)c_rec(p);
    return t;
}
constexpr RecTable REC = make_rec();


}  // namespace woden
