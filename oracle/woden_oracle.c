/* woden_oracle.c -- plain, slow, FP64 CPU predictor.  TEST INFRASTRUCTURE ONLY.
 *
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference
 * legs may build, load or call this file.  It shares no source, header, table or helper
 * with the CUDA library under paper_2005_09316_b200/csrc/, and is never a fallback for it.
 *
 * What it computes is the plain definition (a finite direct sum), one visibility at a time,
 * in the paper's order and notation (citations are PAPER.md line numbers):
 *
 *   V(u_i,v_i,w_i) = sum_j xi_j(u_i,v_i) I_j exp[-2 pi i (u_i l_j + v_i m_j + w_i (n_j - 1))]
 *                                                             Eq 9 (:117) / Eq 11 (:136), B == 1 (:125)
 *   n_j  = sqrt(1 - l_j^2 - m_j^2)                                                        (:115)
 *   I_j  = S0_j (nu / nu0)^alpha_j                 single spectral index per source (:169, :365-367)
 *   (u,v,w) in wavelengths = metres * nu / c       "u,v,w only differ in frequency by a
 *                                                   scaling factor"                        (:161)
 *   point    : xi = 1
 *   Gaussian : xi = exp(-pi^2/(4 ln 2) (kx^2 th_maj^2 + ky^2 th_min^2))                 Eq 12 (:141)
 *              kx =  cos(pa) v + sin(pa) u ;  ky = -sin(pa) v + cos(pa) u            Eq 13-14 (:144-146)
 *   shapelet : xi = sum_q C_q Btilde_{n1_q,n2_q}(kx, ky)                               Eq 15 (:150)
 *              kx = pi/sqrt(2 ln 2) [ cos(pa) v' + sin(pa) u']                          Eq 16 (:152)
 *              ky = pi/sqrt(2 ln 2) [-sin(pa) v' + cos(pa) u']                          Eq 17 (:155)
 *              Btilde_{p1,p2}(kx,ky) = i^(p1+p2) h_{p1}(beta1 kx) h_{p2}(beta2 ky)  Eq 3 (:60), reading G2
 *              h_p(x) = H_p(x) exp(-x^2/2) / sqrt(2^p p!)            Eq 1 (:51) up to the constant
 *                       that the paper's identity B_00 == G (:159) fixes (reading G2)
 *              (u',v') = M_j (u,v,w)^T, or (u,v) when no M_j is given  (:157, reading G4)
 *
 * Implementation rules: double throughout, long double inside h_p; libm sin/cos/pow/exp;
 * Kahan-compensated summation in component order; OpenMP only over the visibility loop.
 *
 * Pins: tests/test_oracle_pins.py (closed forms, brute-force DFTs, mpmath, library Hermite).
 * Parity unpinned against the original WODEN (the paper prints no values): reading G3 (sign
 * of odd orders) and reading G4 (shapelet u',v'); see DESIGN.md.
 */
#include <math.h>
#include <stddef.h>

#define ORACLE_C_LIGHT 299792458.0
#define ORACLE_MAX_ORDER 128

static const double PI = 3.14159265358979323846264338327950288;

typedef struct { double re, im, cre, cim; } kahan_c;

static void kahan_add(kahan_c *a, double re, double im)
{
    double y = re - a->cre, t = a->re + y;
    a->cre = (t - a->re) - y; a->re = t;
    y = im - a->cim; t = a->im + y;
    a->cim = (t - a->im) - y; a->im = t;
}

/* S(nu) = S0 (nu/nu0)^alpha */
static double flux_law(double s0, double alpha, double nu, double nu0)
{
    return s0 * pow(nu / nu0, alpha);
}

/* h_p(x) = H_p(x) exp(-x^2/2)/sqrt(2^p p!) for p = 0..pmax, physicists' Hermite.
 * Unnormalised recurrence H_{p+1} = 2x H_p - 2p H_{p-1} in long double, scaled in the log
 * domain: exp(-x^2/2 - (p ln2 + lgamma(p+1))/2). */
void woden_oracle_hermite_functions(int pmax, double x, double *h_out)
{
    long double xl = (long double)x;
    long double Hm1 = 0.0L, H = 1.0L;
    for (int p = 0; p <= pmax; ++p) {
        long double lognorm = -0.5L * xl * xl
            - 0.5L * ((long double)p * logl(2.0L) + lgammal((long double)p + 1.0L));
        h_out[p] = (double)(H * expl(lognorm));
        long double Hn = 2.0L * xl * H - 2.0L * (long double)p * Hm1;
        Hm1 = H; H = Hn;
    }
}

/* i^k as (re, im) */
static void i_pow(int k, double *re, double *im)
{
    switch (k & 3) {
    case 0: *re = 1.0;  *im = 0.0;  break;
    case 1: *re = 0.0;  *im = 1.0;  break;
    case 2: *re = -1.0; *im = 0.0;  break;
    default: *re = 0.0; *im = -1.0; break;
    }
}

static void split_index(long long flat, int B, int F, int *t, int *f, int *b)
{
    *b = (int)(flat % B);
    long long tf = flat / B;
    *f = (int)(tf % F);
    *t = (int)(tf / F);
}

/* Common driver: kind 0 = points, 1 = Gaussians, 2 = shapelets.
 * vis_index == NULL: all B*T*F visibilities, output index (t*F + f)*B + b.
 * vis_index != NULL: n_index flat indices, output index = position in vis_index.
 * vis is complex128 interleaved (re, im).  accumulate != 0 adds into vis. */
static int predict(int kind, int B, int T, int F,
                   const double *u_m, const double *v_m, const double *w_m,
                   const double *freqs_hz, int n,
                   const double *l, const double *m, const double *s0, const double *alpha,
                   double ref_freq,
                   const double *maj, const double *min_, const double *pa,
                   const double *beta1, const double *beta2, const double *uv_basis,
                   const int *coeff_offset, const int *n1, const int *n2, const double *coeff,
                   const long long *vis_index, long long n_index,
                   double *vis, int accumulate)
{
    if (B <= 0 || T <= 0 || F <= 0 || n < 0) return -2;
    if (!u_m || !v_m || !w_m || !freqs_hz || !vis) return -1;
    if (n > 0 && (!l || !m || !s0 || !alpha)) return -1;
    if (kind == 1 && n > 0 && (!maj || !min_ || !pa)) return -1;
    if (kind == 2 && n > 0 && (!beta1 || !beta2 || !pa || !coeff_offset)) return -1;
    int pmax = 0;
    if (kind == 2 && n > 0) {
        int nc = coeff_offset[n];
        if (nc > 0 && (!n1 || !n2 || !coeff)) return -1;
        for (int q = 0; q < nc; ++q) {
            if (n1[q] < 0 || n2[q] < 0 || n1[q] > ORACLE_MAX_ORDER || n2[q] > ORACLE_MAX_ORDER) return -3;
            if (n1[q] > pmax) pmax = n1[q];
            if (n2[q] > pmax) pmax = n2[q];
        }
    }
    const long long n_out = vis_index ? n_index : (long long)B * T * F;
    const double gauss_const = PI * PI / (4.0 * log(2.0));      /* Eq 12 */
    const double kappa = PI / sqrt(2.0 * log(2.0));             /* Eq 16-17 */

#pragma omp parallel for schedule(dynamic, 64)
    for (long long o = 0; o < n_out; ++o) {
        int t, f, b;
        split_index(vis_index ? vis_index[o] : o, B, F, &t, &f, &b);
        const double nu = freqs_hz[f];
        const double scale = nu / ORACLE_C_LIGHT;               /* metres -> wavelengths (:161) */
        const double u = u_m[(size_t)t * B + b] * scale;
        const double v = v_m[(size_t)t * B + b] * scale;
        const double w = w_m[(size_t)t * B + b] * scale;
        double hx[ORACLE_MAX_ORDER + 1], hy[ORACLE_MAX_ORDER + 1];
        kahan_c V = {0.0, 0.0, 0.0, 0.0};

        for (int j = 0; j < n; ++j) {
            const double nj = sqrt(1.0 - l[j] * l[j] - m[j] * m[j]);
            const double I = flux_law(s0[j], alpha[j], nu, ref_freq);
            const double ph = -2.0 * PI * (u * l[j] + v * m[j] + w * (nj - 1.0));
            double xi_re = 1.0, xi_im = 0.0;
            if (kind == 1) {
                const double kx = cos(pa[j]) * v + sin(pa[j]) * u;
                const double ky = -sin(pa[j]) * v + cos(pa[j]) * u;
                xi_re = exp(-gauss_const * (kx * kx * maj[j] * maj[j] + ky * ky * min_[j] * min_[j]));
            } else if (kind == 2) {
                double up = u, vp = v;
                if (uv_basis) {
                    const double *M = uv_basis + 6 * (size_t)j;
                    up = M[0] * u + M[1] * v + M[2] * w;
                    vp = M[3] * u + M[4] * v + M[5] * w;
                }
                const double kx = kappa * (cos(pa[j]) * vp + sin(pa[j]) * up);
                const double ky = kappa * (-sin(pa[j]) * vp + cos(pa[j]) * up);
                woden_oracle_hermite_functions(pmax, beta1[j] * kx, hx);
                woden_oracle_hermite_functions(pmax, beta2[j] * ky, hy);
                kahan_c xi = {0.0, 0.0, 0.0, 0.0};
                for (int q = coeff_offset[j]; q < coeff_offset[j + 1]; ++q) {
                    double ire, iim;
                    i_pow(n1[q] + n2[q], &ire, &iim);
                    const double bb = coeff[q] * hx[n1[q]] * hy[n2[q]];
                    kahan_add(&xi, bb * ire, bb * iim);
                }
                xi_re = xi.re; xi_im = xi.im;
            }
            const double c = cos(ph), s = sin(ph);
            kahan_add(&V, I * (xi_re * c - xi_im * s), I * (xi_re * s + xi_im * c));
        }
        if (accumulate) { vis[2 * o] += V.re; vis[2 * o + 1] += V.im; }
        else            { vis[2 * o]  = V.re; vis[2 * o + 1]  = V.im; }
    }
    return 0;
}

int woden_oracle_points(int B, int T, int F,
                        const double *u_m, const double *v_m, const double *w_m,
                        const double *freqs_hz, int n,
                        const double *l, const double *m, const double *s0, const double *alpha,
                        double ref_freq,
                        const long long *vis_index, long long n_index,
                        double *vis, int accumulate)
{
    return predict(0, B, T, F, u_m, v_m, w_m, freqs_hz, n, l, m, s0, alpha, ref_freq,
                   NULL, NULL, NULL, NULL, NULL, NULL, NULL, NULL, NULL, NULL,
                   vis_index, n_index, vis, accumulate);
}

int woden_oracle_gaussians(int B, int T, int F,
                           const double *u_m, const double *v_m, const double *w_m,
                           const double *freqs_hz, int n,
                           const double *l, const double *m, const double *s0, const double *alpha,
                           double ref_freq,
                           const double *maj, const double *min_, const double *pa,
                           const long long *vis_index, long long n_index,
                           double *vis, int accumulate)
{
    return predict(1, B, T, F, u_m, v_m, w_m, freqs_hz, n, l, m, s0, alpha, ref_freq,
                   maj, min_, pa, NULL, NULL, NULL, NULL, NULL, NULL, NULL,
                   vis_index, n_index, vis, accumulate);
}

int woden_oracle_shapelets(int B, int T, int F,
                           const double *u_m, const double *v_m, const double *w_m,
                           const double *freqs_hz, int n,
                           const double *l, const double *m, const double *s0, const double *alpha,
                           double ref_freq,
                           const double *beta1, const double *beta2, const double *pa,
                           const double *uv_basis,
                           const int *coeff_offset, const int *n1, const int *n2, const double *coeff,
                           const long long *vis_index, long long n_index,
                           double *vis, int accumulate)
{
    return predict(2, B, T, F, u_m, v_m, w_m, freqs_hz, n, l, m, s0, alpha, ref_freq,
                   NULL, NULL, pa, beta1, beta2, uv_basis, coeff_offset, n1, n2, coeff,
                   vis_index, n_index, vis, accumulate);
}

/* Per-visibility tolerance scale of the north_star parity criterion (reading G12):
 * scale(t,f,b) = sum_k |S_k(nu_f)| * w_k, w_k = 1 for points/Gaussians, sum_q |coeff_q| for a
 * shapelet.  Depends on f only; writes F values, adding into `scale` when accumulate != 0. */
int woden_oracle_tolerance_scale(int F, const double *freqs_hz, int n,
                                 const double *s0, const double *alpha, double ref_freq,
                                 const int *coeff_offset, const double *coeff,
                                 double *scale, int accumulate)
{
    if (F <= 0 || n < 0) return -2;
    if (!freqs_hz || !scale || (n > 0 && (!s0 || !alpha))) return -1;
    for (int f = 0; f < F; ++f) {
        double acc = 0.0;
        for (int j = 0; j < n; ++j) {
            double wgt = 1.0;
            if (coeff_offset) {
                wgt = 0.0;
                for (int q = coeff_offset[j]; q < coeff_offset[j + 1]; ++q) wgt += fabs(coeff[q]);
            }
            acc += fabs(flux_law(s0[j], alpha[j], freqs_hz[f], ref_freq)) * wgt;
        }
        scale[f] = accumulate ? scale[f] + acc : acc;
    }
    return 0;
}

/* ---- the step before the hot path -------------------------------------
 * Baseline (u,v,w) in metres "calculated once per time step" from antenna positions
 * in the local equatorial frame by the standard interferometry rotation (Thompson, Moran & Swenson,
 * cited at PAPER.md:110; reading G14), written as the matrix product
 *   (u,v,w)^T = R(H, d0) (X,Y,Z)^T,   rows of R:  ( sin H,          cos H,         0     )
 *                                                  (-sin d0 cos H,   sin d0 sin H,  cos d0)
 *                                                  ( cos d0 cos H,  -cos d0 sin H,  sin d0)
 * Pairs p < q in p-major order, baseline = antenna p - antenna q.
 * Pinned by tests/test_oracle_pins.py::test_p16_* (length preservation, R orthonormal, w = projection
 * on the source direction, special cases). */
int woden_oracle_uvw(int n_ant, const double *X, const double *Y, const double *Z,
                     int T, const double *hour_angle, double dec0,
                     double *u, double *v, double *w)
{
    if (n_ant < 2 || T <= 0) return -2;
    if (!X || !Y || !Z || !hour_angle || !u || !v || !w) return -1;
    const long long B = (long long)n_ant * (n_ant - 1) / 2;
    for (int t = 0; t < T; ++t) {
        const double H = hour_angle[t];
        const double R[3][3] = {
            { sin(H),              cos(H),             0.0       },
            {-sin(dec0) * cos(H),  sin(dec0) * sin(H), cos(dec0) },
            { cos(dec0) * cos(H), -cos(dec0) * sin(H), sin(dec0) } };
        long long b = 0;
        for (int p = 0; p < n_ant; ++p)
            for (int q = p + 1; q < n_ant; ++q, ++b) {
                const double d[3] = { X[p] - X[q], Y[p] - Y[q], Z[p] - Z[q] };
                double o[3];
                for (int r = 0; r < 3; ++r) o[r] = R[r][0] * d[0] + R[r][1] * d[1] + R[r][2] * d[2];
                u[(size_t)t * B + b] = o[0]; v[(size_t)t * B + b] = o[1]; w[(size_t)t * B + b] = o[2];
            }
    }
    return 0;
}

/* M_j of reading G4: local East / North unit vectors at s = (l, m, n) in the
 * phase-centre (u,v,w) frame; e = (p x s)/|p x s|, north = s x e, p = (0, cos d0, sin d0).
 * Pinned by test_p14_* (orthonormal, perpendicular to s, identity at the phase centre) and
 * test_p16_* (equals re-phasing: uvw about the component's own centre = M_j applied to uvw). */
int woden_oracle_uv_basis(int n, const double *l, const double *m, double dec0, double *M)
{
    if (n < 0) return -2;
    if (n > 0 && (!l || !m || !M)) return -1;
    const double p[3] = { 0.0, cos(dec0), sin(dec0) };
    for (int k = 0; k < n; ++k) {
        const double s[3] = { l[k], m[k], sqrt(1.0 - l[k] * l[k] - m[k] * m[k]) };
        double e[3] = { p[1] * s[2] - p[2] * s[1], p[2] * s[0] - p[0] * s[2], p[0] * s[1] - p[1] * s[0] };
        const double en = sqrt(e[0] * e[0] + e[1] * e[1] + e[2] * e[2]);
        for (int i = 0; i < 3; ++i) e[i] /= en;
        const double nn[3] = { s[1] * e[2] - s[2] * e[1], s[2] * e[0] - s[0] * e[2], s[0] * e[1] - s[1] * e[0] };
        for (int i = 0; i < 3; ++i) { M[6 * (size_t)k + i] = e[i]; M[6 * (size_t)k + 3 + i] = nn[i]; }
    }
    return 0;
}
