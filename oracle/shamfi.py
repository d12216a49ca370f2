"""FP64 CPU oracle of the image-space shapelet fit (SHAMFI, section 2.1, lines 89-102;
truncation weights Eq 25).  TEST INFRASTRUCTURE ONLY, like the rest of oracle/:
only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline legs may import it; it never
imports paper_2005_09316_b200 and shares no code with the CUDA path.

What it computes, literally as the paper states it (Eq 7, :93): a design matrix with one row per
pixel and one column per basis function B_{p1,p2}, p1 + p2 <= p_max, each column the basis function
imaged on the pixel grid and convolved with the restoring beam (:98-100); the coefficients are
`numpy.linalg.lstsq` of that matrix against the pixel values (:96); a list of (beta1, beta2) pairs
is searched by the residual sum of squares of each fit (:102, Fig 3 "(Jy/pixel)^2").

Readings (G17-G19; the paper prints no image-space formula beyond Eq 1-2, 7, 10):
  G17  The image basis is the one whose Fourier transform is exactly what Eq 15-17 evaluate under
       readings G2/G3/G7 (so that fitted coefficients go straight into the predictor with s0 = 1):
           Bimg_{n1,n2}(l, m) = 4 ln2 / (pi beta1 beta2) * h_{n1}(-a x / beta1) h_{n2}(-a y / beta2),
           a = 2 sqrt(2 ln 2),  h_p(t) = H_p(t) exp(-t^2/2) / sqrt(2^p p!),
           x = sin(pa) (l - l0) + cos(pa) (m - m0),  y = cos(pa) (l - l0) - sin(pa) (m - m0)
       (x runs along the major axis, PA from North through East; beta is FWHM-like: B_00 is Eq 10's
       Gaussian with theta = beta, :159, and integrates to one).  A pixel holds Bimg * dl * dm
       (Jy/pixel for a coefficient in Jy).  The minus signs are reading G3's point reflection.
  G18  Restoring beam: Eq 10's Gaussian (bmaj, bmin FWHM, bpa) sampled at the pixel offsets of a
       (2 hw + 1)^2 stencil and divided by its sum ("kernel sums to one", :157); convolution with
       zero padding outside the image ("same" size).  bmaj == 0 means no beam.
  G19  Residual of a fit = sum over pixels of (P - A x)^2.
Pixel (s, t), s = 0..n_l-1 along l, t = 0..n_m-1 along m, is at
  l = l_c + (s - (n_l - 1)/2) dl,  m = m_c + (t - (n_m - 1)/2) dm;  images are [n_m][n_l] (t-major).

The Hermite functions come from the oracle's own long-double routine (woden_oracle.c, pinned by
P8).  Pins of this file: tests/test_shamfi_oracle.py.
"""
from __future__ import annotations

import numpy as np
from scipy.signal import convolve2d

from . import hermite_functions

LN2 = np.log(2.0)
A_FWHM = 2.0 * np.sqrt(2.0 * LN2)


def full_triangle(p_max: int):
    """(n1, n2) of every basis function with n1 + n2 <= p_max, n1-major (Eq 6 count, :84)."""
    n1 = [a for a in range(p_max + 1) for _ in range(p_max + 1 - a)]
    n2 = [b for a in range(p_max + 1) for b in range(p_max + 1 - a)]
    return np.asarray(n1, dtype=np.int32), np.asarray(n2, dtype=np.int32)


def pixel_coordinates(n_l, n_m, dl, dm, l_c=0.0, m_c=0.0):
    """[n_m, n_l] arrays of the pixel centres' l and m."""
    l = l_c + (np.arange(n_l) - (n_l - 1) / 2.0) * dl
    m = m_c + (np.arange(n_m) - (n_m - 1) / 2.0) * dm
    return np.broadcast_to(l[None, :], (n_m, n_l)).copy(), np.broadcast_to(m[:, None], (n_m, n_l)).copy()


def _hermite_table(p_max, t):
    """h_p(t) for p = 0..p_max at every element of the array t: [p_max + 1, *t.shape]."""
    flat = np.asarray(t, dtype=np.float64).ravel()
    out = np.empty((p_max + 1, flat.size))
    for i, v in enumerate(flat):
        out[:, i] = hermite_functions(p_max, float(v))
    return out.reshape((p_max + 1,) + np.shape(t))


def basis_images(n_l, n_m, dl, dm, l_c, m_c, l0, m0, pa, beta1, beta2, p_max):
    """[P, n_m, n_l]: every basis function of reading G17 imaged on the grid (times dl dm)."""
    L, M = pixel_coordinates(n_l, n_m, dl, dm, l_c, m_c)
    x = np.sin(pa) * (L - l0) + np.cos(pa) * (M - m0)
    y = np.cos(pa) * (L - l0) - np.sin(pa) * (M - m0)
    hx = _hermite_table(p_max, -A_FWHM * x / beta1)
    hy = _hermite_table(p_max, -A_FWHM * y / beta2)
    n1, n2 = full_triangle(p_max)
    norm = 4.0 * LN2 / (np.pi * beta1 * beta2) * abs(dl * dm)
    return norm * hx[n1] * hy[n2]


def beam_kernel(dl, dm, bmaj, bmin, bpa, half_width):
    """[2hw+1, 2hw+1] (t-major) restoring-beam stencil of reading G18, unit sum."""
    o = np.arange(-half_width, half_width + 1)
    DL, DM = np.meshgrid(o * dl, o * dm)                        # [t][s]
    xb = np.sin(bpa) * DL + np.cos(bpa) * DM
    yb = np.cos(bpa) * DL - np.sin(bpa) * DM
    with np.errstate(divide="ignore", invalid="ignore"):
        ex = np.where(bmaj > 0, xb ** 2 / bmaj ** 2, np.where(xb == 0, 0.0, np.inf))
        ey = np.where(bmin > 0, yb ** 2 / bmin ** 2, np.where(yb == 0, 0.0, np.inf))
    k = np.exp(-4.0 * LN2 * (ex + ey))                           # Eq 10 (:131)
    return k / k.sum()


def design_matrix(n_l, n_m, dl, dm, l_c, m_c, l0, m0, pa, beta1, beta2, p_max,
                  bmaj=0.0, bmin=0.0, bpa=0.0, half_width=0):
    """[n_m * n_l, P]: Eq 7's matrix, columns convolved with the restoring beam (:98-100)."""
    imgs = basis_images(n_l, n_m, dl, dm, l_c, m_c, l0, m0, pa, beta1, beta2, p_max)
    if bmaj > 0.0:
        ker = beam_kernel(dl, dm, bmaj, bmin, bpa, half_width)
        imgs = np.stack([convolve2d(im, ker, mode="same", boundary="fill", fillvalue=0.0) for im in imgs])
    return imgs.reshape(imgs.shape[0], -1).T.copy()


def render(coeff, *args, **kw):
    """Model image [n_m, n_l] of a coefficient list (full triangle order) = A x."""
    n_l, n_m = args[0], args[1]
    return (design_matrix(*args, **kw) @ np.asarray(coeff, dtype=np.float64)).reshape(n_m, n_l)


def fit(image, n_l, n_m, dl, dm, l_c, m_c, l0, m0, pa, beta1, beta2, p_max,
        bmaj=0.0, bmin=0.0, bpa=0.0, half_width=0):
    """Eq 7 by numpy.linalg.lstsq (:96).  Returns (coeff [P], residual sum of squares, A)."""
    A = design_matrix(n_l, n_m, dl, dm, l_c, m_c, l0, m0, pa, beta1, beta2, p_max, bmaj, bmin, bpa, half_width)
    b = np.asarray(image, dtype=np.float64).reshape(-1)
    x = np.linalg.lstsq(A, b, rcond=None)[0]
    r = b - A @ x
    return x, float(r @ r), A


def grid_search(image, n_l, n_m, dl, dm, l_c, m_c, l0, m0, pa, beta1_list, beta2_list, p_max,
                bmaj=0.0, bmin=0.0, bpa=0.0, half_width=0):
    """Fit every (beta1, beta2) pair of the two equally long lists; the best pair is the one with
    the smallest residual (:102).  Returns (coeff [n, P], residual [n], best index)."""
    coeffs, res = [], []
    for b1, b2 in zip(beta1_list, beta2_list):
        x, r, _ = fit(image, n_l, n_m, dl, dm, l_c, m_c, l0, m0, pa, b1, b2, p_max, bmaj, bmin, bpa, half_width)
        coeffs.append(x)
        res.append(r)
    res = np.asarray(res)
    return np.stack(coeffs), res, int(np.argmin(res))


def truncation_weights(coeff, A):
    """Eq 25 (:279): I_{p1,p2} = sum over pixels |C_{p1,p2} (G * B_{p1,p2})(x_s, y_t)|, with A the
    beam-convolved design matrix of the fit."""
    return np.abs(np.asarray(coeff, dtype=np.float64)) * np.abs(A).sum(axis=0)
