"""Pins of the image-space fit oracle (oracle/shamfi.py; section 2.1, :89-102, Eq 25 :279).
`-m "not gpu"`.  The paper prints no number for the fit, so the pins are closed forms, the paper's
own identities, and the already pinned visibility-side oracle (woden_oracle.c): a plausible mistake in
the image basis (a sign, a swapped beta, the PA sense, the FWHM scaling, the normalisation, the beam's
orientation or normalisation, the pixel indexing) fails at least one of them."""
import numpy as np
import pytest

import oracle
from oracle import shamfi

ARCMIN = np.pi / 180.0 / 60.0
LN2 = np.log(2.0)
C_LIGHT = 299792458.0


def _dft(image, n_l, n_m, dl, dm, l_c, m_c, u, v):
    """sum over pixels of P exp(-2 pi i (u l + v m)), Eq 9's kernel at w = 0, one (u, v) at a time."""
    L, M = shamfi.pixel_coordinates(n_l, n_m, dl, dm, l_c, m_c)
    return np.array([np.sum(image * np.exp(-2j * np.pi * (uu * L + vv * M))) for uu, vv in zip(u, v)])


GRID = dict(n_l=72, n_m=60, dl=-0.45 * ARCMIN, dm=0.5 * ARCMIN, l_c=2.0 * ARCMIN, m_c=-1.0 * ARCMIN)


def test_basis_is_orthogonal_with_the_closed_form_norm():
    # continuum: int Bimg_q Bimg_q' dl dm = 2 ln2 / (pi beta1 beta2) delta_qq' (int h_p h_q = sqrt(pi) delta,
    # P8); the pixel sum is that times dl dm for a well sampled, well contained basis (trapezoid rule on
    # Gaussian-decaying functions converges spectrally).  Rotated, off-centre, rectangular pixels.
    b1, b2, pa = 4.0 * ARCMIN, 3.0 * ARCMIN, 0.7
    g = dict(GRID, n_l=160, n_m=160, dl=-0.25 * ARCMIN, dm=0.25 * ARCMIN)
    B = shamfi.basis_images(**g, l0=2.5 * ARCMIN, m0=-0.5 * ARCMIN, pa=pa, beta1=b1, beta2=b2, p_max=6)
    A = B.reshape(B.shape[0], -1)
    gram = A @ A.T
    expect = 2.0 * LN2 * abs(g["dl"] * g["dm"]) / (np.pi * b1 * b2)
    assert np.abs(gram / expect - np.eye(len(A))).max() < 1e-10
    assert len(A) == 28                                          # Eq 6 at p_max = 6


def test_b00_is_eq10s_gaussian_with_theta_equal_beta():
    # PAPER.md:159 "G(x, y, theta_maj, theta_min) = B_00(x, y, theta_maj, theta_min)"; Eq 10 (:131) is
    # typed here from the paper with the major axis along (sin pa, cos pa) (reading G7), unit integral
    b1, b2, pa, l0, m0 = 6.0 * ARCMIN, 2.5 * ARCMIN, 1.1, 1.0 * ARCMIN, 0.5 * ARCMIN
    L, M = shamfi.pixel_coordinates(**GRID)
    x = (L - l0) * np.sin(pa) + (M - m0) * np.cos(pa)
    y = (L - l0) * np.cos(pa) - (M - m0) * np.sin(pa)
    G = np.exp(-4.0 * LN2 * (x ** 2 / b1 ** 2 + y ** 2 / b2 ** 2))
    G *= 4.0 * LN2 / (np.pi * b1 * b2) * abs(GRID["dl"] * GRID["dm"])
    B00 = shamfi.basis_images(**GRID, l0=l0, m0=m0, pa=pa, beta1=b1, beta2=b2, p_max=0)[0]
    assert np.abs(B00 - G).max() < 1e-15 * G.max() * 10
    assert abs(G.sum() - 1.0) < 1e-9                              # the kernel sums to one (:157)
    # a 7.5 Jy Gaussian fitted with the single (0,0) term returns its integrated flux density
    x00, res, _ = shamfi.fit(7.5 * G, **GRID, l0=l0, m0=m0, pa=pa, beta1=b1, beta2=b2, p_max=0)
    assert abs(x00[0] - 7.5) < 1e-12 and res < 1e-24
    # the PA sense matters: the mirrored angle does not reproduce it
    wrong, res_w, _ = shamfi.fit(7.5 * G, **GRID, l0=l0, m0=m0, pa=-pa, beta1=b1, beta2=b2, p_max=0)
    assert res_w > 1e-6


@pytest.mark.parametrize("pa", [0.0, 0.6, 2.3])
def test_image_model_transforms_to_the_predicted_visibilities(pa):
    # The round trip that makes fitted coefficients usable by the predictor: the direct DFT (Eq 9's
    # kernel, w = 0) of the rendered image equals woden_oracle_shapelets of the same coefficient list
    # (Eq 15-17 under readings G2/G3/G7), including odd orders (whose sign is reading G3's reflection)
    # and the phase of the off-centre position.
    rng = np.random.default_rng(3)
    p_max, b1, b2 = 5, 3.5 * ARCMIN, 2.2 * ARCMIN
    l0, m0 = 1.5 * ARCMIN, -2.0 * ARCMIN
    g = dict(n_l=128, n_m=128, dl=-0.3 * ARCMIN, dm=0.3 * ARCMIN, l_c=1.0 * ARCMIN, m_c=-1.5 * ARCMIN)
    n1, n2 = shamfi.full_triangle(p_max)
    coeff = rng.normal(0, 1, len(n1))
    img = shamfi.render(coeff, g["n_l"], g["n_m"], g["dl"], g["dm"], g["l_c"], g["m_c"], l0, m0, pa, b1, b2, p_max)
    u = rng.uniform(-400, 400, 30); v = rng.uniform(-400, 400, 30)
    got = _dft(img, **g, u=u, v=v)
    um = u[None, :]; vm = v[None, :]; wm = np.zeros((1, 30))
    ref = oracle.predict_shapelets(um, vm, wm, np.array([C_LIGHT]), [l0], [m0], [1.0], [0.0], C_LIGHT,
                                   [b1], [b2], [pa], None, [0, len(n1)], n1, n2, coeff)[0, 0]
    # n - 1 of the off-centre direction multiplies w = 0: no contribution
    assert np.abs(got - ref).max() < 1e-9 * np.abs(coeff).sum()
    assert np.abs(ref).max() > 0.1


def test_single_odd_terms_fix_the_reflection_and_the_axis_pairing():
    # one coefficient at a time, beta1 != beta2: (1,0) and (0,1) are odd in x resp. y
    b1, b2, pa = 4.0 * ARCMIN, 2.0 * ARCMIN, 0.4
    g = dict(n_l=128, n_m=128, dl=-0.25 * ARCMIN, dm=0.25 * ARCMIN, l_c=0.0, m_c=0.0)
    rng = np.random.default_rng(5)
    u = rng.uniform(-300, 300, 12)[None, :]; v = rng.uniform(-300, 300, 12)[None, :]
    for a, b in [(1, 0), (0, 1), (2, 1), (3, 0)]:
        p_max = a + b
        n1, n2 = shamfi.full_triangle(p_max)
        coeff = ((n1 == a) & (n2 == b)).astype(float)
        img = shamfi.render(coeff, g["n_l"], g["n_m"], g["dl"], g["dm"], 0.0, 0.0, 0.0, 0.0, pa, b1, b2, p_max)
        got = _dft(img, **g, u=u[0], v=v[0])
        ref = oracle.predict_shapelets(u, v, 0 * u, np.array([C_LIGHT]), [0.0], [0.0], [1.0], [0.0], C_LIGHT,
                                       [b1], [b2], [pa], None, [0, 1], [a], [b], [1.0])[0, 0]
        assert np.abs(got - ref).max() < 1e-10, (a, b)
        assert np.abs(ref).max() > 0.05


def test_restoring_beam_closed_form_and_orientation():
    # (i) circular beta and circular beam: Gaussians convolve to FWHM^2 = beta^2 + beam^2
    beta, beam = 4.0 * ARCMIN, 3.0 * ARCMIN
    g = dict(n_l=96, n_m=96, dl=-0.25 * ARCMIN, dm=0.25 * ARCMIN, l_c=0.0, m_c=0.0)
    hw = 40                                                       # 10 arcmin = 3.3 beam FWHM: e^-30
    A = shamfi.design_matrix(**g, l0=0.0, m0=0.0, pa=0.3, beta1=beta, beta2=beta, p_max=0,
                             bmaj=beam, bmin=beam, bpa=1.0, half_width=hw)
    L, M = shamfi.pixel_coordinates(**g)
    w2 = beta ** 2 + beam ** 2
    expect = 4.0 * LN2 / (np.pi * w2) * np.exp(-4.0 * LN2 * (L ** 2 + M ** 2) / w2) * abs(g["dl"] * g["dm"])
    inner = (np.abs(L) < 6 * ARCMIN) & (np.abs(M) < 6 * ARCMIN)  # away from the zero-padded edge
    assert np.abs(A[:, 0].reshape(96, 96) - expect)[inner].max() < 1e-9 * expect.max()
    ker = shamfi.beam_kernel(g["dl"], g["dm"], beam, beam, 0.0, hw)
    assert abs(ker.sum() - 1.0) < 1e-15 and ker.shape == (81, 81)
    # (ii) elliptical beam: the transform of a convolved column = (Eq 15-17 of the basis function) x
    # (Eq 12-14 of the beam), both from the pinned visibility-side oracle: fixes the beam's PA sense
    # and FWHM convention
    b1, b2, pa = 3.0 * ARCMIN, 2.0 * ARCMIN, 0.8
    bmaj, bmin, bpa = 3.0 * ARCMIN, 1.5 * ARCMIN, 2.0
    g = dict(n_l=144, n_m=144, dl=-0.2 * ARCMIN, dm=0.2 * ARCMIN, l_c=0.0, m_c=0.0)
    n1, n2 = shamfi.full_triangle(3)
    A = shamfi.design_matrix(**g, l0=0.0, m0=0.0, pa=pa, beta1=b1, beta2=b2, p_max=3,
                             bmaj=bmaj, bmin=bmin, bpa=bpa, half_width=45)
    rng = np.random.default_rng(8)
    u = rng.uniform(-250, 250, 10)[None, :]; v = rng.uniform(-250, 250, 10)[None, :]
    fr = np.array([C_LIGHT])
    env = oracle.predict_gaussians(u, v, 0 * u, fr, [0.0], [0.0], [1.0], [0.0], C_LIGHT, [bmaj], [bmin], [bpa])[0, 0]
    for q in (0, 2, 5, 9):
        got = _dft(A[:, q].reshape(144, 144), **g, u=u[0], v=v[0])
        ref = oracle.predict_shapelets(u, v, 0 * u, fr, [0.0], [0.0], [1.0], [0.0], C_LIGHT, [b1], [b2], [pa], None,
                                       [0, 1], [n1[q]], [n2[q]], [1.0])[0, 0]
        assert np.abs(got - ref * env).max() < 1e-8, q
    assert np.abs(env).min() < 0.9                                  # the beam does something at these (u, v)


def test_planted_model_is_recovered_and_the_residual_picks_its_beta():
    rng = np.random.default_rng(11)
    p_max, pa = 8, 0.9
    b1, b2 = 3.0 * ARCMIN, 2.0 * ARCMIN
    beam = dict(bmaj=1.2 * ARCMIN, bmin=0.8 * ARCMIN, bpa=0.2, half_width=8)
    g = (64, 56, -0.4 * ARCMIN, 0.4 * ARCMIN, 0.5 * ARCMIN, 0.0)
    n1, n2 = shamfi.full_triangle(p_max)
    planted = rng.normal(0, 1, len(n1)) * np.exp(-(n1 + n2) / 4.0)
    img = shamfi.render(planted, *g, 0.3 * ARCMIN, 0.2 * ARCMIN, pa, b1, b2, p_max, **beam)
    x, res, A = shamfi.fit(img, *g, 0.3 * ARCMIN, 0.2 * ARCMIN, pa, b1, b2, p_max, **beam)
    assert np.abs(x - planted).max() < 1e-10 * np.abs(planted).max()
    assert res < 1e-24 * float(img.ravel() @ img.ravel())
    assert A.shape == (64 * 56, 45)
    # grid of (beta1, beta2) pairs around the planted one (Fig 3): smallest residual there
    f1, f2 = np.meshgrid([0.8, 1.0, 1.25], [0.8, 1.0, 1.25], indexing="ij")
    coeffs, resid, best = shamfi.grid_search(img, *g, 0.3 * ARCMIN, 0.2 * ARCMIN, pa, (b1 * f1).ravel(),
                                             (b2 * f2).ravel(), p_max, **beam)
    assert best == 4 and resid[4] < 1e-20 and np.all(np.delete(resid, 4) > 1e6 * max(resid[4], 1e-30))
    # the fit is the least-squares one: the residual image is orthogonal to every column (normal equations)
    noisy = img + rng.normal(0, 1e-3 * np.abs(img).max(), img.shape)
    xn, _, An = shamfi.fit(noisy, *g, 0.3 * ARCMIN, 0.2 * ARCMIN, pa, b1, b2, p_max, **beam)
    r = noisy.ravel() - An @ xn
    assert np.abs(An.T @ r).max() < 1e-12 * np.abs(An.T @ noisy.ravel()).max()


def test_eq25_truncation_weights():
    # I_{p1,p2} = sum_pixels |C (G * B)|: the (0,0) column is positive and sums to one, so
    # its weight is |C_00|; every weight equals the explicit double loop over pixels
    p_max, pa, b1, b2 = 4, 0.5, 3.0 * ARCMIN, 2.5 * ARCMIN
    g = (48, 48, -0.4 * ARCMIN, 0.4 * ARCMIN, 0.0, 0.0)
    beam = dict(bmaj=1.0 * ARCMIN, bmin=1.0 * ARCMIN, bpa=0.0, half_width=7)
    A = shamfi.design_matrix(*g, 0.0, 0.0, pa, b1, b2, p_max, **beam)
    coeff = np.array([(-1.0) ** q * (q + 1.0) for q in range(A.shape[1])])
    w = shamfi.truncation_weights(coeff, A)
    assert abs(w[0] - 1.0) < 1e-6
    for q in (1, 7, 14):
        s = 0.0
        for i in range(A.shape[0]):
            s += abs(coeff[q] * A[i, q])
        assert abs(w[q] - s) < 1e-12 * s
    assert w.shape == (15,) and np.all(w > 0)
