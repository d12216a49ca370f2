"""GPU-vs-oracle parity of the image-space shapelet fit (woden_fit_shapelets; Eq 7,
Eq 25), `-m gpu`, through the C ABI.

What is compared.  The least-squares solution is unique when the design matrix has full rank, and the
library reaches it by refinement with the exact FP64 operator (fit.cu), so for well-conditioned fits the
coefficients themselves are compared: |x_gpu - x_oracle| <= 1e-8 max|x| (DESIGN.md derives it: FP64
operator, contraction <= 0.06 per pass at condition number 10^3, six passes).  For ill-conditioned fits
(a beam much wider than the finest basis structure, the paper's own regime) coefficients of the
undetermined directions are not unique in practice; what is unique is the fitted image A x and the
residual, and those are compared."""
import numpy as np
import pytest

import oracle
from oracle import shamfi
from paper_2005_09316_b200 import inputs

pytestmark = pytest.mark.gpu

ARCMIN = np.pi / 180.0 / 60.0
C_LIGHT = 299792458.0


@pytest.fixture(scope="module")
def ctx():
    from paper_2005_09316_b200 import binding
    c = binding.Woden(0)
    yield c
    c.close()


def _dev(a, dtype=None):
    import torch
    return torch.as_tensor(np.ascontiguousarray(a), dtype=dtype or torch.float64, device="cuda:0")


def _planted(seed, p_max, decay):
    rng = np.random.default_rng(seed)
    n1, n2 = shamfi.full_triangle(p_max)
    return rng.normal(0, 1, len(n1)) * np.exp(-(n1 + n2) / decay)


def _gpu_fit(ctx, img, g, l0, m0, pa, p_max, b1, b2, beam=None, **kw):
    import torch
    out = ctx.fit_shapelets(_dev(img), g[2], g[3], g[4], g[5], l0, m0, pa, p_max, b1, b2, beam=beam, **kw)
    torch.cuda.synchronize()
    ctx.check()
    return [None if t is None else t.cpu().numpy() for t in out]


@pytest.mark.parametrize("n_l,n_m,p_max", [(64, 64, 8), (50, 37, 12), (90, 77, 20), (96, 96, 30)])
def test_noiseless_and_noisy_fits_match_lstsq(ctx, n_l, n_m, p_max):
    # no beam; pixel counts that are not multiples of the 64-pixel K stage, unknown counts (45, 91, 231,
    # 496) that are not multiples of the 128-row tile; basis well sampled and well contained
    pa, l0, m0 = 0.7, 0.4 * ARCMIN, -0.3 * ARCMIN
    pix = 0.4 * ARCMIN
    g = (n_l, n_m, -pix, pix, 0.2 * ARCMIN, 0.1 * ARCMIN)
    ext = min(n_l, n_m) * pix
    beta = ext * 2.3548 / (2.0 * 2.6 * np.sqrt(2 * p_max + 1.0))       # order p_max turning point at 38 % of the extent
    b1, b2 = beta, 0.85 * beta
    planted = _planted(p_max, p_max, 6.0)
    clean = shamfi.render(planted, *g, l0, m0, pa, b1, b2, p_max)
    rng = np.random.default_rng(p_max)
    for img in (clean, clean + rng.normal(0, 0.02 * np.abs(clean).max(), clean.shape)):
        x_ref, res_ref, A = shamfi.fit(img, *g, l0, m0, pa, b1, b2, p_max)
        assert np.linalg.cond(A / np.abs(A).max(axis=0)) < 1e3          # the regime the coefficient tolerance is for
        coeff, resid, _, best = _gpu_fit(ctx, img, g, l0, m0, pa, p_max, [b1], [b2])
        assert np.abs(coeff[0] - x_ref).max() <= 1e-8 * np.abs(x_ref).max()
        assert abs(resid[0] - res_ref) <= 1e-9 * float(img.ravel() @ img.ravel()) + 1e-12 * res_ref
        assert best[0] == 0
    assert np.abs(coeff[0] - planted).max() < 0.2 * np.abs(planted).max()   # and it is the planted model, to the noise


def test_beam_convolved_fit_grid_search_and_eq25_weights(ctx):
    p_max, pa = 10, 1.9
    b1, b2 = 3.2 * ARCMIN, 2.4 * ARCMIN
    beam = (1.3 * ARCMIN, 0.9 * ARCMIN, 0.4, 9)
    g = (72, 66, -0.35 * ARCMIN, 0.35 * ARCMIN, 0.0, 0.3 * ARCMIN)
    l0, m0 = -0.2 * ARCMIN, 0.5 * ARCMIN
    kw = dict(bmaj=beam[0], bmin=beam[1], bpa=beam[2], half_width=beam[3])
    planted = _planted(2, p_max, 4.0)
    rng = np.random.default_rng(21)
    img = shamfi.render(planted, *g, l0, m0, pa, b1, b2, p_max, **kw)
    img = img + rng.normal(0, 1e-3 * np.abs(img).max(), img.shape)
    f1, f2 = np.meshgrid([0.85, 1.0, 1.2], [0.85, 1.0, 1.2], indexing="ij")
    B1, B2 = (b1 * f1).ravel(), (b2 * f2).ravel()
    c_ref, r_ref, best_ref = shamfi.grid_search(img, *g, l0, m0, pa, B1, B2, p_max, **kw)
    coeff, resid, weights, best = _gpu_fit(ctx, img, g, l0, m0, pa, p_max, B1, B2, beam=beam, want_weights=True)
    assert best[0] == best_ref == 4
    power = float(img.ravel() @ img.ravel())
    for k in range(9):
        A = shamfi.design_matrix(*g, l0, m0, pa, B1[k], B2[k], p_max, **kw)
        # the fitted image and the residual are unique: always compared
        assert np.abs(A @ (coeff[k] - c_ref[k])).max() <= 1e-9 * np.abs(img).max(), k
        assert abs(resid[k] - r_ref[k]) <= 1e-9 * power, k
        if np.linalg.cond(A / np.abs(A).max(axis=0)) < 1e3:
            assert np.abs(coeff[k] - c_ref[k]).max() <= 1e-8 * np.abs(c_ref[k]).max(), k
            w_ref = shamfi.truncation_weights(c_ref[k], A)
            assert np.abs(weights[k] - w_ref).max() <= 1e-8 * w_ref.max(), k
    # the stencil really was applied: without the beam the same image fits worse at the planted beta
    _, r_nobeam, _, _ = _gpu_fit(ctx, img, g, l0, m0, pa, p_max, [b1], [b2])
    assert r_nobeam[0] > 10 * resid[4]


def test_ill_conditioned_fit_matches_in_image_space(ctx):
    # a beam as wide as beta damps the high orders by many decades (the paper fits with p_max chosen at a
    # third of the resolution, :183): lstsq and the refined normal equations agree on the fitted image
    p_max, pa = 14, 0.3
    b1 = b2 = 2.0 * ARCMIN
    beam = (2.5 * ARCMIN, 2.0 * ARCMIN, 1.0, 14)
    g = (80, 80, -0.3 * ARCMIN, 0.3 * ARCMIN, 0.0, 0.0)
    kw = dict(bmaj=beam[0], bmin=beam[1], bpa=beam[2], half_width=beam[3])
    planted = _planted(9, p_max, 3.0)
    rng = np.random.default_rng(33)
    img = shamfi.render(planted, *g, 0.0, 0.0, pa, b1, b2, p_max, **kw)
    img = img + rng.normal(0, 1e-3 * np.abs(img).max(), img.shape)
    x_ref, res_ref, A = shamfi.fit(img, *g, 0.0, 0.0, pa, b1, b2, p_max, **kw)
    assert np.linalg.cond(A / np.abs(A).max(axis=0)) > 1e4
    coeff, resid, _, _ = _gpu_fit(ctx, img, g, 0.0, 0.0, pa, p_max, [b1], [b2], beam=beam, n_refine=12)
    power = float(img.ravel() @ img.ravel())
    assert res_ref <= resid[0] <= res_ref + 1e-6 * power           # lstsq's residual is the minimum
    assert np.abs(A @ (coeff[0] - x_ref)).max() <= 2e-3 * np.abs(img).max()
    assert np.all(np.isfinite(coeff[0]))


def test_fit_at_the_orders_of_the_paper(ctx):
    # p_max = 46 is the paper's phase I order (1128 basis functions); 60 is config 4's.
    # 9 and 15 row tiles of 128, 18 and 30 Cholesky panels; fitted image and residual against lstsq,
    # coefficients too when the scaled design matrix is well conditioned.
    for p_max, n in ((46, 150), (60, 200)):
        pa, pix = 0.4, 0.3 * ARCMIN
        g = (n, n, -pix, pix, 0.0, 0.0)
        beta = n * pix * 2.3548 / (2.0 * 2.5 * np.sqrt(2 * p_max + 1.0))
        planted = _planted(p_max, p_max, 8.0)
        rng = np.random.default_rng(p_max)
        img = shamfi.render(planted, *g, 0.0, 0.0, pa, beta, 0.9 * beta, p_max)
        img = img + rng.normal(0, 0.01 * np.abs(img).max(), img.shape)
        x_ref, res_ref, A = shamfi.fit(img, *g, 0.0, 0.0, pa, beta, 0.9 * beta, p_max)
        coeff, resid, _, _ = _gpu_fit(ctx, img, g, 0.0, 0.0, pa, p_max, [beta], [0.9 * beta])
        power = float(img.ravel() @ img.ravel())
        assert np.abs(A @ (coeff[0] - x_ref)).max() <= 1e-8 * np.abs(img).max(), p_max
        assert abs(resid[0] - res_ref) <= 1e-9 * power, p_max
        if np.linalg.cond(A / np.abs(A).max(axis=0)) < 1e3:
            assert np.abs(coeff[0] - x_ref).max() <= 1e-8 * np.abs(x_ref).max(), p_max


def test_round_trip_image_to_fit_to_predicted_visibilities(ctx):
    # image of a planted model -> woden_fit_shapelets -> woden_predict_shapelets, against the oracle
    # predicting the PLANTED coefficients (Eq 15-17): north_star tolerance 1e-4 sum|coeff|
    import torch
    from paper_2005_09316_b200 import binding
    p_max, pa = 16, 2.2
    b1, b2 = 2.6 * ARCMIN, 2.0 * ARCMIN
    l0, m0 = 0.004, -0.003
    g = (96, 96, -0.3 * ARCMIN, 0.3 * ARCMIN, l0, m0)
    planted = _planted(4, p_max, 5.0)
    img = shamfi.render(planted, *g, l0, m0, pa, b1, b2, p_max)
    coeff, resid, _, _ = _gpu_fit(ctx, img, g, l0, m0, pa, p_max, [b1], [b2])
    assert np.abs(coeff[0] - planted).max() <= 1e-8 * np.abs(planted).max()
    wl = inputs.make_config(1)
    u, v, w = wl.u_m, wl.v_m, wl.w_m
    fr = wl.freqs_hz
    n1, n2 = shamfi.full_triangle(p_max)
    d = lambda a, dt=None: _dev(a, dt)
    uvw = binding.Uvw(d(u), d(v), d(w), fr)
    vis = ctx.new_vis(uvw)
    ctx.set_path(0)
    ctx.predict_shapelets(uvw, d([l0]), d([m0]), d([1.0]), d([0.0]), 150e6, d([b1]), d([b2]), d([pa]), None,
                          d([0, len(n1)], torch.int32), len(n1), p_max, d(n1, torch.int32), d(n2, torch.int32),
                          torch.as_tensor(coeff[0], device="cuda:0"), vis)
    torch.cuda.synchronize(); ctx.check()
    ref = oracle.predict_shapelets(u, v, w, fr, [l0], [m0], [1.0], [0.0], 150e6, [b1], [b2], [pa], None,
                                   [0, len(n1)], n1, n2, planted)
    assert np.abs(vis.cpu().numpy() - ref).max() <= 1e-4 * np.abs(planted).sum()
    assert np.abs(ref).max() > 0.1


def test_fit_error_codes(ctx):
    import torch
    from paper_2005_09316_b200 import binding
    img = torch.zeros((16, 16), dtype=torch.float64, device="cuda:0")
    with pytest.raises(binding.WodenError) as e:
        ctx.fit_shapelets(img, 1e-4, 1e-4, 0, 0, 0, 0, 0.0, 87, [1e-3], [1e-3])
    assert e.value.status == binding.WODEN_ERR_ORDER
    with pytest.raises(binding.WodenError) as e:
        ctx.fit_shapelets(img, 0.0, 1e-4, 0, 0, 0, 0, 0.0, 4, [1e-3], [1e-3])
    assert e.value.status == binding.WODEN_ERR_DIM
    with pytest.raises(binding.WodenError) as e:
        ctx.fit_shapelets(img, 1e-4, 1e-4, 0, 0, 0, 0, 0.0, 4, [1e-3], [-1e-3])
    assert e.value.status == binding.WODEN_ERR_DIM
    with pytest.raises(binding.WodenError) as e:
        ctx.fit_shapelets(img, 1e-4, 1e-4, 0, 0, 0, 0, 0.0, 4, [1e-3], [1e-3], beam=(1e-3, 1e-3, 0.0, 25))
    assert e.value.status == binding.WODEN_ERR_DIM
    # an all-zero image fits to zero coefficients and zero residual
    coeff, resid, _, best = ctx.fit_shapelets(img, 1e-4, 1e-4, 0, 0, 0, 0, 0.0, 4, [1e-3, 2e-3], [1e-3, 2e-3])
    torch.cuda.synchronize(); ctx.check()
    assert float(coeff.abs().max()) == 0.0 and float(resid.abs().max()) == 0.0 and int(best[0]) == 0
