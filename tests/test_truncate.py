"""Model truncation (§5.3, Eq 23-24): host-side selection logic, checked by brute force."""
import numpy as np

from paper_2005_09316_b200 import inputs, truncate


def _brute_n_keep(a_sorted, f):
    tot, n, run = sum(a_sorted), 0, 0.0
    for x in a_sorted:                       # Eq 23: largest N with sum_{j<=N} |I_j| <= f * total
        if run + x <= f * tot * (1 + 1e-15):
            run += x; n += 1
        else:
            break
    return n


def test_eq23_eq24_against_brute_force():
    rng = np.random.default_rng(5)
    for _ in range(50):
        a = np.sort(rng.lognormal(0, 1.5, rng.integers(1, 40)))[::-1]
        for f in (0.0, 0.1, 0.5, 0.9, 0.999, 1.0):
            assert truncate.n_keep(a, f) == _brute_n_keep(list(a), f)
    assert truncate.n_keep(np.array([]), 0.5) == 0
    # worked example: |I| = 5, 3, 1, 1 (total 10): f = 0.8 keeps {5, 3}; f = 0.85 still {5, 3}; 0.9 adds one
    a = np.array([5.0, 3.0, 1.0, 1.0])
    assert [truncate.n_keep(a, f) for f in (0.49, 0.5, 0.8, 0.85, 0.9, 1.0)] == [0, 1, 2, 2, 3, 4]


def test_components_keep_the_brightest_by_absolute_flux():
    wl = inputs.make_config(4)               # MS-CLEAN-like: 25 % negative components
    g = truncate.truncate_components(wl.gaussians, 0.5)
    assert 0 < g.n < wl.gaussians.n
    assert np.abs(g.s0_jy).min() >= np.sort(np.abs(wl.gaussians.s0_jy))[::-1][g.n - 1] - 1e-15
    assert (g.s0_jy < 0).any() and g.maj_fwhm_rad.shape == g.l.shape == g.pa_rad.shape
    assert np.abs(g.s0_jy).sum() <= 0.5 * np.abs(wl.gaussians.s0_jy).sum() * (1 + 1e-12)
    full = truncate.truncate_components(wl.points, 1.0)
    assert full.n == wl.points.n and np.array_equal(full.l, wl.points.l)


def test_shapelet_truncation_keeps_csr_consistent():
    wl = inputs.make_config(5)
    s = wl.shapelets
    w = truncate.shapelet_basis_weights(s)
    assert w.shape == s.coeff.shape and (w >= 0).all() and w.max() > 0
    for f in (1.0, 0.6, 0.2):
        t = truncate.truncate_shapelets(s, f, w)
        assert t.coeff_offset[0] == 0 and t.coeff_offset[-1] == t.coeff.size == t.n1.size == t.n2.size
        assert np.all(np.diff(t.coeff_offset) >= 0) and t.n == s.n
        if f == 1.0:
            assert np.array_equal(t.coeff, s.coeff)
        else:
            assert 0 < t.coeff.size < s.coeff.size
    empty = inputs.make_config(2).shapelets                      # a config without shapelets passes through
    assert truncate.truncate_shapelets(empty, 0.5).n == 0
    # the (0,0) weight is |C| * 1 by construction (pixel-sum normalisation of each component's basis)
    j0 = int(s.coeff_offset[0])
    assert s.n1[j0] == 0 and s.n2[j0] == 0
    assert np.isclose(w[j0], abs(s.coeff[j0] * s.s0_jy[0]))
