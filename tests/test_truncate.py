"""Model truncation (section 5.3, Eq 23-24): pins of the oracle (oracle/truncate.py) on the CPU
and, `-m gpu`, parity of woden_truncate_select / woden_shapelet_basis_sums against the oracles."""
import numpy as np
import pytest

from oracle import shamfi
from oracle import truncate as otrunc
from paper_2005_09316_b200 import inputs

ARCMIN = np.pi / 180.0 / 60.0


def _brute_keep(weights, f):
    """Every prefix of the ranked list is tried; the largest admissible one wins (Eq 23 read literally)."""
    w = [abs(float(x)) for x in weights]
    order = sorted(range(len(w)), key=lambda j: (-w[j], j))
    tot = sum(w[j] for j in order)
    best = 0
    for n in range(len(w) + 1):
        if sum(w[j] for j in order[:n]) <= f * tot * (1 + 1e-15):
            best = n
        else:
            break
    return set(order[:best])


def test_eq23_eq24_against_brute_force_and_a_worked_example():
    rng = np.random.default_rng(5)
    for _ in range(40):
        w = rng.lognormal(0, 1.5, rng.integers(1, 40)) * rng.choice([-1.0, 1.0], 1)
        for f in (0.0, 0.1, 0.5, 0.9, 0.999, 1.0):
            got = set(np.flatnonzero(otrunc.keep_mask(w, f)))
            assert got == _brute_keep(w, f) if f < 1.0 else len(got) == w.size
    assert otrunc.n_keep([], 0.5) == 0
    # worked example: |I| = 5, 3, 1, 1 (total 10): f = 0.8 keeps {5, 3}; 0.85 still {5, 3}; 0.9 adds one
    a = [5.0, 3.0, 1.0, 1.0]
    assert [otrunc.n_keep(a, f) for f in (0.49, 0.5, 0.8, 0.85, 0.9, 1.0)] == [0, 1, 2, 2, 3, 4]
    # signs do not matter, order of equal values does: the earlier of two equal components is kept first
    m = otrunc.keep_mask([1.0, -5.0, 1.0, 3.0], 0.9)
    assert m.tolist() == [True, True, False, True]


def test_invariants_of_the_selection():
    rng = np.random.default_rng(6)
    w = rng.normal(0, 1, 500) * rng.lognormal(0, 2, 500)
    tot = np.abs(w).sum()
    prev = 0
    for f in np.linspace(0, 1, 21):
        m = otrunc.keep_mask(w, f)
        kept = np.abs(w[m]).sum()
        assert kept <= f * tot * (1 + 1e-12)
        if m.sum() < w.size:                                     # the next one would not fit
            nxt = np.abs(w[~m]).max()
            assert kept + nxt > f * tot * (1 - 1e-12)
            assert np.abs(w[m]).min() >= nxt if m.any() else True
        assert m.sum() >= prev                                   # monotone in f_comp
        prev = m.sum()
    perm = rng.permutation(w.size)                               # distinct values: the choice is a set of values
    assert np.array_equal(np.sort(w[otrunc.keep_mask(w, 0.6)]), np.sort(w[perm][otrunc.keep_mask(w[perm], 0.6)]))


@pytest.fixture(scope="module")
def ctx():
    from paper_2005_09316_b200 import binding
    c = binding.Woden(0)
    yield c
    c.close()


@pytest.mark.gpu
def test_gpu_selection_is_bit_exact_against_the_oracle(ctx):
    import torch
    rng = np.random.default_rng(9)
    cases = [rng.normal(0, 1, n) * rng.lognormal(0, 2, n) for n in (1, 2, 31, 257, 5000)]
    cases.append(np.array([2.0, -2.0, 2.0, 1.0, -1.0, 2.0]))     # ties
    cases.append(inputs.make_config(4).gaussians.s0_jy)          # 25 % negative, 5660 components
    for w in cases:
        for f in (0.0, 0.3, 0.5, 0.8, 0.999999, 1.0, 2.0):
            keep, nk = ctx.truncate_select(torch.as_tensor(w, device="cuda:0"), f)
            ref = otrunc.keep_mask(w, f)
            assert np.array_equal(keep.cpu().numpy().astype(bool), ref), (w.size, f)
            assert int(nk[0]) == int(ref.sum())
    keep, nk = ctx.truncate_select(torch.zeros(0, dtype=torch.float64, device="cuda:0"), 0.5)
    assert int(nk[0]) == 0 and keep.numel() == 0


@pytest.mark.gpu
def test_gpu_selection_with_non_finite_weights_is_defined_and_reported(ctx):
    # a NaN weight would make the ranking a partial order (slots of the ranked list never written); the library
    # ranks non-finite weights as 0, counts them for woden_check, and the rest of the list is selected as usual
    import torch
    from paper_2005_09316_b200 import binding
    rng = np.random.default_rng(10)
    w = rng.normal(0, 1, 300) * rng.lognormal(0, 1, 300)
    bad = w.copy()
    bad[[3, 77, 150]] = np.nan
    bad[[5, 200]] = [np.inf, -np.inf]
    as_zero = np.where(np.isfinite(bad), bad, 0.0)
    ctx.check()
    for f in (0.2, 0.7, 1.0):
        keep, nk = ctx.truncate_select(torch.as_tensor(bad, device="cuda:0"), f)
        ref = otrunc.keep_mask(as_zero, f)
        assert np.array_equal(keep.cpu().numpy().astype(bool), ref)
        assert int(nk[0]) == int(ref.sum())
        with pytest.raises(binding.WodenError) as e:
            ctx.check()
        assert e.value.status == binding.WODEN_ERR_DATA
        k2 = torch.empty(300, dtype=torch.int32, device="cuda:0"); n2 = torch.empty(1, dtype=torch.int32, device="cuda:0")
        binding.truncate_select_static(torch.as_tensor(bad, device="cuda:0"), f, k2, n2)
        assert torch.equal(k2, keep) and int(n2[0]) == int(nk[0])
    keep, nk = ctx.truncate_select(torch.as_tensor(w, device="cuda:0"), 0.5)     # finite input: nothing reported
    ctx.check()


@pytest.mark.gpu
def test_gpu_eq25_basis_sums_match_the_oracle(ctx):
    # sum_pixels |(G * B_q)| for every basis function: with and without the beam, rotated, rectangular pixels
    for p_max, beam in ((6, None), (9, (1.5 * ARCMIN, 1.0 * ARCMIN, 0.7, 6)), (20, (1.0 * ARCMIN, 1.0 * ARCMIN, 0.0, 4))):
        g = (70, 54, -0.4 * ARCMIN, 0.45 * ARCMIN, 0.3 * ARCMIN, -0.2 * ARCMIN)
        b1, b2, pa = 3.0 * ARCMIN, 2.2 * ARCMIN, 1.2
        kw = {} if beam is None else dict(bmaj=beam[0], bmin=beam[1], bpa=beam[2], half_width=beam[3])
        A = shamfi.design_matrix(*g, 0.1 * ARCMIN, 0.0, pa, b1, b2, p_max, **kw)
        ref = np.abs(A).sum(axis=0)
        got = ctx.shapelet_basis_sums(*g, 0.1 * ARCMIN, 0.0, pa, p_max, b1, b2, beam=beam).cpu().numpy()
        assert np.abs(got - ref).max() <= 1e-11 * ref.max()
        coeff = np.arange(1.0, ref.size + 1) * (-1.0) ** np.arange(ref.size)
        assert np.allclose(np.abs(coeff) * got, shamfi.truncation_weights(coeff, A), rtol=1e-11)


@pytest.mark.gpu
def test_gpu_eq25_weights_of_a_whole_model_match_the_oracle(ctx):
    # woden_shapelet_truncation_weights: |C S0| x sum_pixels |G * B| per listed basis function on the grid and beam
    # of reading G20, against the image-space oracle on the same grid; ragged, unsorted lists,
    # an empty component, no beam / default beam / explicit beam
    from paper_2005_09316_b200 import binding
    rng = np.random.default_rng(21)
    a = 2.0 * np.sqrt(2.0 * np.log(2.0))
    s0 = np.array([1.5, -0.7, 2.0]); b1 = np.array([3.0, 5.0, 2.0]) * ARCMIN; b2 = np.array([2.0, 6.5, 2.0]) * ARCMIN
    pa = np.array([0.4, 2.1, 0.0])
    lists = [[(0, 0), (3, 2), (1, 7), (9, 0), (2, 2)], [], [(0, 12), (5, 5), (0, 0), (11, 1)]]
    off = np.cumsum([0] + [len(x) for x in lists]).astype(np.int32)
    n1 = np.array([p[0] for x in lists for p in x], dtype=np.int32)
    n2 = np.array([p[1] for x in lists for p in x], dtype=np.int32)
    cf = rng.normal(0, 1, n1.size)
    for n_pix, fwhm in ((65, 0.0), (65, 1.5 * ARCMIN)):
        got = ctx.shapelet_truncation_weights(s0, b1, b2, pa, off, n1, n2, cf, n_pix=n_pix, beam_fwhm_rad=fwhm)
        got = got.cpu().numpy()
        npx, beam_fwhm = n_pix, fwhm
        ref = np.zeros(cf.size)
        for j in range(3):
            lo, hi = off[j], off[j + 1]
            if hi == lo:
                continue
            pm = int((n1[lo:hi] + n2[lo:hi]).max())
            half = 1.5 * np.sqrt(2 * pm + 1.0) * max(b1[j], b2[j]) / a
            pix = 2.0 * half / (npx - 1)
            kw = {}
            if beam_fwhm > 0:
                kw = dict(bmaj=beam_fwhm, bmin=beam_fwhm, bpa=0.0, half_width=int(min(24, np.ceil(1.5 * beam_fwhm / pix))))
            A = shamfi.design_matrix(npx, npx, -pix, pix, 0.0, 0.0, 0.0, 0.0, pa[j], b1[j], b2[j], pm, **kw)
            full = np.zeros(A.shape[1])
            q = n1[lo:hi].astype(np.int64) * (pm + 1) - n1[lo:hi].astype(np.int64) * (n1[lo:hi] - 1) // 2 + n2[lo:hi]
            for i, qi in zip(range(lo, hi), q):
                full[:] = 0.0
                full[qi] = cf[i] * s0[j]
                ref[i] = shamfi.truncation_weights(full, A)[qi]
        assert np.abs(got - ref).max() <= 1e-10 * ref.max(), (n_pix, fwhm)
    ctx.check()
    # the defaults of reading G20 are what the header says: 257 pixels, a 2 arcmin beam
    dflt = ctx.shapelet_truncation_weights(s0, b1, b2, pa, off, n1, n2, cf)
    expl = ctx.shapelet_truncation_weights(s0, b1, b2, pa, off, n1, n2, cf, n_pix=binding.WODEN_EQ25_PIXELS,
                                           beam_fwhm_rad=2.0 * ARCMIN)
    import torch
    assert torch.equal(dflt, expl) and float(dflt.min()) > 0.0
    empty = ctx.shapelet_truncation_weights(s0[:0], b1[:0], b2[:0], pa[:0], np.zeros(1, np.int32), n1[:0], n2[:0], cf[:0])
    assert empty.numel() == 0
    with pytest.raises(binding.WodenError) as e:
        ctx.shapelet_truncation_weights(s0[:1], b1[:1], b2[:1], pa[:1], np.array([0, 1], np.int32), np.array([60], np.int32),
                                        np.array([60], np.int32), np.array([1.0]))
    assert e.value.status == binding.WODEN_ERR_ORDER


@pytest.mark.gpu
def test_components_and_shapelets_are_truncated_consistently(ctx):
    from paper_2005_09316_b200 import truncate
    wl = inputs.make_config(4)               # MS-CLEAN-like: 25 % negative components
    g = truncate.truncate_components(ctx, wl.gaussians, 0.5)
    assert 0 < g.n < wl.gaussians.n
    assert np.abs(g.s0_jy).min() >= np.sort(np.abs(wl.gaussians.s0_jy))[::-1][g.n - 1] - 1e-15
    assert (g.s0_jy < 0).any() and g.maj_fwhm_rad.shape == g.l.shape == g.pa_rad.shape
    assert np.abs(g.s0_jy).sum() <= 0.5 * np.abs(wl.gaussians.s0_jy).sum() * (1 + 1e-12)
    full = truncate.truncate_components(ctx, wl.points, 1.0)
    assert full.n == wl.points.n and np.array_equal(full.l, wl.points.l)
    s = inputs.make_config(5).shapelets
    w_dev = truncate.shapelet_basis_weights(ctx, s)          # Eq 25 by the library; stays on the device
    w = w_dev.cpu().numpy()
    assert w.shape == s.coeff.shape and (w >= 0).all() and w.max() > 0
    for f in (1.0, 0.6, 0.2):
        t = truncate.truncate_shapelets(ctx, s, f, w_dev)
        assert t.coeff_offset[0] == 0 and t.coeff_offset[-1] == t.coeff.size == t.n1.size == t.n2.size
        assert np.all(np.diff(t.coeff_offset) >= 0) and t.n == s.n
        if f == 1.0:
            assert np.array_equal(t.coeff, s.coeff)
        else:
            assert 0 < t.coeff.size < s.coeff.size
    empty = inputs.make_config(2).shapelets                      # a config without shapelets passes through
    assert truncate.truncate_shapelets(ctx, empty, 0.5).n == 0
    # the (0,0) basis image is a unit-sum Gaussian: its Eq 25 weight is |C_00| (to the grid's truncation)
    j0 = int(s.coeff_offset[0])
    assert s.n1[j0] == 0 and s.n2[j0] == 0
    assert np.isclose(w[j0], abs(s.coeff[j0] * s.s0_jy[0]), rtol=1e-6)
