"""Pins for the FP64 CPU oracle (oracle/woden_oracle.c) against what the paper and the
mathematics fix -- NOT against itself (SURVEY.md §8(c) pins P1-P15).

Every expected value here is a closed form, a brute-force DFT of an image-space definition,
a library Hermite routine, or an mpmath high-precision evaluation written out independently
of the oracle.  CPU only (`-m "not gpu"`).
"""
import math

import mpmath as mp
import numpy as np
import pytest
from numpy.polynomial import hermite as nph

import oracle
from paper_2005_09316_b200 import inputs

C = 299792458.0
LN2 = math.log(2.0)


def _uvw(T=2, B=7, seed=0, scale=800.0):
    rng = np.random.default_rng(seed)
    return tuple(rng.uniform(-scale, scale, (T, B)) for _ in range(3))


FREQS = np.array([150.0e6, 167.0e6, 167.08e6, 200.3e6])


# ----------------------------------------------------------------------------- P1, P13
def test_p1_phase_centre_point_gives_flux_everywhere():
    # Eq 9 with B == 1: l = m = 0 => V = S(nu) on every (t, f, b).
    u, v, w = _uvw()
    s0, alpha, nu0 = 3.25, -0.7, 150.0e6
    V = oracle.predict_points(u, v, w, FREQS, [0.0], [0.0], [s0], [alpha], nu0)
    assert V.shape == (2, 4, 7)
    expect = s0 * (FREQS / nu0) ** alpha
    assert np.allclose(V.real, expect[None, :, None], rtol=1e-14, atol=0)
    assert np.all(V.imag == 0.0)
    # P13: S(nu0) = S0 exactly; ratio law
    assert V[0, 0, 0].real == pytest.approx(s0, rel=1e-15)
    assert V[0, 3, 0].real / V[0, 1, 0].real == pytest.approx((FREQS[3] / FREQS[1]) ** alpha, rel=1e-14)


# ----------------------------------------------------------------------------- P2
def test_p2_offset_point_matches_mpmath_phase():
    # V = S exp(-2 pi i (u l + v m + w (n - 1))), Eq 9; 40-digit mpmath.
    mp.mp.dps = 40
    u, v, w = _uvw(T=2, B=6, seed=3, scale=1500.0)
    l, m, s0, alpha, nu0 = 0.21, -0.17, 2.0, -0.8, 150.0e6
    V = oracle.predict_points(u, v, w, FREQS, [l], [m], [s0], [alpha], nu0)
    ml, mm = mp.mpf(l), mp.mpf(m)
    mn = mp.sqrt(1 - ml * ml - mm * mm)
    for t in range(2):
        for f, nu in enumerate(FREQS):
            for b in range(6):
                sc = mp.mpf(float(nu)) / mp.mpf(C)
                uu, vv, ww = (mp.mpf(float(a[t, b])) * sc for a in (u, v, w))
                S = mp.mpf(s0) * (mp.mpf(float(nu)) / mp.mpf(nu0)) ** mp.mpf(alpha)
                ref = S * mp.exp(-2j * mp.pi * (uu * ml + vv * mm + ww * (mn - 1)))
                assert abs(V[t, f, b] - complex(ref)) < 2e-11 * s0


def test_p2_sign_convention_small_offset():
    # a source slightly East (l > 0) on an East-West baseline u > 0: phase is -2 pi u l < 0
    u = np.array([[100.0]]); z = np.zeros((1, 1))
    nu = np.array([C])                      # 1 m wavelength: u_lambda = 100
    V = oracle.predict_points(u, z, z, nu, [1e-3], [0.0], [1.0], [0.0], C)
    assert V[0, 0, 0].imag == pytest.approx(-math.sin(2 * math.pi * 0.1), rel=1e-12)
    assert V[0, 0, 0].real == pytest.approx(math.cos(2 * math.pi * 0.1), rel=1e-12)
    # w-term only: V = exp(-2 pi i w (n - 1)), n - 1 < 0 => positive phase
    w = np.array([[1000.0]])
    V = oracle.predict_points(z, z, w, nu, [0.3], [0.0], [1.0], [0.0], C)
    ph = -2 * math.pi * 1000.0 * (math.sqrt(1 - 0.09) - 1.0)
    assert ph > 0
    assert V[0, 0, 0] == pytest.approx(complex(math.cos(ph), math.sin(ph)), abs=1e-11)


# ----------------------------------------------------------------------------- P3
def test_p3_gaussian_closed_forms():
    nu = np.array([C])                      # metres == wavelengths
    z = np.zeros((1, 5))
    # circular: xi = exp(-pi^2 theta^2 (u^2+v^2) / (4 ln2))  (Eq 12)
    theta = 3.0e-3
    u = np.array([[10.0, 50.0, -80.0, 120.0, 0.0]])
    v = np.array([[5.0, -40.0, 60.0, 0.0, 147.0904]])
    for pa in (0.0, 0.4, 2.0):
        V = oracle.predict_gaussians(u, v, z, nu, [0.0], [0.0], [1.0], [0.0], C,
                                     [theta], [theta], [pa])
        expect = np.exp(-math.pi ** 2 * theta ** 2 * (u ** 2 + v ** 2) / (4 * LN2))
        assert np.allclose(V[0, 0].real, expect[0], rtol=1e-13)
        assert np.allclose(V[0, 0].imag, 0.0, atol=1e-16)
    # half power at baseline length k with k theta = 2 ln2 / pi
    k = 2 * LN2 / (math.pi * theta)
    V = oracle.predict_gaussians(np.array([[k]]), np.zeros((1, 1)), np.zeros((1, 1)), nu,
                                 [0.0], [0.0], [1.0], [0.0], C, [theta], [theta], [0.0])
    assert V[0, 0, 0].real == pytest.approx(0.5, rel=1e-13)
    # pa = 0, theta_min = 0: kx = v pairs with theta_maj => depends on v only (Eq 13-14)
    V = oracle.predict_gaussians(u, v, z, nu, [0.0], [0.0], [1.0], [0.0], C, [theta], [0.0], [0.0])
    expect = np.exp(-math.pi ** 2 * theta ** 2 * v ** 2 / (4 * LN2))
    assert np.allclose(V[0, 0].real, expect[0], rtol=1e-13)
    # pa = 90 deg: major axis East-West => depends on u only
    V = oracle.predict_gaussians(u, v, z, nu, [0.0], [0.0], [1.0], [0.0], C,
                                 [theta], [0.0], [math.pi / 2])
    expect = np.exp(-math.pi ** 2 * theta ** 2 * u ** 2 / (4 * LN2))
    assert np.allclose(V[0, 0].real, expect[0], rtol=1e-12)


# ----------------------------------------------------------------------------- P4
def _image_grid(half_width, n):
    x = np.linspace(-half_width, half_width, n)
    return np.meshgrid(x, x, indexing="xy")        # X = l offsets (East), Y = m offsets (North)


def _dft(img, X, Y, u, v):
    """sum_pix img exp(-2 pi i (u x + v y)), the Eq 8 kernel on a flat patch."""
    return np.array([np.sum(img * np.exp(-2j * np.pi * (uu * X + vv * Y))) for uu, vv in zip(u, v)])


def test_p4_gaussian_envelope_is_normalised_dft_of_eq10():
    # Eq 10 with the major axis along (sin pa, cos pa) (PA from North to East,
    # :102/:134), divided by its pixel sum ("kernel sums to one", :157) == Eq 12-14.
    maj, mnr, pa = 4.0e-3, 1.5e-3, 0.7
    X, Y = _image_grid(0.02, 401)
    a = X * math.sin(pa) + Y * math.cos(pa)         # along the major axis
    b = X * math.cos(pa) - Y * math.sin(pa)         # along the minor axis
    img = np.exp(-4 * LN2 * (a ** 2 / maj ** 2 + b ** 2 / mnr ** 2))
    rng = np.random.default_rng(5)
    u = rng.uniform(-150, 150, 12); v = rng.uniform(-150, 150, 12)
    ref = _dft(img, X, Y, u, v) / img.sum()
    V = oracle.predict_gaussians(u[None], v[None], np.zeros((1, 12)), np.array([C]),
                                 [0.0], [0.0], [1.0], [0.0], C, [maj], [mnr], [pa])
    assert np.max(np.abs(V[0, 0] - ref)) < 1e-10
    assert np.max(np.abs(ref.imag)) < 1e-12


# ----------------------------------------------------------------------------- P5
def test_p5_shapelet_00_equals_gaussian():
    # B_00 == G when beta1 = theta_maj, beta2 = theta_min.
    u, v, w = _uvw(T=2, B=9, seed=11, scale=300.0)
    maj, mnr, pa = 2.5e-3, 1.0e-3, 1.1
    l, m = 0.05, -0.02
    G = oracle.predict_gaussians(u, v, w, FREQS, [l], [m], [1.7], [-0.6], 150e6, [maj], [mnr], [pa])
    S = oracle.predict_shapelets(u, v, w, FREQS, [l], [m], [1.7], [-0.6], 150e6, [maj], [mnr], [pa],
                                 None, [0, 1], [0], [0], [1.0])
    assert np.max(np.abs(G - S)) < 1e-14 * 1.7
    assert np.max(np.abs(G)) > 0.1


# ----------------------------------------------------------------------------- P6
def _h_lib(p, x):
    """h_p(x) from numpy's Hermite series evaluator (library routine, not the oracle)."""
    c = np.zeros(p + 1); c[p] = 1.0
    return nph.hermval(x, c) * np.exp(-x * x / 2) / math.sqrt(2.0 ** p * math.factorial(p))


@pytest.mark.parametrize("p1,p2", [(0, 0), (1, 0), (0, 1), (2, 1), (3, 3), (5, 0), (4, 5), (1, 2)])
def test_p6_basis_ft_matches_dft_of_reflected_image_basis(p1, p2):
    # Eq 3 with Eq 16-17 scalings, reading G3: i^(p1+p2) h(beta kappa k) is the
    # e^{-2 pi i ...} transform of the point-reflected image basis h_p(-a x / beta),
    # a = 2 sqrt(2 ln 2), divided by pi beta1 beta2 / (4 ln 2) (the (0,0) integral).
    b1, b2 = 3.0e-3, 2.0e-3
    a = 2 * math.sqrt(2 * LN2)
    half, n = 0.03, 601
    X, Y = _image_grid(half, n)
    dx = 2 * half / (n - 1)
    img = _h_lib(p1, -a * X / b1) * _h_lib(p2, -a * Y / b2)
    rng = np.random.default_rng(100 + 7 * p1 + p2)
    u = rng.uniform(-120, 120, 6); v = rng.uniform(-120, 120, 6)
    ref = _dft(img, X, Y, u, v) * dx * dx / (math.pi * b1 * b2 / (4 * LN2))
    # pa = pi/2: kx = kappa u pairs with beta1 along East (x); ky = -kappa v pairs with beta2.
    # To align the image y axis (North) with +ky use pa such that ky = +kappa v: take
    # the component's axes as (x along l, y along m) => evaluate with explicit rotation below.
    # PA = pi/2 gives kx = u, ky = -v; h_{p2}(-y) = (-1)^p2 h_{p2}(y) fixes the sign.
    V = oracle.predict_shapelets(u[None], v[None], np.zeros((1, 6)), np.array([C]),
                                 [0.0], [0.0], [1.0], [0.0], C, [b1], [b2], [math.pi / 2],
                                 None, [0, 1], [p1], [p2], [1.0])[0, 0]
    V = V * (-1) ** p2
    assert np.max(np.abs(V - ref)) < 5e-9
    # and independently of the oracle: the closed form with library Hermite functions
    kappa = math.pi / math.sqrt(2 * LN2)
    closed = (1j) ** (p1 + p2) * _h_lib(p1, b1 * kappa * u) * _h_lib(p2, b2 * kappa * v)
    assert np.max(np.abs(closed - ref)) < 5e-9
    # unreflected basis gives (-i)^(p1+p2)
    img2 = _h_lib(p1, a * X / b1) * _h_lib(p2, a * Y / b2)
    ref2 = _dft(img2, X, Y, u, v) * dx * dx / (math.pi * b1 * b2 / (4 * LN2))
    assert np.max(np.abs(ref2 - (-1) ** (p1 + p2) * ref)) < 5e-9


# ----------------------------------------------------------------------------- helpers
def _tiny():
    return inputs.make_config(1)


def _shapelet_args(s, sel=None):
    return (s.l, s.m, s.s0_jy, s.alpha)


# ----------------------------------------------------------------------------- P7
def test_p7_hermitian_symmetry_all_types():
    # real sky => V(-u,-v,-w) = conj V(u,v,w); pins the parity handling of i^(n1+n2).
    wl = _tiny()
    Vp = oracle.predict_workload(wl)
    wl2 = inputs.make_config(1)
    wl2.u_m, wl2.v_m, wl2.w_m = -wl.u_m, -wl.v_m, -wl.w_m
    Vm = oracle.predict_workload(wl2)
    scale = oracle.workload_tolerance_scale(wl)[None, :, None]
    assert np.max(np.abs(Vm - np.conj(Vp)) / scale) < 1e-14
    # the shapelet alone, with odd orders present
    s = wl.shapelets
    a = oracle.predict_shapelets(wl.u_m, wl.v_m, wl.w_m, wl.freqs_hz, s.l, s.m, s.s0_jy, s.alpha,
                                 wl.ref_freq_hz, s.beta1_rad, s.beta2_rad, s.pa_rad, s.uv_basis,
                                 s.coeff_offset, s.n1, s.n2, s.coeff)
    b = oracle.predict_shapelets(-wl.u_m, -wl.v_m, -wl.w_m, wl.freqs_hz, s.l, s.m, s.s0_jy, s.alpha,
                                 wl.ref_freq_hz, s.beta1_rad, s.beta2_rad, s.pa_rad, s.uv_basis,
                                 s.coeff_offset, s.n1, s.n2, s.coeff)
    assert np.max(np.abs(b - np.conj(a))) < 1e-13
    assert np.max(np.abs(a.imag)) > 1e-3


# ----------------------------------------------------------------------------- P8
def test_p8_hermite_routine_against_library_and_identities():
    xs = [-31.0, -7.3, -1.0, -1e-3, 0.0, 0.5, 2.2, 9.9, 14.0, 20.0, 40.0]
    for x in xs:
        h = oracle.hermite_functions(100, x)
        for p in (0, 1, 2, 3, 7, 20, 46, 60, 86, 100):
            # library: scipy/numpy Hermite polynomial, normalised in mpmath to avoid overflow
            Hp = mp.hermite(p, mp.mpf(x))
            ref = Hp * mp.exp(-mp.mpf(x) ** 2 / 2) / mp.sqrt(mp.mpf(2) ** p * mp.factorial(p))
            assert abs(h[p] - float(ref)) < 1e-13, (x, p)
    # numpy hermval agreement at moderate order / argument
    x = np.linspace(-6, 6, 25)
    for p in range(0, 31):
        got = np.array([oracle.hermite_functions(p, xx)[p] for xx in x])
        assert np.allclose(got, _h_lib(p, x), rtol=0, atol=2e-13)
    # h_{2m}(0) = (-1)^m sqrt((2m)!)/(2^m m!), h_odd(0) = 0
    h0 = oracle.hermite_functions(40, 0.0)
    for mm in range(0, 21):
        assert h0[2 * mm] == pytest.approx((-1) ** mm * math.sqrt(math.factorial(2 * mm))
                                           / (2 ** mm * math.factorial(mm)), rel=1e-13)
    assert np.all(h0[1::2] == 0.0)
    # orthogonality: int h_p h_q dx = sqrt(pi) delta_pq (trapezoid on a wide fine grid)
    xg = np.linspace(-20, 20, 8001)
    H = np.array([oracle.hermite_functions(30, xx) for xx in xg])      # [x, p]
    G = (H.T @ H) * (xg[1] - xg[0])
    assert np.max(np.abs(G - math.sqrt(math.pi) * np.eye(31))) < 1e-10
    # |h_p| <= 1 for p <= 86 (used by tolerance reading G12)
    xg = np.linspace(-25, 25, 5001)
    H = np.array([oracle.hermite_functions(86, xx) for xx in xg])
    assert np.max(np.abs(H)) <= 1.0 + 1e-15


# ----------------------------------------------------------------------------- P9
def test_p9_additivity_accumulate_and_permutation():
    wl = _tiny()
    p = wl.points
    a = (wl.u_m, wl.v_m, wl.w_m, wl.freqs_hz)
    full = oracle.predict_points(*a, p.l, p.m, p.s0_jy, p.alpha, wl.ref_freq_hz)
    A = oracle.predict_points(*a, p.l[:4], p.m[:4], p.s0_jy[:4], p.alpha[:4], wl.ref_freq_hz)
    Bv = oracle.predict_points(*a, p.l[4:], p.m[4:], p.s0_jy[4:], p.alpha[4:], wl.ref_freq_hz)
    assert np.max(np.abs(full - (A + Bv))) < 1e-13
    acc = A.copy()
    oracle.predict_points(*a, p.l[4:], p.m[4:], p.s0_jy[4:], p.alpha[4:], wl.ref_freq_hz,
                          out=acc, accumulate=True)
    assert np.array_equal(acc, A + Bv)
    perm = np.random.default_rng(1).permutation(wl.n_baselines)
    Vp = oracle.predict_points(wl.u_m[:, perm], wl.v_m[:, perm], wl.w_m[:, perm], wl.freqs_hz,
                               p.l, p.m, p.s0_jy, p.alpha, wl.ref_freq_hz)
    assert np.array_equal(Vp, full[:, :, perm])
    # zero components: overwrite gives zeros
    z = oracle.predict_points(*a, [], [], [], [], wl.ref_freq_hz)
    assert z.shape == full.shape and not z.any()
    # subset evaluation picks the same values, index = (t*F + f)*B + b
    idx = np.array([0, 5, 495, 496, 7935, 1234], dtype=np.int64)
    sub = oracle.predict_points(*a, p.l, p.m, p.s0_jy, p.alpha, wl.ref_freq_hz, vis_index=idx)
    assert np.array_equal(sub, full.reshape(-1)[idx])


# ----------------------------------------------------------------------------- P10
def test_p10_frequency_is_only_a_scale_on_uvw():
    # with alpha = 0, V(s * u_m, nu) = V(u_m, s * nu) for every type.
    wl = _tiny()
    s = 1.0371
    g, sh = wl.gaussians, wl.shapelets
    z = np.zeros
    for kind in ("p", "g", "s"):
        def run(u, v, w, fr):
            if kind == "p":
                c = wl.points
                return oracle.predict_points(u, v, w, fr, c.l, c.m, c.s0_jy, z(c.n), wl.ref_freq_hz)
            if kind == "g":
                return oracle.predict_gaussians(u, v, w, fr, g.l, g.m, g.s0_jy, z(g.n), wl.ref_freq_hz,
                                                g.maj_fwhm_rad, g.min_fwhm_rad, g.pa_rad)
            return oracle.predict_shapelets(u, v, w, fr, sh.l, sh.m, sh.s0_jy, z(sh.n), wl.ref_freq_hz,
                                            sh.beta1_rad, sh.beta2_rad, sh.pa_rad, sh.uv_basis,
                                            sh.coeff_offset, sh.n1, sh.n2, sh.coeff)
        a = run(s * wl.u_m, s * wl.v_m, s * wl.w_m, wl.freqs_hz)
        b = run(wl.u_m, wl.v_m, wl.w_m, s * wl.freqs_hz)
        assert np.max(np.abs(a - b)) < 1e-9 * np.max(np.abs(a)), kind


# ----------------------------------------------------------------------------- P11
def test_p11_basis_counts_eq6():
    # Eq 6 and the counts quoted at :271
    for pmax, cnt in [(5, 21), (40, 861), (46, 1128), (60, 1891), (86, 3828)]:
        assert inputs.basis_count(pmax) == cnt
        n1, n2 = inputs.full_triangle(pmax)
        assert len(n1) == cnt and np.all(n1 + n2 <= pmax) and len(set(zip(n1, n2))) == cnt
    assert 2 * inputs.basis_count(86) == 7656


# ----------------------------------------------------------------------------- P12
def test_p12_position_angle_symmetries():
    u, v, w = _uvw(T=1, B=11, seed=21, scale=250.0)
    fr = np.array([180e6])
    kw = ([0.02], [0.03], [1.0], [0.0], 150e6)
    g0 = oracle.predict_gaussians(u, v, w, fr, *kw, [3e-3], [1e-3], [0.6])
    g1 = oracle.predict_gaussians(u, v, w, fr, *kw, [3e-3], [1e-3], [0.6 + math.pi])
    assert np.max(np.abs(g0 - g1)) < 1e-14
    for (a, b) in [(1, 0), (2, 1), (0, 3), (2, 2)]:
        s0 = oracle.predict_shapelets(u, v, w, fr, *kw, [3e-3], [1e-3], [0.6], None, [0, 1], [a], [b], [1.0])
        s1 = oracle.predict_shapelets(u, v, w, fr, *kw, [3e-3], [1e-3], [0.6 + math.pi], None,
                                      [0, 1], [a], [b], [1.0])
        assert np.max(np.abs(s1 - (-1) ** (a + b) * s0)) < 1e-14
        assert np.max(np.abs(s0)) > 1e-4


# ----------------------------------------------------------------------------- P14
def test_p14_uv_basis_identity_and_orthonormality():
    wl = _tiny()
    s = wl.shapelets
    args = (wl.u_m, wl.v_m, wl.w_m, wl.freqs_hz, s.l, s.m, s.s0_jy, s.alpha, wl.ref_freq_hz,
            s.beta1_rad, s.beta2_rad, s.pa_rad)
    tail = (s.coeff_offset, s.n1, s.n2, s.coeff)
    a = oracle.predict_shapelets(*args, None, *tail)
    ident = np.array([[1.0, 0, 0, 0, 1.0, 0]])
    b = oracle.predict_shapelets(*args, ident, *tail)
    assert np.array_equal(a, b)
    # a non-trivial M changes the answer (so the argument is really used)
    c = oracle.predict_shapelets(*args, s.uv_basis, *tail)
    assert np.max(np.abs(c - a)) > 1e-6
    # generator's M: identity at the phase centre; rows orthonormal and perpendicular to s
    M0 = inputs.local_uv_basis([0.0], [0.0])
    assert np.allclose(M0, ident, atol=1e-15)
    l = np.array([0.1, -0.3, 0.02]); m = np.array([0.2, 0.25, -0.4])
    M = inputs.local_uv_basis(l, m).reshape(-1, 2, 3)
    sv = np.stack([l, m, np.sqrt(1 - l * l - m * m)], axis=1)
    for j in range(3):
        assert np.allclose(M[j] @ M[j].T, np.eye(2), atol=1e-15)
        assert np.allclose(M[j] @ sv[j], 0.0, atol=1e-15)


# ----------------------------------------------------------------------------- P15
def test_p15_oracle_vs_mpmath_brute_force_on_tiny():
    # Whole Tiny config (all three types), 24 visibilities, 30-digit mpmath restatement of
    # Eq 9/11/12-17 with mp.hermite: |delta| <= 1e-11 * sum |S|.
    mp.mp.dps = 30
    wl = _tiny()
    idx = np.random.default_rng(15).choice(wl.n_vis, 24, replace=False).astype(np.int64)
    V = oracle.predict_workload(wl, vis_index=idx)
    scale = oracle.workload_tolerance_scale(wl)
    B, F = wl.n_baselines, wl.n_freqs
    f = lambda x: mp.mpf(float(x))
    kap = mp.pi / mp.sqrt(2 * mp.log(2))
    gc = mp.pi ** 2 / (4 * mp.log(2))
    for o, flat in enumerate(idx):
        b = int(flat % B); fi = int((flat // B) % F); t = int(flat // (B * F))
        nu = f(wl.freqs_hz[fi]); sc = nu / f(C)
        u, v, w = f(wl.u_m[t, b]) * sc, f(wl.v_m[t, b]) * sc, f(wl.w_m[t, b]) * sc
        tot = mp.mpc(0)

        def common(c, j):
            l, m = f(c.l[j]), f(c.m[j])
            n = mp.sqrt(1 - l * l - m * m)
            S = f(c.s0_jy[j]) * (nu / f(wl.ref_freq_hz)) ** f(c.alpha[j])
            return S * mp.exp(-2j * mp.pi * (u * l + v * m + w * (n - 1)))

        for j in range(wl.points.n):
            tot += common(wl.points, j)
        g = wl.gaussians
        for j in range(g.n):
            pa = f(g.pa_rad[j])
            kx = mp.cos(pa) * v + mp.sin(pa) * u
            ky = -mp.sin(pa) * v + mp.cos(pa) * u
            tot += common(g, j) * mp.exp(-gc * (kx ** 2 * f(g.maj_fwhm_rad[j]) ** 2
                                                + ky ** 2 * f(g.min_fwhm_rad[j]) ** 2))
        s = wl.shapelets
        for j in range(s.n):
            M = [f(x) for x in s.uv_basis[j]]
            up = M[0] * u + M[1] * v + M[2] * w
            vp = M[3] * u + M[4] * v + M[5] * w
            pa = f(s.pa_rad[j])
            x = f(s.beta1_rad[j]) * kap * (mp.cos(pa) * vp + mp.sin(pa) * up)
            y = f(s.beta2_rad[j]) * kap * (-mp.sin(pa) * vp + mp.cos(pa) * up)
            xi = mp.mpc(0)
            for q in range(int(s.coeff_offset[j]), int(s.coeff_offset[j + 1])):
                a, bb = int(s.n1[q]), int(s.n2[q])
                ha = mp.hermite(a, x) * mp.exp(-x * x / 2) / mp.sqrt(mp.mpf(2) ** a * mp.factorial(a))
                hb = mp.hermite(bb, y) * mp.exp(-y * y / 2) / mp.sqrt(mp.mpf(2) ** bb * mp.factorial(bb))
                xi += f(s.coeff[q]) * mp.mpc(0, 1) ** (a + bb) * ha * hb
            tot += common(s, j) * xi
        assert abs(V[o] - complex(tot)) <= 1e-11 * scale[fi]


def test_tolerance_scale_definition():
    # reading G12: scale_f = sum |S_k(nu_f)| (x sum |coeff| for shapelets), restated in numpy
    wl = _tiny()
    sc = oracle.workload_tolerance_scale(wl)
    fr = wl.freqs_hz[:, None] / wl.ref_freq_hz
    ref = (np.abs(wl.points.s0_jy) * fr ** wl.points.alpha).sum(1)
    ref += (np.abs(wl.gaussians.s0_jy) * fr ** wl.gaussians.alpha).sum(1)
    ref += (np.abs(wl.shapelets.s0_jy) * fr ** wl.shapelets.alpha).sum(1) * np.abs(wl.shapelets.coeff).sum()
    assert np.allclose(sc, ref, rtol=1e-13)
    # signs: negative fluxes and negative coefficients enter by absolute value (hand-computed case:
    # S = -2 and +3 at nu = ref, alpha irrelevant there; shapelet S = -1.5 with coefficients 1, -2, 0.5)
    fr1 = np.array([wl.ref_freq_hz])
    assert oracle.tolerance_scale(fr1, [-2.0, 3.0], [-0.7, 0.3], wl.ref_freq_hz)[0] == pytest.approx(5.0, rel=1e-15)
    assert oracle.tolerance_scale(fr1, [-1.5], [-0.8], wl.ref_freq_hz, [0, 3], [1.0, -2.0, 0.5])[0] == pytest.approx(
        5.25, rel=1e-15)
    # and at another frequency the law is |s0| (nu/ref)^alpha, never negative
    two = oracle.tolerance_scale(np.array([2.0 * wl.ref_freq_hz]), [-2.0], [-1.0], wl.ref_freq_hz)
    assert two[0] == pytest.approx(1.0, rel=1e-15)
    wl4 = inputs.make_config(4)                                   # 25 % negative components
    sc4 = oracle.tolerance_scale(wl4.freqs_hz[:3], wl4.points.s0_jy, wl4.points.alpha, wl4.ref_freq_hz)
    ref4 = (np.abs(wl4.points.s0_jy) * (wl4.freqs_hz[:3, None] / wl4.ref_freq_hz) ** wl4.points.alpha).sum(1)
    assert (wl4.points.s0_jy < 0).any() and np.allclose(sc4, ref4, rtol=1e-13)


# ----------------------------------------------------------------------------- P16 (NEXT-2)
def test_p16_uvw_rotation_special_cases_lengths_and_projection():
    rng = np.random.default_rng(16)
    n = 7
    X, Y, Z = rng.normal(0, 800.0, (3, n))
    # explicit pair order for 3 antennas: (0,1), (0,2), (1,2); baseline = antenna p - antenna q
    u, v, w = oracle.uvw_from_antennas(X[:3], Y[:3], Z[:3], [0.0], 0.0)
    assert np.allclose(u[0], [Y[0] - Y[1], Y[0] - Y[2], Y[1] - Y[2]], atol=1e-12)      # H = 0, d0 = 0: u = Y
    assert np.allclose(v[0], [Z[0] - Z[1], Z[0] - Z[2], Z[1] - Z[2]], atol=1e-12)      #                v = Z
    assert np.allclose(w[0], [X[0] - X[1], X[0] - X[2], X[1] - X[2]], atol=1e-12)      #                w = X
    u, v, w = oracle.uvw_from_antennas(X[:2], Y[:2], Z[:2], [0.0, np.pi / 2], np.pi / 2)
    assert np.allclose([u[0, 0], v[0, 0], w[0, 0]], [Y[0] - Y[1], -(X[0] - X[1]), Z[0] - Z[1]], atol=1e-12)   # pole
    u, v, w = oracle.uvw_from_antennas(X[:2], Y[:2], Z[:2], [np.pi / 2], 0.0)
    assert np.allclose([u[0, 0], v[0, 0], w[0, 0]], [X[0] - X[1], Z[0] - Z[1], -(Y[0] - Y[1])], atol=1e-12)
    # general case: a rotation preserves length; w is the projection on the source direction
    H = np.array([-0.7, 0.0, 0.3, 2.9]); d0 = np.deg2rad(-37.0)
    u, v, w = oracle.uvw_from_antennas(X, Y, Z, H, d0)
    p, q = inputs.baseline_pairs(n)
    bx, by, bz = X[p] - X[q], Y[p] - Y[q], Z[p] - Z[q]
    assert np.allclose(u * u + v * v + w * w, (bx * bx + by * by + bz * bz)[None, :], rtol=1e-13)
    for t, h in enumerate(H):
        s0 = np.array([np.cos(d0) * np.cos(h), -np.cos(d0) * np.sin(h), np.sin(d0)])     # source direction in XYZ
        assert np.allclose(w[t], bx * s0[0] + by * s0[1] + bz * s0[2], atol=1e-10)
        east = np.array([np.sin(h), np.cos(h), 0.0])                                      # d s0 / dH direction
        assert np.allclose(u[t], bx * east[0] + by * east[1], atol=1e-10)


def test_p16_uv_basis_is_rephasing_to_the_component_centre():
    # the shapelet's u,v are "calculated with a phase-centre ... which corresponds to
    # the central position" of the shapelet.  Reading G4 replaces that by the time-independent M_j;
    # here the two are shown equal using the oracle's own uvw routine at the component's (H_j, d_j).
    rng = np.random.default_rng(61)
    X, Y, Z = rng.normal(0, 900.0, (3, 6))
    d0 = np.deg2rad(-37.0)
    l = np.array([0.0, 0.12, -0.3, 0.02]); m = np.array([0.0, -0.2, 0.25, 0.4])
    M = oracle.shapelet_uv_basis(l, m, d0).reshape(-1, 2, 3)
    assert np.allclose(M[0], [[1, 0, 0], [0, 1, 0]], atol=1e-15)            # identity at the phase centre
    sv = np.stack([l, m, np.sqrt(1 - l * l - m * m)], axis=1)
    for j in range(len(l)):
        assert np.allclose(M[j] @ M[j].T, np.eye(2), atol=1e-15)            # orthonormal rows
        assert np.allclose(M[j] @ sv[j], 0.0, atol=1e-15)                   # perpendicular to s
    for H0 in (-1.1, 0.0, 0.4):
        u0, v0, w0 = oracle.uvw_from_antennas(X, Y, Z, [H0], d0)
        R0 = np.array([[np.sin(H0), np.cos(H0), 0.0],
                       [-np.sin(d0) * np.cos(H0), np.sin(d0) * np.sin(H0), np.cos(d0)],
                       [np.cos(d0) * np.cos(H0), -np.cos(d0) * np.sin(H0), np.sin(d0)]])
        for j in range(len(l)):
            sx = R0.T @ sv[j]                                                # component direction in XYZ
            dj, Hj = np.arcsin(sx[2]), np.arctan2(-sx[1], sx[0])
            uj, vj, _ = oracle.uvw_from_antennas(X, Y, Z, [Hj], dj)
            got = M[j] @ np.stack([u0[0], v0[0], w0[0]])
            assert np.allclose(got[0], uj[0], atol=1e-9) and np.allclose(got[1], vj[0], atol=1e-9)
    # the generator's matrices (used for configs 1, 4, 5) are the same ones
    assert np.allclose(inputs.local_uv_basis(l, m, d0), oracle.shapelet_uv_basis(l, m, d0), atol=1e-15)


def test_oracle_uv_basis_equals_the_generators_independent_construction():
    # predict_workload and the CUDA side each compute M_j (reading G4) with their own routine
    # from (l, m, dec0); the generator builds it a third way (cross products with the celestial pole in numpy,
    # inputs.local_uv_basis).  Pin the oracle's routine to the generator's arrays for the shapelet configs, so a
    # misreading of the basis rotation shared by the two C-side routines cannot pass end-to-end parity unnoticed.
    for cfg in (4, 5, 6):
        wl = inputs.make_config(cfg)
        s = wl.shapelets
        assert s.n > 0 and s.uv_basis is not None
        M = oracle.shapelet_uv_basis(s.l, s.m, wl.meta["dec0_rad"])
        assert M.shape == s.uv_basis.reshape(s.n, 6).shape
        assert np.max(np.abs(M - s.uv_basis.reshape(s.n, 6))) <= 1e-12
        # and it is not the identity-like trivial case: the rows are orthonormal 3-vectors orthogonal to s
        for j in range(s.n):
            e, nvec = M[j, :3], M[j, 3:]
            n_dir = np.sqrt(1.0 - s.l[j] ** 2 - s.m[j] ** 2)
            sdir = np.array([s.l[j], s.m[j], n_dir])
            assert abs(e @ e - 1) < 1e-12 and abs(nvec @ nvec - 1) < 1e-12 and abs(e @ nvec) < 1e-12
            assert abs(e @ sdir) < 1e-12 and abs(nvec @ sdir) < 1e-12
