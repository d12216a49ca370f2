"""Host-side checks of the seeded input generator (SURVEY.md §8(d) recipe)."""
import numpy as np
import pytest

from paper_2005_09316_b200 import inputs

SHAPES = {  # config: (B, T, F, Kp, Kg, Ks, n_coeff)
    1: (496, 1, 16, 10, 2, 1, 21),
    2: (8128, 14, 32, 1000, 0, 0, 0),
    3: (8128, 14, 32, 0, 10000, 0, 0),
    4: (8128, 14, 384, 14340, 5660, 2, 2 * 1891),
    5: (8128, 56, 384, 8000, 2000, 4, 4 * 861),
    6: (8128, 14, 384, 0, 0, 2, 2 * 3828),          # extra: phase II-like
}


@pytest.mark.parametrize("cfg", [1, 2, 3, 4, 5, 6])
def test_config_shapes_and_preconditions(cfg):
    wl = inputs.make_config(cfg)
    B, T, F, Kp, Kg, Ks, P = SHAPES[cfg]
    assert (wl.n_baselines, wl.n_times, wl.n_freqs) == (B, T, F)
    assert (wl.points.n, wl.gaussians.n, wl.shapelets.n, wl.n_coeff) == (Kp, Kg, Ks, P)
    assert wl.u_m.dtype == np.float64 and wl.u_m.flags.c_contiguous
    assert np.allclose(np.diff(wl.freqs_hz), 80e3) and wl.freqs_hz[0] == 167e6
    for c in (wl.points, wl.gaussians, wl.shapelets):
        if c.n:
            assert np.all(c.l ** 2 + c.m ** 2 < 1.0)
    # baseline lengths: |b| <= 2 * 1500 m (A128) or 2 * 500 m (A32), rotation preserves length
    blen = np.sqrt(wl.u_m ** 2 + wl.v_m ** 2 + wl.w_m ** 2)
    assert blen.max() <= {1: 1000.0, 6: 5500.0}.get(cfg, 3000.0)
    assert np.allclose(blen, blen[0][None, :], rtol=1e-12)
    if wl.gaussians.n:
        g = wl.gaussians
        assert np.all(g.min_fwhm_rad <= g.maj_fwhm_rad) and np.all(g.min_fwhm_rad >= 0)
    if wl.shapelets.n:
        s = wl.shapelets
        assert np.all(s.beta1_rad > 0) and np.all(s.beta2_rad > 0)
        assert s.uv_basis.shape == (Ks, 6) and s.coeff_offset[-1] == len(s.coeff)


def test_seeded_determinism_and_hour_angles():
    a, b = inputs.make_config(1), inputs.make_config(1)
    assert np.array_equal(a.u_m, b.u_m) and np.array_equal(a.points.l, b.points.l)
    # T = 1 => HA = 0 => u = East component of the baseline (w has no Y term at H=0)
    wl = inputs.make_config(2)


    assert not np.array_equal(wl.u_m[0], wl.u_m[1])


def test_time_shards_tile_the_observation():
    for world in (1, 2, 3, 4, 8):
        spans = [inputs.time_shard(56, r, world) for r in range(world)]
        assert spans[0][0] == 0 and sum(n for _, n in spans) == 56
        for (t0, n), (t1, _) in zip(spans, spans[1:]):
            assert t0 + n == t1
    # a rank's shard equals the same rows of the full observation
    full = inputs.make_config(2)
    t0, n = inputs.time_shard(14, 1, 2)
    part = inputs.make_config(2, t_index0=t0, n_times=n, n_times_total=14)
    assert np.allclose(part.u_m, full.u_m[t0:t0 + n], rtol=0, atol=1e-9)
    assert np.array_equal(part.points.l, full.points.l)


def test_subset_indices_cover_declared_rows():
    wl = inputs.make_config(2)
    idx = inputs.subset_indices(wl, n_random=1000)
    assert idx.dtype == np.int64 and np.all(np.diff(idx) > 0) and idx.max() < wl.n_vis
    B, F, T = wl.n_baselines, wl.n_freqs, wl.n_times
    for t in (0, T - 1):
        for f in (0, F // 2, F - 1):
            row = (t * F + f) * B + np.arange(B)
            assert np.isin(row, idx).all()
