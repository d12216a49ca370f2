"""NEXT-5: the 1-D shapelet series by recurrence and by the paper's look-up tables
(PAPER.md:159), both against the oracle's long-double Hermite routine; `-m gpu`."""
import numpy as np
import pytest

import oracle

pytestmark = pytest.mark.gpu


@pytest.mark.parametrize("p_max", [0, 5, 40, 86, 100])
def test_series_recurrence_and_lut_against_the_oracle(p_max):
    import torch
    from paper_2005_09316_b200 import binding
    ctx = binding.Woden(0)
    rng = np.random.default_rng(p_max)
    x = np.concatenate([rng.uniform(-14, 14, 1500), [0.0, -0.0, 1e-3, -31.99, 31.99, 35.0, -40.0]]).astype(np.float32)
    c = (rng.normal(0, 1, p_max + 1) * np.exp(-np.arange(p_max + 1) / 10.0)).astype(np.float32)
    ref = np.array([np.dot(c.astype(np.float64), oracle.hermite_functions(p_max, float(v))) for v in x])
    xd, cd = torch.as_tensor(x, device="cuda:0"), torch.as_tensor(c, device="cuda:0")
    scale = np.abs(c).sum()
    rec = ctx.shapelet_series(binding.WODEN_BASIS_RECURRENCE, xd, cd).cpu().numpy()
    assert np.abs(rec - ref).max() <= 1e-5 * scale
    for dx in (2.0 ** -7, 2.0 ** -10):
        lut = ctx.shapelet_series(binding.WODEN_BASIS_LUT, xd, cd, lut_dx=dx, lut_x_max=32.0).cpu().numpy()
        inside = np.abs(x) < 32.0
        bound = dx * dx * (2 * p_max + 1) * 1.09 / 8 * scale + 2e-6 * scale
        assert np.abs(lut - ref)[inside].max() <= bound, (dx, np.abs(lut - ref)[inside].max(), bound)
        assert np.all(lut[~inside] == 0.0) and np.abs(ref[~inside]).max() < 1e-30     # beyond the table: underflowed anyway
    ctx.close()
