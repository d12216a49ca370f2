"""GPU gain calibration and peel (woden_calibrate_gains / woden_peel; section 5.1, Eq 18-22)
against the numpy oracle (oracle/calibrate.py), `-m gpu`."""
import numpy as np
import pytest

import oracle
from oracle import calibrate as ocal
from paper_2005_09316_b200 import inputs, truncate

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def ctx():
    from paper_2005_09316_b200 import binding
    c = binding.Woden(0)
    yield c
    c.close()


def _dev(a):
    import torch
    return torch.as_tensor(np.ascontiguousarray(a), device="cuda:0")


@pytest.mark.parametrize("n_ant", [2, 3, 9, 33, 64, 65, 100, 128])      # 65-128: the register-resident kernel
def test_gains_match_the_oracle_on_random_cells(ctx, n_ant):
    import torch
    rng = np.random.default_rng(n_ant)
    nb = n_ant * (n_ant - 1) // 2
    ideal = (rng.normal(0, 3, (2, 3, nb)) + 1j * rng.normal(0, 3, (2, 3, nb))).astype(np.complex64)
    gam = (1 + 0.2 * rng.normal(0, 1, (2, 3, n_ant))) * np.exp(1j * rng.normal(0, 0.4, (2, 3, n_ant)))
    i, j = ocal.baseline_pairs(n_ant)
    noise = 0.05 * (rng.normal(0, 1, ideal.shape) + 1j * rng.normal(0, 1, ideal.shape))
    data = (gam[..., i] * np.conj(gam[..., j]) * ideal + noise).astype(np.complex64)
    g = ctx.calibrate_gains(n_ant, _dev(data), _dev(ideal), 10)
    torch.cuda.synchronize()
    ref = ocal.calibrate(data, ideal, n_ant, 10)
    assert g.shape == ref.shape
    assert np.abs(g.cpu().numpy() - ref).max() <= 1e-9 * max(1.0, np.abs(ref).max())
    out = ctx.peel(n_ant, _dev(data), _dev(ideal), g)
    torch.cuda.synchronize()
    assert np.abs(out.cpu().numpy() - ocal.peel(data, ideal, ref)).max() <= 2e-6 * np.abs(data).max()
    # fewer iterations: every Gauss-Newton step agrees, not only the converged answer
    g1 = ctx.calibrate_gains(n_ant, _dev(data), _dev(ideal), 1)
    assert np.abs(g1.cpu().numpy() - ocal.calibrate(data, ideal, n_ant, 1)).max() <= 1e-10


def test_planted_gains_recovered_and_identity(ctx):
    import torch
    rng = np.random.default_rng(77)
    n_ant, nb = 40, 780
    ideal = (rng.normal(0, 2, (5, nb)) + 1j * rng.normal(0, 2, (5, nb))).astype(np.complex64)
    g = ctx.calibrate_gains(n_ant, _dev(ideal), _dev(ideal), 10)
    assert np.abs(g.cpu().numpy() - 1.0).max() <= 1e-12
    gam = (1 + 0.1 * rng.normal(0, 1, (5, n_ant))) * np.exp(1j * rng.normal(0, 0.3, (5, n_ant)))
    i, j = ocal.baseline_pairs(n_ant)
    data = (gam[:, i] * np.conj(gam[:, j]) * ideal.astype(np.complex128)).astype(np.complex64)
    g = ctx.calibrate_gains(n_ant, _dev(data), _dev(ideal), 10).cpu().numpy()
    prod = g[:, i] * np.conj(g[:, j])
    assert np.abs(prod - gam[:, i] * np.conj(gam[:, j])).max() <= 2e-6        # complex64 data rounding
    res = ctx.peel(n_ant, _dev(data), _dev(ideal), _dev(g)).cpu().numpy()
    assert np.abs(res).max() <= 5e-6 * np.abs(data).max()


def test_peeling_a_predicted_sky_with_a_truncated_model(ctx):
    # the paper's experiment in miniature (section 5): "observed" = full sky through the predictor,
    # model = the truncated sky (Eq 23-24) through the predictor; fit gains per cell, subtract
    import torch
    from paper_2005_09316_b200 import binding
    wl = inputs.make_config(2, n_times=2)
    n_ant = 128
    uvw = binding.Uvw(_dev(wl.u_m), _dev(wl.v_m), _dev(wl.w_m), wl.freqs_hz[:3])
    p = wl.points
    full = ctx.new_vis(uvw)
    ctx.predict_points(uvw, _dev(p.l), _dev(p.m), _dev(p.s0_jy), _dev(p.alpha), wl.ref_freq_hz, full)
    pt = truncate.truncate_components(ctx, p, 0.8)
    model = ctx.new_vis(uvw)
    ctx.predict_points(uvw, _dev(pt.l), _dev(pt.m), _dev(pt.s0_jy), _dev(pt.alpha), wl.ref_freq_hz, model)
    g = ctx.calibrate_gains(n_ant, full, model, 10)
    res = ctx.peel(n_ant, full, model, g)
    torch.cuda.synchronize(); ctx.check()
    fh, mh = full.cpu().numpy(), model.cpu().numpy()
    ref = ocal.calibrate(fh[0, :2], mh[0, :2], n_ant, 10)                    # two cells through lstsq (16256 x 256)
    assert np.abs(g.cpu().numpy()[0, :2] - ref).max() <= 1e-8
    r = res.cpu().numpy()
    assert np.abs(r[0, :2] - ocal.peel(fh[0, :2], mh[0, :2], ref)).max() <= 2e-6 * np.abs(fh).max()
    # calibration can only lower the residual power relative to subtracting the raw model
    assert np.sum(np.abs(r) ** 2) <= np.sum(np.abs(fh - mh) ** 2) * (1 + 1e-6)


def test_calibrate_argument_errors(ctx):
    import torch
    from paper_2005_09316_b200 import binding
    z = torch.zeros((1, 1), dtype=torch.complex64, device="cuda:0")
    with pytest.raises(ValueError):
        ctx.calibrate_gains(3, z, z)
    big = torch.zeros((1, 201 * 200 // 2), dtype=torch.complex64, device="cuda:0")
    with pytest.raises(binding.WodenError) as e:
        ctx.calibrate_gains(201, big, big)                                    # W would not fit shared memory
    assert e.value.status == binding.WODEN_ERR_DIM


def test_largest_supported_array_matches_the_oracle(ctx):
    # 200 antennas: the triangle of W fills one CTA's shared memory (one cell per SM); one and three passes
    import torch
    n_ant = 200
    rng = np.random.default_rng(200)
    nb = n_ant * (n_ant - 1) // 2
    ideal = (rng.normal(0, 3, (1, nb)) + 1j * rng.normal(0, 3, (1, nb))).astype(np.complex64)
    gam = (1 + 0.1 * rng.normal(0, 1, (1, n_ant))) * np.exp(1j * rng.normal(0, 0.3, (1, n_ant)))
    i, j = ocal.baseline_pairs(n_ant)
    data = (gam[..., i] * np.conj(gam[..., j]) * ideal).astype(np.complex64)
    for n_iter in (1, 3):
        g = ctx.calibrate_gains(n_ant, _dev(data), _dev(ideal), n_iter)
        torch.cuda.synchronize()
        ref = ocal.calibrate(data, ideal, n_ant, n_iter)
        assert np.abs(g.cpu().numpy() - ref).max() <= 1e-9 * max(1.0, np.abs(ref).max())
