"""Pins for the gain-calibration oracle (oracle/calibrate.py; section 5.1, Eq 18-22) against
what the mathematics fixes, not against itself."""
import numpy as np

from oracle import calibrate as ocal


def _cell(seed, n=9):
    rng = np.random.default_rng(seed)
    nb = n * (n - 1) // 2
    ideal = rng.normal(0, 3, nb) + 1j * rng.normal(0, 3, nb)
    gam = (1 + 0.2 * rng.normal(0, 1, n)) * np.exp(1j * rng.normal(0, 0.4, n))
    return rng, ideal, gam


def test_identity_data_gives_unit_gains_and_zero_residual():
    _, ideal, _ = _cell(0)
    g = ocal.calibrate(ideal, ideal, 9)
    assert np.allclose(g, 1.0, atol=1e-14)
    assert np.abs(ocal.peel(ideal, ideal, g)).max() < 1e-13


def test_planted_gains_are_recovered_up_to_the_overall_phase():
    _, ideal, gam = _cell(1)
    data = ocal.model_vis(gam, ideal)                       # Eq 19 with g + e = gamma
    g = ocal.calibrate(data, ideal, 9, n_iter=10)           # :235 "converged after 10 iterations"
    i, j = ocal.baseline_pairs(9)
    assert np.abs(g[i] * np.conj(g[j]) - gam[i] * np.conj(gam[j])).max() < 1e-10
    assert np.abs(ocal.peel(data, ideal, g)).max() < 1e-9
    phase = g[0] / gam[0]
    assert abs(abs(phase) - 1) < 1e-10 and np.allclose(g, gam * phase, atol=1e-10)


def test_design_matrix_is_the_jacobian_of_eq18():
    # Eq 21 is the first-order expansion of Eq 19 - Eq 18: A must equal dM/d(Re g, Im g) at g
    _, ideal, gam = _cell(2, n=6)
    A = ocal.design_matrix(gam, ideal)
    n, h = 6, 1e-6
    for k in range(2 * n):
        dg = np.zeros(n, dtype=complex)
        dg[k % n] = h if k < n else 1j * h
        dM = (ocal.model_vis(gam + dg, ideal) - ocal.model_vis(gam - dg, ideal)) / (2 * h)
        assert np.allclose(A[:, k], np.concatenate([dM.real, dM.imag]), atol=1e-8), k
    # the overall phase is unconstrained: e_i = i g_i is a null vector of A (why Eq 22 needs lstsq)
    null = np.concatenate([(1j * gam).real, (1j * gam).imag])
    assert np.abs(A @ null).max() < 1e-12
    assert np.linalg.matrix_rank(A) == 2 * n - 1


def test_step_is_least_squares_and_minimum_norm_and_objective_falls():
    rng, ideal, gam = _cell(3)
    data = ocal.model_vis(gam, ideal) + 0.05 * (rng.normal(0, 1, ideal.size) + 1j * rng.normal(0, 1, ideal.size))
    g = np.ones(9, dtype=complex)
    cost = [np.sum(np.abs(data - ocal.model_vis(g, ideal)) ** 2)]
    for _ in range(10):
        e = ocal.gain_step(g, data, ideal)
        A = ocal.design_matrix(g, ideal)
        R = data - ocal.model_vis(g, ideal)
        x = np.concatenate([e.real, e.imag])
        grad = A.T @ (A @ x - np.concatenate([R.real, R.imag]))          # normal equations of Eq 22
        assert np.abs(grad).max() < 1e-9 * np.abs(A).max() ** 2
        assert abs(np.sum((np.conj(1j * g) * e).real)) < 1e-10           # no component along the gauge direction
        g = g + e
        cost.append(np.sum(np.abs(data - ocal.model_vis(g, ideal)) ** 2))
    assert cost[-1] < 0.05 * cost[0] and all(b <= a * (1 + 1e-9) for a, b in zip(cost[3:], cost[4:]))


def test_cells_are_independent_and_shapes_broadcast():
    rng, ideal, gam = _cell(4, n=5)
    ideal2 = np.stack([ideal, ideal[::-1]]).reshape(1, 2, -1)
    data2 = np.stack([ocal.model_vis(gam, ideal), ocal.model_vis(np.conj(gam), ideal[::-1])]).reshape(1, 2, -1)
    g = ocal.calibrate(data2, ideal2, 5)
    assert g.shape == (1, 2, 5)
    assert np.allclose(g[0, 0], ocal.calibrate(data2[0, 0], ideal2[0, 0], 5), atol=0)
    assert np.abs(ocal.peel(data2, ideal2, g)).max() < 1e-9
