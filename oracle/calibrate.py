"""Plain numpy FP64 oracle of the per-antenna gain fit and peel of PAPER.md section 5.1
(Eq 18-22).  TEST INFRASTRUCTURE ONLY: only tests/ and bench.py's reference legs
may import it; it shares no code with paper_2005_09316_b200/csrc/calibrate.cu (which solves the
reduced N x N normal equations by conjugate gradients instead of a dense least-squares routine).

Per (time, frequency) cell, in the paper's order and notation:

    M_ij = g_i g_j^* I_ij                     Eq 18 (:215; the printed g_i g_i^* is a typo, reading G15)
    R_ij = V_ij - M_ij                        Eq 20 (:223)
    R_ij ~ e_i g_j^* I_ij + g_i e_j^* I_ij    Eq 21 (:229; first-order expansion of Eq 19 - Eq 18,
                                              the printed subscripts are garbled, reading G15)
    A x = b with x = (Re e_1..Re e_N, Im e_1..Im e_N), b = (Re R, Im R)
    x = [A^T A]^-1 A^T b                      Eq 22 (:233) -- A^T A is singular (the overall phase
                                              of the gains is not constrained), so the step is the
                                              minimum-norm least-squares solution (numpy.linalg.lstsq,
                                              a library primitive; reading G16)
    g <- g + e, 10 times from g = 1           (:235 "converged after 10 iterations")

Baselines are all pairs i < j in i-major order (the order of woden_uvw).  The cubic-spline smoothing
of the gains across the band (:237) is not part of this oracle (not built).

Pins (tests/test_calibrate_oracle.py): V = I gives g = 1; planted gains are recovered up to the
overall phase; the design matrix equals the numerical Jacobian of Eq 18; each step is the
Gauss-Newton step of the true residual.
"""
from __future__ import annotations

import numpy as np


def baseline_pairs(n_ant: int):
    i, j = np.triu_indices(n_ant, k=1)
    return i.astype(np.int64), j.astype(np.int64)


def model_vis(g: np.ndarray, ideal: np.ndarray) -> np.ndarray:
    """Eq 18: M_ij = g_i g_j^* I_ij for one cell; g [N] complex, ideal [B] complex."""
    i, j = baseline_pairs(g.shape[0])
    return g[i] * np.conj(g[j]) * ideal


def design_matrix(g: np.ndarray, ideal: np.ndarray) -> np.ndarray:
    """A of Eq 21-22 for one cell: [2B, 2N], rows (Re R_ij ..., Im R_ij ...), columns
    (Re e_1..Re e_N, Im e_1..Im e_N), from R_ij = a e_i + b e_j^*, a = g_j^* I_ij, b = g_i I_ij."""
    n = g.shape[0]
    i, j = baseline_pairs(n)
    nb = i.shape[0]
    a = np.conj(g[j]) * ideal
    b = g[i] * ideal
    A = np.zeros((2 * nb, 2 * n))
    rows = np.arange(nb)
    # Re(a e_i) = Re a Re e_i - Im a Im e_i ; Im(a e_i) = Im a Re e_i + Re a Im e_i
    A[rows, i] += a.real
    A[rows, n + i] += -a.imag
    A[nb + rows, i] += a.imag
    A[nb + rows, n + i] += a.real
    # Re(b e_j^*) = Re b Re e_j + Im b Im e_j ; Im(b e_j^*) = Im b Re e_j - Re b Im e_j
    A[rows, j] += b.real
    A[rows, n + j] += b.imag
    A[nb + rows, j] += b.imag
    A[nb + rows, n + j] += -b.real
    return A


def gain_step(g: np.ndarray, data: np.ndarray, ideal: np.ndarray) -> np.ndarray:
    """One pass of Eq 20-22 for one cell: the additive gain errors e [N]."""
    n = g.shape[0]
    R = data - model_vis(g, ideal)
    bvec = np.concatenate([R.real, R.imag])
    x, *_ = np.linalg.lstsq(design_matrix(g, ideal), bvec, rcond=None)
    return x[:n] + 1j * x[n:]


def calibrate(data: np.ndarray, ideal: np.ndarray, n_ant: int, n_iter: int = 10) -> np.ndarray:
    """Gains [..., N] complex128 for visibilities [..., B] (one independent fit per leading cell)."""
    data = np.asarray(data, dtype=np.complex128)
    ideal = np.asarray(ideal, dtype=np.complex128)
    nb = n_ant * (n_ant - 1) // 2
    if data.shape != ideal.shape or data.shape[-1] != nb:
        raise ValueError("data and ideal must be [..., n_ant (n_ant - 1) / 2]")
    lead = data.shape[:-1]
    d2, i2 = data.reshape(-1, nb), ideal.reshape(-1, nb)
    out = np.ones((d2.shape[0], n_ant), dtype=np.complex128)
    for c in range(d2.shape[0]):
        g = out[c]
        for _ in range(n_iter):
            g = g + gain_step(g, d2[c], i2[c])
        out[c] = g
    return out.reshape(lead + (n_ant,))


def peel(data: np.ndarray, ideal: np.ndarray, gains: np.ndarray) -> np.ndarray:
    """Residual V_ij - g_i g_j^* I_ij (Eq 20 with the fitted gains), per cell."""
    n = gains.shape[-1]
    i, j = baseline_pairs(n)
    return np.asarray(data, dtype=np.complex128) - gains[..., i] * np.conj(gains[..., j]) * ideal
