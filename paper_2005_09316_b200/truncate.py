"""Model truncation of PAPER.md §5.3 (Eq 23-25): host-side selection of which sky
components / shapelet basis functions to keep.  Not on the GPU hot path: it only shortens the
component arrays and coefficient lists that `woden_predict_*` take (sparse lists go through the
same shapelet kernel, which skips empty coefficient chunks).

Eq 23-24: sort by |I_j| descending and keep the largest N_comp with
    sum_{j <= N_comp} |I_j|  <=  f_comp * sum_{j <= N_tot} |I_j|.
For a point source or Gaussian I_j is its integrated flux density (:275).  For a shapelet basis
function the paper sums the absolute value of the restoring-beam-convolved, coefficient-weighted
basis image over the fitted pixels (Eq 25, :277-280); the restoring beam and the fitted image are
not available here, so `shapelet_basis_weights` uses the unconvolved basis on a
synthetic grid -- a stand-in with the same structure, stated in DESIGN.md.
"""
from __future__ import annotations

import dataclasses
from typing import Optional

import numpy as np

from .inputs import Components


def n_keep(abs_flux: np.ndarray, f_comp: float) -> int:
    """N_comp of Eq 23 for |I_j| already sorted in descending order (Eq 24)."""
    a = np.asarray(abs_flux, dtype=np.float64)
    if a.size == 0:
        return 0
    if np.any(np.diff(a) > 0):
        raise ValueError("abs_flux must be sorted in descending order (Eq 24)")
    if f_comp >= 1.0:
        return int(a.size)
    csum = np.cumsum(a)
    return int(np.searchsorted(csum, f_comp * csum[-1] * (1.0 + 1e-15), side="right"))


def keep_indices(weights: np.ndarray, f_comp: float) -> np.ndarray:
    """Indices (ascending, i.e. original order) of the components Eq 23-24 keep."""
    w = np.abs(np.asarray(weights, dtype=np.float64))
    order = np.argsort(-w, kind="stable")
    return np.sort(order[: n_keep(w[order], f_comp)])


def truncate_components(c: Components, f_comp: float) -> Components:
    """Points or Gaussians: I_j = integrated flux density at the reference frequency (:275)."""
    idx = keep_indices(c.s0_jy, f_comp)
    out = {}
    for f in dataclasses.fields(c):
        v = getattr(c, f.name)
        out[f.name] = None if v is None else np.ascontiguousarray(v[idx])
    return Components(**out)


def _abs_hermite_sums(p_max: int, beta: float, half_width: float, n_pix: int) -> np.ndarray:
    """sum over pixels of |h_p(a x / beta)|, p = 0..p_max, a = 2 sqrt(2 ln 2) (image-space basis of
    Eq 1-2 under the FWHM-like beta of Eq 15-17 / reading G2), on n_pix pixels over +-half_width."""
    x = np.linspace(-half_width, half_width, n_pix) * (2.0 * np.sqrt(2.0 * np.log(2.0)) / beta)
    out = np.empty(p_max + 1)
    hm, h = np.zeros_like(x), np.exp(-0.5 * x * x)          # normalised recurrence of h_p
    for p in range(p_max + 1):
        out[p] = np.abs(h).sum()
        hm, h = h, np.sqrt(2.0 / (p + 1)) * x * h - np.sqrt(p / (p + 1.0)) * hm
    return out


def shapelet_basis_weights(s: Components, n_pix: int = 257) -> np.ndarray:
    """Stand-in for Eq 25: |C_{p1,p2}| * sum_pixels |B_{p1,p2}| per listed basis function, with the
    pixel-sum normalisation of each component's basis (1 / sum of its (0,0) term) so that weights
    of different components are comparable.  Grid: +-1.5 sqrt(2 p_max + 1) beta / a per axis."""
    w = np.zeros(s.coeff.shape[0])
    for j in range(s.n):
        lo, hi = int(s.coeff_offset[j]), int(s.coeff_offset[j + 1])
        if hi == lo:
            continue
        pm = int(max(s.n1[lo:hi].max(), s.n2[lo:hi].max()))
        a = 2.0 * np.sqrt(2.0 * np.log(2.0))
        sx = _abs_hermite_sums(pm, s.beta1_rad[j], 1.5 * np.sqrt(2 * pm + 1.0) * s.beta1_rad[j] / a, n_pix)
        sy = _abs_hermite_sums(pm, s.beta2_rad[j], 1.5 * np.sqrt(2 * pm + 1.0) * s.beta2_rad[j] / a, n_pix)
        w[lo:hi] = np.abs(s.coeff[lo:hi] * s.s0_jy[j]) * sx[s.n1[lo:hi]] * sy[s.n2[lo:hi]] / (sx[0] * sy[0])
    return w


def truncate_shapelets(s: Components, f_comp: float, weights: Optional[np.ndarray] = None) -> Components:
    """Keep the basis functions Eq 23-24 select, ranked over ALL shapelet components together
    (the paper's N_tot counts basis functions of both lobes, :271).  Components are kept even
    when all their basis functions go (empty CSR range)."""
    if s.n == 0 or s.coeff is None:
        return s
    if weights is None:
        weights = shapelet_basis_weights(s)
    idx = keep_indices(weights, f_comp)
    owner = np.searchsorted(s.coeff_offset, idx, side="right") - 1
    counts = np.bincount(owner, minlength=s.n)
    off = np.zeros(s.n + 1, dtype=np.int32)
    off[1:] = np.cumsum(counts)
    return dataclasses.replace(s, coeff_offset=off, n1=np.ascontiguousarray(s.n1[idx]),
                               n2=np.ascontiguousarray(s.n2[idx]), coeff=np.ascontiguousarray(s.coeff[idx]))
