"""Model truncation of PAPER.md section 5.3 (Eq 23-25): which sky components / shapelet
basis functions to keep.  The method's arithmetic runs in the library -- woden_truncate_select (Eq 23-24:
ranking and the cumulative absolute flux) and woden_shapelet_basis_sums / woden_fit_shapelets (Eq 25: the
restoring-beam-convolved basis images) -- this module only marshals arrays in and slices the component
lists with the returned flags.  Sparse coefficient lists go through the same shapelet predictor, which
skips empty coefficient chunks.
"""
from __future__ import annotations

import dataclasses
from typing import Optional

import numpy as np

from .inputs import ARCMIN, Components

# Eq 25 needs "the pixels used during the model fit" and the restoring beam (:279-281).  The BASELINE
# configs draw their coefficients instead of fitting an image, so a grid and a beam are chosen for them
# (reading G20): EQ25_PIXELS^2 pixels over +-1.5 sqrt(2 p_max + 1) max(beta) / a per axis
# (1.5 times the highest order's turning point) and a circular beam of EQ25_BEAM_FWHM (the ~2 arcmin
# resolution of a 3 km array at 180 MHz).
EQ25_PIXELS = 257
EQ25_BEAM_FWHM = 2.0 * ARCMIN


def keep_indices(ctx, weights, f_comp: float) -> np.ndarray:
    """Indices (ascending) of the components Eq 23-24 keep: woden_truncate_select's flags."""
    import torch
    w = torch.as_tensor(np.ascontiguousarray(weights, dtype=np.float64), device=f"cuda:{ctx.device}")
    keep, _ = ctx.truncate_select(w, f_comp)
    return np.flatnonzero(keep.cpu().numpy())


def _take(c: Components, idx) -> Components:
    out = {}
    for f in dataclasses.fields(c):
        v = getattr(c, f.name)
        out[f.name] = None if v is None else np.ascontiguousarray(v[idx])
    return Components(**out)


def truncate_components(ctx, c: Components, f_comp: float) -> Components:
    """Points or Gaussians: I_j = integrated flux density at the reference frequency (:275)."""
    return _take(c, keep_indices(ctx, c.s0_jy, f_comp))


def shapelet_basis_weights(ctx, s: Components, beam_fwhm_rad: float = EQ25_BEAM_FWHM,
                           n_pix: int = EQ25_PIXELS) -> np.ndarray:
    """Eq 25 per listed basis function: |C_{p1,p2}| * sum_pixels |(G * B_{p1,p2})| with the beam-convolved
    basis images of woden_shapelet_basis_sums on the grid of reading G20."""
    w = np.zeros(s.coeff.shape[0])
    a = 2.0 * np.sqrt(2.0 * np.log(2.0))
    for j in range(s.n):
        lo, hi = int(s.coeff_offset[j]), int(s.coeff_offset[j + 1])
        if hi == lo:
            continue
        pm = int((s.n1[lo:hi] + s.n2[lo:hi]).max())
        half = 1.5 * np.sqrt(2 * pm + 1.0) * max(s.beta1_rad[j], s.beta2_rad[j]) / a
        pix = 2.0 * half / (n_pix - 1)
        beam = None
        if beam_fwhm_rad > 0.0:
            beam = (beam_fwhm_rad, beam_fwhm_rad, 0.0, int(min(24, np.ceil(1.5 * beam_fwhm_rad / pix))))
        sums = ctx.shapelet_basis_sums(n_pix, n_pix, -pix, pix, 0.0, 0.0, 0.0, 0.0, s.pa_rad[j], pm,
                                       s.beta1_rad[j], s.beta2_rad[j], beam=beam,
                                       device=f"cuda:{ctx.device}").cpu().numpy()
        n1, n2 = s.n1[lo:hi].astype(np.int64), s.n2[lo:hi].astype(np.int64)
        q = n1 * (pm + 1) - n1 * (n1 - 1) // 2 + n2             # index in the full triangle, n1-major
        w[lo:hi] = np.abs(s.coeff[lo:hi] * s.s0_jy[j]) * sums[q]
    return w


def truncate_shapelets(ctx, s: Components, f_comp: float, weights: Optional[np.ndarray] = None) -> Components:
    """Keep the basis functions Eq 23-24 select, ranked over ALL shapelet components together
    (the paper's N_tot counts basis functions of both lobes, :271).  Components are kept even
    when all their basis functions go (empty CSR range)."""
    if s.n == 0 or s.coeff is None:
        return s
    if weights is None:
        weights = shapelet_basis_weights(ctx, s)
    idx = keep_indices(ctx, weights, f_comp)
    owner = np.searchsorted(s.coeff_offset, idx, side="right") - 1
    counts = np.bincount(owner, minlength=s.n)
    off = np.zeros(s.n + 1, dtype=np.int32)
    off[1:] = np.cumsum(counts)
    return dataclasses.replace(s, coeff_offset=off, n1=np.ascontiguousarray(s.n1[idx]),
                               n2=np.ascontiguousarray(s.n2[idx]), coeff=np.ascontiguousarray(s.coeff[idx]))
