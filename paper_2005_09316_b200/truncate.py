"""Model truncation of PAPER.md section 5.3 (Eq 23-25): which sky components / shapelet
basis functions to keep.  The method's arithmetic runs in the library -- woden_truncate_select (Eq 23-24:
ranking and the cumulative absolute flux) and woden_shapelet_truncation_weights / woden_fit_shapelets (Eq 25: |C S0| times the absolute pixel sums of
the restoring-beam-convolved basis images) -- this module only marshals arrays in and slices the component
lists with the returned flags.  Sparse coefficient lists go through the same shapelet predictor, which
skips empty coefficient chunks.
"""
from __future__ import annotations

import dataclasses
from typing import Optional

import numpy as np

from .inputs import Components

# Eq 25 needs "the pixels used during the model fit" and the restoring beam (:279-281).  The BASELINE
# configs draw their coefficients instead of fitting an image, so the library chooses a grid and a beam for them
# (reading G20; defaults WODEN_EQ25_PIXELS / WODEN_EQ25_BEAM_FWHM_RAD in include/woden_b200.h).


def keep_indices(ctx, weights, f_comp: float) -> np.ndarray:
    """Indices (ascending) of the components Eq 23-24 keep: woden_truncate_select's flags.  `weights` is a host
    array or a float64 device tensor (as shapelet_basis_weights returns)."""
    import torch
    if isinstance(weights, torch.Tensor):
        w = weights.to(device=f"cuda:{ctx.device}", dtype=torch.float64).contiguous()
    else:
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


def shapelet_basis_weights(ctx, s: Components, beam_fwhm_rad: float = -1.0, n_pix: int = 0):
    """Eq 25 per listed basis function, computed by the library (woden_shapelet_truncation_weights): a device
    float64 tensor [n_coeff].  beam_fwhm_rad < 0 / n_pix = 0 take the library's defaults, beam_fwhm_rad = 0 no beam."""
    return ctx.shapelet_truncation_weights(s.s0_jy, s.beta1_rad, s.beta2_rad, s.pa_rad, s.coeff_offset, s.n1, s.n2,
                                           s.coeff, n_pix=n_pix, beam_fwhm_rad=beam_fwhm_rad)


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
