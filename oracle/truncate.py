"""FP64 CPU oracle of the model truncation of PAPER.md section 5.3 (Eq 23-25, :267-284).  TEST
INFRASTRUCTURE ONLY, like the rest of oracle/.  Plain loops in the paper's order:

  Eq 24: order the components by |I_j|, largest first (equal values keep their original order);
  Eq 23: N_comp = the largest N with  sum_{j <= N} |I_j| <= f_comp * sum_{j <= N_tot} |I_j|
         (the running sum in that order, FP64; compared with f_comp * total * (1 + 1e-15), one rounding
         of slack so that f_comp = an exact partial-sum ratio keeps the component that reaches it);
  Eq 25: the weight of a shapelet basis function = sum over the fitted pixels of
         |C_{p1,p2} (G * B_{p1,p2})(x_s, y_t)|  -- oracle.shamfi.truncation_weights on the design matrix.
Pins: tests/test_truncate.py (brute force, a worked example, invariants)."""
from __future__ import annotations

import numpy as np


def ranked_order(weights) -> np.ndarray:
    """Indices that put |weights| in descending order, ties in original order (Eq 24)."""
    w = np.abs(np.asarray(weights, dtype=np.float64))
    return np.argsort(-w, kind="stable")


def n_keep(abs_sorted, f_comp: float) -> int:
    """N_comp of Eq 23 for |I_j| already in descending order."""
    a = [float(x) for x in abs_sorted]
    if f_comp >= 1.0:
        return len(a)
    total = 0.0
    for x in a:
        total += x
    limit = f_comp * total * (1.0 + 1e-15)
    run, n = 0.0, 0
    for x in a:
        run += x
        if run <= limit:
            n += 1
        else:
            break
    return n


def keep_mask(weights, f_comp: float) -> np.ndarray:
    """Boolean mask of the components Eq 23-24 keep."""
    w = np.abs(np.asarray(weights, dtype=np.float64))
    order = ranked_order(w)
    mask = np.zeros(w.size, dtype=bool)
    mask[order[: n_keep(w[order], f_comp)]] = True
    return mask
