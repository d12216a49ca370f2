"""Pins against the only numbers the paper prints for this path (tests/golden/
paper_printed_values.txt, each line citing its PAPER.md passage): basis counts (Eq 6) and the
MS CLEAN component split that shapes config 4."""
import os

import numpy as np

import oracle
from paper_2005_09316_b200 import inputs

HERE = os.path.dirname(os.path.abspath(__file__))


def _golden():
    out = {}
    for line in open(os.path.join(HERE, "golden", "paper_printed_values.txt")):
        line = line.split("#", 1)[0].strip()
        if line:
            k, v = line.split()
            out[k] = float(v)
    return out


def test_basis_counts_match_the_papers_printed_totals():
    g = _golden()
    p2 = int(g["p_max_phase2"])
    # Eq 6 evaluated by the generator's triangle, not by retyping the formula
    n1, n2 = inputs.full_triangle(p2)
    assert len(n1) == len(set(zip(n1.tolist(), n2.tolist())))          # no duplicates
    assert int(g["n_lobes"]) * len(n1) == int(g["n_basis_two_lobes_pmax86"])
    assert np.all(n1 + n2 <= p2) and (n1 + n2).max() == p2              # "<=" reading G5
    assert inputs.basis_count(int(g["p_max_phase1"])) == len(inputs.full_triangle(int(g["p_max_phase1"]))[0])


def test_config4_component_split_follows_the_papers_ms_clean_model():
    g = _golden()
    assert g["n_msclean_point"] + g["n_msclean_gaussian"] == g["n_msclean_total"]
    wl = inputs.make_config(4)
    n = wl.points.n + wl.gaussians.n
    assert n == 20000
    # SURVEY.md section 8 fixes 14 340 : 5 660, the paper's 4540 : 1791 to within 0.02 %
    assert abs(wl.points.n / n - g["n_msclean_point"] / g["n_msclean_total"]) < 2e-4
    assert wl.shapelets.n == int(g["n_lobes"])


def test_oracle_accepts_the_papers_largest_model():
    # two lobes x p_max = 86 (7656 basis functions): the oracle evaluates it without overflow
    g = _golden()
    p = int(g["p_max_phase2"])
    n1, n2 = inputs.full_triangle(p)
    P = len(n1)
    rng = np.random.default_rng(86)
    u = np.array([[0.0, 40.0, -900.0, 2900.0]]); v = np.array([[0.0, -25.0, 700.0, 300.0]]); w = np.zeros((1, 4))
    cf = np.concatenate([rng.normal(0, 1, P) * np.exp(-(n1 + n2) / 10.0) for _ in range(2)])
    off = np.array([0, P, 2 * P])
    V = oracle.predict_shapelets(u, v, w, np.array([180e6]), np.array([-0.004, 0.004]), np.zeros(2),
                                 np.ones(2), np.zeros(2), 180e6, np.full(2, 10 * inputs.ARCMIN),
                                 np.full(2, 10 * inputs.ARCMIN), np.zeros(2), None, off,
                                 np.tile(n1, 2), np.tile(n2, 2), cf)
    assert V.shape == (1, 1, 4) and np.all(np.isfinite(V.view(np.float64)))
    # at (u,v) = 0 only even-even orders survive and h_p(0) has a closed form (P8): real-valued
    assert abs(V[0, 0, 0].imag) < 1e-12 * abs(V[0, 0, 0].real)
