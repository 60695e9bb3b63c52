"""Pins of the oracle's single-element integrator (element k seen from field point k; PAPER.md L193-196
item a, the unit of the accuracy protocol of L68 / L149) and of the Duffy-mapped rectangle rules on
triangles (L163-169).  `-m "not gpu"`."""
from __future__ import annotations

import numpy as np
import pytest

import oracle
from conftest import read_golden
from paper_1606_03743_b200 import synth

TRI, RECT = 0, 1


def _pairs(kind, n, seed, dr):
    et, verts = synth.random_elements(kind, n, seed)
    cen, _, L = oracle.geometry(et, verts)
    dirs = synth.isotropic_directions(np.random.default_rng(seed + 1), n)
    return et, verts, cen + dirs * (dr * L)[:, None]


@pytest.mark.parametrize("kind", [TRI, RECT])
def test_pairs_equal_the_summed_path_on_one_element_meshes(kind):
    et, verts, P = _pairs(kind, 40, 31 + kind, np.geomspace(0.4, 3000.0, 40))
    sigma = np.random.default_rng(2).uniform(-2.0, 2.0, 40)
    dr = oracle.default_policy(True)
    for method in (0, 1, 2, 3, 4, -1):
        got = oracle.evaluate_pairs(et, verts, P, method, sigma=sigma, dr=dr)
        for k in range(40):
            one = oracle.evaluate(et[k:k + 1], verts[k:k + 1], sigma[k:k + 1], P[k:k + 1], method, dr=dr, want_counts=True)
            assert got["phi"][k] == one["phi"][0] and np.array_equal(got["E"][k], one["E"][0])
            assert got["Sphi"][k] == one["Sphi"][0] and got["SE"][k] == one["SE"][0]
            if method == -1:
                assert (got["used"][k] == 5) == (one["nana"][0] == 1)
    # method 5 = the closed form, whatever the distance
    ana = oracle.evaluate_pairs(et, verts, P, 5)
    for k in range(0, 40, 7):
        ip, ie = oracle.analytic(kind, verts[k], P[k])
        assert abs(ana["phi"][k] - oracle.coulomb_k() * ip) <= 4e-16 * abs(ana["phi"][k])
        assert np.abs(ana["E"][k] - oracle.coulomb_k() * ie).max() <= 4e-16 * np.linalg.norm(ana["E"][k])
    assert np.all(ana["used"] == 5)


@pytest.mark.parametrize("level", [0, 1, 2, 3, 4])
def test_duffy_mapped_rule_weights_nodes_and_reduced_degree(level):
    """w' = (1 + y) w: sum 1, all positive, nodes inside the triangle; exact for triangle monomials up
    to (D - 1)/2 (D = degree of the rectangle rule; the tensor rule B1 reaches 2), wrong beyond, and
    in particular wrong at the degree the triangle rule of the same level integrates exactly."""
    bary, w = oracle.duffy_nodes(level)
    assert abs(w.sum() - 1.0) < 1e-15 and np.all(w > 0)
    assert np.all(bary > -1e-15) and np.allclose(bary.sum(axis=1), 1.0, atol=1e-15)
    n_rect, D = oracle.rule_info(RECT, level)
    _, D_tri = oracle.rule_info(TRI, level)
    assert len(w) == n_rect
    exact_to = max((D - 1) // 2, 2 if level == 0 else 0)
    for d in range(exact_to + 1):
        for a in range(d + 1):
            assert abs(oracle.duffy_monomial_residual(level, a, d - a)) < 1e-16, (level, a, d - a)
    worst_next = max(abs(oracle.duffy_monomial_residual(level, a, exact_to + 1 - a)) for a in range(exact_to + 2))
    assert worst_next > 1e-9, (level, worst_next)
    assert exact_to < D_tri
    assert max(abs(oracle.duffy_monomial_residual(level, a, D_tri - a)) for a in range(D_tri + 1)) > 1e-6


def test_duffy_7_point_rule_at_dr_100_is_the_printed_1e_minus_8():
    """Soft pin (L169, golden file): field error of the Duffy-mapped 7-point rectangle rule on random
    triangles at DR = 100 'about 1e-8', against 'few times 1e-15' for the 7-point triangle rule."""
    rows = dict(read_golden("paper_duffy.txt"))
    et, verts, P = _pairs(TRI, 1000, 5, np.full(1000, 100.0))
    ref = oracle.evaluate_pairs(et, verts, P, 4)                       # N = 33 in long double: exact at DR = 100
    def field_err(method):
        r = oracle.evaluate_pairs(et, verts, P, method, precision="double")
        return float((np.abs(r["E"] - ref["E"]).sum(axis=1) / np.linalg.norm(ref["E"], axis=1)).mean())
    duffy, tri = field_err(oracle.DUFFY + 1), field_err(1)
    printed = float(rows["duffy_rect7_field_error_dr100"])
    assert printed / 4 < duffy < printed * 4, duffy                    # "about 1e-8": 5.8e-9
    assert tri < float(rows["tri7_field_error_dr100"]), tri            # "few times 1e-15": 1.9e-15
    # the error falls like DR^-(d+1) with the REDUCED degree d = 2 of the mapped rule, not with d = 5
    et, verts, P2 = _pairs(TRI, 1000, 5, np.full(1000, 200.0))
    ref2 = oracle.evaluate_pairs(et, verts, P2, 4)
    r2 = oracle.evaluate_pairs(et, verts, P2, oracle.DUFFY + 1)
    duffy2 = float((np.abs(r2["E"] - ref2["E"]).sum(axis=1) / np.linalg.norm(ref2["E"], axis=1)).mean())
    assert 6.0 < duffy / duffy2 < 10.0, duffy / duffy2                 # 2^3 = 8


def test_duffy_method_leaves_rectangles_alone():
    et, verts, P = _pairs(RECT, 30, 77, np.geomspace(3.0, 300.0, 30))
    for level in range(5):
        a = oracle.evaluate_pairs(et, verts, P, oracle.DUFFY + level)
        b = oracle.evaluate_pairs(et, verts, P, level)
        assert np.array_equal(a["phi"], b["phi"]) and np.array_equal(a["E"], b["E"])


def test_pairs_argument_checks():
    et, verts, P = _pairs(TRI, 3, 1, np.full(3, 10.0))
    for bad in (6, 7, 13, -2):
        with pytest.raises(ValueError):
            oracle.evaluate_pairs(et, verts, P, bad)
    with pytest.raises(ValueError):
        oracle.evaluate_pairs(et, verts, P, -1)                        # adaptive needs limits
