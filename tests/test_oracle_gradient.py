"""Pins of the oracle's field gradient G_ij = dE_i/dx_j (derivatives of the field from
the same point charges).  The oracle formula is pinned by things other than itself: central
differences of the (separately pinned) oracle field, the point-charge closed form in the far
field, the charged-sphere closed form, and Laplace's equation (trace = 0)."""
from __future__ import annotations

import numpy as np
import pytest

import oracle
from paper_1606_03743_b200 import synth

IDX = {(0, 0): 0, (1, 1): 1, (2, 2): 2, (0, 1): 3, (1, 0): 3, (0, 2): 4, (2, 0): 4, (1, 2): 5, (2, 1): 5}


def full(G6):
    return np.array([[G6[IDX[(i, j)]] for j in range(3)] for i in range(3)])


@pytest.mark.parametrize("level", [0, 1, 2, 3, 4])
def test_gradient_is_derivative_of_field(level):
    c = synth.config4(scale=0.0005, ntracks=3, npts_per_track=4)      # mixed mesh, smooth sigma
    pts = c["pts"][:6]
    g = oracle.evaluate_gradient(c["etype"], c["verts"], c["sigma"], pts, level)
    h = 1e-4
    for j, P in enumerate(pts):
        num = np.zeros((3, 3))
        for ax in range(3):
            d = np.zeros(3)
            d[ax] = h
            Ep = oracle.evaluate(c["etype"], c["verts"], c["sigma"], (P + d)[None], level)["E"][0]
            Em = oracle.evaluate(c["etype"], c["verts"], c["sigma"], (P - d)[None], level)["E"][0]
            num[:, ax] = (Ep - Em) / (2 * h)
        # central differences: O(h^2) truncation, ~1e-16/h rounding, both relative to SG
        assert np.max(np.abs(full(g["G"][j]) - num)) <= 2e-6 * g["SG"][j]


@pytest.mark.parametrize("kind", [synth.TRI, synth.RECT])
def test_far_field_point_charge_limit(kind):
    c = synth.config5(kind, m=64, dr_lo=300.0, dr_hi=3e4)
    etype, verts = c["etype"], c["verts"]
    cen = synth.element_centroids(etype, verts)[0]
    area = 0.5 * 0.8 if kind == synth.TRI else 1.0                    # the two config-5 elements
    k = oracle.coulomb_k()
    g = oracle.evaluate_gradient(etype, verts, c["sigma"], c["pts"], 1)
    for j, P in enumerate(c["pts"]):
        d = P - cen
        r = np.linalg.norm(d)
        exact = k * area * (np.eye(3) / r ** 3 - 3.0 * np.outer(d, d) / r ** 5)
        # deviation of a finite element from a point charge: O(DR^-2)
        assert np.max(np.abs(full(g["G"][j]) - exact)) <= 5.0 / c["ratio"][j] ** 2 * g["SG"][j]


def test_traceless_and_denominator():
    c = synth.config2(nside=4, m=50)
    g = oracle.evaluate_gradient(c["etype"], c["verts"], c["sigma"], c["pts"], 2)
    assert np.all(np.abs(g["G"][:, :3].sum(axis=1)) <= 1e-15 * g["SG"])      # Laplace: div E = 0
    assert np.all(g["SG"] > 0)
    assert np.all(np.abs(g["G"]).max(axis=1) <= 2.0 * g["SG"])               # |delta - 3 dd/r^2| <= 2


def test_charged_sphere_gradient():
    c = synth.config1()
    pts = c["pts"][:20]
    g = oracle.evaluate_gradient(c["etype"], c["verts"], c["sigma"], pts, 1)
    areas = 0.5 * np.linalg.norm(np.cross(c["verts"][:, 1] - c["verts"][:, 0], c["verts"][:, 2] - c["verts"][:, 0]), axis=1)
    Q = float((c["sigma"] * areas).sum())
    k = oracle.coulomb_k()
    for j, P in enumerate(pts):
        r = np.linalg.norm(P)
        exact = k * Q * (np.eye(3) / r ** 3 - 3.0 * np.outer(P, P) / r ** 5)
        # faceted sphere vs point charge with the same total charge: multipoles l >= 6 only
        # (Phi deviates <= 1.6e-5 at r = 1.5; two derivatives cost a factor (l+2)(l+3)/6 = 12)
        assert np.max(np.abs(full(g["G"][j]) - exact)) <= 5e-4 * np.abs(exact).max()


def test_adaptive_uses_per_pair_rule_and_rejects_analytic():
    c = synth.config5(synth.TRI, m=40, dr_lo=30.0, dr_hi=70.0)         # all pairs in the N = 12 band
    dr = oracle.default_policy(False)
    ga = oracle.evaluate_gradient(c["etype"], c["verts"], c["sigma"], c["pts"], -1, dr=dr)
    g2 = oracle.evaluate_gradient(c["etype"], c["verts"], c["sigma"], c["pts"], 2)
    g1 = oracle.evaluate_gradient(c["etype"], c["verts"], c["sigma"], c["pts"], 1)
    assert np.array_equal(ga["G"], g2["G"]) and not np.array_equal(ga["G"], g1["G"])
    with pytest.raises(ValueError):
        oracle.evaluate_gradient(c["etype"], c["verts"], c["sigma"], c["pts"], -1, dr=dr, levels_mask=63)
