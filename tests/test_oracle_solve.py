"""Pins of the oracle's BEM solve (the linear system for the unknown charge densities).
The direct solve is pinned by physics and by an independent code path: the capacitance of a sphere,
and the residual computed with oracle.evaluate (field-point sum) instead of the assembled matrix."""
from __future__ import annotations

import numpy as np

import oracle
from paper_1606_03743_b200 import synth

EPS0 = 8.8541878128e-12


def _areas(verts):
    return 0.5 * np.linalg.norm(np.cross(verts[:, 1] - verts[:, 0], verts[:, 2] - verts[:, 0]), axis=1)


def test_unit_potential_sphere_capacitance():
    """Sphere of radius R at potential V: sigma = eps0 V / R, Q = 4 pi eps0 R V (textbook)."""
    c = synth.config1(level=2, m=1)                      # 320 flat triangles, R = 1
    V = np.full(len(c["etype"]), 1.0)
    sigma, A = oracle.solve(c["etype"], c["verts"], V, oracle.default_policy(False))
    Q = float((sigma * _areas(c["verts"])).sum())
    assert abs(Q / (4 * np.pi * EPS0) - 1.0) < 2e-2       # flat facets inside the sphere: slightly smaller capacitance
    assert np.all(sigma > 0) and sigma.std() / sigma.mean() < 0.1
    assert abs(sigma.mean() / EPS0 - 1.0) < 3e-2
    # finer mesh: closer
    c3 = synth.config1(level=3, m=1)
    s3, _ = oracle.solve(c3["etype"], c3["verts"], np.ones(len(c3["etype"])), oracle.default_policy(False))
    Q3 = float((s3 * _areas(c3["verts"])).sum())
    assert abs(Q3 / (4 * np.pi * EPS0) - 1.0) < abs(Q / (4 * np.pi * EPS0) - 1.0)


def test_solution_reproduces_the_potential_through_the_field_point_sum():
    """A sigma = V checked with the other oracle path: evaluate() at the centroids (adaptive)."""
    c = synth.config4(scale=0.0004, ntracks=1, npts_per_track=2)     # small mixed mesh
    n = len(c["etype"])
    cen = synth.element_centroids(c["etype"], c["verts"])
    V = 100.0 * np.cos(cen[:, 2] / 5.0) + 10.0 * cen[:, 0]
    dr = oracle.default_policy(False)
    sigma, A = oracle.solve(c["etype"], c["verts"], V, dr)
    back = oracle.evaluate(c["etype"], c["verts"], sigma, cen, -1, dr=dr)["phi"]
    assert np.max(np.abs(back - V)) <= 1e-9 * np.max(np.abs(V))
    assert n > 100 and np.linalg.cond(A) < 1e4
