"""Pins of the oracle's linearly varying charge density (q_i = w_i A sigma(Q_i))."""
from __future__ import annotations

import numpy as np
import pytest

import oracle
from paper_1606_03743_b200 import synth


def _mesh():
    et, vt = synth.random_elements(synth.TRI, 7, 21)
    er, vr = synth.random_elements(synth.RECT, 5, 22)
    return np.concatenate([et, er]), np.concatenate([vt, vr])


def test_constant_vertex_values_reduce_to_constant_sigma():
    etype, verts = _mesh()
    rng = np.random.default_rng(1)
    sigma = rng.uniform(-1, 1, len(etype))
    pts = 3.0 + rng.random((9, 3))
    for level in range(5):
        a = oracle.evaluate_linear(etype, verts, np.repeat(sigma[:, None], 3, axis=1), pts, level)
        b = oracle.evaluate(etype, verts, sigma, pts, level)
        assert np.max(np.abs(a["phi"] - b["phi"])) <= 1e-15 * np.max(b["Sphi"])
        assert np.max(np.abs(a["E"] - b["E"])) <= 1e-15 * np.max(b["SE"])


def test_superposition_in_the_vertex_values():
    etype, verts = _mesh()
    rng = np.random.default_rng(2)
    s1, s2 = rng.uniform(-1, 1, (len(etype), 3)), rng.uniform(-1, 1, (len(etype), 3))
    pts = 3.0 + rng.random((5, 3))
    a = oracle.evaluate_linear(etype, verts, s1, pts, 2)["phi"]
    b = oracle.evaluate_linear(etype, verts, s2, pts, 2)["phi"]
    c = oracle.evaluate_linear(etype, verts, 2.0 * s1 - 3.0 * s2, pts, 2)
    assert np.max(np.abs(c["phi"] - (2.0 * a - 3.0 * b))) <= 1e-14 * np.max(c["Sphi"])


@pytest.mark.parametrize("kind", [synth.TRI, synth.RECT])
@pytest.mark.parametrize("level", [0, 2, 4])
def test_far_field_monopole_and_dipole_closed_forms(kind, level):
    """Total charge and dipole moment of a linear density have closed forms
    (triangle: Int l_i l_j = A (1 + delta_ij) / 12; rectangle: Int x^2 = 1/3 on [-1,1]);
    every rule is exact for them (degree >= 3), and far away Phi -> k (Q/r + p.d/r^3)."""
    etype, verts = synth.random_elements(kind, 1, 31 + kind)
    A_, B_, C_ = verts[0]
    sv = np.array([[0.7, -0.4, 1.9]])
    if kind == synth.TRI:
        area = 0.5 * np.linalg.norm(np.cross(B_ - A_, C_ - A_))
        cen = (A_ + B_ + C_) / 3.0
        Q = area * sv.mean()
        p = area / 12.0 * sum(sv[0, i] * (v - cen) for i, v in enumerate((A_, B_, C_)))
    else:
        e1, e2 = B_ - A_, C_ - A_
        area = np.linalg.norm(e1) * np.linalg.norm(e2)
        cen = A_ + 0.5 * e1 + 0.5 * e2
        s_c = sv[0, 0] + 0.5 * (sv[0, 1] - sv[0, 0]) + 0.5 * (sv[0, 2] - sv[0, 0])
        Q = area * s_c
        p = area / 12.0 * ((sv[0, 1] - sv[0, 0]) * e1 + (sv[0, 2] - sv[0, 0]) * e2)
    k = oracle.coulomb_k()
    rng = np.random.default_rng(3)
    d = synth.isotropic_directions(rng, 6) * 400.0
    r = np.linalg.norm(d, axis=1)
    got = oracle.evaluate_linear(etype, verts, sv, cen + d, level)
    want = k * (Q / r + d @ p / r ** 3)
    # next term of the expansion: quadrupole, relative size (L/r)^2
    assert np.max(np.abs(got["phi"] - want) / got["Sphi"]) <= 3.0 / 400.0 ** 2


def test_converges_to_a_fine_piecewise_constant_subdivision():
    """Linear sigma on one triangle vs 4^k flat sub-triangles carrying sigma at their centroids:
    the piecewise-constant model converges to it with O(h^2), i.e. 4x per subdivision level."""
    A_, B_, C_ = np.array([0.0, 0, 0]), np.array([1.0, 0, 0]), np.array([0.3, 0.8, 0])
    sv = np.array([[1.0, 2.0, -0.5]])
    pts = np.array([[0.4, 0.3, 2.0], [2.5, -1.0, 0.7]])
    got = oracle.evaluate_linear(np.zeros(1, dtype=np.uint8), np.array([[A_, B_, C_]]), sv, pts, 4)
    M2 = np.array([[1.0, 0.3], [0.0, 0.8]])                       # in-plane coordinates of (s, t)
    tris = [(A_, B_, C_)]
    errs = []
    for k in range(1, 6):
        nxt = []
        for a, b, c in tris:
            ab, bc, ca = (a + b) / 2, (b + c) / 2, (c + a) / 2
            nxt += [(a, ab, ca), (ab, b, bc), (ca, bc, c), (ab, bc, ca)]
        tris = nxt
        if k < 4:
            continue
        fv = np.array(tris)
        st = np.linalg.solve(M2, fv.mean(axis=1)[:, :2].T).T
        fs = sv[0, 0] + st[:, 0] * (sv[0, 1] - sv[0, 0]) + st[:, 1] * (sv[0, 2] - sv[0, 0])
        ref = oracle.evaluate(np.zeros(len(fv), dtype=np.uint8), fv, fs, pts, 4)
        errs.append((np.max(np.abs(got["phi"] - ref["phi"]) / ref["Sphi"]),
                     np.max(np.abs(got["E"] - ref["E"]).max(axis=1) / ref["SE"])))
    (p4, e4), (p5, e5) = errs
    assert p5 <= 1e-4 and e5 <= 1e-3
    assert 3.0 < p4 / p5 < 5.0 and 3.0 < e4 / e5 < 5.0
