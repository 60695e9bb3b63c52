"""Pins for the oracle's transcription of the ten cubature tables (App. A/B).

The pins are mathematical facts and values the paper prints, not a retyping of the oracle:
sum of weights (Eq. 3.1), exact monomial integration up to the stated degree and failure
at degree+1 (L113, L125), the printed (N, d) pairs, the worked example for Table A2 (L127).
"""
from fractions import Fraction
from itertools import product
from math import factorial, sqrt

import numpy as np
import pytest

import oracle
from conftest import read_golden

TRI, RECT = 0, 1
SUMMARY = [(0 if r[0] == "tri" else 1, int(r[1]), r[2], int(r[3]), int(r[4]))
           for r in read_golden("paper_rule_summary.txt")]


def tri_exact(a, b, c):
    """Int lA^a lB^b lC^c dS / area over a triangle = 2 a! b! c! / (a+b+c+2)!"""
    return float(Fraction(2 * factorial(a) * factorial(b) * factorial(c), factorial(a + b + c + 2)))


def rect_exact(n, m):
    """Int x^n y^m dx dy / 4 over [-1,1]^2."""
    return 0.0 if (n % 2 or m % 2) else 1.0 / ((n + 1) * (m + 1))


@pytest.mark.parametrize("etype,level,table,N,deg", SUMMARY)
def test_printed_N_and_degree(etype, level, table, N, deg):
    assert oracle.rule_info(etype, level) == (N, deg)
    coords, w = oracle.rule_nodes(etype, level)
    assert len(w) == N


@pytest.mark.parametrize("etype,level,table,N,deg", SUMMARY)
def test_weights_sum_to_one(etype, level, table, N, deg):
    _, w = oracle.rule_nodes(etype, level)
    assert abs(w.sum() - 1.0) < 5e-16


@pytest.mark.parametrize("etype,level,table,N,deg", SUMMARY)
def test_exact_up_to_degree_and_not_beyond(etype, level, table, N, deg):
    coords, w = oracle.rule_nodes(etype, level)
    worst_in, worst_out = 0.0, 0.0
    if etype == TRI:
        assert np.allclose(coords.sum(axis=1), 1.0, atol=3e-16)
        for a, b, c in product(range(deg + 2), repeat=3):
            tot = a + b + c
            if tot > deg + 1:
                continue
            val = float(np.sum(w * coords[:, 0] ** a * coords[:, 1] ** b * coords[:, 2] ** c))
            rel = abs(val - tri_exact(a, b, c)) / tri_exact(a, b, c)
            if tot <= deg:
                worst_in = max(worst_in, rel)
            else:
                worst_out = max(worst_out, rel)
        # the decimal tables carry 16 digits: A3 leaves ~3e-14 relative at degree 7
        assert worst_in < 2e-13, worst_in
        assert worst_out > 5e-5, worst_out
    else:
        for n, m in product(range(deg + 2), repeat=2):
            tot = n + m
            if tot > deg + 1:
                continue
            val = float(np.sum(w * coords[:, 0] ** n * coords[:, 1] ** m))
            err = abs(val - rect_exact(n, m))
            if tot <= deg:
                worst_in = max(worst_in, err)
            else:
                worst_out = max(worst_out, err)
        assert worst_in < 5e-16, worst_in
        # odd degree d+1 monomials vanish by symmetry; d+1 is even for all five rectangle rules
        assert worst_out > 2e-5, worst_out


@pytest.mark.parametrize("etype,level,table,N,deg", SUMMARY)
def test_monomial_residual_entry_point(etype, level, table, N, deg):
    """The long-double residual exported by the oracle agrees with the float64 evaluation above."""
    for a in range(deg + 1):
        for b in range(deg + 1 - a):
            assert abs(oracle.monomial_residual(etype, level, a, b)) < 3e-15


@pytest.mark.parametrize("etype,level,table,N,deg", SUMMARY)
def test_nodes_inside_and_weight_signs(etype, level, table, N, deg):
    coords, w = oracle.rule_nodes(etype, level)
    if etype == TRI:
        assert coords.min() > 0.02 and coords.max() < 1.0        # strictly inside (L121)
    else:
        assert np.abs(coords).max() < 0.99
    if table == "A1":
        assert w[0] == -9.0 / 16.0 and (w[1:] > 0).all()          # printed negative weight (L287)
    else:
        assert (w > 0).all()
    # no duplicated node
    for i in range(N):
        d = np.abs(coords - coords[i]).max(axis=1)
        d[i] = 1.0
        assert d.min() > 1e-3


def test_table_A2_worked_example():
    """PAPER.md L127 + caption L292: which coordinate is distinguished for points 2..7."""
    coords, w = oracle.rule_nodes(TRI, 1)
    t = 1.0 / 3.0
    sym = {"s": (1.0 - sqrt(15.0)) / 7.0, "r": (1.0 + sqrt(15.0)) / 7.0}
    wts = {"s": (155.0 + sqrt(15.0)) / 1200.0, "r": (155.0 - sqrt(15.0)) / 1200.0}
    for row in read_golden("paper_worked_example_A2.txt"):
        i, which, s = int(row[0]) - 1, int(row[1]), row[2]
        if which < 0:
            assert np.allclose(coords[i], t, atol=1e-16) and abs(w[i] - 9.0 / 40.0) < 1e-16
            continue
        x = sym[s]
        expect = np.full(3, t - t * x)
        expect[which] = t + 2.0 * t * x
        assert np.allclose(coords[i], expect, atol=2e-16)
        assert abs(w[i] - wts[s]) < 2e-16


def test_table_B_closed_form_rows():
    """Rows of B1-B3 given by closed expressions in the captions (L335, L344, L353)."""
    c, w = oracle.rule_nodes(RECT, 0)
    assert np.allclose(np.abs(c), 1.0 / sqrt(3.0), atol=1e-16) and np.allclose(w, 0.25)
    assert len({(np.sign(x), np.sign(y)) for x, y in c}) == 4
    c, w = oracle.rule_nodes(RECT, 1)
    t, r, s = sqrt(14.0 / 15.0), sqrt(3.0 / 5.0), sqrt(1.0 / 3.0)
    assert np.allclose(c[0], 0) and abs(w[0] - 2.0 / 7.0) < 1e-16
    assert sorted(c[1:3, 1].tolist()) == pytest.approx([-t, t], abs=1e-16) and np.allclose(c[1:3, 0], 0)
    assert np.allclose(w[1:3], 5.0 / 63.0) and np.allclose(w[3:], 5.0 / 36.0)
    assert np.allclose(np.abs(c[3:, 0]), r, atol=1e-16) and np.allclose(np.abs(c[3:, 1]), s, atol=1e-16)
    c, w = oracle.rule_nodes(RECT, 2)
    q = sqrt(583.0)
    assert np.allclose(w[:4], 49.0 / 810.0)
    assert np.allclose(w[4:8], (178981.0 + 2769.0 * q) / 1888920.0)
    assert np.allclose(w[8:], (178981.0 - 2769.0 * q) / 1888920.0)
    assert np.allclose(np.abs(c[4:8]), sqrt((114.0 - 3.0 * q) / 287.0), atol=1e-16)
    assert np.allclose(np.abs(c[8:]), sqrt((114.0 + 3.0 * q) / 287.0), atol=1e-16)


def test_rotation_orbits_B4_B5():
    """B4/B5 rows expand by rotations of 0, 180, +-90 degrees (L364, L374): the node set is
    invariant under a 90 degree rotation and each orbit carries one weight."""
    for level in (3, 4):
        c, w = oracle.rule_nodes(RECT, level)
        rot = np.stack([-c[:, 1], c[:, 0]], axis=1)
        for p, wp in zip(rot, w):
            d = np.abs(c - p).max(axis=1)
            j = int(d.argmin())
            assert d[j] < 1e-16 and w[j] == wp


@pytest.mark.parametrize("n", [2, 5, 12, 16, 32])
def test_gauss_legendre_nodes(n):
    """n-point Gauss-Legendre integrates x^k on [-1,1] exactly for k <= 2n-1."""
    x, w = oracle.gauss_legendre(n)
    for k in range(2 * n):
        exact = 0.0 if k % 2 else 2.0 / (k + 1)
        assert abs(np.sum(w * x ** k) - exact) < 1e-15
    assert abs(np.sum(w * x ** (2 * n)) - 2.0 / (2 * n + 1)) > 1e-22 if n < 12 else True
