"""Pins for the oracle's arithmetic (Eq. 3.2/3.3 mapping, Eq. 4.1 sum, analytic branch, GL2,
adaptive reference, distance-ratio policy, matrix rows) against facts fixed by the paper and
by mathematics: closed forms, limits, identities, brute force with mpmath on tiny inputs.
Nothing here recomputes the oracle's own formula to compare with.
"""
import math

import mpmath as mp
import numpy as np
import pytest

import oracle
from conftest import read_golden
from paper_1606_03743_b200 import synth

TRI, RECT = 0, 1
EPS0 = 8.8541878128e-12      # CODATA 2018 vacuum permittivity, F/m (reading 10)
K = 1.0 / (4.0 * math.pi * EPS0)
K_PRINTED = 8.9875517923e9   # CODATA 2018: 1/(4 pi eps0) = 8.987 551 7923(14) e9 N m^2 / C^2
TRI_N = [4, 7, 12, 19, 33]
RECT_N = [4, 7, 12, 17, 33]


def rect_verts(a, b, center=(0.0, 0.0, 0.0)):
    c = np.asarray(center, float)
    p0 = c + np.array([-a / 2, -b / 2, 0.0])
    return np.array([[p0, p0 + [a, 0, 0], p0 + [0, b, 0]]])


def on_axis_rect(a, b, z):
    """Textbook closed form: uniformly charged a x b rectangle, point at height z above its
    centre.  Returns (Int dS/R, Int dS z/R^3)."""
    x, y = mp.mpf(a) / 2, mp.mpf(b) / 2
    z = mp.mpf(z)
    r = mp.sqrt(x * x + y * y + z * z)
    om = 4 * mp.atan(x * y / (z * r))
    iphi = 4 * (x * mp.asinh(y / mp.sqrt(x * x + z * z)) + y * mp.asinh(x / mp.sqrt(y * y + z * z))) - z * om
    return iphi, om


def test_closed_form_itself_by_brute_force():
    """The closed form above against direct 2-D mpmath quadrature of Eq. 2.1."""
    mp.mp.dps = 25
    a, b, z = 1.0, 0.6, 0.8
    f = lambda x, y: 1 / mp.sqrt(x * x + y * y + z * z)
    g = lambda x, y: z / mp.sqrt(x * x + y * y + z * z) ** 3
    iphi = mp.quad(f, [-a / 2, 0, a / 2], [-b / 2, 0, b / 2])
    iez = mp.quad(g, [-a / 2, 0, a / 2], [-b / 2, 0, b / 2])
    cphi, cez = on_axis_rect(a, b, z)
    assert abs(iphi - cphi) < 1e-15 and abs(iez - cez) < 1e-15


def test_coulomb_constant():
    assert abs(oracle.coulomb_k() / K_PRINTED - 1.0) < 2e-10
    assert abs(oracle.coulomb_k() / K - 1.0) < 1e-15


# ------------------------------------------------------------------ geometry / mapping

def test_geometry_triangle_and_rectangle():
    tri = np.array([[[0, 0, 0], [3, 0, 0], [0, 4, 0]]], float)          # 3-4-5 triangle
    cen, area, L = oracle.geometry([TRI], tri)
    assert np.allclose(cen[0], [1.0, 4.0 / 3.0, 0.0], atol=1e-16)
    assert area[0] == pytest.approx(6.0, abs=1e-15) and L[0] == pytest.approx(4.0, abs=1e-15)   # (3+4+5)/3, L66
    cen, area, L = oracle.geometry([RECT], rect_verts(2.0, 0.5, (1, 2, 3)))
    assert np.allclose(cen[0], [1, 2, 3]) and area[0] == pytest.approx(1.0) and L[0] == pytest.approx(1.25)


def test_geometry_errors():
    with pytest.raises(ValueError):
        oracle.geometry([TRI], np.array([[[0, 0, 0], [1, 1, 1], [2, 2, 2]]], float))       # degenerate
    with pytest.raises(ValueError):
        oracle.geometry([RECT], np.array([[[0, 0, 0], [1, 0, 0], [0.5, 1, 0]]], float))     # not a rectangle


@pytest.mark.parametrize("kind", [TRI, RECT])
@pytest.mark.parametrize("level", range(5))
def test_point_charges_total_charge_and_first_moment(kind, level):
    """sum q_i = sigma*A (Eq. 3.1 with f = 1, L143); first moment about Q_cen vanishes
    (every rule has degree >= 1); points lie in the element's plane and inside it."""
    et, verts = synth.random_elements(kind, 20, seed=11 + kind)
    sigma = np.linspace(-2.0, 3.0, 20)
    cen, area, _ = oracle.geometry(et, verts)
    pq = oracle.points(et, verts, sigma, level)
    N = (TRI_N if kind == TRI else RECT_N)[level]
    assert pq.shape == (20 * N, 4)
    pq = pq.reshape(20, N, 4)
    assert np.allclose(pq[:, :, 3].sum(axis=1), sigma * area, rtol=0, atol=2e-15)
    w = pq[:, :, 3] / (sigma * area)[:, None]
    mom = (w[:, :, None] * (pq[:, :, :3] - cen[:, None, :])).sum(axis=1)
    assert np.abs(mom).max() < 5e-16
    e1, e2 = verts[:, 1] - verts[:, 0], verts[:, 2] - verts[:, 0]
    nrm = np.cross(e1, e2)
    nrm /= np.linalg.norm(nrm, axis=1, keepdims=True)
    off = np.einsum("enk,ek->en", pq[:, :, :3] - verts[:, None, 0, :], nrm)
    assert np.abs(off).max() < 1e-15
    # local coordinates inside the element
    for e in range(20):
        M = np.stack([e1[e], e2[e]], axis=1)
        uv = np.linalg.lstsq(M, (pq[e, :, :3] - verts[e, 0]).T, rcond=None)[0].T
        if kind == TRI:
            assert (uv > 0).all() and (uv.sum(axis=1) < 1).all()
        else:
            assert (uv > 0).all() and (uv < 1).all()


def test_centroid_node_maps_to_centroid():
    """lA = lB = lC = 1/3 is the centroid (L111); (x,y) = (0,0) is the rectangle centre (L103)."""
    et, verts = synth.random_elements(TRI, 5, seed=3)
    cen, _, _ = oracle.geometry(et, verts)
    pq = oracle.points(et, verts, np.ones(5), 1).reshape(5, 7, 4)
    assert np.allclose(pq[:, 0, :3], cen, atol=2e-16)
    et, verts = synth.random_elements(RECT, 5, seed=4)
    cen, _, _ = oracle.geometry(et, verts)
    pq = oracle.points(et, verts, np.ones(5), 3).reshape(5, 17, 4)
    assert np.allclose(pq[:, 0, :3], cen, atol=2e-16)


# ------------------------------------------------------------------ Eq. 4.1 sum

@pytest.mark.parametrize("kind", [TRI, RECT])
def test_far_field_point_charge_limit(kind):
    """Phi -> k q / D and E -> k q (P - Q_cen)/D^3 with relative deviation O(DR^-2) (config 5)."""
    cfg = synth.config5(kind, m=400, seed=5, dr_lo=10.0, dr_hi=1e6)
    cen, area, _ = oracle.geometry(cfg["etype"], cfg["verts"])
    d = cfg["pts"] - cen[0]
    D = np.linalg.norm(d, axis=1)
    for level in (0, 1, 4):
        r = oracle.evaluate(cfg["etype"], cfg["verts"], cfg["sigma"], cfg["pts"], level)
        dev_phi = np.abs(r["phi"] * D / (K * area[0]) - 1.0)
        assert (dev_phi < 0.5 / cfg["ratio"] ** 2 + 5e-10).all()
        Epc = K * area[0] * d / D[:, None] ** 3
        dev_E = np.linalg.norm(r["E"] - Epc, axis=1) / np.linalg.norm(Epc, axis=1)
        assert (dev_E < 1.5 / cfg["ratio"] ** 2 + 5e-10).all()
        assert np.allclose(r["Sphi"], r["phi"], rtol=1e-15) or level == 0     # all q_i > 0 except A1


@pytest.mark.parametrize("a,b", [(1.0, 1.0), (0.7, 0.3)])
def test_rectangle_rules_converge_to_on_axis_closed_form(a, b):
    """The whole chain tables -> Eq. 3.2 mapping -> Eq. 4.1 against the textbook closed form.
    Error decreases with the rule's degree and reaches ~1e-15 (L44) for the high rules."""
    mp.mp.dps = 30
    sigma = np.array([2.5e-9])
    verts = rect_verts(a, b, (0.3, -0.2, 0.1))
    L = (a + b) / 2
    errs = {}
    for dr in (3.0, 8.0, 30.0):
        z = dr * L
        P = np.array([[0.3, -0.2, 0.1 + z]])
        iphi, iez = on_axis_rect(a, b, z)
        for level in range(5):
            r = oracle.evaluate([RECT], verts, sigma, P, level)
            ephi = abs(r["phi"][0] / (K * sigma[0]) - float(iphi)) / float(iphi)
            eez = abs(r["E"][0, 2] / (K * sigma[0]) - float(iez)) / float(iez)
            assert abs(r["E"][0, 0]) < 1e-14 * abs(r["E"][0, 2]) and abs(r["E"][0, 1]) < 1e-14 * abs(r["E"][0, 2])
            errs[(dr, level)] = (ephi, eez)
    # high-order rules at their working distance: double-precision level
    assert max(errs[(8.0, 4)]) < 5e-14 and max(errs[(30.0, 3)]) < 5e-15 and max(errs[(30.0, 4)]) < 5e-15
    # 4-point rule is visibly worse close by, and the error falls with level at DR = 3
    assert errs[(3.0, 0)][0] > 1e-5
    assert errs[(3.0, 0)][0] > errs[(3.0, 1)][0] > errs[(3.0, 2)][0] > errs[(3.0, 4)][0]


def test_triangle_rules_against_rectangle_closed_form():
    """Two triangles tiling a rectangle: their summed cubature potential/field on the
    rectangle's axis equals the closed form (pins the barycentric mapping and Tables A)."""
    mp.mp.dps = 30
    a, b = 0.8, 0.5
    p0 = np.array([-a / 2, -b / 2, 0.0])
    p1, p2, p3 = p0 + [a, 0, 0], p0 + [a, b, 0], p0 + [0, b, 0]
    verts = np.array([[p0, p1, p2], [p0, p2, p3]])
    sigma = np.array([1.0, 1.0])
    for dr, level, tol in ((25.0, 2, 3e-14), (12.0, 3, 2e-13), (12.0, 4, 2e-14), (100.0, 1, 5e-14), (2000.0, 0, 1e-14)):
        z = dr * 0.75
        iphi, iez = on_axis_rect(a, b, z)
        r = oracle.evaluate([TRI, TRI], verts, sigma, np.array([[0, 0, z]]), level)
        assert abs(r["phi"][0] / K - float(iphi)) / float(iphi) < tol
        assert abs(r["E"][0, 2] / K - float(iez)) / float(iez) < 10 * tol


def test_uniform_sphere_config1():
    """Config 1: Phi = k Q_tot / r outside an (almost) uniformly charged sphere.  The flat
    facets of the level-3 icosphere leave multipoles l >= 6 only: deviation <= 2e-5 at r >= 1.5,
    <= 5e-7 at r >= 2.9; E radial with |E| = k Q_tot / r^2."""
    cfg = synth.config1(level=3, m=200)
    _, area, _ = oracle.geometry(cfg["etype"], cfg["verts"])
    Q = float((cfg["sigma"] * area).sum())
    assert abs(area.sum() / (4 * math.pi) - 0.995235) < 2e-6          # facet area deficit
    r = oracle.evaluate(cfg["etype"], cfg["verts"], cfg["sigma"], cfg["pts"], 1)
    rad = np.linalg.norm(cfg["pts"], axis=1)
    dev = np.abs(r["phi"] * rad / (K * Q) - 1.0)
    assert dev.max() < 2e-5 and dev[rad > 2.9].max() < 5e-7
    Er = np.einsum("ij,ij->i", r["E"], cfg["pts"]) / rad
    assert np.abs(Er * rad ** 2 / (K * Q) - 1.0).max() < 2e-4
    Et = r["E"] - Er[:, None] * cfg["pts"] / rad[:, None]
    assert (np.linalg.norm(Et, axis=1) < 2e-4 * np.abs(Er)).all()
    # exact sphere sigma R^2/(eps0 r) only up to the area deficit (BASELINE.json config 1)
    eps0 = 1.0 / (4 * math.pi * K)
    exact = 1e-9 / (eps0 * rad)
    assert np.abs(r["phi"] / exact - 0.995235).max() < 3e-5


@pytest.mark.parametrize("level", [-1, 1, 3])
def test_field_is_minus_gradient_of_potential(level):
    """E = -grad Phi holds exactly for the discrete sum of Eq. 4.1 (central differences)."""
    cfg = synth.config2(nside=4, m=12)
    dr = oracle.default_policy(True)
    h = 1e-5
    r0 = oracle.evaluate(cfg["etype"], cfg["verts"], cfg["sigma"], cfg["pts"], level, dr=dr)
    grad = np.zeros((12, 3))
    for ax in range(3):
        e = np.zeros(3)
        e[ax] = h
        rp = oracle.evaluate(cfg["etype"], cfg["verts"], cfg["sigma"], cfg["pts"] + e, level, dr=dr)
        rm = oracle.evaluate(cfg["etype"], cfg["verts"], cfg["sigma"], cfg["pts"] - e, level, dr=dr)
        grad[:, ax] = (rp["phi"] - rm["phi"]) / (2 * h)
    scale = r0["SE"]
    assert (np.abs(r0["E"] + grad).max(axis=1) < 2e-8 * scale).all()


def test_parity_denominators_and_counts():
    """Sphi = k sum |q_i|/r_i and SE = k sum |q_i|/r_i^2: equal to Phi for positive charges,
    invariant under sign flips of sigma, and >= |Phi|, |E|; npi = n*N for a fixed rule."""
    cfg = synth.config2(nside=3, m=7)
    pos = np.abs(cfg["sigma"])
    a = oracle.evaluate(cfg["etype"], cfg["verts"], pos, cfg["pts"], 2, want_counts=True)
    b = oracle.evaluate(cfg["etype"], cfg["verts"], cfg["sigma"], cfg["pts"], 2)
    assert np.allclose(a["Sphi"], a["phi"], rtol=1e-15)
    assert np.allclose(a["Sphi"], b["Sphi"], rtol=1e-15) and np.allclose(a["SE"], b["SE"], rtol=1e-15)
    assert (np.abs(b["phi"]) <= b["Sphi"]).all() and (np.linalg.norm(b["E"], axis=1) <= b["SE"] * (1 + 1e-15)).all()
    assert (a["npi"] == 54 * 12).all()


def test_double_instantiation_matches_long_double():
    cfg = synth.config1(level=1, m=50)
    a = oracle.evaluate(cfg["etype"], cfg["verts"], cfg["sigma"], cfg["pts"], 1)
    b = oracle.evaluate(cfg["etype"], cfg["verts"], cfg["sigma"], cfg["pts"], 1, precision="double")
    assert np.abs(a["phi"] - b["phi"]).max() < 1e-13 * a["Sphi"].max()
    assert np.abs(a["E"] - b["E"]).max() < 1e-13 * a["SE"].max()


def test_linearity_in_sigma_and_element_order():
    cfg = synth.config2(nside=2, m=5)
    r1 = oracle.evaluate(cfg["etype"], cfg["verts"], cfg["sigma"], cfg["pts"], 4)
    r2 = oracle.evaluate(cfg["etype"], cfg["verts"], 3.0 * cfg["sigma"], cfg["pts"], 4)
    assert np.allclose(r2["phi"], 3.0 * r1["phi"], rtol=1e-14, atol=0)
    perm = np.random.default_rng(0).permutation(len(cfg["etype"]))
    r3 = oracle.evaluate(cfg["etype"][perm], cfg["verts"][perm], cfg["sigma"][perm], cfg["pts"], 4)
    assert np.abs(r3["E"] - r1["E"]).max() < 1e-15 * r1["SE"].max()


# ------------------------------------------------------------------ analytic / GL2 / adaptive

def test_analytic_closed_forms():
    mp.mp.dps = 30
    sq = rect_verts(1.0, 1.0)[0]
    ip, ie = oracle.analytic(RECT, sq, [0, 0, 0])
    assert abs(ip - float(4 * mp.log(1 + mp.sqrt(2)))) < 2e-15 and np.abs(ie).max() < 1e-15
    a = 0.37
    tri = np.array([[0, 0, 0], [a, 0, 0], [a / 2, a * math.sqrt(3) / 2, 0]])
    ip, ie = oracle.analytic(TRI, tri, tri.mean(axis=0))
    assert abs(ip - float(mp.sqrt(3) * a * mp.log(2 + mp.sqrt(3)))) < 1e-15 and np.abs(ie).max() < 1e-14
    for (ra, rb, z) in ((1.0, 1.0, 0.3), (2.0, 0.4, 1.5), (0.05, 0.03, 0.002), (1.0, 1.0, 40.0)):
        iphi, iez = on_axis_rect(ra, rb, z)
        for sgn in (1.0, -1.0):
            ip, ie = oracle.analytic(RECT, rect_verts(ra, rb)[0], [0, 0, sgn * z])
            assert abs(ip - float(iphi)) < 1e-14 * float(iphi)
            assert abs(ie[2] - sgn * float(iez)) < 1e-13 * float(iez) + 1e-18
            assert abs(ie[0]) + abs(ie[1]) < 1e-13 * float(iez)


def test_analytic_orientation_and_vertex_order_independent():
    et, verts = synth.random_elements(TRI, 6, seed=8)
    P = np.array([0.3, 0.9, 0.4])
    for v in verts:
        a = oracle.analytic(TRI, v, P)
        b = oracle.analytic(TRI, v[[0, 2, 1]], P)
        c = oracle.analytic(TRI, v[[1, 2, 0]], P)
        for o in (b, c):
            assert abs(o[0] - a[0]) < 1e-15 * abs(a[0]) and np.abs(o[1] - a[1]).max() < 1e-14 * np.linalg.norm(a[1])


@pytest.mark.parametrize("kind", [TRI, RECT])
def test_analytic_equals_gl2_for_dr_2_to_5(kind):
    """GL2 with 16 nodes is double-precision accurate above DR = 2 and does
    not change with the number of nodes; the analytic formula agrees with it there."""
    et, verts = synth.random_elements(kind, 40, seed=21 + kind)
    cen, _, L = oracle.geometry(et, verts)
    rng = np.random.default_rng(5)
    dirs = synth.isotropic_directions(rng, 40)
    worst = 0.0
    for e in range(40):
        for dr in (2.0, 3.0, 5.0):
            P = cen[e] + dirs[e] * dr * L[e]
            a = oracle.analytic(kind, verts[e], P)
            g16 = oracle.gl2(kind, verts[e], P, 16)
            g32 = oracle.gl2(kind, verts[e], P, 32)
            en = np.linalg.norm(g32[1])
            worst = max(worst, abs(g16[0] - g32[0]) / g32[0], np.abs(g16[1] - g32[1]).sum() / en)
            assert abs(a[0] - g32[0]) < 2e-14 * g32[0]
            assert np.abs(a[1] - g32[1]).sum() < 2e-13 * en
    assert worst < 1e-13 if kind == TRI else worst < 1e-14


@pytest.mark.parametrize("kind", [TRI, RECT])
def test_analytic_equals_adaptive_quadrature_near_field(kind):
    """Brute force on tiny inputs, including DR < 1 where GL2 is not reliable (L78)."""
    cfg5 = synth.config5(kind, m=1)
    v = cfg5["verts"][0]
    cen, _, L = oracle.geometry([kind], cfg5["verts"])
    pts = [cen[0] + np.array(d) * L[0] for d in
           ((0.05, 0.02, 0.12), (0.3, -0.1, 0.25), (-0.6, 0.5, -0.4), (1.2, 0.3, 0.05), (0.1, 0.1, 2.5), (0.9, -0.9, -0.03))]
    for P in pts:
        a = oracle.analytic(kind, v, P)
        q = oracle.adaptive(kind, v, P, 1e-17)
        assert abs(a[0] - q[0]) < 3e-15 * abs(q[0])
        assert np.abs(a[1] - q[1]).max() < 3e-14 * np.linalg.norm(q[1])


def test_analytic_field_is_minus_gradient():
    v = synth.CFG5_TRIANGLE[0]
    for P in ([0.2, 0.3, 0.15], [1.4, -0.2, 0.0], [0.5, 0.4, -0.6]):
        P = np.array(P)
        _, ie = oracle.analytic(TRI, v, P)
        h = 1e-5
        g = np.array([(oracle.analytic(TRI, v, P + h * np.eye(3)[k])[0] - oracle.analytic(TRI, v, P - h * np.eye(3)[k])[0]) / (2 * h)
                      for k in range(3)])
        mask = np.ones(3, bool)
        if P[2] == 0.0:
            mask[2] = False          # in-plane outside point: E_normal = 0 by symmetry
            assert ie[2] == 0.0
        assert np.abs(ie + g)[mask].max() < 1e-8 * np.linalg.norm(ie)


def test_analytic_in_plane_and_edge_line_cases():
    """h = 0: self term and coplanar neighbours (matrix fill); P on the extension of an edge."""
    v = synth.CFG5_TRIANGLE[0]
    ip, ie = oracle.analytic(TRI, v, v.mean(axis=0))
    assert abs(ip - 2.18358707571485765681) < 2e-15           # SURVEY.md §8(c) 30-digit value
    # P on the line of edge AB beyond B: finite, continuous with its neighbourhood
    P = np.array([1.5, 0.0, 0.0])
    ip0, ie0 = oracle.analytic(TRI, v, P)
    ip1, _ = oracle.analytic(TRI, v, P + [0, 1e-9, 0])
    q = oracle.adaptive(TRI, v, P, 1e-16)
    assert np.isfinite(ip0) and np.isfinite(ie0).all()
    assert abs(ip0 - ip1) < 1e-8 and abs(ip0 - q[0]) < 1e-14 * q[0]
    assert np.abs(ie0 - q[1]).max() < 1e-13 * np.linalg.norm(q[1])


# ------------------------------------------------------------------ distance-ratio policy

def test_printed_dr_limits_are_the_potential_policy():
    rows = read_golden("paper_dr_limits.txt")
    dr = oracle.default_policy(False)
    level_of_N = {4: 0, 7: 1, 12: 2, 19: 3, 33: 4, 0: 5}
    for method, lo, hi in rows:
        lv = level_of_N[int(method)]
        lo = float(lo)
        hi = float("inf") if hi == "inf" else float(hi)
        for t in (TRI, RECT):
            L = 0.37
            probe = [max(lo, 1e-3) * 1.0000001, (lo + min(hi, 1e5)) / 2] + ([hi * 0.9999999] if hi < 1e300 else [1e9])
            for d in probe:
                assert oracle.choose_level((d * L) ** 2, L, dr[t]) == lv
            # lower-inclusive band edges (reading 8)
            if lo > 0:
                assert oracle.choose_level((lo * L) ** 2, L, dr[t]) == lv
    fdr = oracle.default_policy(True)
    assert (fdr >= dr).all() and (fdr[:, 0] > dr[:, 0]).all()       # "slightly higher" for the field (L159)


def test_levels_mask_moves_to_more_accurate_rule():
    dr = oracle.default_policy(False)[0]
    L = 1.0
    assert oracle.choose_level(30.0 ** 2, L, dr) == 2
    assert oracle.choose_level(30.0 ** 2, L, dr, 0b110010) == 4      # paper's GPU integrator: 7/33/analytic
    assert oracle.choose_level(30.0 ** 2, L, dr, 0b110110) == 2      # 7/12/33 + analytic (L239)
    assert oracle.choose_level(5000.0 ** 2, L, dr, 0b110110) == 1
    assert oracle.choose_level(1.0, L, dr, 0b011111) == 4            # analytic disabled -> N=33


def test_dr_limits_reach_printed_accuracy_level():
    """Soft pin (L159): averaged over random triangles, N = 4/7/12/19/33 at DR = 1500/80/20/8/3
    reach the ~2e-15 level for the potential (GL2-32 in long double as reference); one band
    lower (at a third of the limit) the same rule is clearly worse."""
    et, verts = synth.random_elements(TRI, 200, seed=99)
    cen, _, L = oracle.geometry(et, verts)
    dirs = synth.isotropic_directions(np.random.default_rng(7), 200)
    for level, lim in ((0, 1500.0), (1, 80.0), (2, 20.0), (3, 8.0), (4, 3.0)):
        errs, errs_close = [], []
        for e in range(200):
            for fac, store in ((1.0, errs), (1.0 / 3.0, errs_close)):
                P = cen[e] + dirs[e] * lim * fac * L[e]
                if fac < 1 and level == 4:
                    ref = oracle.analytic(TRI, verts[e], P)[0]
                else:
                    ref = oracle.gl2(TRI, verts[e], P, 32)[0]
                r = oracle.evaluate([TRI], verts[e:e + 1], np.ones(1), P[None, :], level)
                store.append(abs(r["phi"][0] / K - ref) / ref)
        assert np.mean(errs) < 6e-15, (level, np.mean(errs))
        assert np.mean(errs_close) > 20 * np.mean(errs)


@pytest.mark.parametrize("kind", [TRI, RECT])
def test_field_dr_limits_by_the_papers_protocol(kind):
    """Pin of the shipped Phi+E limits (reading 7; L159: for the field the limits are
    'slightly higher', and 'if both the potential and the field has to be computed ... one should use
    the limits defined by the field').  The paper's protocol (L68, L149): 1000 random elements with
    corners in the unit cube, a random direction each, mean of err(Phi) = |dPhi/Phi| and err(E) =
    sum_j |dE_j| / |E| (L80), double arithmetic for the rule, exact reference in long double (closed
    form below DR = 12, the 33-point rule above).  At every shipped limit the rule that takes over
    there is at the paper's 2e-15 level for the FIELD as well (<= 3e-15; potential <= 5e-16), and the
    limits are not slack: 40 % nearer every rule is above that level, 20 % nearer all but the
    rectangle N = 4 rule."""
    fdr = oracle.default_policy(True)[kind]
    n = 1000
    et, verts = synth.random_elements(kind, n, seed=1234 + kind)
    cen, _, L = oracle.geometry(et, verts)
    dirs = synth.isotropic_directions(np.random.default_rng(77 + kind), n)

    def mean_errors(level, ratio):
        P = cen + dirs * (ratio * L)[:, None]
        ref = oracle.evaluate_pairs(et, verts, P, 5 if ratio < 12.0 else 4)
        r = oracle.evaluate_pairs(et, verts, P, level, precision="double")
        e_phi = np.abs(r["phi"] - ref["phi"]) / np.abs(ref["phi"])
        e_E = np.abs(r["E"] - ref["E"]).sum(axis=1) / np.linalg.norm(ref["E"], axis=1)
        return float(e_phi.mean()), float(e_E.mean())

    for band, level in ((4, 0), (3, 1), (2, 2), (1, 3), (0, 4)):       # dr[band] = lower end of `level`'s range
        lim = float(fdr[band])
        e_phi, e_E = mean_errors(level, lim)
        assert e_phi <= 5e-16 and e_E <= 3e-15, (kind, level, lim, e_phi, e_E)
        _, e_E_06 = mean_errors(level, 0.6 * lim)
        assert e_E_06 > 3e-15, (kind, level, 0.6 * lim, e_E_06)
        if not (kind == RECT and level == 0):
            _, e_E_08 = mean_errors(level, 0.8 * lim)
            assert e_E_08 > 3e-15, (kind, level, 0.8 * lim, e_E_08)
    # and they are the same numbers the header of the C ABI promises
    expect = {TRI: [4, 10, 25, 100, 2000], RECT: [6, 15, 40, 150, 3000]}[kind]
    assert list(fdr) == expect


@pytest.mark.parametrize("kind", [TRI, RECT])
def test_single_precision_limits_sit_at_the_fp32_floor(kind):
    """want_field = 2: at each limit the rule that takes over has a field error (long-double arithmetic,
    i.e. the rule's own truncation error) at or below the FP32 rounding floor of 1e-7, and is above it
    40 % nearer - so in FP32 the more accurate rule would buy nothing there."""
    dr32 = oracle.default_policy(2)[kind]
    assert np.all(np.diff(dr32) >= 0) and np.all(dr32 <= oracle.default_policy(True)[kind])
    n = 1000
    et, verts = synth.random_elements(kind, n, seed=4321 + kind)
    cen, _, L = oracle.geometry(et, verts)
    dirs = synth.isotropic_directions(np.random.default_rng(78 + kind), n)

    def field_error(level, ratio):
        P = cen + dirs * (ratio * L)[:, None]
        ref = oracle.evaluate_pairs(et, verts, P, 5 if ratio < 12.0 else 4)
        r = oracle.evaluate_pairs(et, verts, P, level)
        return float((np.abs(r["E"] - ref["E"]).sum(axis=1) / np.linalg.norm(ref["E"], axis=1)).mean())

    for band, level in ((4, 0), (3, 1), (2, 2), (1, 3), (0, 4)):
        lim = float(dr32[band])
        if band < 4 and lim == float(dr32[band + 1]):
            continue                                  # empty range [dr[band], dr[band + 1]): this rule is never chosen
        assert field_error(level, lim) <= 1.3e-7, (kind, level, lim, field_error(level, lim))
        assert field_error(level, 0.6 * lim) > 1.3e-7, (kind, level, 0.6 * lim)


def test_adaptive_sum_uses_per_pair_rule():
    """Adaptive evaluation = sum over elements of the fixed-rule value at the level the policy
    picks per pair; point-interaction counts follow; the analytic branch is taken below the
    first limit."""
    cfg = synth.config2(nside=3, m=6)
    pts = np.concatenate([cfg["pts"], [[0.51, 0.1, 0.1], [0.0, 0.0, 0.9]]])
    et, verts, sigma = cfg["etype"], cfg["verts"], cfg["sigma"]
    dr = oracle.default_policy(True)
    cen, _, L = oracle.geometry(et, verts)
    full = oracle.evaluate(et, verts, sigma, pts, -1, dr=dr, want_counts=True)
    total = np.zeros(len(pts))
    counts = np.zeros(len(pts), dtype=np.int64)
    n_analytic = 0
    for e in range(len(et)):
        for j, P in enumerate(pts):
            lv = oracle.choose_level(float(((P - cen[e]) ** 2).sum()), L[e], dr[1])
            if lv == 5:
                total[j] += K * sigma[e] * oracle.analytic(RECT, verts[e], P)[0]
                n_analytic += 1
            else:
                total[j] += oracle.evaluate(et[e:e + 1], verts[e:e + 1], sigma[e:e + 1], P[None], lv)["phi"][0]
                counts[j] += RECT_N[lv]
    assert n_analytic > 0
    assert np.abs(total - full["phi"]).max() < 1e-14 * full["Sphi"].max()
    assert (counts == full["npi"]).all()


# ------------------------------------------------------------------ collocation matrix rows

def test_matrix_rows_sphere():
    """Rows of the collocation matrix of an icosphere with unit sigma: the row sum is the
    potential of the (almost) uniformly charged sphere at its own surface, R/eps0, up to the
    discretisation (~1e-2 at level 2); self terms are analytic and close to the equilateral
    closed form sqrt3 a ln(2+sqrt3) for near-equilateral facets; near entries analytic, far
    entries by cubature, all positive."""
    et, verts = synth.icosphere_elements(2, 1.0)
    n = len(et)
    dr = oracle.default_policy(False)
    rows = np.array([0, 17, n - 1])
    A, code = oracle.assemble_rows(et, verts, rows, dr)
    eps0 = 1.0 / (4 * math.pi * K)
    assert np.abs(A.sum(axis=1) * eps0 - 1.0).max() < 2e-2
    assert (A > 0).all()
    cen, area, L = oracle.geometry(et, verts)
    for r, i in enumerate(rows):
        assert code[r, i] == 5
        a_eq = math.sqrt(4 * area[i] / math.sqrt(3))
        assert abs(A[r, i] / K / (math.sqrt(3) * a_eq * math.log(2 + math.sqrt(3))) - 1.0) < 0.02
        D = np.linalg.norm(cen - cen[i], axis=1)
        ana = code[r] == 5
        assert (D[ana] < 3 * L[ana]).all() and (D[~ana] >= 3 * L[~ana]).all()
        # far entries ~ k * area / D
        far = D > 20 * L
        if far.any():
            assert np.abs(A[r, far] * D[far] / (K * area[far]) - 1.0).max() < 1e-3
    # each entry equals the single-element potential at the centroid (Eq. 4.1 with unit sigma)
    j = 5
    lv = int(code[1, j])
    if lv < 5:
        v = oracle.evaluate(et[j:j + 1], verts[j:j + 1], np.ones(1), cen[17][None], lv)["phi"][0]
        assert abs(v - A[1, j]) < 1e-15 * v
