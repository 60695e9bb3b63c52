"""-m gpu: the few-field-point path (m <= 64: elements across the lanes, per-pair rule choice, partial sums
combined with warp shuffles).  Per-pair choice means the result must match the per-pair oracle whatever
allow_upgrade says, and the interaction counters must match it exactly."""
from __future__ import annotations

import numpy as np
import pytest

import oracle
from paper_1606_03743_b200 import synth
from gpu_common import TOL_F64, Gpu, parity_errors

pytestmark = pytest.mark.gpu


@pytest.mark.parametrize("m", [1, 2, 3, 4, 5, 13, 16, 32, 63, 64])
def test_adaptive_few_points_incl_near_field(m):
    c = synth.config4(scale=0.003, ntracks=8, npts_per_track=9)
    rng = np.random.default_rng(100 + m)
    pts = c["pts"][rng.choice(len(c["pts"]), m, replace=False)].copy()
    # pull one point close to the wall so that the analytic branch and N = 33 / 19 are exercised
    cen = synth.element_centroids(c["etype"], c["verts"])
    pts[0] = cen[len(cen) // 3] * (1.0 - 0.004)
    g = Gpu(c["etype"], c["verts"])
    pol = g.b.bemcub_default_policy(True)
    ref = oracle.evaluate(c["etype"], c["verts"], c["sigma"], pts, -1, dr=oracle.default_policy(True), want_counts=True)
    for want_E in (True, False):
        phi, E = g.eval(c["sigma"], pts, -1, policy=pol, want_E=want_E)
        err = parity_errors(phi, E, ref)
        assert err["phi"] <= 1e-10 and err.get("E", 0.0) <= 1e-10, (m, want_E, err)    # analytic pairs: 1e-10
        assert ref["nana"][0] > 0
        far = np.flatnonzero(ref["nana"] == 0)                                          # no analytic pair: 1e-12
        if len(far):
            sub = {k: v[far] for k, v in ref.items()}
            e2 = parity_errors(phi[far], None if E is None else E[far], sub)
            assert e2["phi"] <= TOL_F64 and e2.get("E", 0.0) <= TOL_F64, (m, e2)
    st = g.stats()
    assert st["point_interactions"] == int(ref["npi"].sum())
    assert st["analytic_pairs"] > 0
    g.close()


@pytest.mark.parametrize("level", [0, 3, 4])
def test_fixed_rule_few_points_mixed_mesh(level):
    et, vt = synth.random_elements(synth.TRI, 333, 51)
    er, vr = synth.random_elements(synth.RECT, 222, 52)
    etype, verts = np.concatenate([et, er]), np.concatenate([vt, vr])
    rng = np.random.default_rng(53)
    sigma = rng.uniform(-1, 1, len(etype))
    pts = 3.0 + 2.0 * rng.random((7, 3))
    g = Gpu(etype, verts)
    phi, E = g.eval(sigma, pts, level)
    err = parity_errors(phi, E, oracle.evaluate(etype, verts, sigma, pts, level))
    assert err["phi"] <= TOL_F64 and err["E"] <= TOL_F64, err
    nt, nr = oracle.rule_info(0, level)[0], oracle.rule_info(1, level)[0]
    assert g.stats()["point_interactions"] == (333 * nt + 222 * nr) * 7
    g.close()


@pytest.mark.parametrize("m", [1, 2, 7])
def test_few_point_calls_are_bit_reproducible(m):
    """The CTAs of eval_few_kernel finish in any order; the last one of a pass adds their sums in CTA
    order, so repeated calls return the same bits."""
    c = synth.config4(scale=0.02, ntracks=3, npts_per_track=5)
    g = Gpu(c["etype"], c["verts"])
    pol = g.b.bemcub_default_policy(True)
    pts = c["pts"][:m].copy()
    a_phi, a_E = g.eval(c["sigma"], pts, -1, policy=pol)
    for _ in range(4):
        b_phi, b_E = g.eval(c["sigma"], pts, -1, policy=pol)
        assert np.array_equal(a_phi, b_phi) and np.array_equal(a_E, b_E)
    g.close()


@pytest.mark.parametrize("n_el", [1, 2, 33])
@pytest.mark.parametrize("m", [1, 2, 3])
def test_tiny_meshes_few_points(n_el, m):
    """Fewer elements than threads (most CTAs of eval_few_kernel have nothing to add, the last one still
    sums all of them), triangles and rectangles mixed, every rule level and the distance-ratio choice."""
    et, vt = synth.random_elements(synth.TRI, n_el, 71)
    er, vr = synth.random_elements(synth.RECT, n_el, 72)
    etype, verts = np.concatenate([et, er]), np.concatenate([vt, vr])
    rng = np.random.default_rng(73 + m)
    sigma = rng.uniform(-1, 1, len(etype))
    pts = 2.0 + 3.0 * rng.random((m, 3))
    g = Gpu(etype, verts)
    for level in (0, 1, 2, 3, 4):
        phi, E = g.eval(sigma, pts, level)
        err = parity_errors(phi, E, oracle.evaluate(etype, verts, sigma, pts, level))
        assert err["phi"] <= TOL_F64 and err["E"] <= TOL_F64, (level, err)
    pol = g.b.bemcub_default_policy(True)
    ref = oracle.evaluate(etype, verts, sigma, pts, -1, dr=oracle.default_policy(True), want_counts=True)
    phi, E = g.eval(sigma, pts, -1, policy=pol)
    err = parity_errors(phi, E, ref)
    assert err["phi"] <= 1e-10 and err["E"] <= 1e-10, err
    assert g.stats()["point_interactions"] == int(ref["npi"].sum())
    g.close()


def test_sigma_null_reuses_the_charges_of_the_previous_call():
    c = synth.config4(scale=0.003, ntracks=12, npts_per_track=9)       # 108 points: the tiled path
    g = Gpu(c["etype"], c["verts"])
    torch, b = g.torch, g.b
    h = g.ctx.handle
    pol = b.bemcub_default_policy(True)
    d_sigma = torch.as_tensor(c["sigma"]).cuda()
    pts = c["pts"]
    d_all = torch.as_tensor(pts).cuda()
    m = len(pts)
    phi = torch.empty(m, dtype=torch.float64, device="cuda")
    E = torch.empty((m, 3), dtype=torch.float64, device="cuda")
    # no charges yet: error
    with pytest.raises(Exception):
        b.bemcub_eval(h, None, -1, pol, m, d_all, phi, E, b.F64)
    b.bemcub_eval(h, d_sigma, -1, pol, m, d_all, phi, E, b.F64)
    first = (phi.clone(), E.clone())
    launches_full = g.stats()["last_eval_launches"]
    # same call without sigma: identical bits, fewer launches (no expansion)
    b.bemcub_eval(h, None, -1, pol, m, d_all, phi, E, b.F64)
    torch.cuda.synchronize()
    assert torch.equal(phi, first[0]) and torch.equal(E, first[1])
    assert g.stats()["last_eval_launches"] < launches_full
    # point by point, as a tracker would: parity with the oracle
    ref = oracle.evaluate(c["etype"], c["verts"], c["sigma"], pts[:5], -1, dr=oracle.default_policy(True))
    for j in range(5):
        p1 = torch.empty(1, dtype=torch.float64, device="cuda")
        e1 = torch.empty((1, 3), dtype=torch.float64, device="cuda")
        b.bemcub_eval(h, None, -1, pol, 1, d_all[j:j + 1].contiguous(), p1, e1, b.F64)
        torch.cuda.synchronize()
        assert abs(p1.item() - ref["phi"][j]) <= TOL_F64 * ref["Sphi"][j]
        assert np.max(np.abs(e1.cpu().numpy()[0] - ref["E"][j])) <= TOL_F64 * ref["SE"][j]
    # another rule with the kept sigma: its level is expanded on demand
    b.bemcub_eval(h, None, 3, None, m, d_all, phi, E, b.F64)
    torch.cuda.synchronize()
    ref3 = oracle.evaluate(c["etype"], c["verts"], c["sigma"], pts, 3)
    err = parity_errors(phi.cpu().numpy(), E.cpu().numpy(), ref3)
    assert err["phi"] <= TOL_F64 and err["E"] <= TOL_F64, err
    # few points with the kept sigma: on the fly (nothing expanded for level 0) and from kept points (level 3) agree with the oracle
    for level in (0, 3):
        p4 = torch.empty(4, dtype=torch.float64, device="cuda")
        e4 = torch.empty((4, 3), dtype=torch.float64, device="cuda")
        b.bemcub_eval(h, None, level, None, 4, d_all[:4].contiguous(), p4, e4, b.F64)
        torch.cuda.synchronize()
        r4 = oracle.evaluate(c["etype"], c["verts"], c["sigma"], pts[:4], level)
        e = parity_errors(p4.cpu().numpy(), e4.cpu().numpy(), r4)
        assert e["phi"] <= TOL_F64 and e["E"] <= TOL_F64, (level, e)
    # a new mesh drops the kept sigma
    b.bemcub_set_elements(h, g.n, g.d_type, g.d_verts)
    with pytest.raises(Exception):
        b.bemcub_eval(h, None, 1, None, m, d_all, phi, E, b.F64)
    g.close()
