"""-m gpu parity of bemcub_eval_linear (charge density linear over each element) with the
oracle; same bar as the constant-sigma path."""
from __future__ import annotations

import numpy as np
import pytest

import oracle
from paper_1606_03743_b200 import synth
from gpu_common import TOL_F32, TOL_F64, Gpu, parity_errors

pytestmark = pytest.mark.gpu


def run_linear(g, sigma_v, pts, rule, policy=None, precision=0):
    torch, b = g.torch, g.b
    m = len(pts)
    d_sv = torch.as_tensor(np.ascontiguousarray(sigma_v)).cuda()
    d_pts = torch.as_tensor(np.ascontiguousarray(pts)).cuda()
    phi = torch.full((m,), float("nan"), dtype=torch.float64, device="cuda")
    E = torch.full((m, 3), float("nan"), dtype=torch.float64, device="cuda")
    b.bemcub_eval_linear(g.ctx.handle, d_sv, rule, policy, m, d_pts, phi, E, precision)
    torch.cuda.synchronize()
    return phi.cpu().numpy(), E.cpu().numpy()


def _mixed(n_tri, n_rect):
    et, vt = synth.random_elements(synth.TRI, n_tri, 41)
    er, vr = synth.random_elements(synth.RECT, n_rect, 42)
    return np.concatenate([et, er]), np.concatenate([vt, vr])


@pytest.mark.parametrize("precision", [0, 1])
@pytest.mark.parametrize("level", [0, 1, 2, 3, 4])
def test_fixed_rules_mixed_mesh(level, precision):
    etype, verts = _mixed(301, 215)
    rng = np.random.default_rng(7)
    sv = rng.uniform(-1.0, 1.0, (len(etype), 3))
    pts = 3.0 + 4.0 * rng.random((777, 3))
    g = Gpu(etype, verts)
    phi, E = run_linear(g, sv, pts, level, precision=precision)
    err = parity_errors(phi, E, oracle.evaluate_linear(etype, verts, sv, pts, level))
    tol = TOL_F32 if precision else TOL_F64
    assert err["phi"] <= tol and err["E"] <= tol, err
    g.close()


@pytest.mark.parametrize("allow_upgrade", [0, 1])
def test_adaptive_cfg4_small(allow_upgrade):
    c = synth.config4(scale=0.002, ntracks=40, npts_per_track=53)
    n = len(c["etype"])
    rng = np.random.default_rng(8)
    sv = c["sigma"][:, None] * (1.0 + 0.3 * rng.uniform(-1.0, 1.0, (n, 3)))
    g = Gpu(c["etype"], c["verts"])
    pol = g.b.bemcub_default_policy(True)
    pol.allow_upgrade = allow_upgrade
    pol.use_levels_mask = 0b011111
    phi, E = run_linear(g, sv, c["pts"], -1, policy=pol)
    ref = oracle.evaluate_linear(c["etype"], c["verts"], sv, c["pts"], -1, dr=oracle.default_policy(True), levels_mask=0b011111)
    err = parity_errors(phi, E, ref)
    assert err["phi"] <= TOL_F64 and err["E"] <= TOL_F64, err
    # the analytic branch is for constant sigma only
    bad = g.b.bemcub_default_policy(True)
    with pytest.raises(Exception):
        run_linear(g, sv, c["pts"], -1, policy=bad)
    g.close()


@pytest.mark.parametrize("m", [1, 4, 5, 64])
def test_few_field_points_take_the_shuffle_path(m):
    """m <= 64 dispatches bemcub_eval_linear to eval_few_kernel (elements across the lanes, points on the
    fly with the linear density, per-pair rule): fixed rule and the distance-ratio choice."""
    c = synth.config4(scale=0.003, ntracks=8, npts_per_track=9)
    n = len(c["etype"])
    rng = np.random.default_rng(60 + m)
    sv = c["sigma"][:, None] * (1.0 + 0.3 * rng.uniform(-1.0, 1.0, (n, 3)))
    pts = c["pts"][rng.choice(len(c["pts"]), m, replace=False)].copy()
    g = Gpu(c["etype"], c["verts"])
    for level in (1, 4):
        phi, E = run_linear(g, sv, pts, level)
        assert g.stats()["last_eval_launches"] == 1                       # eval_few_kernel alone (its last CTA adds the CTAs)
        err = parity_errors(phi, E, oracle.evaluate_linear(c["etype"], c["verts"], sv, pts, level))
        assert err["phi"] <= TOL_F64 and err["E"] <= TOL_F64, (m, level, err)
    pol = g.b.bemcub_default_policy(True)
    pol.use_levels_mask = 0b011111
    for up in (0, 1):                                                      # no effect on this path: per-pair rule
        pol.allow_upgrade = up
        phi, E = run_linear(g, sv, pts, -1, policy=pol)
        ref = oracle.evaluate_linear(c["etype"], c["verts"], sv, pts, -1, dr=oracle.default_policy(True), levels_mask=0b011111)
        err = parity_errors(phi, E, ref)
        assert err["phi"] <= TOL_F64 and err["E"] <= TOL_F64, (m, up, err)
    g.close()
