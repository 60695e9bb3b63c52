"""-m gpu parity of bemcub_eval_gradient (field gradient from the point charges) against
the oracle: max_ab |dG_ab| <= 1e-12 * k sum|q_i|/r_i^3 per field point; Phi and E of the same call keep
their own bar."""
from __future__ import annotations

import numpy as np
import pytest

import oracle
from paper_1606_03743_b200 import synth
from gpu_common import TOL_F64, Gpu, parity_errors

pytestmark = pytest.mark.gpu


def run_grad(g, sigma, pts, rule, policy=None, want_phiE=True):
    torch, b = g.torch, g.b
    m = len(pts)
    d_sigma = torch.as_tensor(np.ascontiguousarray(sigma)).cuda()
    d_pts = torch.as_tensor(np.ascontiguousarray(pts)).cuda()
    phi = torch.full((m,), float("nan"), dtype=torch.float64, device="cuda") if want_phiE else None
    E = torch.full((m, 3), float("nan"), dtype=torch.float64, device="cuda") if want_phiE else None
    G = torch.full((m, 6), float("nan"), dtype=torch.float64, device="cuda")
    b.bemcub_eval_gradient(g.ctx.handle, d_sigma, rule, policy, m, d_pts, phi, E, G)
    torch.cuda.synchronize()
    return (phi.cpu().numpy() if want_phiE else None, E.cpu().numpy() if want_phiE else None, G.cpu().numpy())


def check(G, ref):
    assert np.all(np.isfinite(G))
    err = float((np.abs(G - ref["G"]).max(axis=1) / ref["SG"]).max())
    assert err <= TOL_F64, err
    return err


@pytest.mark.parametrize("level", [0, 1, 2, 3, 4])
def test_cfg2_fixed_rules(level):
    c = synth.config2()
    g = Gpu(c["etype"], c["verts"])
    phi, E, G = run_grad(g, c["sigma"], c["pts"], level)
    check(G, oracle.evaluate_gradient(c["etype"], c["verts"], c["sigma"], c["pts"], level))
    err = parity_errors(phi, E, oracle.evaluate(c["etype"], c["verts"], c["sigma"], c["pts"], level))
    assert err["phi"] <= TOL_F64 and err["E"] <= TOL_F64
    assert np.all(np.abs(G[:, :3].sum(axis=1)) <= 1e-15 * np.abs(G).max(axis=1) + 1e-300)   # traceless
    g.close()


@pytest.mark.parametrize("n_tri,n_rect,m", [(1, 0, 1), (3, 2, 33), (129, 70, 257), (700, 613, 1031)])
def test_ragged_shapes(n_tri, n_rect, m):
    et, vt = synth.random_elements(synth.TRI, n_tri, 11)
    er, vr = synth.random_elements(synth.RECT, n_rect, 12)
    etype, verts = np.concatenate([et, er]), np.concatenate([vt, vr])
    rng = np.random.default_rng(13)
    sigma = rng.uniform(-1, 1, len(etype))
    pts = 3.0 + 4.0 * rng.random((m, 3))
    g = Gpu(etype, verts)
    _, _, G = run_grad(g, sigma, pts, 1, want_phiE=False)
    check(G, oracle.evaluate_gradient(etype, verts, sigma, pts, 1))
    g.close()


@pytest.mark.parametrize("allow_upgrade", [0, 1])
def test_cfg4_small_adaptive(allow_upgrade):
    c = synth.config4(scale=0.002, ntracks=40, npts_per_track=53)
    g = Gpu(c["etype"], c["verts"])
    pol = g.b.bemcub_default_policy(True)
    pol.allow_upgrade = allow_upgrade
    pol.use_levels_mask = 0b011111                       # cubature levels only
    phi, E, G = run_grad(g, c["sigma"], c["pts"], -1, policy=pol)
    dr = oracle.default_policy(True)
    check(G, oracle.evaluate_gradient(c["etype"], c["verts"], c["sigma"], c["pts"], -1, dr=dr, levels_mask=0b011111))
    err = parity_errors(phi, E, oracle.evaluate(c["etype"], c["verts"], c["sigma"], c["pts"], -1, dr=dr, levels_mask=0b011111))
    assert err["phi"] <= TOL_F64 and err["E"] <= TOL_F64
    g.close()


def test_rejects_analytic_branch_and_fp32():
    c = synth.config1(level=1, m=40)
    g = Gpu(c["etype"], c["verts"])
    pol = g.b.bemcub_default_policy(True)               # mask 63: analytic enabled
    with pytest.raises(Exception):
        run_grad(g, c["sigma"], c["pts"], -1, policy=pol)
    g.close()
