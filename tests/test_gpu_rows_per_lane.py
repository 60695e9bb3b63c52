"""-m gpu: the R = 2 and R = 4 instantiations of the plain evaluation kernels against the oracle.

plan_splits (csrc/bemcub.cu) gives every lane R field points only when a call has tiles enough to keep
all warps busy; the other parity tests are too small for that and run R = 1.  What full-size calls run -
eval_fixed_kernel<T, 4 | 2, Phi+E | Phi | gradient> and eval_adaptive_kernel<T, 4 | 2, ...> (FP64 where
the paired kernel does not apply, FP32, potential only on triangles, gradient) - differs from R = 1 in
load_field_points<R>, store_partial<R> and the ragged last tile of 32 R points.  Every case here is
sized by plan_splits' own rule for the instantiation it names, asserts through
bemcub_stats.field_points_per_lane that it got there, and has a field-point count that is not a
multiple of 32 R.  Eq. 4.1; tolerances as everywhere: 1e-12 / 1e-5 of k sum|q|/r
(1e-10 where the oracle's sum used the analytic form)."""
from __future__ import annotations

import numpy as np
import pytest

import oracle
from paper_1606_03743_b200 import synth
from gpu_common import TOL_ANALYTIC, TOL_F32, TOL_F64, Gpu, assert_parity

pytestmark = pytest.mark.gpu


def _sample(m, count, seed):
    """Seeded subset that holds the whole first and the whole last tile (a fixed rule keeps the caller's order)."""
    rng = np.random.default_rng(seed)
    mid = rng.choice(np.arange(300, m - 300), count - 600, replace=False)
    return np.sort(np.concatenate([np.arange(300), mid, np.arange(m - 300, m)]))


def _sub(ref, sel):
    return {k: v[sel] for k, v in ref.items()}


def _split_parity(phi, E, ref, tol, what):
    ana = ref["nana"] > 0
    for sel, t in ((~ana, tol), (ana, max(tol, TOL_ANALYTIC))):
        if sel.any():
            assert_parity(phi[sel], None if E is None else E[sel], _sub(ref, sel), t, f"{what} analytic={t != tol}")


# ------------------------------------------------------------------ eval_fixed_kernel<T, R, Phi+E | Phi>
@pytest.mark.parametrize("scale,level,want_R", [(0.04, 1, 4), (0.01, 3, 2)])
def test_fixed_rule_R4_and_R2(scale, level, want_R):
    """40000 (R = 4) / 10000 (R = 2) mixed elements x 10010 track points: 79 tiles of 128 (the last holds 26)
    or 157 tiles of 64 (the last 26); FP64 and FP32, Phi + E and Phi only.  (plan_splits: tiles x min(n / 32,
    512) splits must reach 16 items for each of the 1776 warps: 79 x 512 does, 79 x 312 does not, 157 x 312 does.)"""
    c = synth.config4(scale=scale, ntracks=10, npts_per_track=1001)
    m = len(c["pts"])
    assert m % (32 * want_R) != 0
    g = Gpu(c["etype"], c["verts"])
    idx = _sample(m, 2000, 7 + want_R)
    ref = oracle.evaluate(c["etype"], c["verts"], c["sigma"], c["pts"][idx], level)
    for precision, tol in ((0, TOL_F64), (1, TOL_F32)):
        for want_E in (True, False):
            phi, E = g.eval(c["sigma"], c["pts"], level, precision=precision, want_E=want_E)
            st = g.stats()
            assert g.b.bemcub_last_path(g.ctx.handle) == g.b.PATH_FIXED
            assert st["field_points_per_lane"] == want_R, (st["field_points_per_lane"], want_R)
            assert np.all(np.isfinite(phi)) and (E is None or np.all(np.isfinite(E)))
            assert_parity(phi[idx], None if E is None else E[idx], ref, tol, f"fixed R={want_R} p{precision} E={want_E}")
    g.close()


# ------------------------------------------------------------------ eval_adaptive_kernel<double, R>
@pytest.mark.parametrize("ntracks,npts,want_R", [(30, 950, 4), (15, 1000, 2)])
@pytest.mark.parametrize("allow_upgrade", [0, 1])
def test_plain_adaptive_f64_R4_and_R2(ntracks, npts, want_R, allow_upgrade):
    """The FP64 distance-ratio kernel where the paired one does not apply (analytic limits below a distance
    ratio of 2): 5027 mixed elements x 28500 (R = 4: 223 tiles, the last of 84) or 15000 points (R = 2:
    235 tiles, the last of 24); the oracle on every point (field points are Morton-sorted into tiles,
    so a sample could not name the last tile)."""
    c = synth.config4(scale=0.005, ntracks=ntracks, npts_per_track=npts)
    m = len(c["pts"])
    assert m % (32 * want_R) != 0
    dr = oracle.default_policy(True).copy()
    dr[:, 0] = 1.9
    g = Gpu(c["etype"], c["verts"])
    pol = g.b.make_policy(dr, allow_upgrade, g.b.ALL_LEVELS)
    ref = oracle.evaluate(c["etype"], c["verts"], c["sigma"], c["pts"], -1, dr=dr, want_counts=True)
    assert int(ref["nana"].sum()) > 0
    for want_E in (True, False):
        phi, E = g.eval(c["sigma"], c["pts"], -1, policy=pol, want_E=want_E)
        st = g.stats()
        assert g.b.bemcub_last_path(g.ctx.handle) == g.b.PATH_ADAPTIVE
        assert st["field_points_per_lane"] == want_R, (st["field_points_per_lane"], want_R)
        _split_parity(phi, E, ref, TOL_F64, f"adaptive f64 R={want_R} upgrade={allow_upgrade} E={want_E}")
        if not allow_upgrade:
            assert st["point_interactions"] == int(ref["npi"].sum())
            assert st["analytic_pairs"] == int(ref["nana"].sum())
    g.close()


# ------------------------------------------------------------------ eval_adaptive_kernel<float, R>
@pytest.mark.parametrize("ntracks,npts,want_R", [(30, 950, 4), (15, 1000, 2)])
def test_adaptive_f32_R4_and_R2(ntracks, npts, want_R):
    c = synth.config4(scale=0.005, ntracks=ntracks, npts_per_track=npts)
    dr32 = oracle.default_policy(2)
    g = Gpu(c["etype"], c["verts"])
    pol = g.b.bemcub_default_policy(g.b.POLICY_FIELD_F32)
    ref = oracle.evaluate(c["etype"], c["verts"], c["sigma"], c["pts"], -1, dr=dr32, want_counts=True)
    for want_E in (True, False):
        phi, E = g.eval(c["sigma"], c["pts"], -1, policy=pol, precision=1, want_E=want_E)
        assert g.b.bemcub_last_path(g.ctx.handle) == g.b.PATH_ADAPTIVE
        assert g.stats()["field_points_per_lane"] == want_R
        assert_parity(phi, E, ref, TOL_F32, f"adaptive f32 R={want_R} E={want_E}")
    g.close()


# ------------------------------------------------------------------ eval_adaptive_kernel<double, R, Phi> on triangles
@pytest.mark.parametrize("m,want_R", [(28500, 4), (15000, 2)])
def test_potential_only_on_triangles_R4_and_R2(m, want_R):
    """A potential-only call on a mesh of triangles alone stays on the plain kernel (it is the mat-vec of a
    solve): level-4 icosphere (5120 triangles), field points from 1.02 to 4 radii, default potential limits."""
    etype, verts = synth.icosphere_elements(4)
    rng = np.random.default_rng(4100 + want_R)
    sigma = rng.uniform(-1e-9, 1e-9, len(etype))
    pts = synth.isotropic_directions(rng, m) * np.exp(rng.uniform(np.log(1.02), np.log(4.0), m))[:, None]
    g = Gpu(etype, verts)
    pol = g.b.bemcub_default_policy(g.b.POLICY_POTENTIAL)
    ref = oracle.evaluate(etype, verts, sigma, pts, -1, dr=oracle.default_policy(False), want_counts=True)
    assert int(ref["nana"].sum()) > 0
    phi, _ = g.eval(sigma, pts, -1, policy=pol, want_E=False)
    assert g.b.bemcub_last_path(g.ctx.handle) == g.b.PATH_ADAPTIVE
    assert g.stats()["field_points_per_lane"] == want_R
    _split_parity(phi, None, ref, TOL_F64, f"potential only, triangles, R={want_R}")
    g.close()


# ------------------------------------------------------------------ gradient kernels at R = 2
def _run_grad(g, sigma, pts, rule, policy):
    torch, b = g.torch, g.b
    m = len(pts)
    d_sigma = torch.as_tensor(np.ascontiguousarray(sigma)).cuda()
    d_pts = torch.as_tensor(np.ascontiguousarray(pts)).cuda()
    phi = torch.full((m,), float("nan"), dtype=torch.float64, device="cuda")
    E = torch.full((m, 3), float("nan"), dtype=torch.float64, device="cuda")
    G = torch.full((m, 6), float("nan"), dtype=torch.float64, device="cuda")
    b.bemcub_eval_gradient(g.ctx.handle, d_sigma, rule, policy, m, d_pts, phi, E, G)
    torch.cuda.synchronize()
    return phi.cpu().numpy(), E.cpu().numpy(), G.cpu().numpy()


def test_gradient_fixed_rule_R2():
    c = synth.config4(scale=0.02, ntracks=10, npts_per_track=1001)
    m = len(c["pts"])
    g = Gpu(c["etype"], c["verts"])
    idx = _sample(m, 1500, 21)
    phi, E, G = _run_grad(g, c["sigma"], c["pts"], 1, None)
    assert g.stats()["field_points_per_lane"] == 2
    assert np.all(np.isfinite(G))
    rg = oracle.evaluate_gradient(c["etype"], c["verts"], c["sigma"], c["pts"][idx], 1)
    assert float((np.abs(G[idx] - rg["G"]).max(axis=1) / rg["SG"]).max()) <= TOL_F64
    assert_parity(phi[idx], E[idx], oracle.evaluate(c["etype"], c["verts"], c["sigma"], c["pts"][idx], 1), TOL_F64, "gradient fixed R=2")
    g.close()


def test_gradient_adaptive_R2():
    c = synth.config4(scale=0.005, ntracks=15, npts_per_track=1000)
    g = Gpu(c["etype"], c["verts"])
    pol = g.b.bemcub_default_policy(True)
    pol.use_levels_mask = 0b011111                       # cubature levels only (L273)
    phi, E, G = _run_grad(g, c["sigma"], c["pts"], -1, pol)
    assert g.b.bemcub_last_path(g.ctx.handle) == g.b.PATH_ADAPTIVE
    assert g.stats()["field_points_per_lane"] == 2
    dr = oracle.default_policy(True)
    rg = oracle.evaluate_gradient(c["etype"], c["verts"], c["sigma"], c["pts"], -1, dr=dr, levels_mask=0b011111)
    assert np.all(np.isfinite(G))
    assert float((np.abs(G - rg["G"]).max(axis=1) / rg["SG"]).max()) <= TOL_F64
    assert_parity(phi, E, oracle.evaluate(c["etype"], c["verts"], c["sigma"], c["pts"], -1, dr=dr, levels_mask=0b011111),
                  TOL_F64, "gradient adaptive R=2")
    g.close()
