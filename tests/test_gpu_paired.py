"""-m gpu parity tests of eval_paired_kernel (csrc/kernels_paired.cuh): the distance-ratio evaluation with the
rectangle rules' points taken in symmetric pairs (App. B, Eq. 3.2, Eq. 4.1).  The kernel is taken
for FP64 Phi + E distance-ratio calls on meshes with rectangles (bemcub_last_path says which kernel ran):
with 160- or 96-point tiles once there are field points enough - these cases are sized for that while the
oracle still needs only seconds - and with 32-point tiles below (every adaptive case of test_gpu_eval.py on a
mixed mesh).  Same acceptance protocol as everywhere (gpu_common.py)."""
import numpy as np
import pytest

import oracle
from paper_1606_03743_b200 import synth

from gpu_common import Gpu, TOL_ANALYTIC, TOL_F64, parity_errors

pytestmark = pytest.mark.gpu


def _split_parity(phi, E, ref, what):
    """1e-12 where the oracle's sum used no analytic pair, 1e-10 elsewhere."""
    assert np.all(np.isfinite(phi)) and np.all(np.isfinite(E)), what
    ephi = np.abs(phi - ref["phi"]) / ref["Sphi"]
    eE = np.abs(E - ref["E"]).max(axis=1) / ref["SE"]
    tol = np.where(ref["nana"] > 0, TOL_ANALYTIC, TOL_F64)
    assert np.all(ephi <= tol), f"{what}: potential {ephi.max():.3e}"
    assert np.all(eE <= tol), f"{what}: field {eE.max():.3e}"
    return float(ephi.max()), float(eE.max())


@pytest.mark.parametrize("allow_upgrade,ntracks", [(0, 150), (1, 150), (0, 191), (1, 191)])
def test_mixed_mesh_far_field(allow_upgrade, ntracks):
    """Config 4 in small (4000 rectangles + 1000 triangles; 22 500 track points: tiles of 96, or 36 481: tiles
    of 160 - the launch configuration of the full-size bench - each with a ragged last tile): paired rectangles
    of the 7- and 12-point rules next to median-form and plain triangle points in the same stages."""
    c = synth.config4(scale=0.005, ntracks=ntracks, npts_per_track=ntracks)
    g = Gpu(c["etype"], c["verts"])
    pol = g.b.bemcub_default_policy(True)
    pol.allow_upgrade = allow_upgrade
    phi, E = g.eval(c["sigma"], c["pts"], -1, policy=pol)
    assert g.b.bemcub_last_path(g.ctx.handle) == g.b.PATH_PAIRED
    ref = oracle.evaluate(c["etype"], c["verts"], c["sigma"], c["pts"], -1, dr=oracle.default_policy(True), want_counts=True)
    _split_parity(phi, E, ref, f"mixed mesh upgrade={allow_upgrade}")
    st = g.stats()
    if allow_upgrade:
        assert st["point_interactions"] >= int(ref["npi"].sum())
    else:
        assert st["point_interactions"] == int(ref["npi"].sum()) and st["analytic_pairs"] == int(ref["nana"].sum())
    # potential only (out_E = NULL, the mat-vec of a solve): the paired / median forms without their field part
    phi2, _ = g.eval(c["sigma"], c["pts"], -1, policy=pol, want_E=False)
    assert g.b.bemcub_last_path(g.ctx.handle) == g.b.PATH_PAIRED
    assert np.max(np.abs(phi2 - ref["phi"]) / ref["Sphi"]) <= TOL_F64
    st2 = g.stats()
    assert st2["fp64_instructions"] < 12 * st2["point_interactions"]
    if not allow_upgrade:
        assert st2["point_interactions"] == int(ref["npi"].sum())
    g.close()


def _near_points(etype, verts, m, seed, hmin, hmax):
    """Field points from hmin to hmax mean sides off random elements of the mesh (along the normal, with a
    lateral offset of up to one side): every distance-ratio band, the analytic one included."""
    cen, L = synth.mean_side_and_centre(etype, verts)
    rng = np.random.default_rng(seed)
    pick = rng.integers(0, len(etype), m)
    e1 = verts[pick, 1] - verts[pick, 0]
    e2 = verts[pick, 2] - verts[pick, 0]
    nrm = np.cross(e1, e2)
    nrm /= np.linalg.norm(nrm, axis=1)[:, None]
    h = L[pick] * np.exp(rng.uniform(np.log(hmin), np.log(hmax), m))
    lat = rng.uniform(-0.5, 0.5, (m, 2))
    return np.ascontiguousarray(cen[pick] + nrm * h[:, None] + lat[:, :1] * e1 + lat[:, 1:] * e2)


@pytest.mark.parametrize("allow_upgrade", [0, 1])
def test_cube_surface_all_bands(allow_upgrade):
    """6144 squares (the config-2 mesh), 22 000 field points from 0.3 to 300 sides off the surface: all five
    paired rules, the analytic branch, tiles that straddle limits (upgrades, or pair by pair)."""
    c = synth.config2(m=8)
    etype, verts, sigma = c["etype"], c["verts"], c["sigma"]
    pts = _near_points(etype, verts, 22000, 31, 0.3, 300.0)
    g = Gpu(etype, verts)
    pol = g.b.bemcub_default_policy(True)
    pol.allow_upgrade = allow_upgrade
    phi, E = g.eval(sigma, pts, -1, policy=pol)
    assert g.b.bemcub_last_path(g.ctx.handle) == g.b.PATH_PAIRED
    ref = oracle.evaluate(etype, verts, sigma, pts, -1, dr=oracle.default_policy(True), want_counts=True)
    _split_parity(phi, E, ref, f"cube upgrade={allow_upgrade}")
    assert int(ref["nana"].sum()) > 0 and len(np.unique(ref["npi"])) > 100
    if not allow_upgrade:
        st = g.stats()
        assert st["point_interactions"] == int(ref["npi"].sum()) and st["analytic_pairs"] == int(ref["nana"].sum())
    g.close()


def test_pairs_down_to_a_distance_ratio_of_two_and_the_fallback():
    """A policy whose analytic limit for rectangles is exactly 2 still takes the paired kernel (|d| < |D| holds
    there: the outermost pair of the 33-point rule sits 0.7 sides from the centre); per-pair policy, so every
    pair uses the oracle's rule and the comparison is at the 1e-12 bar even at these close ranges.  One with a
    lower limit, or without the analytic branch, must fall back to the plain kernel."""
    c = synth.config2(m=8)
    etype, verts, sigma = c["etype"], c["verts"], c["sigma"]
    pts = _near_points(etype, verts, 22000, 32, 1.0, 60.0)
    g = Gpu(etype, verts)
    dr = np.array([[2.0, 4.0, 8.0, 20.0, 100.0], [2.0, 4.0, 8.0, 20.0, 100.0]])
    ref = oracle.evaluate(etype, verts, sigma, pts, -1, dr=dr, want_counts=True)
    phi, E = g.eval(sigma, pts, -1, policy=g.b.make_policy(dr, 0))
    assert g.b.bemcub_last_path(g.ctx.handle) == g.b.PATH_PAIRED
    _split_parity(phi, E, ref, "limits 2/4/8/20/100")
    assert g.stats()["point_interactions"] == int(ref["npi"].sum())
    dr_low = dr.copy()
    dr_low[1, 0] = 1.9
    phi, E = g.eval(sigma, pts, -1, policy=g.b.make_policy(dr_low, 0))
    assert g.b.bemcub_last_path(g.ctx.handle) == g.b.PATH_ADAPTIVE
    assert g.stats()["field_points_per_lane"] == 2                    # eval_adaptive_kernel<double, 2>: 22000 points
    ref_low = oracle.evaluate(etype, verts, sigma, pts, -1, dr=dr_low, want_counts=True)
    _split_parity(phi, E, ref_low, "fallback: rectangle analytic limit 1.9")
    assert g.stats()["point_interactions"] == int(ref_low["npi"].sum())
    phi, E = g.eval(sigma, pts, -1, policy=g.b.make_policy(dr, 0, 0b011111))
    assert g.b.bemcub_last_path(g.ctx.handle) == g.b.PATH_ADAPTIVE
    ref_cub = oracle.evaluate(etype, verts, sigma, pts, -1, dr=dr, levels_mask=0b011111, want_counts=True)
    _split_parity(phi, E, ref_cub, "fallback: no analytic branch")
    assert g.stats()["point_interactions"] == int(ref_cub["npi"].sum())
    g.close()


@pytest.mark.parametrize("allow_upgrade", [0, 1])
def test_triangles_only_seven_point_rule_on_the_medians(allow_upgrade):
    """A triangle mesh (level-4 icosphere, 5120 triangles) takes the same kernel for its 7-point rule, whose
    points are the centroid and two orbits on the medians (Q = C + kappa (V - C)); the other triangle rules
    stay plain point records.  Field points from 0.5 to 400 sides off the surface: every band."""
    etype, verts = synth.icosphere_elements(4, 1.0)
    rng = np.random.default_rng(41)
    sigma = rng.uniform(-1.0, 1.0, len(etype))
    pts = _near_points(etype, verts, 22000, 42, 0.5, 400.0)
    g = Gpu(etype, verts)
    pol = g.b.bemcub_default_policy(True)
    pol.allow_upgrade = allow_upgrade
    phi, E = g.eval(sigma, pts, -1, policy=pol)
    assert g.b.bemcub_last_path(g.ctx.handle) == g.b.PATH_PAIRED
    ref = oracle.evaluate(etype, verts, sigma, pts, -1, dr=oracle.default_policy(True), want_counts=True)
    _split_parity(phi, E, ref, f"triangles upgrade={allow_upgrade}")
    st = g.stats()
    if not allow_upgrade:
        assert st["point_interactions"] == int(ref["npi"].sum()) and st["analytic_pairs"] == int(ref["nana"].sum())
    assert st["fp64_instructions"] < 18 * st["point_interactions"]          # the median form executed fewer
    # without the 7-point level nothing is left to pair on a triangle mesh
    pol.use_levels_mask = 0b111101
    g.eval(sigma, pts, -1, policy=pol)
    assert g.b.bemcub_last_path(g.ctx.handle) == g.b.PATH_ADAPTIVE
    g.close()


def test_level_mask_and_reproducibility():
    """Rule levels switched off (7 -> 12, 17 -> 33 points) and repeated calls: same bits every time."""
    c = synth.config4(scale=0.005, ntracks=150, npts_per_track=150)
    g = Gpu(c["etype"], c["verts"])
    mask = 0b110101
    pol = g.b.bemcub_default_policy(True)
    pol.use_levels_mask = mask
    a_phi, a_E = g.eval(c["sigma"], c["pts"], -1, policy=pol)
    assert g.b.bemcub_last_path(g.ctx.handle) == g.b.PATH_PAIRED
    ref = oracle.evaluate(c["etype"], c["verts"], c["sigma"], c["pts"], -1, dr=oracle.default_policy(True), levels_mask=mask,
                          want_counts=True)
    _split_parity(a_phi, a_E, ref, "mask 110101")
    for _ in range(3):
        b_phi, b_E = g.eval(c["sigma"], c["pts"], -1, policy=pol)
        assert np.array_equal(a_phi, b_phi) and np.array_equal(a_E, b_E)
    g.close()
