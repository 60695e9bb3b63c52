"""-m gpu parity tests of bemcub_eval (steps a1, a2, a3, a4, a6 of DESIGN.md §2) against the CPU
oracle, element by element on the same seeded inputs, through the C ABI."""
import numpy as np
import pytest

import oracle
from paper_1606_03743_b200 import synth

from gpu_common import Gpu, TOL_F32, TOL_F64, assert_parity, parity_errors

pytestmark = pytest.mark.gpu


def _mixed_mesh(n_tri, n_rect, seed):
    tt, tv = synth.random_elements(synth.TRI, n_tri, seed)
    rt, rv = synth.random_elements(synth.RECT, n_rect, seed + 1)
    etype = np.concatenate([tt, rt])
    verts = np.concatenate([tv, rv], axis=0)
    perm = np.random.default_rng(seed + 2).permutation(len(etype))
    return np.ascontiguousarray(etype[perm]), np.ascontiguousarray(verts[perm])


def _far_points(m, seed, lo=3.0, hi=8.0):
    rng = np.random.default_rng(seed)
    d = synth.isotropic_directions(rng, m)
    return np.ascontiguousarray(0.5 + d * rng.uniform(lo, hi, m)[:, None])


# ------------------------------------------------------------------ a1: preprocessing
@pytest.mark.parametrize("n_tri,n_rect", [(50, 0), (0, 50), (37, 41)])
def test_geometry_and_expanded_points(n_tri, n_rect):
    etype, verts = _mixed_mesh(n_tri, n_rect, 11)
    n = len(etype)
    sigma = np.random.default_rng(5).uniform(-1, 1, n)
    g = Gpu(etype, verts)
    torch, b = g.torch, g.b
    cen = torch.empty((n, 3), dtype=torch.float64, device="cuda")
    area = torch.empty(n, dtype=torch.float64, device="cuda")
    L = torch.empty(n, dtype=torch.float64, device="cuda")
    b.bemcub_get_geometry(g.ctx.handle, cen, area, L)
    torch.cuda.synchronize()
    ocen, oarea, oL = oracle.geometry(etype, verts)
    np.testing.assert_allclose(cen.cpu().numpy(), ocen, rtol=0, atol=4e-16)
    np.testing.assert_allclose(area.cpu().numpy(), oarea, rtol=4e-16)
    np.testing.assert_allclose(L.cpu().numpy(), oL, rtol=4e-16)
    d_sigma = torch.as_tensor(sigma).cuda()
    for level in range(5):
        ntri, _ = oracle.rule_info(0, level)
        nrect, _ = oracle.rule_info(1, level)
        stride = max(ntri if n_tri else 0, nrect if n_rect else 0)
        out = torch.full((n * stride, 4), float("nan"), dtype=torch.float64, device="cuda")
        got_stride = b.bemcub_expand_points(g.ctx.handle, d_sigma, level, out)
        torch.cuda.synchronize()
        assert got_stride == stride
        got = out.cpu().numpy().reshape(n, stride, 4)
        ref = oracle.points(etype, verts, sigma, level)  # concatenated, N_e points per element
        pos = 0
        for e in range(n):
            N = ntri if etype[e] == 0 else nrect
            np.testing.assert_allclose(got[e, :N, :3], ref[pos:pos + N, :3], rtol=0, atol=5e-16)
            np.testing.assert_allclose(got[e, :N, 3], ref[pos:pos + N, 3], rtol=5e-16, atol=0)
            assert np.all(got[e, N:, 3] == 0.0)            # padding carries no charge
            np.testing.assert_allclose(got[e, N:, :3], np.broadcast_to(ocen[e], (stride - N, 3)), atol=4e-16)
            pos += N
        assert pos == len(ref)
    g.close()


# ------------------------------------------------------------------ configs 1 and 2, fixed rules
def test_cfg1_icosphere_n7_f64():
    c = synth.config1()
    g = Gpu(c["etype"], c["verts"])
    phi, E = g.eval(c["sigma"], c["pts"], 1)
    ref = oracle.evaluate(c["etype"], c["verts"], c["sigma"], c["pts"], 1)
    assert_parity(phi, E, ref, TOL_F64, "cfg1")
    # exact sphere: Phi = k Q_tot / r up to the l >= 6 multipoles of the icosphere
    _, area, _ = oracle.geometry(c["etype"], c["verts"])
    r = np.linalg.norm(c["pts"], axis=1)
    point = oracle.coulomb_k() * 1e-9 * area.sum() / r
    assert np.max(np.abs(phi / point - 1.0)) < 2e-5
    assert g.stats()["point_interactions"] == 1280 * 7 * 1000
    g.close()


@pytest.mark.parametrize("level", [0, 1, 2, 3, 4])
@pytest.mark.parametrize("precision", [0, 1])
def test_cfg2_cube_all_rules(level, precision):
    c = synth.config2()                        # the configuration's full 10^4 field points at every rule
    assert len(c["pts"]) == 10000
    g = Gpu(c["etype"], c["verts"])
    phi, E = g.eval(c["sigma"], c["pts"], level, precision=precision)
    ref = oracle.evaluate(c["etype"], c["verts"], c["sigma"], c["pts"], level)
    assert_parity(phi, E, ref, TOL_F64 if precision == 0 else TOL_F32, f"cfg2 L{level} p{precision}")
    g.close()


# ------------------------------------------------------------------ ragged / edge shapes
@pytest.mark.parametrize("n_tri,n_rect,m", [(1, 0, 1), (0, 1, 5), (3, 2, 33), (129, 70, 257), (700, 613, 1031),
                                              (5, 5, 20000)])
@pytest.mark.parametrize("level", [1, 3])
def test_ragged_shapes_fixed(n_tri, n_rect, m, level):
    etype, verts = _mixed_mesh(n_tri, n_rect, 100 + n_tri)
    sigma = np.random.default_rng(9).uniform(-1e-9, 1e-9, len(etype))
    pts = _far_points(m, 17)
    g = Gpu(etype, verts)
    for precision, tol in ((0, TOL_F64), (1, TOL_F32)):
        phi, E = g.eval(sigma, pts, level, precision=precision)
        ref = oracle.evaluate(etype, verts, sigma, pts, level)
        assert_parity(phi, E, ref, tol, f"ragged n={len(etype)} m={m} L{level} p{precision}")
    # potential only (out_E = NULL) runs the 12-instruction kernel (q/r folded into one FMA): same
    # potential up to the rounding of that one operation, and the same parity bar
    phi2, _ = g.eval(sigma, pts, level, want_E=False)
    assert_parity(phi2, None, ref, TOL_F64, "potential only")
    assert np.all(np.abs(phi2 - g.eval(sigma, pts, level)[0]) <= 1e-14 * ref["Sphi"])
    g.close()


def test_empty_inputs():
    etype, verts = _mixed_mesh(4, 4, 3)
    g = Gpu(etype, verts)
    phi, E = g.eval(np.ones(8), np.zeros((0, 3)), 1)           # m = 0: no-op
    assert phi.shape == (0,) and E.shape == (0, 3)
    g.close()
    g0 = Gpu(np.zeros(0, dtype=np.uint8), np.zeros((0, 3, 3)))  # n = 0: zero potential and field
    phi, E = g0.eval(np.zeros(0), _far_points(10, 1), 1)
    assert np.all(phi == 0.0) and np.all(E == 0.0)
    g0.close()


def test_error_codes():
    g = Gpu(*_mixed_mesh(2, 2, 8))
    b, torch = g.b, g.torch
    h = g.ctx.handle
    bad = np.zeros((1, 3, 3))
    bad[0, 1] = [1, 0, 0]
    bad[0, 2] = [2, 0, 0]                                         # collinear triangle
    for etype, verts, code in ((np.array([0], np.uint8), bad, b.ERR_DEGENERATE_ELEMENT),
                               (np.array([1], np.uint8), np.array([[[0, 0, 0], [1, 0, 0], [0.5, 1, 0]]], float),
                                b.ERR_NOT_RECTANGLE),
                               (np.array([7], np.uint8), np.array([[[0, 0, 0], [1, 0, 0], [0, 1, 0]]], float),
                                b.ERR_INVALID_ARG)):
        with pytest.raises(b.BemcubError) as ei:
            b.bemcub_set_elements(h, 1, torch.as_tensor(etype).cuda(), torch.as_tensor(verts).cuda())
        assert ei.value.code == code
        with pytest.raises(b.BemcubError) as ei:                  # the ctx holds no mesh after a failure
            g.eval(np.ones(1), _far_points(3, 1), 1)
        assert ei.value.code == b.ERR_NO_ELEMENTS
    g.close()
    g = Gpu(*_mixed_mesh(2, 2, 8))
    with pytest.raises(g.b.BemcubError) as ei:
        g.eval(np.ones(4), _far_points(3, 1), 9)
    assert ei.value.code == g.b.ERR_BAD_RULE
    with pytest.raises(g.b.BemcubError) as ei:
        g.eval(np.ones(4), _far_points(3, 1), -1, policy=None)   # adaptive needs a policy
    assert ei.value.code == g.b.ERR_INVALID_ARG
    g.close()


def test_host_entry_points_match_device_path():
    c = synth.config1(m=500)
    g = Gpu(c["etype"], c["verts"])
    phi_d, E_d = g.eval(c["sigma"], c["pts"], 1)
    b = g.b
    ctx2 = b.Context(0)
    b.bemcub_set_elements_host(ctx2.handle, len(c["etype"]), c["etype"], c["verts"])
    phi_h, E_h = np.zeros(500), np.zeros((500, 3))
    b.bemcub_eval_host(ctx2.handle, c["sigma"], 1, None, 500, c["pts"], phi_h, E_h)
    assert np.array_equal(phi_h, phi_d) and np.array_equal(E_h, E_d)
    ctx2.close()
    g.close()


# ------------------------------------------------------------------ a2 + a4: adaptive mode
def _assert_parity_split(phi, E, ref, what):
    """1e-12 on the field points whose oracle sum used no analytic pair, 1e-10 on the others."""
    ana = ref["nana"] > 0
    for sel, tol in ((~ana, TOL_F64), (ana, 1e-10)):
        if sel.any():
            sub = {k: v[sel] for k, v in ref.items()}
            assert_parity(phi[sel], None if E is None else E[sel], sub, tol, f"{what} analytic={tol == 1e-10}")


def _policy(b, want_field, allow_upgrade, mask=63, dr=None):
    p = b.bemcub_default_policy(want_field)
    if dr is not None:
        p = b.make_policy(dr, allow_upgrade, mask)
    p.allow_upgrade = int(allow_upgrade)
    p.use_levels_mask = mask
    return p


@pytest.mark.parametrize("kind", [0, 1])
@pytest.mark.parametrize("allow_upgrade", [0, 1])
def test_cfg5_single_element_adaptive(kind, allow_upgrade):
    """All six branches (analytic, N = 33 ... 4) on one element: DR log-uniform in [0.3, 1e4]."""
    c = synth.config5(kind, m=20000, dr_lo=0.3, dr_hi=1e4)
    g = Gpu(c["etype"], c["verts"])
    pol = _policy(g.b, True, allow_upgrade)
    dr = oracle.default_policy(True)
    phi, E = g.eval(c["sigma"], c["pts"], -1, policy=pol)
    ref = oracle.evaluate(c["etype"], c["verts"], c["sigma"], c["pts"], -1, dr=dr, want_counts=True)
    assert_parity(phi, E, ref, TOL_F64, f"cfg5 kind={kind} upgrade={allow_upgrade}")
    st = g.stats()
    if not allow_upgrade:                                           # exact per-pair policy: same work
        assert st["point_interactions"] == int(ref["npi"].sum())
    else:
        assert st["point_interactions"] >= int(ref["npi"].sum())
    assert st["analytic_pairs"] > 0
    g.close()


@pytest.mark.parametrize("allow_upgrade", [0, 1])
@pytest.mark.parametrize("mask", [63, 0b110110])   # all levels | the paper's GPU set 7/12/33 + analytic (L239)
def test_cfg4_small_mixed_adaptive(allow_upgrade, mask):
    """Config 4 shrunk to ~2000 elements: elements are large, so field points see every band,
    including the analytic one; triangles and rectangles mixed; several tiles and splits."""
    c = synth.config4(scale=0.002, ntracks=40, npts_per_track=53)
    g = Gpu(c["etype"], c["verts"])
    pol = _policy(g.b, True, allow_upgrade, mask)
    dr = oracle.default_policy(True)
    phi, E = g.eval(c["sigma"], c["pts"], -1, policy=pol)
    ref = oracle.evaluate(c["etype"], c["verts"], c["sigma"], c["pts"], -1, dr=dr, levels_mask=mask,
                          want_counts=True)
    assert_parity(phi, E, ref, TOL_F64, f"cfg4-small upgrade={allow_upgrade} mask={mask}")
    if not allow_upgrade:
        assert g.stats()["point_interactions"] == int(ref["npi"].sum())
    g.close()


def test_adaptive_policy_potential_limits_and_custom():
    """want_field = 0 limits (L159) and a custom policy with wide near bands."""
    etype, verts = _mixed_mesh(150, 150, 77)
    sigma = np.random.default_rng(1).uniform(-1e-9, 1e-9, 300)
    rng = np.random.default_rng(2)
    pts = np.ascontiguousarray(rng.uniform(-3.0, 4.0, (3001, 3)))
    g = Gpu(etype, verts)
    for dr, want_field in ((None, False), (np.array([[5, 12, 30, 120, 2500.0], [7, 18, 45, 200, 4000.0]]), True)):
        for up in (0, 1):
            pol = _policy(g.b, want_field, up, dr=dr)
            odr = oracle.default_policy(want_field) if dr is None else dr
            phi, E = g.eval(sigma, pts, -1, policy=pol)
            ref = oracle.evaluate(etype, verts, sigma, pts, -1, dr=odr, want_counts=True)
            # points may fall inside the element cloud; the analytic branch handles them: 1e-10 where a
            # point used it, 1e-12 on all the others
            _assert_parity_split(phi, E, ref, (up, want_field))
    g.close()


# ------------------------------------------------------------------ full-size config 4 (bench launch config)
def test_cfg4_full_size_sampled():
    """10^6 elements x 10^6 field points, adaptive, the exact call bench.py times; the oracle recomputes
    1024 field points one by one: 768 drawn from a seed plus the first and the last 128 points of the
    evaluation (Morton) order, i.e. the first tile and the ragged last one."""
    c = synth.config4()
    n, m = len(c["etype"]), len(c["pts"])
    assert n == 1_000_000 and m == 1_000_000
    g = Gpu(c["etype"], c["verts"])
    pol = _policy(g.b, True, 1)
    phi, E = g.eval(c["sigma"], c["pts"], -1, policy=pol)
    assert g.b.bemcub_last_path(g.ctx.handle) == g.b.PATH_PAIRED       # the kernel bench.py times ...
    assert g.stats()["field_points_per_lane"] == 5                     # ... in the instantiation it times: <5, 8>
    assert np.all(np.isfinite(phi)) and np.all(np.isfinite(E))
    ppp_upgrade = g.stats()["point_interactions"] / (float(n) * m)
    # Morton order of the field points, recomputed here (30-bit keys on the bounding box, as DESIGN.md
    # section 2 describes) only to pick the sample: points of the first and of the last tile
    lo, hi = c["pts"].min(axis=0), c["pts"].max(axis=0)
    q = np.minimum(((c["pts"] - lo) / (hi - lo) * 1024.0).astype(np.int64), 1023)
    key = np.zeros(m, dtype=np.int64)
    for bit in range(10):
        for k in range(3):
            key |= ((q[:, k] >> bit) & 1) << (3 * bit + k)
    order = np.argsort(key, kind="stable")
    idx = np.unique(np.concatenate([order[:128], order[-128:],
                                    np.random.default_rng(160603749).choice(m, 768, replace=False)]))
    ref = oracle.evaluate(c["etype"], c["verts"], c["sigma"], c["pts"][idx], -1, dr=oracle.default_policy(True),
                          want_counts=True)
    assert int(ref["nana"].sum()) == 0                                  # config 4 has no near-field pair (DR_min = 18)
    assert_parity(phi[idx], E[idx], ref, TOL_F64, "cfg4 full")
    # the method's own work (per-pair policy) on the sample, and what the tiles execute beside it
    ppp_own = ref["npi"].sum() / (float(n) * len(idx))
    assert 7.2 < ppp_own < 7.6 and ppp_own <= ppp_upgrade < 1.05 * ppp_own, (ppp_own, ppp_upgrade)
    # allow_upgrade = 0 on the sampled points: the device counter equals the oracle's count exactly
    pol0 = _policy(g.b, True, 0)
    phi0, E0 = g.eval(c["sigma"], c["pts"][idx], -1, policy=pol0)
    assert g.stats()["point_interactions"] == int(ref["npi"].sum())
    assert_parity(phi0, E0, ref, TOL_F64, "cfg4 sample, per-pair policy")
    g.close()


# ------------------------------------------------------------------ potential only (out_E = NULL: 12-instruction kernels)
@pytest.mark.parametrize("precision", [0, 1])
def test_potential_only_fixed_matches_oracle(precision):
    c = synth.config2()
    g = Gpu(c["etype"], c["verts"])
    phi, _ = g.eval(c["sigma"], c["pts"], 2, precision=precision, want_E=False)
    ref = oracle.evaluate(c["etype"], c["verts"], c["sigma"], c["pts"], 2)
    assert_parity(phi, None, ref, TOL_F32 if precision else TOL_F64, "cfg2 potential only")
    g.close()


@pytest.mark.parametrize("level", [2, 3])
@pytest.mark.parametrize("allow_upgrade", [0, 1])
def test_potential_only_adaptive_with_analytic_branch(allow_upgrade, level):
    """Field points = element centroids of a sphere (the mat-vec of a BEM solve): self terms and
    neighbours go through the analytic branch.  Level 3 is the regression case of a field point
    sitting exactly on the centroid node of a rule that OTHER points of its tile use (0 * inf)."""
    c = synth.config1(level=level, m=1)
    cen = synth.element_centroids(c["etype"], c["verts"])
    sigma = np.random.default_rng(5).uniform(0.5, 1.5, len(c["etype"]))
    g = Gpu(c["etype"], c["verts"])
    pol = _policy(g.b, False, allow_upgrade)
    phi, _ = g.eval(sigma, cen, -1, policy=pol, want_E=False)
    ref = oracle.evaluate(c["etype"], c["verts"], sigma, cen, -1, dr=oracle.default_policy(False))
    err = parity_errors(phi, None, ref)
    assert err["phi"] <= 1e-10, err          # analytic entries: BASELINE.json's 1e-10 (every centroid has its self term)
    # with E as well: same potential; E itself is not compared - on the element's own surface the
    # normal field jumps by sigma/eps0 and its sign hangs on the rounding of h = n.(P - V0) ~ 1e-17
    phi2, E2 = g.eval(sigma, cen, -1, policy=pol)
    err2 = parity_errors(phi2, None, ref)
    assert np.all(np.isfinite(E2)) and err2["phi"] <= 1e-10, err2
    g.close()


def test_results_are_bit_reproducible():
    """Work items are pulled from an atomic queue, so WHICH warp computes an item varies from run to
    run; what an item computes, the split sums and their order do not: outputs are bit-identical."""
    c = synth.config4(scale=0.01, ntracks=100, npts_per_track=100)
    g = Gpu(c["etype"], c["verts"])
    pol = _policy(g.b, True, 1)
    a_phi, a_E = g.eval(c["sigma"], c["pts"], -1, policy=pol)
    for _ in range(3):
        b_phi, b_E = g.eval(c["sigma"], c["pts"], -1, policy=pol)
        assert np.array_equal(a_phi, b_phi) and np.array_equal(a_E, b_E)
    f_phi, f_E = g.eval(c["sigma"], c["pts"], 2)
    f2_phi, f2_E = g.eval(c["sigma"], c["pts"], 2)
    assert np.array_equal(f_phi, f2_phi) and np.array_equal(f_E, f2_E)
    g.close()


def test_non_finite_field_points_do_not_spoil_their_tile():
    """A NaN / inf field point gives NaN for itself only: the other points of its tile keep the rule
    choice (and the parity) they would have had."""
    c = synth.config4(scale=0.002, ntracks=20, npts_per_track=50)
    pts = c["pts"].copy()
    bad = np.array([3, 200, 777])
    pts[3, 0] = np.nan
    pts[200, 1] = np.inf
    pts[777] = [-np.inf, np.nan, 0.0]
    g = Gpu(c["etype"], c["verts"])
    pol = _policy(g.b, True, 1)
    phi, E = g.eval(c["sigma"], pts, -1, policy=pol)
    good = np.setdiff1d(np.arange(len(pts)), bad)
    assert not np.any(np.isfinite(phi[bad]))
    ref = oracle.evaluate(c["etype"], c["verts"], c["sigma"], pts[good], -1, dr=oracle.default_policy(True))
    assert_parity(phi[good], E[good], ref, TOL_F64, "tile mates of non-finite points")
    g.close()


# ------------------------------------------------------------------ sharding by contiguous ranges
@pytest.mark.parametrize("world", [2, 3, 8])
def test_sub_ranges_reproduce_the_full_call(world):
    """What every rank of a multi-GPU job does (bench.py --gpus N, multi.my_range): bemcub_eval on its
    contiguous range of the field points, bemcub_assemble_rows on its range of the rows.  Fixed rule:
    the concatenation is bit-identical to the single full call (a field point's sum does not depend on
    its tile mates).  Adaptive: tiles differ, so the pieces agree with the oracle at the parity bar."""
    c = synth.config4(scale=0.004, ntracks=30, npts_per_track=41)
    m = len(c["pts"])
    g = Gpu(c["etype"], c["verts"])
    full_phi, full_E = g.eval(c["sigma"], c["pts"], 1)
    pol = _policy(g.b, True, 1)
    ref = oracle.evaluate(c["etype"], c["verts"], c["sigma"], c["pts"], -1, dr=oracle.default_policy(True), want_counts=True)
    parts_phi, parts_E = [], []
    for r in range(world):
        lo, hi = synth.shard_range(m, r, world)
        p1, e1 = g.eval(c["sigma"], c["pts"][lo:hi], 1)
        parts_phi.append(p1)
        parts_E.append(e1)
        pa, ea = g.eval(c["sigma"], c["pts"][lo:hi], -1, policy=pol)
        _assert_parity_split(pa, ea, {k: v[lo:hi] for k, v in ref.items()}, f"rank {r}/{world}")
    assert np.array_equal(np.concatenate(parts_phi), full_phi) and np.array_equal(np.concatenate(parts_E), full_E)
    # matrix rows
    n = g.n
    pol0 = _policy(g.b, False, 0)
    torch = g.torch
    A = torch.empty((n, n), dtype=torch.float64, device="cuda")
    g.b.bemcub_assemble(g.ctx.handle, pol0, A, n)
    pieces = []
    for r in range(world):
        lo, hi = synth.shard_range(n, r, world)
        rows = torch.empty((hi - lo, n), dtype=torch.float64, device="cuda")
        g.b.bemcub_assemble_rows(g.ctx.handle, pol0, lo, hi - lo, rows, n)
        pieces.append(rows)
    torch.cuda.synchronize()
    assert torch.equal(torch.cat(pieces, dim=0), A)                      # per-pair policy: bit-identical
    g.close()


# ------------------------------------------------------------------ FP32 with the distance-ratio choice
@pytest.mark.parametrize("allow_upgrade", [0, 1])
def test_adaptive_f32_small_mixed_and_single_element(allow_upgrade):
    """BEMCUB_RULE_ADAPTIVE with BEMCUB_F32: rule choice and analytic branch in FP64, points and
    interactions in FP32, with the limits of BEMCUB_POLICY_FIELD_F32.  Parity 1e-5 against the
    long-double oracle under the same limits; with allow_upgrade = 0 the same interaction count; and
    the result is as accurate as FP32 allows (the limits are not too low)."""
    dr32 = oracle.default_policy(2)
    for c in (synth.config4(scale=0.002, ntracks=40, npts_per_track=53),
              synth.config5(synth.TRI, m=20000, dr_lo=0.3, dr_hi=1e4),
              synth.config5(synth.RECT, m=20000, dr_lo=0.3, dr_hi=1e4)):
        g = Gpu(c["etype"], c["verts"])
        pol = g.b.bemcub_default_policy(g.b.POLICY_FIELD_F32)
        assert [list(pol.dr[0]), list(pol.dr[1])] == dr32.tolist()
        pol.allow_upgrade = allow_upgrade
        ref = oracle.evaluate(c["etype"], c["verts"], c["sigma"], c["pts"], -1, dr=dr32, want_counts=True)
        for want_E in (True, False):
            phi, E = g.eval(c["sigma"], c["pts"], -1, policy=pol, precision=1, want_E=want_E)
            assert_parity(phi, E, ref, TOL_F32, f"adaptive f32 {c['name']} upgrade={allow_upgrade}")
            if not allow_upgrade:
                assert g.stats()["point_interactions"] == int(ref["npi"].sum())
        # against the accurate answer (FP64 limits, long double): at the FP32 rounding floor
        exact = oracle.evaluate(c["etype"], c["verts"], c["sigma"], c["pts"], -1, dr=oracle.default_policy(True))
        phi, E = g.eval(c["sigma"], c["pts"], -1, policy=pol, precision=1)
        e_phi = np.abs(phi - exact["phi"]) / exact["Sphi"]
        e_E = np.abs(E - exact["E"]).max(axis=1) / exact["SE"]
        assert e_phi.mean() <= 2e-7 and e_E.mean() <= 4e-7, (c["name"], e_phi.mean(), e_E.mean())
        g.close()
