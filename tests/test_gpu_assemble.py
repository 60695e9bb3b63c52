"""-m gpu parity tests of bemcub_assemble / bemcub_assemble_rows (step a5 of DESIGN.md §2): dense
collocation matrix entries against the CPU oracle.  Tolerances (BASELINE.json north_star):
1e-12 relative for cubature entries, 1e-10 for entries computed by the analytic formula."""
import numpy as np
import pytest

import oracle
from paper_1606_03743_b200 import synth

from gpu_common import Gpu, TOL_ANALYTIC, TOL_F64

pytestmark = pytest.mark.gpu


def _check_rows(got, ref, code, what):
    assert np.all(np.isfinite(got)), what
    rel = np.abs(got - ref) / np.abs(ref)
    cub, ana = code < 5, code == 5
    if cub.any():
        assert rel[cub].max() <= TOL_F64, f"{what}: cubature entries {rel[cub].max():.3e}"
    if ana.any():
        assert rel[ana].max() <= TOL_ANALYTIC, f"{what}: analytic entries {rel[ana].max():.3e}"
    return float(rel[cub].max()) if cub.any() else 0.0, float(rel[ana].max()) if ana.any() else 0.0


def _assemble(g, policy, n, ld=None):
    ld = n if ld is None else ld
    out = g.torch.full((n, ld), float("nan"), dtype=g.torch.float64, device="cuda")
    g.b.bemcub_assemble(g.ctx.handle, policy, out, ld)
    g.torch.cuda.synchronize()
    return out


@pytest.mark.parametrize("allow_upgrade", [0, 1])
def test_icosphere_level3_full_matrix(allow_upgrade):
    etype, verts = synth.icosphere_elements(3, 1.0)
    n = len(etype)
    g = Gpu(etype, verts)
    pol = g.b.bemcub_default_policy(False)
    pol.allow_upgrade = allow_upgrade
    A = _assemble(g, pol, n, ld=n + 5).cpu().numpy()      # ld > n: padding columns stay untouched
    assert np.all(np.isnan(A[:, n:]))
    ref, code = oracle.assemble_rows(etype, verts, np.arange(n), oracle.default_policy(False))
    _check_rows(A[:, :n], ref, code, f"level-3 matrix upgrade={allow_upgrade}")
    st = g.stats()
    assert st["analytic_pairs"] >= int((code == 5).sum())
    if not allow_upgrade:
        assert st["analytic_pairs"] == int((code == 5).sum())
    # sanity: row sums = potential of the unit-sigma sphere on its surface ~ R/eps0
    rows = A[:, :n].sum(axis=1)
    assert np.all(np.abs(rows * 8.8541878128e-12 - 1.0) < 2e-2)
    g.close()


def test_mixed_mesh_rows_api_and_ragged_tiles():
    """Triangles and rectangles mixed, n not a multiple of 32, a row window that starts and ends
    inside tiles; random elements overlap in space so every band (and the analytic one) occurs."""
    tt, tv = synth.random_elements(synth.TRI, 211, 5)
    rt, rv = synth.random_elements(synth.RECT, 190, 6)
    etype = np.concatenate([tt, rt])
    verts = np.concatenate([tv * 4.0, rv * 4.0 + 1.0], axis=0)
    n = len(etype)
    g = Gpu(etype, verts)
    for up in (0, 1):
        pol = g.b.bemcub_default_policy(False)
        pol.allow_upgrade = up
        row0, nrows = 37, 263
        out = g.torch.full((nrows, n), float("nan"), dtype=g.torch.float64, device="cuda")
        g.b.bemcub_assemble_rows(g.ctx.handle, pol, row0, nrows, out, n)
        g.torch.cuda.synchronize()
        ref, code = oracle.assemble_rows(etype, verts, np.arange(row0, row0 + nrows), oracle.default_policy(False))
        # overlapping random elements: a centroid may lie very close to another element's plane;
        # the analytic entries then carry the 1e-10 tolerance
        _check_rows(out.cpu().numpy(), ref, code, f"mixed rows upgrade={up}")
    g.close()


@pytest.mark.parametrize("mask", [0b101011, 0b110101, 0b100100])
@pytest.mark.parametrize("allow_upgrade", [0, 1])
def test_level_masks_and_row_groups(mask, allow_upgrade):
    """use_levels_mask with rule levels switched off (a wanted level maps to the next more accurate one
    that is enabled; with N = 33 off, the groups that straddle the analytic limit have no cubature rule to
    fall back on and take the per-pair path), on a spatially ordered mesh whose 128-row tiles straddle
    every limit of L159 (level-4 icosphere, 5120 triangles: L = 0.08, so the limits 3 / 8 / 20 L lie inside
    a tile's reach; a row window that starts inside a 32-row group): every entry against the oracle.  (The
    printed limits are kept: where a tile takes a more accurate rule than the pair asks for, the two differ
    by the truncation error of the pair's rule, which is below the parity bar only at limits made for it.)"""
    etype, verts = synth.icosphere_elements(4, 1.0)
    n = len(etype)
    g = Gpu(etype, verts)
    dr = oracle.default_policy(False)
    pol = g.b.make_policy(dr, allow_upgrade, mask)
    row0, nrows = 1000 + 13, 3 * 128 + 57
    out = g.torch.full((nrows, n), float("nan"), dtype=g.torch.float64, device="cuda")
    g.b.bemcub_assemble_rows(g.ctx.handle, pol, row0, nrows, out, n)
    g.torch.cuda.synchronize()
    ref, code = oracle.assemble_rows(etype, verts, np.arange(row0, row0 + nrows), dr, levels_mask=mask)
    _check_rows(out.cpu().numpy(), ref, code, f"mask {mask:06b} upgrade={allow_upgrade}")
    assert len(np.unique(code)) >= 2
    st = g.stats()
    if not allow_upgrade:
        assert st["analytic_pairs"] == int((code == 5).sum())
        npts = np.array([4, 7, 12, 19, 33])
        assert st["point_interactions"] == int(npts[code[code < 5]].sum())
    g.close()


def test_element_order_does_not_matter():
    """The rows of a call are taken in Morton order of their centroids, so a mesh handed over in random
    element order is filled with (nearly) the point count of the spatially ordered one - a tile of rows that
    spans the whole sphere would take the 33-point rule everywhere - and every entry still agrees with the
    oracle; a row window of the shuffled mesh too."""
    etype, verts = synth.icosphere_elements(4, 1.0)
    n = len(etype)
    perm = np.random.default_rng(7).permutation(n)
    g0 = Gpu(etype, verts)
    pol = g0.b.bemcub_default_policy(False)
    _assemble(g0, pol, n)
    ordered_pts = g0.stats()["point_interactions"]
    g0.close()
    g = Gpu(etype[perm].copy(), verts[perm].copy())
    A = _assemble(g, pol, n).cpu().numpy()
    shuffled_pts = g.stats()["point_interactions"]
    assert shuffled_pts <= 1.05 * ordered_pts, (shuffled_pts, ordered_pts)
    rows = np.random.default_rng(8).choice(n, 96, replace=False)
    ref, code = oracle.assemble_rows(etype[perm], verts[perm], rows, oracle.default_policy(False))
    _check_rows(A[rows], ref, code, "shuffled mesh")
    row0, nrows = 777, 1000
    out = g.torch.full((nrows, n), float("nan"), dtype=g.torch.float64, device="cuda")
    g.b.bemcub_assemble_rows(g.ctx.handle, pol, row0, nrows, out, n)
    g.torch.cuda.synchronize()
    assert np.array_equal(out.cpu().numpy()[:5], A[row0:row0 + 5]) or np.allclose(out.cpu().numpy(), A[row0:row0 + nrows], rtol=1e-12, atol=0)
    assert bool(g.torch.isfinite(out).all())
    g.close()


def test_cfg3_level5_full_size_sampled_rows():
    """Config 3 at full size (20480 x 20480, 3.36 GB) in the launch configuration bench.py uses;
    the oracle recomputes 72 rows: row 0, row n-1, the two rows at four 64-row tile boundaries, and
    62 seeded ones."""
    c = synth.config3()
    n = len(c["etype"])
    assert n == 20480
    g = Gpu(c["etype"], c["verts"])
    pol = g.b.bemcub_default_policy(False)
    A = _assemble(g, pol, n)
    edges = np.array([0, 63, 64, 127, 128, 10239, 10240, n - 65, n - 64, n - 1])
    rows = np.unique(np.concatenate([edges, np.random.default_rng(160603750).choice(n, 62, replace=False)]))
    assert len(rows) >= 64
    got = A[g.torch.as_tensor(rows).cuda()].cpu().numpy()
    ref, code = oracle.assemble_rows(c["etype"], c["verts"], rows, oracle.default_policy(False))
    cub, ana = _check_rows(got, ref, code, "cfg3 sampled rows")
    # about 67 analytic entries per row with the L159 limits
    per_row = (code == 5).sum(axis=1)
    assert 40 <= per_row.mean() <= 100
    # no NaN anywhere in the 3.36 GB
    assert bool(g.torch.isfinite(A).all())
    del A
    g.close()
