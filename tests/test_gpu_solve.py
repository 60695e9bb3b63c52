"""-m gpu: bemcub_solve (matrix-free GMRES around the potential-only kernel) against the oracle's direct
solve of the same collocation system.  The converged solution is unique; the bar is
|sigma_gpu - sigma_ref|_inf <= cond(A) * rel_tol * |sigma_ref|_inf (here with a safety factor), rel_tol = 1e-12."""
from __future__ import annotations

import numpy as np
import pytest

import oracle
from paper_1606_03743_b200 import synth
from gpu_common import Gpu

pytestmark = pytest.mark.gpu


def gpu_solve(g, V, pol, rel_tol=1e-12, max_matvecs=200, x0=None):
    torch, b = g.torch, g.b
    d_V = torch.as_tensor(np.ascontiguousarray(V)).cuda()
    d_s = torch.zeros(len(V), dtype=torch.float64, device="cuda") if x0 is None else torch.as_tensor(x0.copy()).cuda()
    mv, res, ok = b.bemcub_solve(g.ctx.handle, pol, d_V, d_s, rel_tol, max_matvecs)
    return d_s.cpu().numpy(), mv, res, ok


@pytest.mark.parametrize("allow_upgrade", [0, 1])
def test_unit_potential_sphere(allow_upgrade):
    c = synth.config1(level=3, m=1)
    n = len(c["etype"])
    V = np.ones(n)
    ref, A = oracle.solve(c["etype"], c["verts"], V, oracle.default_policy(False))
    g = Gpu(c["etype"], c["verts"])
    pol = g.b.bemcub_default_policy(False)
    pol.allow_upgrade = allow_upgrade
    sigma, mv, res, ok = gpu_solve(g, V, pol)
    assert ok and res <= 1e-12 and mv < 60, (mv, res)
    assert np.max(np.abs(sigma - ref)) <= 1e-10 * np.max(np.abs(ref))
    g.close()


def test_mixed_mesh_nonuniform_potential_and_warm_start():
    c = synth.config4(scale=0.002, ntracks=1, npts_per_track=2)
    cen = synth.element_centroids(c["etype"], c["verts"])
    V = 100.0 * np.cos(cen[:, 2] / 5.0) + 10.0 * cen[:, 0]
    ref, A = oracle.solve(c["etype"], c["verts"], V, oracle.default_policy(False))
    g = Gpu(c["etype"], c["verts"])
    pol = g.b.bemcub_default_policy(False)
    sigma, mv, res, ok = gpu_solve(g, V, pol, max_matvecs=400)
    assert ok and res <= 1e-12, (mv, res)
    assert np.max(np.abs(sigma - ref)) <= 1e-9 * np.max(np.abs(ref))
    # warm start from the solution: converged after the first residual evaluation
    _, mv2, res2, ok2 = gpu_solve(g, V, pol, rel_tol=1e-10, x0=sigma)
    assert ok2 and mv2 == 1
    # a mat-vec limit that is too small is reported, with a usable iterate; the budget is exact and the
    # residual returned is the true residual of the sigma returned (checked through the oracle's matrix)
    for limit in (1, 2, 5, 6):
        s3, mv3, res3, ok3 = gpu_solve(g, V, pol, max_matvecs=limit)
        assert not ok3 and mv3 == limit and np.all(np.isfinite(s3)), (limit, mv3)
        true_res = np.linalg.norm(V - A @ s3) / np.linalg.norm(V)
        assert abs(res3 - true_res) <= 1e-9 * max(true_res, 1e-30) + 1e-12, (limit, res3, true_res)
        assert res3 <= 1.0 + 1e-12
    g.close()


@pytest.mark.parametrize("n_odd", [False, True])
def test_stored_matrix_solve_matches_the_matrix_free_one(n_odd):
    """bemcub_solve_storage: with 8 n^2 bytes allowed the solve fills the matrix once and every mat-vec is
    the GEMV kernel; the same system, so the same solution (against the oracle at the same bar, and against
    the matrix-free solve far below it); an odd n takes the GEMV's scalar path; a budget that is too small,
    and budget 0, fall back to the matrix-free mat-vec."""
    c = synth.config4(scale=0.002, ntracks=1, npts_per_track=2)
    etype, verts = (c["etype"][:-1], c["verts"][:-1]) if n_odd else (c["etype"], c["verts"])
    n = len(etype)
    assert (n % 2 == 1) == n_odd
    cen = synth.element_centroids(etype, verts)
    V = 100.0 * np.cos(cen[:, 2] / 5.0) + 10.0 * cen[:, 0]
    ref, A = oracle.solve(etype, verts, V, oracle.default_policy(False))
    g = Gpu(etype, verts)
    pol = g.b.bemcub_default_policy(False)
    free, mv_free, _, ok = gpu_solve(g, V, pol, max_matvecs=400)
    assert ok
    l0 = g.stats()["kernel_launches"]
    g.b.bemcub_solve_storage(g.ctx.handle, 8 * n * n)
    kept, mv_kept, res, ok = gpu_solve(g, V, pol, max_matvecs=400)
    launches_kept = g.stats()["kernel_launches"] - l0
    assert ok and res <= 1e-12, (mv_kept, res)
    assert np.max(np.abs(kept - ref)) <= 1e-9 * np.max(np.abs(ref))
    assert np.max(np.abs(kept - free)) <= 1e-10 * np.max(np.abs(ref))
    assert abs(mv_kept - mv_free) <= 2
    # the true residual of the returned iterate, through the oracle's matrix
    assert np.linalg.norm(V - A @ kept) / np.linalg.norm(V) <= 1e-10
    l1 = g.stats()["kernel_launches"]
    g.b.bemcub_solve_storage(g.ctx.handle, 8 * n * n - 1)          # one byte short: matrix-free again
    again, mv_again, _, ok = gpu_solve(g, V, pol, max_matvecs=400)
    launches_free = g.stats()["kernel_launches"] - l1
    assert ok and mv_again == mv_free and np.array_equal(again, free)
    assert launches_free > launches_kept                             # an evaluation is several launches, a GEMV one
    g.b.bemcub_solve_storage(g.ctx.handle, 0)
    with pytest.raises(Exception):
        g.b.bemcub_solve_storage(g.ctx.handle, -1)
    g.close()


@pytest.mark.parametrize("n_tri,ld_extra", [(640, 0), (641, 0), (641, 3), (37, 1)])
def test_matvec_against_numpy(n_tri, ld_extra):
    """bemcub_matvec on a random matrix (even / odd n, padded ld: vector and scalar paths) against numpy in
    long double; and on the assembled matrix it reproduces the potential-only evaluation at the centroids."""
    etype, verts = synth.random_elements(synth.TRI, n_tri, 11)
    n, ld = n_tri, n_tri + ld_extra
    g = Gpu(etype, verts)
    torch = g.torch
    rng = np.random.default_rng(3)
    A = rng.standard_normal((n, ld))
    x = rng.standard_normal(n)
    d_y = torch.full((n,), float("nan"), dtype=torch.float64, device="cuda")
    g.b.bemcub_matvec(g.ctx.handle, torch.as_tensor(A).cuda(), ld, torch.as_tensor(x).cuda(), d_y)
    torch.cuda.synchronize()
    ref = (A[:, :n].astype(np.longdouble) @ x.astype(np.longdouble)).astype(np.float64)
    scale = np.abs(A[:, :n]) @ np.abs(x)
    assert np.max(np.abs(d_y.cpu().numpy() - ref) / scale) <= 1e-14
    # the assembled matrix times sigma = Phi at the centroids for that sigma (L34)
    pol = g.b.bemcub_default_policy(False)
    M = torch.empty((n, n), dtype=torch.float64, device="cuda")
    g.b.bemcub_assemble(g.ctx.handle, pol, M, n)
    g.b.bemcub_matvec(g.ctx.handle, M, n, torch.as_tensor(x).cuda(), d_y)
    torch.cuda.synchronize()
    cen = synth.element_centroids(etype, verts)
    r = oracle.evaluate(etype, verts, x, cen, -1, dr=oracle.default_policy(False))
    assert np.max(np.abs(d_y.cpu().numpy() - r["phi"]) / r["Sphi"]) <= 1e-10
    with pytest.raises(Exception):
        g.b.bemcub_matvec(g.ctx.handle, M, n - 1, torch.as_tensor(x).cuda(), d_y)
    g.close()


def test_zero_rhs_and_argument_errors():
    c = synth.config1(level=1, m=1)
    g = Gpu(c["etype"], c["verts"])
    pol = g.b.bemcub_default_policy(False)
    sigma, mv, res, ok = gpu_solve(g, np.zeros(len(c["etype"])), pol, x0=np.ones(len(c["etype"])))
    assert ok and np.all(sigma == 0.0)
    with pytest.raises(Exception):
        gpu_solve(g, np.ones(len(c["etype"])), pol, rel_tol=0.0)
    g.close()
