"""-m gpu: bemcub_eval_few_noalloc, the few-point evaluation for callers that may not allocate.

Some users of this library drive it from a place where cudaMalloc is off limits: a particle tracker
embedded in an application that has given all device memory to its own pool, or a loop sharing the
GPU with other streams that a cudaMalloc (a device-wide synchronisation) would stall.  For them the
library has one entry point whose scratch - the CTAs' partial sums and the kernel's counters - is a
fixed array inside the library image instead of ctx-owned cudaMalloc memory (include/bemcub.h).

The array is shared by every call and keeps what the last call left in it, so the case worth testing
is two calls in a row with different shapes: a 64-point call (the maximum; every pass counter and
every partial-sum slot used) followed by a 5-point call that would pick up stale counters or stale
sums if the entry point did not clear / overwrite what it must.  Both are compared with bemcub_eval
on the same inputs (same kernel and grid: the bits agree; the assertion that counts is the parity
tolerance of the other GPU tests, 1e-12 of k sum|q|/r, 1e-10 where analytic pairs are involved).

The file sorts last on purpose (pytest -x would otherwise hide every later test behind a failure
here) and needs nothing from the tests before it: it passes alone in a fresh process as well.
"""
from __future__ import annotations

import numpy as np
import pytest

import oracle
from paper_1606_03743_b200 import synth
from gpu_common import TOL_ANALYTIC, TOL_F64, Gpu, parity_errors

pytestmark = pytest.mark.gpu


def _mesh_and_points():
    c = synth.config4(scale=0.003, ntracks=8, npts_per_track=9)
    rng = np.random.default_rng(4242)
    pts = c["pts"][rng.choice(len(c["pts"]), 64, replace=False)].copy()
    cen = synth.element_centroids(c["etype"], c["verts"])
    pts[0] = cen[len(cen) // 3] * (1.0 - 0.004)  # one point at the wall: analytic branch, N = 33 / 19
    pts[3] = cen[len(cen) // 2] * (1.0 - 0.004)
    return c, pts


def test_two_calls_in_a_row_match_bemcub_eval_and_allocate_nothing():
    c, pts = _mesh_and_points()
    g = Gpu(c["etype"], c["verts"])
    torch, b, h = g.torch, g.b, g.ctx.handle
    pol = b.bemcub_default_policy(True)
    d_sigma = torch.as_tensor(c["sigma"]).cuda()
    d_sigma2 = torch.as_tensor(-0.5 * c["sigma"][::-1].copy()).cuda()
    d_pts = torch.as_tensor(pts).cuda()
    shapes = [(64, 0, d_sigma), (5, 3, d_sigma2)]  # (m, first point, charges): the second call differs in all three
    out = [(torch.full((m,), float("nan"), dtype=torch.float64, device="cuda"),
            torch.full((m, 3), float("nan"), dtype=torch.float64, device="cuda")) for m, _, _ in shapes]

    def run_pair():
        for (m, j0, sg), (phi, E) in zip(shapes, out):
            b.bemcub_eval_few_noalloc(h, sg, b.RULE_ADAPTIVE, pol, m, d_pts[j0:j0 + m], phi, E)

    # Set-up call (asks the runtime for the array's address on this device, loads the kernels), then the
    # two calls under test back to back on one stream; free device memory must not move across them.
    run_pair()
    torch.cuda.synchronize()
    for phi, E in out:
        phi.fill_(float("nan"))
        E.fill_(float("nan"))
    torch.cuda.synchronize()
    free_before = torch.cuda.mem_get_info(0)[0]
    run_pair()
    torch.cuda.synchronize()
    free_after = torch.cuda.mem_get_info(0)[0]
    assert free_after == free_before, (free_before, free_after)
    got = [(phi.cpu().numpy(), E.cpu().numpy()) for phi, E in out]

    # the existing path on the same inputs, after the fact (it allocates its scratch on first use)
    for (m, j0, sg), (phi, E) in zip(shapes, got):
        sigma = sg.cpu().numpy()
        want_phi, want_E = g.eval(sigma, pts[j0:j0 + m], b.RULE_ADAPTIVE, policy=pol)
        assert b.bemcub_last_path(h) == b.PATH_FEW
        ref = oracle.evaluate(c["etype"], c["verts"], sigma, pts[j0:j0 + m], -1, dr=oracle.default_policy(True),
                              want_counts=True)
        assert np.all(np.isfinite(phi)) and np.all(np.isfinite(E))
        # against bemcub_eval, in the parity units of the other tests (the oracle supplies the denominators only)
        err = parity_errors(phi, E, {"phi": want_phi, "E": want_E, "Sphi": ref["Sphi"], "SE": ref["SE"]})
        assert err["phi"] <= TOL_F64 and err["E"] <= TOL_F64, (m, err)
        assert np.array_equal(phi, want_phi) and np.array_equal(E, want_E), m  # same kernel, same grid
        # ... and against the oracle itself, so that agreeing with a wrong bemcub_eval would not pass
        err = parity_errors(phi, E, ref)
        assert err["phi"] <= TOL_ANALYTIC and err["E"] <= TOL_ANALYTIC, (m, err)
    g.close()


def test_potential_only_fixed_rule_and_one_point_calls():
    c, pts = _mesh_and_points()
    g = Gpu(c["etype"], c["verts"])
    torch, b, h = g.torch, g.b, g.ctx.handle
    d_sigma = torch.as_tensor(c["sigma"]).cuda()
    far = np.ascontiguousarray(pts[8:10])           # fixed rules have no near-field switch: stay off the wall
    d_far = torch.as_tensor(far).cuda()
    for m, level in ((2, 1), (1, 4), (2, 2)):
        phi = torch.full((m,), float("nan"), dtype=torch.float64, device="cuda")
        b.bemcub_eval_few_noalloc(h, d_sigma, level, None, m, d_far[:m], phi, None)
        torch.cuda.synchronize()
        want_phi, _ = g.eval(c["sigma"], far[:m], level, want_E=False)
        ref = oracle.evaluate(c["etype"], c["verts"], c["sigma"], far[:m], level)
        err = np.abs(phi.cpu().numpy() - want_phi) / ref["Sphi"]
        assert err.max() <= TOL_F64, (m, level, err)
        assert parity_errors(phi.cpu().numpy(), None, ref)["phi"] <= TOL_F64
    g.close()


def test_sizes_beyond_the_fixed_scratch_are_refused():
    c, pts = _mesh_and_points()
    g = Gpu(c["etype"], c["verts"])
    torch, b, h = g.torch, g.b, g.ctx.handle
    d_sigma = torch.as_tensor(c["sigma"]).cuda()
    more = np.concatenate([pts, pts[:1] + 0.01])    # 65 points
    d_pts = torch.as_tensor(more).cuda()
    phi = torch.full((65,), 7.0, dtype=torch.float64, device="cuda")
    E = torch.full((65, 3), 7.0, dtype=torch.float64, device="cuda")
    with pytest.raises(b.BemcubError) as ei:
        b.bemcub_eval_few_noalloc(h, d_sigma, 1, None, 65, d_pts, phi, E)
    assert ei.value.code == b.ERR_FIXED_SCRATCH
    assert "64 field points" in str(ei.value)
    torch.cuda.synchronize()
    assert bool((phi == 7.0).all()) and bool((E == 7.0).all())       # nothing was enqueued
    with pytest.raises(b.BemcubError) as ei:                          # sigma is required: nothing is kept for reuse
        b.bemcub_eval_few_noalloc(h, None, 1, None, 4, d_pts, phi, E)
    assert ei.value.code == b.ERR_INVALID_ARG
    b.bemcub_eval_few_noalloc(h, d_sigma, 1, None, 0, None, None, None)  # m = 0: no-op
    g.close()
