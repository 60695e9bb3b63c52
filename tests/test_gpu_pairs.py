"""-m gpu parity of bemcub_eval_pairs (element k seen from field point k, no sum; PAPER.md L193-196
item a) with oracle.evaluate_pairs: every method (rule levels, closed form, distance-ratio choice,
Duffy-mapped rectangle rules, L163-169), both element types, FP64 and FP32."""
from __future__ import annotations

import numpy as np
import pytest

import oracle
from paper_1606_03743_b200 import synth
from gpu_common import TOL_ANALYTIC, TOL_F32, TOL_F64, torch_cuda

pytestmark = pytest.mark.gpu


def _pairs(kind, n, seed, lo, hi):
    et, verts = synth.random_elements(kind, n, seed)
    cen, _, L = oracle.geometry(et, verts)
    rng = np.random.default_rng(seed + 1)
    dirs = synth.isotropic_directions(rng, n)
    ratio = np.exp(rng.uniform(np.log(lo), np.log(hi), n))
    return et, verts, np.ascontiguousarray(cen + dirs * (ratio * L)[:, None])


def run_pairs(et, verts, pts, method, sigma=None, policy=None, precision=0, want_E=True):
    torch = torch_cuda()
    from paper_1606_03743_b200 import bemcub as b
    K = len(et)
    ctx = b.Context(0)
    d = lambda a: torch.as_tensor(np.ascontiguousarray(a)).cuda()
    phi = torch.full((K,), float("nan"), dtype=torch.float64, device="cuda")
    E = torch.full((K, 3), float("nan"), dtype=torch.float64, device="cuda") if want_E else None
    b.bemcub_eval_pairs(ctx.handle, K, d(et) if K else None, d(verts) if K else None, None if sigma is None else d(sigma),
                        method, policy, d(pts) if K else None, phi if K else None, E if K else None, precision)
    torch.cuda.synchronize()
    st = b.bemcub_get_stats(ctx.handle)
    ctx.close()
    return phi.cpu().numpy(), (E.cpu().numpy() if want_E else None), st


def _check(phi, E, ref, tol, what):
    assert np.all(np.isfinite(phi)) and (E is None or np.all(np.isfinite(E))), what
    e_phi = np.abs(phi - ref["phi"]) / ref["Sphi"]
    assert e_phi.max() <= tol, (what, float(e_phi.max()))
    if E is not None:
        e_E = np.abs(E - ref["E"]).max(axis=1) / ref["SE"]
        assert e_E.max() <= tol, (what, float(e_E.max()))


@pytest.mark.parametrize("kind", [synth.TRI, synth.RECT], ids=["tri", "rect"])
@pytest.mark.parametrize("precision", [0, 1], ids=["f64", "f32"])
def test_every_rule_level_and_duffy(kind, precision):
    et, verts, P = _pairs(kind, 5003, 300 + kind, 2.0, 1e4)          # 5003: ragged last block
    sigma = np.random.default_rng(9).uniform(-2.0, 2.0, len(et))
    tol = TOL_F32 if precision else TOL_F64
    for method in list(range(5)) + [8 + l for l in range(5)]:
        phi, E, st = run_pairs(et, verts, P, method, sigma=sigma, precision=precision)
        ref = oracle.evaluate_pairs(et, verts, P, method, sigma=sigma)
        _check(phi, E, ref, tol, f"kind {kind} method {method} p{precision}")
        assert st["last_eval_launches"] == 1
    phi, _, _ = run_pairs(et, verts, P, 2, sigma=None, want_E=False)     # unit density, potential only
    ref = oracle.evaluate_pairs(et, verts, P, 2)
    _check(phi, None, ref, TOL_F64, "unit sigma, no E")


@pytest.mark.parametrize("kind", [synth.TRI, synth.RECT], ids=["tri", "rect"])
def test_closed_form_and_distance_ratio_choice(kind):
    from paper_1606_03743_b200 import bemcub as b
    et, verts, P = _pairs(kind, 4000, 310 + kind, 0.3, 10.0)
    phi, E, _ = run_pairs(et, verts, P, b.METHOD_ANALYTIC)
    ref = oracle.evaluate_pairs(et, verts, P, 5)
    _check(phi, E, ref, TOL_ANALYTIC, "closed form")
    # adaptive: all six branches; the pair's own distance ratio decides, exactly as in the oracle
    et, verts, P = _pairs(kind, 20000, 320 + kind, 0.3, 1e4)
    for want_field in (False, True):
        pol = b.bemcub_default_policy(want_field)
        phi, E, _ = run_pairs(et, verts, P, b.RULE_ADAPTIVE, policy=pol)
        ref = oracle.evaluate_pairs(et, verts, P, -1, dr=oracle.default_policy(want_field))
        ana = ref["used"] == 5
        assert ana.any() and (~ana).any() and len(np.unique(ref["used"])) == 6
        for sel, tol in ((ana, TOL_ANALYTIC), (~ana, TOL_F64)):
            sub = {k: v[sel] for k, v in ref.items()}
            _check(phi[sel], E[sel], sub, tol, f"adaptive want_field={want_field}")
    # the paper's GPU set of levels (L239): 7 / 12 / 33 + closed form
    pol = b.bemcub_default_policy(True)
    pol.use_levels_mask = 0b110110
    phi, E, _ = run_pairs(et, verts, P, b.RULE_ADAPTIVE, policy=pol)
    ref = oracle.evaluate_pairs(et, verts, P, -1, dr=oracle.default_policy(True), levels_mask=0b110110)
    assert set(np.unique(ref["used"])) == {1, 2, 4, 5}
    _check(phi, E, ref, TOL_ANALYTIC, "levels mask")


def test_edge_cases():
    from paper_1606_03743_b200 import bemcub as b
    et, verts, P = _pairs(synth.TRI, 7, 1, 5.0, 50.0)
    phi, E, _ = run_pairs(et[:0], verts[:0], P[:0], 1)                    # no pairs: no-op
    assert phi.shape == (0,)
    bad = verts.copy()
    bad[3] = [[0.0, 0.0, 0.0], [1.0, 0.0, 0.0], [2.0, 0.0, 0.0]]           # collinear triangle: area exactly 0
    phi, E, _ = run_pairs(et, bad, P, 1)
    assert np.isnan(phi[3]) and np.all(np.isnan(E[3]))
    ok = np.arange(7) != 3
    ref = oracle.evaluate_pairs(et[ok], verts[ok], P[ok], 1)
    _check(phi[ok], E[ok], ref, TOL_F64, "neighbours of a degenerate element")
    torch = torch_cuda()
    ctx = b.Context(0)
    d = lambda a: torch.as_tensor(np.ascontiguousarray(a)).cuda()
    out = torch.empty(7, dtype=torch.float64, device="cuda")
    for method in (6, 7, 13, -2):
        with pytest.raises(b.BemcubError) as ei:
            b.bemcub_eval_pairs(ctx.handle, 7, d(et), d(verts), None, method, None, d(P), out, None)
        assert ei.value.code == b.ERR_BAD_RULE
    with pytest.raises(b.BemcubError) as ei:                              # adaptive needs a policy
        b.bemcub_eval_pairs(ctx.handle, 7, d(et), d(verts), None, b.RULE_ADAPTIVE, None, d(P), out, None)
    assert ei.value.code == b.ERR_INVALID_ARG
    ctx.close()
