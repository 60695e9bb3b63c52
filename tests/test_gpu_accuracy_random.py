"""-m gpu: the paper's random-element accuracy protocol (L68, L149; Figs. 8-10) on the GPU results.
300 random triangles / rectangles (corners in the unit cube, L68), a field point in a random
direction at each distance ratio of a grid, one element per call; mean relative error of each rule
against the exact integral (oracle, long double: closed form below DR = 10, 33-point rule above).
Soft pins: the printed triangle-potential limits (L159) and the aspect-ratio statement (L161)."""
from __future__ import annotations

import numpy as np
import pytest

import oracle
from paper_1606_03743_b200 import synth

pytestmark = pytest.mark.gpu

N_ELEM = 300
DR_GRID = np.array([3.0, 8.0, 20.0, 80.0, 300.0, 1500.0])
ALL_ANALYTIC = np.full((2, 5), 1e300)


def _aspect_ratio(kind, v):
    if kind == synth.TRI:
        a, b, c = np.linalg.norm(v[1] - v[0]), np.linalg.norm(v[2] - v[1]), np.linalg.norm(v[0] - v[2])
        longest = max(a, b, c)
        area = 0.5 * np.linalg.norm(np.cross(v[1] - v[0], v[2] - v[0]))
        return longest / (2.0 * area / longest)           # longest side / its height (L80)
    a, b = np.linalg.norm(v[1] - v[0]), np.linalg.norm(v[2] - v[0])
    return max(a, b) / min(a, b)


@pytest.mark.parametrize("kind", [synth.TRI, synth.RECT], ids=["triangles", "rectangles"])
def test_random_element_protocol(kind):
    import torch
    from paper_1606_03743_b200 import bemcub as b

    etype, verts = synth.random_elements(kind, N_ELEM, 160603750 + kind)
    rng = np.random.default_rng(160603760 + kind)
    ctx = b.Context(0)
    h = ctx.handle
    err_phi = np.zeros((5, N_ELEM, len(DR_GRID)))
    err_E = np.zeros_like(err_phi)
    ar = np.zeros(N_ELEM)
    one = torch.ones(1, dtype=torch.float64, device="cuda")
    for e in range(N_ELEM):
        et, vt = etype[e:e + 1], verts[e:e + 1]
        ar[e] = _aspect_ratio(kind, vt[0])
        cen = synth.element_centroids(et, vt)[0]
        if kind == synth.TRI:
            L = (np.linalg.norm(vt[0, 1] - vt[0, 0]) + np.linalg.norm(vt[0, 2] - vt[0, 1]) + np.linalg.norm(vt[0, 0] - vt[0, 2])) / 3.0
        else:
            L = 0.5 * (np.linalg.norm(vt[0, 1] - vt[0, 0]) + np.linalg.norm(vt[0, 2] - vt[0, 0]))
        pts = cen + synth.isotropic_directions(rng, len(DR_GRID)) * (DR_GRID * L)[:, None]
        lo = oracle.evaluate(et, vt, np.ones(1), pts, -1, dr=ALL_ANALYTIC)
        hi = oracle.evaluate(et, vt, np.ones(1), pts, 4)
        near = DR_GRID < 10.0
        phi_x = np.where(near, lo["phi"], hi["phi"])
        E_x = np.where(near[:, None], lo["E"], hi["E"])
        b.bemcub_set_elements(h, 1, torch.as_tensor(et).cuda(), torch.as_tensor(vt).cuda())
        d_pts = torch.as_tensor(pts).cuda()
        phi = torch.empty(len(pts), dtype=torch.float64, device="cuda")
        E = torch.empty((len(pts), 3), dtype=torch.float64, device="cuda")
        for level in range(5):
            b.bemcub_eval(h, one, level, None, len(pts), d_pts, phi, E, b.F64)
            torch.cuda.synchronize()
            err_phi[level, e] = np.abs(phi.cpu().numpy() - phi_x) / np.abs(phi_x)
            err_E[level, e] = np.abs(E.cpu().numpy() - E_x).sum(axis=1) / np.linalg.norm(E_x, axis=1)
    ctx.close()
    mean_phi, mean_E = err_phi.mean(axis=1), err_E.mean(axis=1)
    print("\nmean relative error, %s (rows: rule level 0..4, columns: DR = %s)" % ("triangles" if kind == synth.TRI else "rectangles", DR_GRID))
    for level in range(5):
        print("  L%d Phi " % level + " ".join(f"{v:9.2e}" for v in mean_phi[level]) + "   E " + " ".join(f"{v:9.2e}" for v in mean_E[level]))
    col = {dr: i for i, dr in enumerate(DR_GRID)}
    if kind == synth.TRI:
        # L159: N = 4 / 7 / 12 / 19 / 33 reach the 2e-15 level at DR = 1500 / 80 / 20 / 8 / 3
        for level, dr in ((0, 1500.0), (1, 80.0), (2, 20.0), (3, 8.0), (4, 3.0)):
            assert mean_phi[level, col[dr]] <= 1e-14, (level, dr, mean_phi[level, col[dr]])
            if level < 4:   # ... and are far from it one grid step nearer
                assert mean_phi[level, col[dr] - 1] > 1e-13, (level, mean_phi[level, col[dr] - 1])
        # L161, Fig. 10: the triangle rules degrade with the aspect ratio.  (7-point rule, field; at
        # the figure's DR = 300 the FP64 results already sit at the rounding floor for every aspect
        # ratio, so the statement is checked at DR = 20, where the rule's own error dominates.)
        e7 = err_E[1, :, col[20.0]]
        print("  7-point rule, field, DR = 20: mean error AR < 3: %.2e   AR > 10: %.2e" % (e7[ar < 3].mean(), e7[ar > 10].mean()))
        assert e7[ar > 10].mean() > 3.0 * e7[ar < 3].mean()
    else:
        for level, dr in ((0, 1500.0), (1, 300.0), (2, 80.0), (3, 20.0), (4, 8.0)):
            assert mean_phi[level, col[dr]] <= 1e-14, (level, dr, mean_phi[level, col[dr]])
