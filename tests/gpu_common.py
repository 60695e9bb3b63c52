"""Shared helpers of the `-m gpu` parity tests: run the CUDA path through the C-ABI binding on
seeded inputs and compare with the CPU oracle using the acceptance protocol of DESIGN.md §5
(SURVEY.md §8(c)): per field point

    |dPhi| <= tol * k * sum|q_i|/r_i        max_j |dE_j| <= tol * k * sum|q_i|/r_i^2

tol = 1e-12 (FP64) or 1e-5 (FP32) -- BASELINE.json north_star.  The denominators come from the
oracle.  Nothing here is imported by the product."""
from __future__ import annotations

import numpy as np

TOL_F64 = 1e-12
TOL_F32 = 1e-5
TOL_ANALYTIC = 1e-10


def torch_cuda():
    import torch
    assert torch.cuda.is_available(), "the -m gpu tests need a CUDA device"
    return torch


class Gpu:
    """One bemcub ctx on cuda:0 with a mesh loaded; thin convenience over the C-ABI binding."""

    def __init__(self, etype, verts):
        torch = torch_cuda()
        from paper_1606_03743_b200 import bemcub
        self.torch, self.b = torch, bemcub
        self.ctx = bemcub.Context(0)
        self.n = len(etype)
        self.d_type = torch.as_tensor(np.ascontiguousarray(etype, dtype=np.uint8)).cuda()
        self.d_verts = torch.as_tensor(np.ascontiguousarray(verts, dtype=np.float64)).cuda()
        bemcub.bemcub_set_elements(self.ctx.handle, self.n, self.d_type if self.n else None,
                                   self.d_verts if self.n else None)

    def eval(self, sigma, pts, rule, policy=None, precision=0, want_E=True):
        torch, b = self.torch, self.b
        m = len(pts)
        d_sigma = torch.as_tensor(np.ascontiguousarray(sigma, dtype=np.float64)).cuda()
        d_pts = torch.as_tensor(np.ascontiguousarray(pts, dtype=np.float64)).cuda()
        phi = torch.full((m,), float("nan"), dtype=torch.float64, device="cuda")
        E = torch.full((m, 3), float("nan"), dtype=torch.float64, device="cuda") if want_E else None
        b.bemcub_eval(self.ctx.handle, d_sigma if self.n else None, rule, policy, m, d_pts if m else None,
                      phi if m else None, E if (m and want_E) else None, precision)
        torch.cuda.synchronize()
        return phi.cpu().numpy(), (E.cpu().numpy() if want_E else None)

    def stats(self):
        return self.b.bemcub_get_stats(self.ctx.handle)

    def close(self):
        self.ctx.close()


def parity_errors(phi, E, ref):
    """Worst per-point errors in units of the parity denominators."""
    ephi = np.abs(phi - ref["phi"]) / ref["Sphi"]
    out = {"phi": float(ephi.max()) if len(ephi) else 0.0}
    if E is not None:
        eE = np.abs(E - ref["E"]).max(axis=1) / ref["SE"]
        out["E"] = float(eE.max()) if len(eE) else 0.0
    return out


def assert_parity(phi, E, ref, tol, what=""):
    assert np.all(np.isfinite(phi)), f"{what}: non-finite potential"
    if E is not None:
        assert np.all(np.isfinite(E)), f"{what}: non-finite field"
    err = parity_errors(phi, E, ref)
    assert err["phi"] <= tol, f"{what}: potential parity {err['phi']:.3e} > {tol:g}"
    if E is not None:
        assert err["E"] <= tol, f"{what}: field parity {err['E']:.3e} > {tol:g}"
    return err
