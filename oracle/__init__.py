"""ORACLE — TEST INFRASTRUCTURE ONLY (see bem_oracle.cpp's header).

ctypes loader for the plain CPU oracle of arXiv 1606.03743's hot path.  Only `tests/`,
`__graft_entry__.smoke()` and `bench.py`'s `cpu_baseline` / `--impl reference` legs may import
this package.  It imports nothing from `paper_1606_03743_b200` and the CUDA path imports
nothing from here.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
from pathlib import Path

import numpy as np

_HERE = Path(__file__).resolve().parent
_SO = _HERE / "liboracle.so"
_SRC = [_HERE / "bem_oracle.cpp", _HERE / "rule_tables.hpp"]

ANALYTIC = 5          # level code of the analytic branch
ALL_LEVELS = 0b111111


def build(force: bool = False) -> Path:
    """Compile liboracle.so with g++ (no CUDA)."""
    if not force and _SO.exists() and all(_SO.stat().st_mtime >= s.stat().st_mtime for s in _SRC):
        return _SO
    # -ffp-contract=off: the double-typed rule decision forms D^2 with separately rounded products
    # (reading 8) on every host, also where the compiler would otherwise contract to FMAs
    cmd = ["g++", "-O2", "-std=c++17", "-ffp-contract=off", "-fopenmp", "-shared", "-fPIC",
           str(_SRC[0]), "-o", str(_SO)]
    subprocess.run(cmd, check=True, cwd=_HERE)
    return _SO


_lib = None


def lib() -> C.CDLL:
    global _lib
    if _lib is None:
        build()
        L = C.CDLL(str(_SO))
        L.orc_coulomb_k.restype = C.c_double
        L.orc_rule_monomial_residual.restype = C.c_double
        L.orc_points.restype = C.c_int64
        L.orc_duffy_monomial_residual.restype = C.c_double
        _lib = L
    return _lib


def _p(a, t=C.c_double):
    return None if a is None else a.ctypes.data_as(C.POINTER(t))


def _f64(a):
    return np.ascontiguousarray(a, dtype=np.float64)


def coulomb_k() -> float:
    return lib().orc_coulomb_k()


def num_threads() -> int:
    return lib().orc_num_threads()


def rule_info(etype: int, level: int):
    n, d = C.c_int(), C.c_int()
    rc = lib().orc_rule_info(etype, level, C.byref(n), C.byref(d))
    if rc:
        raise ValueError(f"orc_rule_info rc={rc}")
    return n.value, d.value


def rule_nodes(etype: int, level: int):
    n, _ = rule_info(etype, level)
    coords = np.zeros((n, 3 if etype == 0 else 2))
    w = np.zeros(n)
    lib().orc_rule_nodes(etype, level, _p(coords), _p(w))
    return coords, w


def monomial_residual(etype: int, level: int, a: int, b: int) -> float:
    return lib().orc_rule_monomial_residual(etype, level, a, b)


def geometry(etype, verts):
    etype = np.ascontiguousarray(etype, dtype=np.uint8)
    verts = _f64(verts)
    n = len(etype)
    cen, area, L = np.zeros((n, 3)), np.zeros(n), np.zeros(n)
    rc = lib().orc_geometry(C.c_int64(n), _p(etype, C.c_uint8), _p(verts), _p(cen), _p(area), _p(L))
    if rc:
        raise ValueError(f"orc_geometry rc={rc}")
    return cen, area, L


def points(etype, verts, sigma, level: int):
    etype = np.ascontiguousarray(etype, dtype=np.uint8)
    verts, sigma = _f64(verts), _f64(sigma)
    n = len(etype)
    cnt = lib().orc_points(C.c_int64(n), _p(etype, C.c_uint8), _p(verts), _p(sigma), level, None)
    if cnt < 0:
        raise ValueError(f"orc_points rc={cnt}")
    out = np.zeros((cnt, 4))
    lib().orc_points(C.c_int64(n), _p(etype, C.c_uint8), _p(verts), _p(sigma), level, _p(out))
    return out


def default_policy(want_field) -> np.ndarray:
    """dr[2][5]; want_field 0 / False: printed potential limits (L159), 1 / True: Phi+E limits,
    2: limits for single-precision evaluation."""
    dr = np.zeros((2, 5))
    rc = lib().orc_default_policy(_p(dr), int(want_field))
    if rc:
        raise ValueError(f"orc_default_policy rc={rc}")
    return dr


def choose_level(D2: float, L: float, dr5, levels_mask: int = ALL_LEVELS) -> int:
    dr5 = _f64(dr5)
    return lib().orc_choose_level(C.c_double(D2), C.c_double(L), _p(dr5), levels_mask)


def evaluate(etype, verts, sigma, pts, level: int, dr=None, levels_mask: int = ALL_LEVELS,
             precision: str = "long double", nthreads: int = 0, want_counts: bool = False):
    """Eq. 4.1 summed over all elements at every field point.

    level 0..4 = fixed rule (N = 4, 7, 12, 19|17, 33); level -1 = per-pair rule by distance
    ratio with limits dr[2][5].  Returns dict(phi[m], E[m][3], Sphi[m], SE[m][, npi[m], nana[m]]) where
    Sphi = k*sum|q_i|/r_i and SE = k*sum|q_i|/r_i^2 are the parity denominators, npi the point-charge
    interactions and nana the analytic pairs each field point used (want_counts).
    """
    etype = np.ascontiguousarray(etype, dtype=np.uint8)
    verts, sigma, pts = _f64(verts), _f64(sigma), _f64(pts)
    n, m = len(etype), len(pts)
    assert verts.shape == (n, 3, 3) and sigma.shape == (n,) and pts.shape == (m, 3)
    phi, E, Sphi, SE = np.zeros(m), np.zeros((m, 3)), np.zeros(m), np.zeros(m)
    npi = np.zeros(m, dtype=np.int64) if want_counts else None
    nana = np.zeros(m, dtype=np.int64) if want_counts else None
    drp = None if dr is None else _f64(dr)
    rc = lib().orc_eval(C.c_int64(n), _p(etype, C.c_uint8), _p(verts), _p(sigma), level,
                        _p(drp), levels_mask, C.c_int64(m), _p(pts), _p(phi), _p(E), _p(Sphi),
                        _p(SE), _p(npi, C.c_int64), _p(nana, C.c_int64),
                        0 if precision == "long double" else 1, nthreads)
    if rc:
        raise ValueError(f"orc_eval rc={rc}")
    out = dict(phi=phi, E=E, Sphi=Sphi, SE=SE)
    if want_counts:
        out["npi"] = npi
        out["nana"] = nana
    return out


def solve(etype, verts, potential, dr, levels_mask: int = ALL_LEVELS):
    """Charge densities of the BEM collocation system: sum_j A_ij sigma_j = V_i with
    A from assemble_rows (per-pair rule by distance ratio, analytic self/near terms), solved
    directly (LAPACK via numpy) - the plain definition of what the iterative GPU solver converges to."""
    n = len(etype)
    A, _ = assemble_rows(etype, verts, np.arange(n), dr, levels_mask)
    return np.linalg.solve(A, _f64(potential)), A


CUBATURE_LEVELS = 0b011111


def evaluate_gradient(etype, verts, sigma, pts, level: int, dr=None, levels_mask: int = CUBATURE_LEVELS):
    """Field gradient G_ij = dE_i/dx_j of the Eq. 4.1 point charges, long double.
    Returns dict(G[m][6] in the order xx, yy, zz, xy, xz, yz; SG[m] = k*sum|q_i|/r_i^3)."""
    etype = np.ascontiguousarray(etype, dtype=np.uint8)
    verts, sigma, pts = _f64(verts), _f64(sigma), _f64(pts)
    n, m = len(etype), len(pts)
    G, SG = np.zeros((m, 6)), np.zeros(m)
    drp = None if dr is None else _f64(dr)
    rc = lib().orc_eval_gradient(C.c_int64(n), _p(etype, C.c_uint8), _p(verts), _p(sigma), level, _p(drp),
                                 levels_mask, C.c_int64(m), _p(pts), _p(G), _p(SG))
    if rc:
        raise ValueError(f"orc_eval_gradient rc={rc}")
    return dict(G=G, SG=SG)


def evaluate_linear(etype, verts, sigma_v, pts, level: int, dr=None, levels_mask: int = CUBATURE_LEVELS):
    """Eq. 4.1 with a charge density that varies linearly over each element:
    sigma_v[n][3] = values at the three stored vertices, q_i = w_i A sigma(Q_i).  Long double."""
    etype = np.ascontiguousarray(etype, dtype=np.uint8)
    verts, sigma_v, pts = _f64(verts), _f64(sigma_v), _f64(pts)
    n, m = len(etype), len(pts)
    assert sigma_v.shape == (n, 3)
    phi, E, Sphi, SE = np.zeros(m), np.zeros((m, 3)), np.zeros(m), np.zeros(m)
    drp = None if dr is None else _f64(dr)
    rc = lib().orc_eval_linear(C.c_int64(n), _p(etype, C.c_uint8), _p(verts), _p(sigma_v), level, _p(drp),
                               levels_mask, C.c_int64(m), _p(pts), _p(phi), _p(E), _p(Sphi), _p(SE))
    if rc:
        raise ValueError(f"orc_eval_linear rc={rc}")
    return dict(phi=phi, E=E, Sphi=Sphi, SE=SE)


DUFFY = 8             # method code of the Duffy-mapped rectangle rule of level l: DUFFY + l


def evaluate_pairs(etype, verts, pts, method: int, sigma=None, dr=None, levels_mask: int = ALL_LEVELS,
                   precision: str = "long double"):
    """Element k seen from field point k (no sum over elements; PAPER.md L193-196 item a, the unit of
    the accuracy protocol of L68/L149).  method 0..4 = cubature level, 5 = analytic closed form,
    -1 = by distance ratio (dr[2][5]), DUFFY + l = rectangle rule of level l (Duffy-mapped on
    triangles, L163-169).  Returns dict(phi[K], E[K][3], Sphi[K], SE[K], used[K])."""
    etype = np.ascontiguousarray(etype, dtype=np.uint8)
    verts, pts = _f64(verts), _f64(pts)
    K = len(etype)
    assert verts.shape == (K, 3, 3) and pts.shape == (K, 3)
    sg = None if sigma is None else _f64(sigma)
    phi, E, Sphi, SE = np.zeros(K), np.zeros((K, 3)), np.zeros(K), np.zeros(K)
    used = np.zeros(K, dtype=np.uint8)
    drp = None if dr is None else _f64(dr)
    rc = lib().orc_eval_pairs(C.c_int64(K), _p(etype, C.c_uint8), _p(verts), _p(sg), method, _p(drp), levels_mask,
                              _p(pts), _p(phi), _p(E), _p(Sphi), _p(SE), _p(used, C.c_uint8),
                              0 if precision == "long double" else 1)
    if rc:
        raise ValueError(f"orc_eval_pairs rc={rc}")
    return dict(phi=phi, E=E, Sphi=Sphi, SE=SE, used=used)


def duffy_nodes(level: int):
    """Duffy-mapped rectangle rule on the reference triangle: (bary[N][3], w[N])."""
    n, _ = rule_info(1, level)
    bary, w = np.zeros((n, 3)), np.zeros(n)
    rc = lib().orc_duffy_nodes(level, _p(bary), _p(w))
    if rc:
        raise ValueError(f"orc_duffy_nodes rc={rc}")
    return bary, w


def duffy_monomial_residual(level: int, a: int, b: int) -> float:
    return lib().orc_duffy_monomial_residual(level, a, b)


def _single(fn, etype, verts9, P, *extra):
    verts9, P = _f64(verts9).reshape(9), _f64(P).reshape(3)
    ip = C.c_double()
    ie = np.zeros(3)
    rc = fn(int(etype), _p(verts9), _p(P), *extra[:1], C.byref(ip), _p(ie), *extra[1:])
    if rc:
        raise ValueError(f"oracle rc={rc}")
    return ip.value, ie


def analytic(etype, verts9, P, precision: str = "long double"):
    verts9, P = _f64(verts9).reshape(9), _f64(P).reshape(3)
    ip, ie = C.c_double(), np.zeros(3)
    rc = lib().orc_analytic(int(etype), _p(verts9), _p(P), C.byref(ip), _p(ie),
                            0 if precision == "long double" else 1)
    if rc:
        raise ValueError(f"orc_analytic rc={rc}")
    return ip.value, ie


def gl2(etype, verts9, P, ngl: int = 16):
    verts9, P = _f64(verts9).reshape(9), _f64(P).reshape(3)
    ip, ie = C.c_double(), np.zeros(3)
    rc = lib().orc_gl2(int(etype), _p(verts9), _p(P), ngl, C.byref(ip), _p(ie))
    if rc:
        raise ValueError(f"orc_gl2 rc={rc}")
    return ip.value, ie


def adaptive(etype, verts9, P, reltol: float = 1e-17):
    verts9, P = _f64(verts9).reshape(9), _f64(P).reshape(3)
    ip, ie, err = C.c_double(), np.zeros(3), C.c_double()
    rc = lib().orc_adaptive(int(etype), _p(verts9), _p(P), C.c_double(reltol), C.byref(ip), _p(ie),
                            C.byref(err))
    if rc:
        raise ValueError(f"orc_adaptive rc={rc}")
    return ip.value, ie, err.value


def gauss_legendre(n: int):
    x, w = np.zeros(n), np.zeros(n)
    lib().orc_gauss_legendre(n, _p(x), _p(w))
    return x, w


def assemble_rows(etype, verts, rows, dr, levels_mask: int = ALL_LEVELS, nthreads: int = 0):
    etype = np.ascontiguousarray(etype, dtype=np.uint8)
    verts, dr = _f64(verts), _f64(dr)
    rows = np.ascontiguousarray(rows, dtype=np.int64)
    n = len(etype)
    out = np.zeros((len(rows), n))
    code = np.zeros((len(rows), n), dtype=np.uint8)
    rc = lib().orc_assemble_rows(C.c_int64(n), _p(etype, C.c_uint8), _p(verts), _p(dr), levels_mask,
                                 C.c_int64(len(rows)), _p(rows, C.c_int64), _p(out), _p(code, C.c_uint8),
                                 0, nthreads)
    if rc:
        raise ValueError(f"orc_assemble_rows rc={rc}")
    return out, code
