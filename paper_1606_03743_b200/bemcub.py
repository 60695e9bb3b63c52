"""Thin ctypes binding of the bemcub C ABI (include/bemcub.h): argument marshalling only.

Every function below has the name and the argument order of its C counterpart; device buffers
are passed as torch CUDA tensors (or raw integer addresses) and only their `data_ptr()` crosses
the boundary.  All arithmetic of the hot path runs in the CUDA kernels of libbemcub.so.  There is
no CPU fallback: if the library cannot be loaded the import of this module fails loudly.
"""
from __future__ import annotations

import ctypes as C
from pathlib import Path

import numpy as np

from . import build as _build

TRI, RECT = 0, 1
RULE_ADAPTIVE = -1
LEVEL_ANALYTIC = 5
METHOD_ANALYTIC, METHOD_DUFFY_L0 = 5, 8
F64, F32 = 0, 1
ALL_LEVELS = 63

OK = 0
ERR_INVALID_ARG, ERR_DEGENERATE_ELEMENT, ERR_NOT_RECTANGLE = -1, -2, -3
ERR_BAD_RULE, ERR_CUDA, ERR_NOMEM, ERR_NO_ELEMENTS = -4, -5, -6, -7


class bemcub_policy(C.Structure):
    _fields_ = [("dr", (C.c_double * 5) * 2), ("allow_upgrade", C.c_int32), ("use_levels_mask", C.c_int32)]


class bemcub_stats(C.Structure):
    _fields_ = [("kernel_launches", C.c_int64), ("point_interactions", C.c_int64),
                ("analytic_pairs", C.c_int64), ("last_eval_launches", C.c_int64),
                ("kernel_cycles", C.c_int64), ("kernel_ns", C.c_int64), ("fp64_instructions", C.c_int64),
                ("field_points_per_lane", C.c_int64)]


class BemcubError(RuntimeError):
    def __init__(self, code: int, where: str):
        self.code = code
        super().__init__(f"{where}: {strerror(code)} (code {code})")


def _load() -> C.CDLL:
    path = _build.LIB
    if _build.is_stale():
        try:
            _build.build()
        except Exception as exc:  # no nvcc on this box and no prebuilt library
            if not Path(path).exists():
                raise ImportError(f"libbemcub.so is missing and could not be built: {exc}") from exc
    if _build.override_active():
        import sys
        print(f"bemcub: BEMCUB_LIB is set - loading {path}, which is NOT rebuilt from csrc/ and may not match it",
              file=sys.stderr, flush=True)
    lib = C.CDLL(str(path))
    vp, i64, dbl = C.c_void_p, C.c_int64, C.c_double
    PP = C.POINTER(bemcub_policy)
    sig = {
        "bemcub_create": [C.POINTER(vp), C.c_int, vp],
        "bemcub_destroy": [vp],
        "bemcub_default_policy": [PP, C.c_int],
        "bemcub_set_elements": [vp, i64, vp, vp],
        "bemcub_eval": [vp, vp, C.c_int, PP, i64, vp, vp, vp, C.c_int],
        "bemcub_eval_few_noalloc": [vp, vp, C.c_int, PP, i64, vp, vp, vp],
        "bemcub_eval_gradient": [vp, vp, C.c_int, PP, i64, vp, vp, vp, vp],
        "bemcub_eval_pairs": [vp, i64, vp, vp, vp, C.c_int, PP, vp, vp, vp, C.c_int],
        "bemcub_eval_linear": [vp, vp, C.c_int, PP, i64, vp, vp, vp, C.c_int],
        "bemcub_solve": [vp, PP, vp, vp, dbl, C.c_int, C.POINTER(C.c_int), C.POINTER(dbl)],
        "bemcub_solve_storage": [vp, i64],
        "bemcub_matvec": [vp, vp, i64, vp, vp],
        "bemcub_assemble": [vp, PP, vp, i64],
        "bemcub_assemble_rows": [vp, PP, i64, i64, vp, i64],
        "bemcub_set_elements_host": [vp, i64, vp, vp],
        "bemcub_eval_host": [vp, vp, C.c_int, PP, i64, vp, vp, vp, C.c_int],
        "bemcub_rule_info": [C.c_int, C.c_int, C.POINTER(C.c_int), C.POINTER(C.c_int)],
        "bemcub_rule_points": [C.c_int, C.c_int, vp, vp],
        "bemcub_expand_points": [vp, vp, C.c_int, vp, C.POINTER(C.c_int)],
        "bemcub_get_geometry": [vp, vp, vp, vp],
        "bemcub_fp64_peak": [vp, dbl, C.POINTER(dbl)],
        "bemcub_fp64_issue_sweep": [vp, dbl, vp, vp],
        "bemcub_inner_loop_rate": [vp, dbl, C.POINTER(dbl)],
        "bemcub_get_stats": [vp, C.POINTER(bemcub_stats)],
        "bemcub_reset_stats": [vp],
        "bemcub_last_path": [vp, C.POINTER(C.c_int)],
        "bemcub_set_timing": [vp, C.c_int],
        "bemcub_get_timing": [vp, C.POINTER(dbl), C.POINTER(dbl)],
    }
    for name, args in sig.items():
        fn = getattr(lib, name)
        fn.argtypes = args
        fn.restype = C.c_int
    lib.bemcub_strerror.argtypes = [C.c_int]
    lib.bemcub_strerror.restype = C.c_char_p
    return lib


_lib = _load()
EXPORTED = ["bemcub_create", "bemcub_destroy", "bemcub_default_policy", "bemcub_set_elements", "bemcub_eval", "bemcub_eval_few_noalloc",
            "bemcub_eval_gradient", "bemcub_eval_linear", "bemcub_eval_pairs", "bemcub_solve", "bemcub_solve_storage", "bemcub_matvec",
            "bemcub_assemble", "bemcub_assemble_rows", "bemcub_set_elements_host", "bemcub_eval_host",
            "bemcub_rule_info", "bemcub_rule_points", "bemcub_expand_points", "bemcub_get_geometry",
            "bemcub_fp64_peak", "bemcub_fp64_issue_sweep", "bemcub_inner_loop_rate", "bemcub_get_stats", "bemcub_reset_stats", "bemcub_last_path", "bemcub_set_timing",
            "bemcub_get_timing", "bemcub_strerror"]


def library_path() -> str:
    return str(_build.LIB)


def bemcub_strerror(code: int) -> str:
    return _lib.bemcub_strerror(code).decode()


strerror = bemcub_strerror


def _check(rc: int, where: str) -> None:
    if rc != OK:
        raise BemcubError(rc, where)


def _dptr(t):
    """Device address of a torch CUDA tensor (must be contiguous), an int address, or None."""
    if t is None:
        return None
    if isinstance(t, int):
        return C.c_void_p(t)
    if not t.is_cuda or not t.is_contiguous():
        raise ValueError("device buffers must be contiguous CUDA tensors")
    return C.c_void_p(t.data_ptr())


def _hptr(a):
    """Host address of a contiguous numpy array / CPU torch tensor, or None."""
    if a is None:
        return None
    if isinstance(a, np.ndarray):
        if not a.flags["C_CONTIGUOUS"]:
            raise ValueError("host buffers must be C-contiguous")
        return C.c_void_p(a.ctypes.data)
    if a.is_cuda or not a.is_contiguous():
        raise ValueError("host buffers must be contiguous CPU tensors")
    return C.c_void_p(a.data_ptr())


def _policy_ptr(policy):
    return None if policy is None else C.byref(policy)


# ---- one Python function per C entry point ---------------------------------------------------

def bemcub_create(device: int = 0, cuda_stream: int = 0) -> C.c_void_p:
    ctx = C.c_void_p()
    _check(_lib.bemcub_create(C.byref(ctx), device, C.c_void_p(cuda_stream)), "bemcub_create")
    return ctx


def bemcub_destroy(ctx) -> None:
    _check(_lib.bemcub_destroy(ctx), "bemcub_destroy")


POLICY_POTENTIAL, POLICY_FIELD, POLICY_FIELD_F32 = 0, 1, 2


def bemcub_default_policy(want_field) -> bemcub_policy:
    p = bemcub_policy()
    _check(_lib.bemcub_default_policy(C.byref(p), int(want_field)), "bemcub_default_policy")
    return p


def make_policy(dr, allow_upgrade: bool = True, use_levels_mask: int = ALL_LEVELS) -> bemcub_policy:
    """bemcub_policy from dr[2][5] (marshalling helper, no arithmetic)."""
    p = bemcub_policy()
    for t in range(2):
        for b in range(5):
            p.dr[t][b] = float(dr[t][b])
    p.allow_upgrade = int(allow_upgrade)
    p.use_levels_mask = int(use_levels_mask)
    return p


def bemcub_set_elements(ctx, n: int, etype, verts) -> None:
    _check(_lib.bemcub_set_elements(ctx, n, _dptr(etype), _dptr(verts)), "bemcub_set_elements")


def bemcub_eval(ctx, sigma, rule_id: int, policy, m: int, field_pts, out_phi, out_E, precision: int = F64) -> None:
    _check(_lib.bemcub_eval(ctx, _dptr(sigma), rule_id, _policy_ptr(policy), m, _dptr(field_pts), _dptr(out_phi),
                            _dptr(out_E), precision), "bemcub_eval")


ERR_FIXED_SCRATCH = -9
ERR_TOO_MANY_ELEMENTS = -10
NOALLOC_MAX_M = 64


def bemcub_eval_few_noalloc(ctx, sigma, rule_id: int, policy, m: int, field_pts, out_phi, out_E) -> None:
    """bemcub_eval for at most NOALLOC_MAX_M field points without any device allocation by the library
    (for tracking loops that run where cudaMalloc is off limits: memory owned by the application's pool,
    or a device-wide stall nobody can afford).  Its scratch is one fixed array per GPU shared by every
    ctx and stream: do not let two such calls run on a GPU at the same time.  See include/bemcub.h."""
    _check(_lib.bemcub_eval_few_noalloc(ctx, _dptr(sigma), rule_id, _policy_ptr(policy), m, _dptr(field_pts),
                                        _dptr(out_phi), _dptr(out_E)), "bemcub_eval_few_noalloc")


def bemcub_eval_gradient(ctx, sigma, rule_id: int, policy, m: int, field_pts, out_phi, out_E, out_G) -> None:
    _check(_lib.bemcub_eval_gradient(ctx, _dptr(sigma), rule_id, _policy_ptr(policy), m, _dptr(field_pts),
                                     _dptr(out_phi), _dptr(out_E), _dptr(out_G)), "bemcub_eval_gradient")


def bemcub_eval_pairs(ctx, npairs: int, etype, verts, sigma, method: int, policy, field_pts, out_phi, out_E,
                      precision: int = F64) -> None:
    _check(_lib.bemcub_eval_pairs(ctx, npairs, _dptr(etype), _dptr(verts), _dptr(sigma), method, _policy_ptr(policy),
                                  _dptr(field_pts), _dptr(out_phi), _dptr(out_E), precision), "bemcub_eval_pairs")


def bemcub_eval_linear(ctx, sigma_vertex, rule_id: int, policy, m: int, field_pts, out_phi, out_E,
                       precision: int = F64) -> None:
    _check(_lib.bemcub_eval_linear(ctx, _dptr(sigma_vertex), rule_id, _policy_ptr(policy), m, _dptr(field_pts),
                                   _dptr(out_phi), _dptr(out_E), precision), "bemcub_eval_linear")


ERR_NOT_CONVERGED = -8


def bemcub_solve(ctx, policy, rhs_potential, sigma, rel_tol: float, max_matvecs: int):
    """Returns (mat-vecs used, final relative residual, converged)."""
    mv, res = C.c_int(), C.c_double()
    rc = _lib.bemcub_solve(ctx, _policy_ptr(policy), _dptr(rhs_potential), _dptr(sigma), rel_tol, max_matvecs,
                           C.byref(mv), C.byref(res))
    if rc not in (0, ERR_NOT_CONVERGED):
        _check(rc, "bemcub_solve")
    return mv.value, res.value, rc == 0


def bemcub_matvec(ctx, matrix, ld: int, x, y) -> None:
    _check(_lib.bemcub_matvec(ctx, _dptr(matrix), ld, _dptr(x), _dptr(y)), "bemcub_matvec")


PATH_NONE, PATH_FIXED, PATH_ADAPTIVE, PATH_PAIRED, PATH_FEW = 0, 1, 2, 3, 4


def bemcub_last_path(ctx) -> int:
    v = C.c_int()
    _check(_lib.bemcub_last_path(ctx, C.byref(v)), "bemcub_last_path")
    return v.value


def bemcub_solve_storage(ctx, max_matrix_bytes: int) -> None:
    _check(_lib.bemcub_solve_storage(ctx, max_matrix_bytes), "bemcub_solve_storage")


def bemcub_assemble(ctx, policy, out_matrix, ld: int) -> None:
    _check(_lib.bemcub_assemble(ctx, _policy_ptr(policy), _dptr(out_matrix), ld), "bemcub_assemble")


def bemcub_assemble_rows(ctx, policy, row0: int, nrows: int, out_rows, ld: int) -> None:
    _check(_lib.bemcub_assemble_rows(ctx, _policy_ptr(policy), row0, nrows, _dptr(out_rows), ld),
           "bemcub_assemble_rows")


def bemcub_set_elements_host(ctx, n: int, host_type, host_verts) -> None:
    _check(_lib.bemcub_set_elements_host(ctx, n, _hptr(host_type), _hptr(host_verts)), "bemcub_set_elements_host")


def bemcub_eval_host(ctx, host_sigma, rule_id: int, policy, m: int, host_field_pts, host_phi, host_E,
                     precision: int = F64) -> None:
    _check(_lib.bemcub_eval_host(ctx, _hptr(host_sigma), rule_id, _policy_ptr(policy), m, _hptr(host_field_pts),
                                 _hptr(host_phi), _hptr(host_E), precision), "bemcub_eval_host")


def bemcub_rule_info(elem_type: int, rule_id: int):
    n, d = C.c_int(), C.c_int()
    _check(_lib.bemcub_rule_info(elem_type, rule_id, C.byref(n), C.byref(d)), "bemcub_rule_info")
    return n.value, d.value


def bemcub_rule_points(elem_type: int, rule_id: int):
    n, _ = bemcub_rule_info(elem_type, rule_id)
    coords = np.zeros((n, 3 if elem_type == TRI else 2))
    w = np.zeros(n)
    _check(_lib.bemcub_rule_points(elem_type, rule_id, _hptr(coords), _hptr(w)), "bemcub_rule_points")
    return coords, w


def bemcub_expand_points(ctx, sigma, rule_id: int, out_xyzq) -> int:
    stride = C.c_int()
    _check(_lib.bemcub_expand_points(ctx, _dptr(sigma), rule_id, _dptr(out_xyzq), C.byref(stride)),
           "bemcub_expand_points")
    return stride.value


def bemcub_get_geometry(ctx, out_cen, out_area, out_L) -> None:
    _check(_lib.bemcub_get_geometry(ctx, _dptr(out_cen), _dptr(out_area), _dptr(out_L)), "bemcub_get_geometry")


def bemcub_fp64_peak(ctx, seconds: float) -> float:
    v = C.c_double()
    _check(_lib.bemcub_fp64_peak(ctx, seconds, C.byref(v)), "bemcub_fp64_peak")
    return v.value


PEAK_VARIANTS = 18
PEAK_MIXES = ("DFMA", "DADD", "DMUL", "mix 8 DFMA : 6 DMUL : 4 DADD", "DFMA, 3 distinct vector-register sources (model evidence)",
              "DFMA + 1 IMAD per 2 DFMA, DFMAs counted (model evidence)")
PEAK_WARPS = (8, 16, 32)


def bemcub_fp64_issue_sweep(ctx, seconds_per_variant: float):
    """(rates[18] FP64 lane-instructions/s, sm_mhz[18]); index = mix * 3 + occupancy."""
    rates, mhz = np.zeros(PEAK_VARIANTS), np.zeros(PEAK_VARIANTS)
    _check(_lib.bemcub_fp64_issue_sweep(ctx, seconds_per_variant, _hptr(rates), _hptr(mhz)), "bemcub_fp64_issue_sweep")
    return rates, mhz


def bemcub_inner_loop_rate(ctx, seconds: float) -> float:
    v = C.c_double()
    _check(_lib.bemcub_inner_loop_rate(ctx, seconds, C.byref(v)), "bemcub_inner_loop_rate")
    return v.value


def bemcub_get_stats(ctx) -> dict:
    s = bemcub_stats()
    _check(_lib.bemcub_get_stats(ctx, C.byref(s)), "bemcub_get_stats")
    return {k: getattr(s, k) for k, _ in bemcub_stats._fields_}


def bemcub_set_timing(ctx, enable: bool) -> None:
    _check(_lib.bemcub_set_timing(ctx, int(enable)), "bemcub_set_timing")


def bemcub_get_timing(ctx):
    """(ms of the whole call, ms of its dominant kernel) of the most recent timed call."""
    a, b = C.c_double(), C.c_double()
    _check(_lib.bemcub_get_timing(ctx, C.byref(a), C.byref(b)), "bemcub_get_timing")
    return a.value, b.value


def bemcub_reset_stats(ctx) -> None:
    _check(_lib.bemcub_reset_stats(ctx), "bemcub_reset_stats")


class Context:
    """RAII wrapper: owns one bemcub_ctx bound to a device and to torch's current stream."""

    def __init__(self, device: int = 0, stream: int | None = None):
        if stream is None:
            import torch
            stream = torch.cuda.current_stream(device).cuda_stream
        self.device = device
        self.handle = bemcub_create(device, stream)

    def close(self):
        if self.handle is not None:
            bemcub_destroy(self.handle)
            self.handle = None

    def __enter__(self):
        return self

    def __exit__(self, *exc):
        self.close()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass
