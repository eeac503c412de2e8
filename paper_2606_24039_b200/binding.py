"""Thin ctypes binding of the C ABI in include/tmpc.h — argument marshalling only.

Every step of the path runs in the CUDA kernels behind libtmpc.so; PyTorch is used here for device memory and
streams.  There is no CPU fallback: if libtmpc.so is missing or no CUDA device is present the calls raise.
The functions carry the names of the C entry points (tmpc_setup, tmpc_linearize, tmpc_factor, tmpc_admm_solve,
tmpc_backward, ...); `Solver` bundles a handle with its workspace and tensors for convenience.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libtmpc.so")
TMPC_MAX_NG = 32
TMPC_F32, TMPC_F64 = 0, 1
TMPC_MODEL_NONE, TMPC_MODEL_BICYCLE, TMPC_MODEL_SRB = 0, 1, 2
TMPC_LIN_SEQUENTIAL, TMPC_LIN_CYCLIC_REDUCTION, TMPC_LIN_AUTO = 0, 1, 2
TMPC_BWD_REFACTOR_REFINE, TMPC_BWD_ADMM_REUSE_FACTOR = 0, 1
TMPC_SOLVE_ZG_GIVEN = 1
EXPORTS = ["tmpc_workspace_bytes", "tmpc_setup", "tmpc_linearize", "tmpc_factor", "tmpc_admm_solve", "tmpc_backward",
           "tmpc_kkt_solve", "tmpc_host_staging_bytes", "tmpc_admm_solve_host", "tmpc_destroy", "tmpc_status_string",
           "tmpc_launch_count", "tmpc_measure_peak", "tmpc_admm_solve_adaptive", "tmpc_sqp_solve", "tmpc_backward_dgamma", "tmpc_admm_solve_static"]


class TmpcConfig(C.Structure):
    _fields_ = [("batch", C.c_int32), ("N", C.c_int32), ("nx", C.c_int32), ("nu", C.c_int32), ("ng", C.c_int32),
                ("dtype", C.c_int32), ("model", C.c_int32), ("linsolve", C.c_int32),
                ("sigma", C.c_double), ("rho_bar", C.c_double), ("rho_eq_scale", C.c_double), ("alpha", C.c_double),
                ("slack_gamma", C.c_double), ("slack_lambda", C.c_double),
                ("eps_active_abs", C.c_double), ("eps_active_rel", C.c_double),
                ("wheelbase", C.c_double), ("dt", C.c_double),
                ("g_lo", C.c_double * TMPC_MAX_NG), ("g_hi", C.c_double * TMPC_MAX_NG),
                ("g_is_selection", C.c_int32), ("g_col", C.c_int32 * TMPC_MAX_NG), ("soft_row", C.c_uint8 * TMPC_MAX_NG),
                ("model_params", C.c_double * 16)]


class TmpcQp(C.Structure):
    _fields_ = [("D", C.c_void_p), ("D_bstride", C.c_int64), ("E", C.c_void_p), ("E_bstride", C.c_int64), ("q", C.c_void_p),
                ("Am", C.c_void_p), ("Ap", C.c_void_p), ("b", C.c_void_p), ("x_init", C.c_void_p),
                ("G", C.c_void_p), ("G_bstride", C.c_int64), ("lo", C.c_void_p), ("hi", C.c_void_p)]


class TmpcState(C.Structure):
    _fields_ = [("x", C.c_void_p), ("zg", C.c_void_p), ("yf", C.c_void_p), ("yg", C.c_void_p), ("xi", C.c_void_p)]


class TmpcAdaptive(C.Structure):
    _fields_ = [("max_iters", C.c_int32), ("check_every", C.c_int32), ("adapt_rho", C.c_int32), ("reserved", C.c_int32),
                ("eps_abs", C.c_double), ("eps_rel", C.c_double), ("rho_ratio", C.c_double), ("rho_min", C.c_double), ("rho_max", C.c_double)]


class TmpcSqpOpts(C.Structure):
    _fields_ = [("max_sqp", C.c_int32), ("admm_iters", C.c_int32), ("n_alpha", C.c_int32), ("reserved", C.c_int32), ("eps_c", C.c_double), ("eta", C.c_double)]


class TmpcInfo(C.Structure):
    _fields_ = [("r_prim", C.c_void_p), ("r_dual", C.c_void_p), ("objective", C.c_void_p), ("status", C.c_void_p)]


_LIB = None


def lib():
    """Loads libtmpc.so (built in-tree by __graft_entry__.build()).  Raises if it is missing: no fallback."""
    global _LIB
    if _LIB is None:
        if not os.path.exists(LIB_PATH):
            raise RuntimeError(f"{LIB_PATH} not built: run `python -c 'import __graft_entry__ as g; g.build()'` (no CPU fallback)")
        L = C.CDLL(LIB_PATH)
        L.tmpc_status_string.restype = C.c_char_p
        L.tmpc_status_string.argtypes = [C.c_int]
        L.tmpc_launch_count.restype = C.c_int64
        L.tmpc_launch_count.argtypes = [C.c_void_p]
        L.tmpc_workspace_bytes.argtypes = [C.c_void_p, C.POINTER(C.c_size_t)]
        L.tmpc_host_staging_bytes.argtypes = [C.c_void_p, C.POINTER(C.c_size_t)]
        L.tmpc_setup.argtypes = [C.c_void_p, C.c_void_p, C.c_size_t, C.c_void_p, C.POINTER(C.c_void_p)]
        L.tmpc_linearize.argtypes = [C.c_void_p] * 4
        L.tmpc_factor.argtypes = [C.c_void_p] * 2
        L.tmpc_admm_solve.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_int32, C.c_int32, C.c_void_p]
        L.tmpc_backward.argtypes = [C.c_void_p] * 5 + [C.c_int32, C.c_int32, C.c_void_p, C.c_void_p]
        L.tmpc_kkt_solve.argtypes = [C.c_void_p] * 3
        L.tmpc_admm_solve_host.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_int32, C.c_int32, C.c_void_p, C.c_void_p, C.c_size_t]
        L.tmpc_destroy.argtypes = [C.c_void_p]
        L.tmpc_admm_solve_static.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_int32, C.c_int32, C.c_void_p, C.c_void_p]
        L.tmpc_backward_dgamma.argtypes = [C.c_void_p] * 5
        L.tmpc_sqp_solve.argtypes = [C.c_void_p] * 9
        L.tmpc_admm_solve_adaptive.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.c_int32, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p]
        L.tmpc_measure_peak.argtypes = [C.c_int32, C.c_void_p, C.c_void_p, C.c_int32, C.POINTER(C.c_double)]
        _LIB = L
    return _LIB


class TmpcError(RuntimeError):
    pass


def _check(rc: int, what: str):
    if rc != 0:
        raise TmpcError(f"{what}: {lib().tmpc_status_string(rc).decode()} (status {rc})")


def make_config(w, batch=None, dtype=None, linsolve=TMPC_LIN_SEQUENTIAL, eps_abs=None, eps_rel=None) -> TmpcConfig:
    """TmpcConfig from a workloads.QPData."""
    c = TmpcConfig()
    dt = w.dtype if dtype is None else dtype
    c.batch, c.N, c.nx, c.nu, c.ng = (w.B if batch is None else batch), w.N, w.nx, w.nu, w.ng
    c.dtype = TMPC_F64 if dt == "f64" else TMPC_F32
    c.model, c.linsolve = w.model, linsolve
    c.sigma, c.rho_bar, c.rho_eq_scale, c.alpha = w.sigma, w.rho_bar, w.rho_eq_scale, w.alpha
    c.slack_gamma, c.slack_lambda = w.gamma, w.lam
    tol = 1e-8 if dt == "f64" else 1e-4
    c.eps_active_abs = tol if eps_abs is None else eps_abs
    c.eps_active_rel = tol if eps_rel is None else eps_rel
    c.wheelbase, c.dt = w.wheelbase, w.dt
    c.g_is_selection = int(w.G is None and w.g_col is not None and w.model != 1)      # (the bicycle model writes a dense G)
    if getattr(w, 'model_params', None) is not None:
        for i, v in enumerate(w.model_params):
            c.model_params[i] = float(v)
    for r in range(w.ng):
        c.soft_row[r] = int(w.soft[r])
        if c.g_is_selection:
            c.g_col[r] = int(w.g_col[r])
        if w.g_lo is not None:
            c.g_lo[r], c.g_hi[r] = w.g_lo[r], w.g_hi[r]
    return c


def tmpc_workspace_bytes(cfg: TmpcConfig) -> int:
    n = C.c_size_t()
    _check(lib().tmpc_workspace_bytes(C.byref(cfg), C.byref(n)), "tmpc_workspace_bytes")
    return n.value


def tmpc_host_staging_bytes(cfg: TmpcConfig) -> int:
    n = C.c_size_t()
    _check(lib().tmpc_host_staging_bytes(C.byref(cfg), C.byref(n)), "tmpc_host_staging_bytes")
    return n.value


def tmpc_setup(cfg: TmpcConfig, workspace_ptr: int, nbytes: int, stream_ptr: int) -> int:
    h = C.c_void_p()
    _check(lib().tmpc_setup(C.byref(cfg), workspace_ptr, nbytes, stream_ptr, C.byref(h)), "tmpc_setup")
    return h.value


def tmpc_linearize(h, xbar_ptr, ref_ptr, qp: TmpcQp):
    _check(lib().tmpc_linearize(h, xbar_ptr, ref_ptr, C.byref(qp)), "tmpc_linearize")


def tmpc_factor(h, qp: TmpcQp):
    _check(lib().tmpc_factor(h, C.byref(qp)), "tmpc_factor")


def tmpc_admm_solve(h, qp: TmpcQp, st: TmpcState, iters: int, flags: int = 0, info: TmpcInfo | None = None):
    _check(lib().tmpc_admm_solve(h, C.byref(qp), C.byref(st), iters, flags, C.byref(info) if info is not None else None), "tmpc_admm_solve")


def tmpc_backward(h, qp, st, dLdx_ptr, dLdxi_ptr, mode, iters, dq_ptr, dxinit_ptr):
    _check(lib().tmpc_backward(h, C.byref(qp), C.byref(st), dLdx_ptr, dLdxi_ptr, mode, iters, dq_ptr, dxinit_ptr), "tmpc_backward")


def tmpc_kkt_solve(h, eta_ptr, xt_ptr):
    _check(lib().tmpc_kkt_solve(h, eta_ptr, xt_ptr), "tmpc_kkt_solve")


def tmpc_admm_solve_host(h, qp, st, iters, flags, info, staging_ptr, staging_bytes):
    _check(lib().tmpc_admm_solve_host(h, C.byref(qp), C.byref(st), iters, flags, C.byref(info) if info is not None else None,
                                      staging_ptr, staging_bytes), "tmpc_admm_solve_host")


def tmpc_destroy(h):
    lib().tmpc_destroy(h)


def tmpc_launch_count(h) -> int:
    return int(lib().tmpc_launch_count(h))


TMPC_PEAK_FFMA2, TMPC_PEAK_FFMA, TMPC_PEAK_DFMA, TMPC_PEAK_LDS = 0, 1, 2, 3


def tmpc_measure_peak(what: int, scratch_ptr: int, stream_ptr: int, reps: int = 5) -> float:
    out = C.c_double()
    _check(lib().tmpc_measure_peak(what, scratch_ptr, stream_ptr, reps, C.byref(out)), "tmpc_measure_peak")
    return out.value


def tmpc_admm_solve_adaptive(h, qp, st, ad: TmpcAdaptive, flags=0, info=None, iters_ptr=None, converged_ptr=None, rho_ptr=None):
    _check(lib().tmpc_admm_solve_adaptive(h, C.byref(qp), C.byref(st), C.byref(ad), flags, C.byref(info) if info is not None else None,
                                          iters_ptr, converged_ptr, rho_ptr), "tmpc_admm_solve_adaptive")


def tmpc_sqp_solve(h, qp, st, ref_ptr, opts: TmpcSqpOpts, iters_ptr=None, converged_ptr=None, alpha_ptr=None, kkt_ptr=None):
    _check(lib().tmpc_sqp_solve(h, C.byref(qp), C.byref(st), ref_ptr, C.byref(opts), iters_ptr, converged_ptr, alpha_ptr, kkt_ptr), "tmpc_sqp_solve")


def tmpc_backward_dgamma(h, qp, st, dq_ptr, out_ptr):
    _check(lib().tmpc_backward_dgamma(h, C.byref(qp), C.byref(st), dq_ptr, out_ptr), "tmpc_backward_dgamma")


TMPC_STATIC_SCRATCH_BYTES = 8 << 20
TMPC_E_STATIC_LIMIT = 7


def tmpc_admm_solve_static(cfg: TmpcConfig, qp: TmpcQp, st: TmpcState, iters: int, flags: int = 0, info: TmpcInfo | None = None, stream_ptr=None):
    """Allocation-free factor + solve on the library's static device scratch (see include/tmpc.h); no handle, no workspace."""
    _check(lib().tmpc_admm_solve_static(C.byref(cfg), C.byref(qp), C.byref(st), iters, flags, C.byref(info) if info is not None else None, stream_ptr),
           "tmpc_admm_solve_static")
