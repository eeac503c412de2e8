"""ctypes front-end of the CPU oracle (oracle/tmpc_oracle.cpp).  TEST INFRASTRUCTURE ONLY.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may import
this package; the product path (paper_2606_24039_b200) never does.  This file marshals numpy arrays
into the C entry points and holds none of the method's arithmetic.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

from .build import build as _build

_LIB = None
MAXR = 64


class Cfg(C.Structure):
    _fields_ = [
        ("N", C.c_int32), ("nx", C.c_int32), ("nu", C.c_int32), ("ng", C.c_int32),
        ("band", C.c_int32), ("g_sel", C.c_int32), ("zg_given", C.c_int32), ("model", C.c_int32),
        ("sigma", C.c_double), ("rho_bar", C.c_double), ("rho_eq_scale", C.c_double), ("alpha", C.c_double),
        ("gamma", C.c_double), ("lam", C.c_double), ("eps_abs", C.c_double), ("eps_rel", C.c_double),
        ("wheelbase", C.c_double), ("dt", C.c_double),
        ("g_lo", C.c_double * MAXR), ("g_hi", C.c_double * MAXR),
        ("g_col", C.c_int32 * MAXR), ("soft", C.c_uint8 * MAXR), ("model_params", C.c_double * 16),
    ]


def lib():
    global _LIB
    if _LIB is None:
        _LIB = C.CDLL(_build())
        assert _LIB.orc_sizeof_cfg() == C.sizeof(Cfg), "oracle Cfg layout mismatch"
        _LIB.orc_project.argtypes = [C.c_int] + [C.c_double] * 6 + [C.POINTER(C.c_double)] * 2
        _LIB.orc_project.restype = None
    return _LIB


def _p(a):
    if a is None:
        return None
    assert a.dtype == np.float64 and a.flags["C_CONTIGUOUS"]
    return a.ctypes.data_as(C.c_void_p)


def _c(a):
    return None if a is None else np.ascontiguousarray(a, dtype=np.float64)


def make_cfg(w, band=None, zg_given=0, eps_abs=1e-8, eps_rel=1e-8, **over) -> Cfg:
    """Cfg from a workloads.QPData (plus overrides such as rho_bar=..., lam=...)."""
    c = Cfg()
    c.N, c.nx, c.nu, c.ng = w.N, w.nx, w.nu, w.ng
    nz = (w.N + 1) * (w.nx + w.nu)
    c.band = int(nz > 512) if band is None else int(band)
    c.g_sel = int(w.g_col is not None and w.G is None and w.model != 1)      # (the bicycle model writes a dense G)
    c.zg_given = zg_given
    c.model = w.model
    c.sigma, c.rho_bar, c.rho_eq_scale, c.alpha = w.sigma, w.rho_bar, w.rho_eq_scale, w.alpha
    c.gamma, c.lam = w.gamma, w.lam
    c.eps_abs, c.eps_rel = eps_abs, eps_rel
    c.wheelbase, c.dt = w.wheelbase, w.dt
    for r in range(w.ng):
        c.soft[r] = int(w.soft[r])
        if c.g_sel:
            c.g_col[r] = int(w.g_col[r])
        if w.g_lo is not None:
            c.g_lo[r], c.g_hi[r] = w.g_lo[r], w.g_hi[r]
    if getattr(w, 'model_params', None) is not None:
        for i, v in enumerate(w.model_params):
            c.model_params[i] = float(v)
    for k, v in over.items():
        setattr(c, k, v)
    return c


def _dims(w):
    n = w.nx + w.nu
    T = w.N + 1
    return n, T, T * n, w.nx + w.N * w.nx, T * w.ng


def _bs(a, b):
    """Per-problem view of a [B|1,...] array."""
    return a[b if a.shape[0] > 1 else 0]


def assemble_S(w, cfg, b=0) -> np.ndarray:
    n, T, nz, mf, mg = _dims(w)
    S = np.zeros((nz, nz))
    D, E, Am, Ap = _c(_bs(w.D, b)), _c(_bs(w.E, b)), _c(w.Am[b]), _c(w.Ap[b])
    G = None if cfg.g_sel else _c(_bs(w.G, b))
    lib().orc_assemble_S(C.byref(cfg), _p(D), _p(E), _p(Am), _p(Ap), _p(G), _p(S))
    return S


def solve_S(w, cfg, eta, b=0) -> np.ndarray:
    n, T, nz, mf, mg = _dims(w)
    xt = np.zeros(nz)
    D, E, Am, Ap = _c(_bs(w.D, b)), _c(_bs(w.E, b)), _c(w.Am[b]), _c(w.Ap[b])
    G = None if cfg.g_sel else _c(_bs(w.G, b))
    rc = lib().orc_solve_S(C.byref(cfg), _p(D), _p(E), _p(Am), _p(Ap), _p(G), _p(_c(eta)), _p(xt))
    assert rc == 0
    return xt


def project(soft, v, lo, hi, rho, gamma, lam):
    z, xi = C.c_double(), C.c_double()
    lib().orc_project(int(soft), v, lo, hi, rho, gamma, lam, C.byref(z), C.byref(xi))
    return z.value, xi.value


def new_state(w, B=None):
    n, T, nz, mf, mg = _dims(w)
    B = w.B if B is None else B
    return dict(x=np.zeros((B, T, n)), zg=np.zeros((B, T, w.ng)), yf=np.zeros((B, mf)), yg=np.zeros((B, T, w.ng)),
                xi=np.zeros((B, T, w.ng)))


def admm(w, cfg, iters=None, state=None, nthreads=1):
    """Alg. 3 on every problem of the batch.  Returns (state dict, info [B,4] = r_prim, r_dual, objective, min pivot)."""
    n, T, nz, mf, mg = _dims(w)
    iters = w.iters if iters is None else iters
    st = new_state(w) if state is None else {k: _c(v).copy() for k, v in state.items()}
    info = np.zeros((w.B, 4))
    D, E, G = _c(w.D), _c(w.E), (None if cfg.g_sel else _c(w.G))
    sD = 0 if D.shape[0] == 1 else D[0].size
    sE = 0 if E.shape[0] == 1 else E[0].size
    sG = 0 if (G is None or G.shape[0] == 1) else G[0].size
    q, Am, Ap, b, xi0, lo, hi = _c(w.q), _c(w.Am), _c(w.Ap), _c(w.b), _c(w.x_init), _c(w.lo), _c(w.hi)
    f = lib().orc_admm_batch
    f.argtypes = [C.c_void_p, C.c_int, C.c_int, C.c_void_p, C.c_int64, C.c_void_p, C.c_int64] + [C.c_void_p] * 6 + \
                 [C.c_int64] + [C.c_void_p] * 7 + [C.c_int, C.c_void_p]
    rc = f(C.byref(cfg), w.B, nthreads, _p(D), sD, _p(E), sE, _p(q), _p(Am), _p(Ap), _p(b), _p(xi0), _p(G), sG, _p(lo), _p(hi),
           _p(st["x"]), _p(st["zg"]), _p(st["yf"]), _p(st["yg"]), _p(st["xi"]), iters, _p(info))
    return st, info, rc


def admm_rows(w, cfg, soft_rows, iters, state=None):
    """Alg. 3 with a per-row soft flag array soft_rows [B,T,ng] (uint8) instead of the per-row-type mask (adjoint QP, eq. 67)."""
    n, T, nz, mf, mg = _dims(w)
    st = new_state(w) if state is None else {k: _c(v).copy() for k, v in state.items()}
    info = np.zeros((w.B, 4))
    f = lib().orc_admm_rows
    f.argtypes = [C.c_void_p] * 17 + [C.c_int, C.c_void_p]
    sr = np.ascontiguousarray(soft_rows, dtype=np.uint8)
    rc = 0
    for b in range(w.B):
        D, E = _c(_bs(w.D, b)), _c(_bs(w.E, b))
        G = None if cfg.g_sel else _c(_bs(w.G, b))
        rc |= f(C.byref(cfg), _p(D), _p(E), _p(_c(w.q[b])), _p(_c(w.Am[b])), _p(_c(w.Ap[b])), _p(_c(w.b[b])), _p(_c(w.x_init[b])), _p(G),
                _p(_c(w.lo[b])), _p(_c(w.hi[b])), sr[b].ctypes.data_as(C.c_void_p), _p(st["x"][b]), _p(st["zg"][b]), _p(st["yf"][b]),
                _p(st["yg"][b]), _p(st["xi"][b]), iters, _p(info[b]))
    return st, info, rc


class Adaptive(C.Structure):
    _fields_ = [("max_iters", C.c_int32), ("check_every", C.c_int32), ("adapt_rho", C.c_int32), ("pad", C.c_int32),
                ("eps_abs", C.c_double), ("eps_rel", C.c_double), ("ratio", C.c_double), ("rho_min", C.c_double), ("rho_max", C.c_double)]


def make_adaptive(max_iters, eps_abs=1e-3, eps_rel=1e-3, check_every=25, ratio=5.0, rho_min=1e-6, rho_max=1e6, adapt_rho=1) -> Adaptive:
    """Defaults of PAPER.md:303 (k_rho^iter = 25, k_rho^ratio = 5, rho_bar in [1e-6, 1e6])."""
    return Adaptive(max_iters, check_every, adapt_rho, 0, eps_abs, eps_rel, ratio, rho_min, rho_max)


def admm_adaptive(w, cfg, ad, state=None, max_log=256):
    """f1 on every problem.  Returns (state, info [B,8] = r_prim, r_dual, objective, min pivot, iterations, final rho_bar, converged,
    #log rows, log [B,max_log,8] = k, r_prim, r_dual, np, nd, rho before, rho after, converged, rc)."""
    n, T, nz, mf, mg = _dims(w)
    assert lib().orc_sizeof_adaptive() == C.sizeof(Adaptive)
    st = new_state(w) if state is None else {k: _c(v).copy() for k, v in state.items()}
    info = np.zeros((w.B, 8)); log = np.zeros((w.B, max_log, 8))
    f = lib().orc_admm_adaptive
    f.argtypes = [C.c_void_p] * 19 + [C.c_int]
    rc = 0
    for b in range(w.B):
        D, E = _c(_bs(w.D, b)), _c(_bs(w.E, b))
        G = None if cfg.g_sel else _c(_bs(w.G, b))
        rc |= f(C.byref(cfg), C.byref(ad), _p(D), _p(E), _p(_c(w.q[b])), _p(_c(w.Am[b])), _p(_c(w.Ap[b])), _p(_c(w.b[b])), _p(_c(w.x_init[b])), _p(G),
                _p(_c(w.lo[b])), _p(_c(w.hi[b])), _p(st["x"][b]), _p(st["zg"][b]), _p(st["yf"][b]), _p(st["yg"][b]), _p(st["xi"][b]),
                _p(info[b]), _p(log[b]), max_log)
    return st, info, log, rc


class SqpOpt(C.Structure):
    _fields_ = [("max_sqp", C.c_int32), ("admm_iters", C.c_int32), ("n_alpha", C.c_int32), ("pad", C.c_int32), ("eps_c", C.c_double), ("eta", C.c_double)]


def sqp_linesearch_bicycle(w, cfg, max_sqp=10, admm_iters=50, eps_c=1e-3, n_alpha=8, eta=0.4, xbar0=None):
    """f2 on every problem.  Returns (state with x = final iterate, info [B,5] = iterations, converged, stationarity, |f|_inf, violation,
    log [B,max_sqp,10] = alpha, mu, phi0, phi(alpha), c1, dl, accepted, stat, |f|_inf, viol, rc)."""
    n, T, nz, mf, mg = _dims(w)
    assert lib().orc_sizeof_sqpopt() == C.sizeof(SqpOpt)
    op = SqpOpt(max_sqp, admm_iters, n_alpha, 0, eps_c, eta)
    st = new_state(w); st["x"] = _c(w.xbar0 if xbar0 is None else xbar0).copy()
    info = np.zeros((w.B, 5)); log = np.zeros((w.B, max_sqp, 10))
    D, E, q, x0, ref = _c(w.D[0]), _c(w.E[0]), _c(w.q), _c(w.x_init), _c(w.stage_ref)
    fn = lib().orc_sqp_ls_bicycle
    fn.argtypes = [C.c_void_p] * 14
    rc = 0
    for b in range(w.B):
        rc |= fn(C.byref(cfg), C.byref(op), _p(D), _p(E), _p(q[b]), _p(x0[b]), _p(ref[b]), _p(st["x"][b]), _p(st["zg"][b]), _p(st["yf"][b]),
                 _p(st["yg"][b]), _p(st["xi"][b]), _p(info[b]), _p(log[b]))
    return st, info, log, rc


def backward(w, cfg, state, dLdx, dLdxi=None, with_dgamma=False):
    """O-5 on every problem.  Returns dq [B,T,n], dxinit [B,nx], counts [B,2], rc [B] (and dL/dgamma_xi [B], eq. 66, with with_dgamma)."""
    n, T, nz, mf, mg = _dims(w)
    dq = np.zeros((w.B, T, n))
    dxi = np.zeros((w.B, w.nx))
    counts = np.zeros((w.B, 2), dtype=np.int32)
    rcs = np.zeros(w.B, dtype=np.int32)
    f = lib().orc_backward
    f.argtypes = [C.c_void_p] * 20
    dgam = np.zeros(w.B)
    for b in range(w.B):
        D, E = _c(_bs(w.D, b)), _c(_bs(w.E, b))
        G = None if cfg.g_sel else _c(_bs(w.G, b))
        args = [_c(w.q[b]), _c(w.Am[b]), _c(w.Ap[b]), _c(w.b[b]), _c(w.x_init[b])]
        lo, hi = _c(w.lo[b]), _c(w.hi[b])
        x, yg, xi = _c(state["x"][b]), _c(state["yg"][b]), _c(state["xi"][b])
        gx = _c(dLdx[b])
        gxi = None if dLdxi is None else _c(dLdxi[b])
        rcs[b] = f(C.byref(cfg), _p(D), _p(E), *[_p(a) for a in args], _p(G), _p(lo), _p(hi), _p(x), _p(yg), _p(xi), _p(gx), _p(gxi),
                   _p(dq[b]), _p(dxi[b]), counts[b].ctypes.data_as(C.c_void_p), dgam[b:b + 1].ctypes.data_as(C.c_void_p))
    if with_dgamma:
        return dq, dxi, counts, rcs, dgam
    return dq, dxi, counts, rcs


def classify(w, cfg, state, b=0):
    n, T, nz, mf, mg = _dims(w)
    cls = np.zeros(mg, dtype=np.int32)
    f = lib().orc_classify
    f.argtypes = [C.c_void_p] * 15
    D, E = _c(_bs(w.D, b)), _c(_bs(w.E, b))
    G = None if cfg.g_sel else _c(_bs(w.G, b))
    f(C.byref(cfg), _p(D), _p(E), _p(_c(w.q[b])), _p(_c(w.Am[b])), _p(_c(w.Ap[b])), _p(_c(w.b[b])), _p(_c(w.x_init[b])), _p(G),
      _p(_c(w.lo[b])), _p(_c(w.hi[b])), _p(_c(state["x"][b])), _p(_c(state["yg"][b])), _p(_c(state["xi"][b])), cls.ctypes.data_as(C.c_void_p))
    return cls.reshape(T, w.ng)


def bicycle_residual(cfg, vk, vk1):
    f = np.zeros(4)
    fn = lib().orc_bicycle_residual
    fn.argtypes = [C.c_void_p] * 4
    fn(C.byref(cfg), _p(_c(vk)), _p(_c(vk1)), _p(f))
    return f


def bicycle_linearize(w, cfg, xbar, b=0):
    n, T, nz, mf, mg = _dims(w)
    Am = np.zeros((w.N, 4, 6)); Ap = np.zeros((w.N, 4, 6)); bb = np.zeros((w.N, 4))
    G = np.zeros((T, 3, 6)); lo = np.zeros((T, 3)); hi = np.zeros((T, 3))
    fn = lib().orc_bicycle_linearize
    fn.argtypes = [C.c_void_p] * 9
    fn(C.byref(cfg), _p(_c(xbar)), _p(_c(w.stage_ref[b])), _p(Am), _p(Ap), _p(bb), _p(G), _p(lo), _p(hi))
    return Am, Ap, bb, G, lo, hi


def sqp_bicycle(w, cfg, n_sqp=None, iters=None, nthreads=1, with_fnorm=False):
    """O-4 on every problem.  Returns (state dict with x = final xbar, info [B,4], rc[, fnorm [B,n_sqp+1]])."""
    n, T, nz, mf, mg = _dims(w)
    n_sqp = w.sqp_iters if n_sqp is None else n_sqp
    iters = w.iters if iters is None else iters
    st = new_state(w)
    st["x"] = _c(w.xbar0).copy()
    info = np.zeros((w.B, 4))
    D, E, q, x0, ref = _c(w.D[0]), _c(w.E[0]), _c(w.q), _c(w.x_init), _c(w.stage_ref)
    if with_fnorm:
        fn = lib().orc_sqp_bicycle
        fn.argtypes = [C.c_void_p] * 11 + [C.c_int, C.c_int, C.c_void_p, C.c_void_p]
        fnorm = np.zeros((w.B, n_sqp + 1))
        rc = 0
        for b in range(w.B):
            rc |= fn(C.byref(cfg), _p(D), _p(E), _p(q[b]), _p(x0[b]), _p(ref[b]), _p(st["x"][b]), _p(st["zg"][b]), _p(st["yf"][b]),
                     _p(st["yg"][b]), _p(st["xi"][b]), n_sqp, iters, _p(info[b]), _p(fnorm[b]))
        return st, info, rc, fnorm
    fn = lib().orc_sqp_bicycle_batch
    fn.argtypes = [C.c_void_p, C.c_int, C.c_int] + [C.c_void_p] * 10 + [C.c_int, C.c_int, C.c_void_p]
    rc = fn(C.byref(cfg), w.B, nthreads, _p(D), _p(E), _p(q), _p(x0), _p(ref), _p(st["x"]), _p(st["zg"]), _p(st["yf"]), _p(st["yg"]),
            _p(st["xi"]), n_sqp, iters, _p(info))
    return st, info, rc


def srb_step(cfg, x, u):
    """x+ = Phi(x, u): one RK4 step of the SRB humanoid dynamics."""
    out = np.zeros(12)
    fn = lib().orc_srb_step
    fn.argtypes = [C.c_void_p] * 4
    fn(C.byref(cfg), _p(_c(x)), _p(_c(u)), _p(out))
    return out


def srb_linearize(w, cfg, xbar):
    Am = np.zeros((w.N, 12, 18)); Ap = np.zeros((w.N, 12, 18)); b = np.zeros((w.N, 12))
    fn = lib().orc_srb_linearize
    fn.argtypes = [C.c_void_p] * 5
    fn(C.byref(cfg), _p(_c(xbar)), _p(Am), _p(Ap), _p(b))
    return Am, Ap, b


def sqp_linesearch_srb(w, cfg, max_sqp=10, admm_iters=50, eps_c=1e-3, n_alpha=8, eta=0.4, xbar0=None):
    """f2 for the SRB model on every problem; same returns as sqp_linesearch_bicycle."""
    n, T, nz, mf, mg = _dims(w)
    assert lib().orc_sizeof_sqpopt() == C.sizeof(SqpOpt)
    op = SqpOpt(max_sqp, admm_iters, n_alpha, 0, eps_c, eta)
    st = new_state(w); st["x"] = _c(w.xbar0 if xbar0 is None else xbar0).copy()
    info = np.zeros((w.B, 5)); log = np.zeros((w.B, max_sqp, 10))
    D, E = _c(w.D[0]), _c(w.E[0])
    fn = lib().orc_sqp_ls_srb
    fn.argtypes = [C.c_void_p] * 15
    rc = 0
    for b in range(w.B):
        rc |= fn(C.byref(cfg), C.byref(op), _p(D), _p(E), _p(_c(w.q[b])), _p(_c(w.x_init[b])), _p(_c(w.lo[b])), _p(_c(w.hi[b])), _p(st["x"][b]),
                 _p(st["zg"][b]), _p(st["yf"][b]), _p(st["yg"][b]), _p(st["xi"][b]), _p(info[b]), _p(log[b]))
    return st, info, log, rc


def sqp_srb(w, cfg, n_sqp=None, iters=None):
    """O-4 for the SRB model on every problem (selection rows with the workload's constant bounds).  Returns (state with x = final xbar, info, rc)."""
    n_sqp = w.sqp_iters if n_sqp is None else n_sqp
    iters = w.iters if iters is None else iters
    st = new_state(w); st["x"] = _c(w.xbar0).copy()
    info = np.zeros((w.B, 4))
    D, E = _c(w.D[0]), _c(w.E[0])
    fn = lib().orc_sqp_srb
    fn.argtypes = [C.c_void_p] * 12 + [C.c_int, C.c_int, C.c_void_p]
    rc = 0
    for b in range(w.B):
        rc |= fn(C.byref(cfg), _p(D), _p(E), _p(_c(w.q[b])), _p(_c(w.x_init[b])), _p(_c(w.lo[b])), _p(_c(w.hi[b])), _p(st["x"][b]), _p(st["zg"][b]),
                 _p(st["yf"][b]), _p(st["yg"][b]), _p(st["xi"][b]), n_sqp, iters, _p(info[b]))
    return st, info, rc
