"""`Solver`: a tmpc handle + its workspace + the device tensors of one batch of QPs.  Marshalling only —
no arithmetic of the method happens in Python (uploads, pointer packing, and the fixed-count SQP call sequence
tmpc_linearize -> tmpc_factor -> tmpc_admm_solve of SURVEY.md 3.5)."""
from __future__ import annotations

import numpy as np
import torch

from . import binding as B


def _tdtype(dt: str):
    return torch.float64 if dt == "f64" else torch.float32


class Solver:
    def __init__(self, w, dtype=None, device="cuda:0", linsolve=B.TMPC_LIN_SEQUENTIAL, stream=None, eps_abs=None, eps_rel=None):
        if not torch.cuda.is_available():
            raise RuntimeError("tmpc needs a CUDA device: there is no CPU fallback")
        B.lib()
        self.w = w
        self.dt = w.dtype if dtype is None else dtype
        self.td = _tdtype(self.dt)
        self.dev = torch.device(device)
        self.cfg = B.make_config(w, dtype=self.dt, linsolve=linsolve, eps_abs=eps_abs, eps_rel=eps_rel)
        self.stream = stream if stream is not None else torch.cuda.current_stream(self.dev)
        nbytes = B.tmpc_workspace_bytes(self.cfg)
        self.workspace = torch.empty(nbytes + 256, dtype=torch.uint8, device=self.dev)
        base = self.workspace.data_ptr()
        self.ws_ptr = (base + 255) // 256 * 256
        self.h = B.tmpc_setup(self.cfg, self.ws_ptr, nbytes, self.stream.cuda_stream)
        self.t = {}
        self.upload(w)
        self.reset_state()
        Bn = w.B
        self.info = dict(r_prim=torch.zeros(Bn, dtype=self.td, device=self.dev), r_dual=torch.zeros(Bn, dtype=self.td, device=self.dev),
                         objective=torch.zeros(Bn, dtype=self.td, device=self.dev), status=torch.zeros(Bn, dtype=torch.int32, device=self.dev))

    # ---- device tensors
    def _up(self, a):
        return torch.from_numpy(np.ascontiguousarray(a)).to(self.td).to(self.dev)

    def upload(self, w):
        T, n, nx, ng, N, Bn = w.T, w.n, w.nx, w.ng, w.N, w.B
        t = self.t
        t["D"], t["E"], t["q"], t["x_init"] = self._up(w.D), self._up(w.E), self._up(w.q), self._up(w.x_init)
        if w.model == 0:
            t["Am"], t["Ap"], t["b"], t["lo"], t["hi"] = self._up(w.Am), self._up(w.Ap), self._up(w.b), self._up(w.lo), self._up(w.hi)
            t["G"] = self._up(w.G) if w.G is not None else None
        elif w.model == B.TMPC_MODEL_SRB:                 # box bounds on u (selection rows): tmpc_linearize writes Am, Ap, b only
            z = lambda *s: torch.zeros(*s, dtype=self.td, device=self.dev)
            t["Am"], t["Ap"], t["b"] = z(Bn, N, nx, n), z(Bn, N, nx, n), z(Bn, N, nx)
            t["G"], t["lo"], t["hi"] = None, self._up(w.lo), self._up(w.hi)
            t["stage_ref"] = self._up(w.stage_ref)
        else:
            z = lambda *s: torch.zeros(*s, dtype=self.td, device=self.dev)
            t["Am"], t["Ap"], t["b"] = z(Bn, N, nx, n), z(Bn, N, nx, n), z(Bn, N, nx)
            t["G"], t["lo"], t["hi"] = z(Bn, T, ng, n), z(Bn, T, ng), z(Bn, T, ng)
            t["stage_ref"] = self._up(w.stage_ref)
        self.qp = self.make_qp(t)

    def make_qp(self, t) -> B.TmpcQp:
        q = B.TmpcQp()
        q.D, q.D_bstride = t["D"].data_ptr(), (0 if t["D"].shape[0] == 1 else t["D"][0].numel())
        q.E, q.E_bstride = t["E"].data_ptr(), (0 if t["E"].shape[0] == 1 else t["E"][0].numel())
        q.q, q.Am, q.Ap, q.b, q.x_init = t["q"].data_ptr(), t["Am"].data_ptr(), t["Ap"].data_ptr(), t["b"].data_ptr(), t["x_init"].data_ptr()
        if t["G"] is not None:
            q.G, q.G_bstride = t["G"].data_ptr(), (0 if t["G"].shape[0] == 1 else t["G"][0].numel())
        else:
            q.G, q.G_bstride = None, 0
        q.lo, q.hi = t["lo"].data_ptr(), t["hi"].data_ptr()
        return q

    def reset_state(self, x0=None):
        w = self.w
        z = lambda *s: torch.zeros(*s, dtype=self.td, device=self.dev)
        mf = w.nx + w.N * w.nx
        self.s = dict(x=z(w.B, w.T, w.n) if x0 is None else self._up(x0), zg=z(w.B, w.T, w.ng), yf=z(w.B, mf), yg=z(w.B, w.T, w.ng), xi=z(w.B, w.T, w.ng))
        self.st = B.TmpcState(*[self.s[k].data_ptr() for k in ("x", "zg", "yf", "yg", "xi")])

    def set_state(self, state):
        for k in ("x", "zg", "yf", "yg", "xi"):
            self.s[k].copy_(self._up(state[k]).reshape(self.s[k].shape))

    def _info(self):
        i = self.info
        return B.TmpcInfo(i["r_prim"].data_ptr(), i["r_dual"].data_ptr(), i["objective"].data_ptr(), i["status"].data_ptr())

    # ---- the five entry points
    def linearize(self, xbar=None):
        xb = self.s["x"] if xbar is None else xbar
        B.tmpc_linearize(self.h, xb.data_ptr(), self.t["stage_ref"].data_ptr(), self.qp)

    def factor(self):
        B.tmpc_factor(self.h, self.qp)

    def admm_solve(self, iters=None, flags=0):
        B.tmpc_admm_solve(self.h, self.qp, self.st, self.w.iters if iters is None else iters, flags, self._info())

    def solve(self, iters=None):
        """configs 1-3: tmpc_factor + tmpc_admm_solve."""
        self.factor()
        self.admm_solve(iters)

    def solve_adaptive(self, max_iters, eps_abs=1e-3, eps_rel=1e-3, check_every=25, ratio=5.0, rho_min=1e-6, rho_max=1e6, adapt_rho=True, flags=0):
        """f1: tmpc_factor + tmpc_admm_solve_adaptive (paper defaults of PAPER.md:303).  Returns dict(iters, converged, rho) as numpy arrays."""
        w = self.w
        self.factor()
        it = torch.zeros(w.B, dtype=torch.int32, device=self.dev); cv = torch.zeros(w.B, dtype=torch.int32, device=self.dev)
        rho = torch.zeros(w.B, dtype=self.td, device=self.dev)
        ad = B.TmpcAdaptive(int(max_iters), int(check_every), int(bool(adapt_rho)), 0, eps_abs, eps_rel, ratio, rho_min, rho_max)
        B.tmpc_admm_solve_adaptive(self.h, self.qp, self.st, ad, flags, self._info(), it.data_ptr(), cv.data_ptr(), rho.data_ptr())
        torch.cuda.synchronize(self.dev)
        return dict(iters=it.cpu().numpy(), converged=cv.cpu().numpy(), rho=rho.cpu().double().numpy())

    def sqp(self, n_sqp=None, iters=None):
        """configs 4-5: n_sqp x (linearize at xbar = current x -> factor -> ADMM warm start), full steps (reading A-26)."""
        for _ in range(self.w.sqp_iters if n_sqp is None else n_sqp):
            self.linearize()
            self.factor()
            self.admm_solve(iters)

    def sqp_linesearch(self, max_sqp=10, admm_iters=50, eps_c=1e-3, n_alpha=8, eta=0.4):
        """f2: tmpc_sqp_solve from the current state.  Returns dict(iters, converged, alpha [B,max_sqp], kkt [B,3]) as numpy arrays."""
        w = self.w
        it = torch.zeros(w.B, dtype=torch.int32, device=self.dev); cv = torch.zeros(w.B, dtype=torch.int32, device=self.dev)
        al = torch.zeros(w.B, max_sqp, dtype=self.td, device=self.dev); kk = torch.zeros(w.B, 3, dtype=self.td, device=self.dev)
        B.tmpc_sqp_solve(self.h, self.qp, self.st, self.t["stage_ref"].data_ptr(), B.TmpcSqpOpts(max_sqp, admm_iters, n_alpha, 0, eps_c, eta),
                         it.data_ptr(), cv.data_ptr(), al.data_ptr(), kk.data_ptr())
        torch.cuda.synchronize(self.dev)
        return dict(iters=it.cpu().numpy(), converged=cv.cpu().numpy(), alpha=al.cpu().double().numpy(), kkt=kk.cpu().double().numpy())

    def backward(self, dLdx, dLdxi=None, mode=B.TMPC_BWD_REFACTOR_REFINE, iters=None):
        w = self.w
        if iters is None:
            iters = (4 if self.dt == "f64" else 8) if mode == B.TMPC_BWD_REFACTOR_REFINE else 1000
        dq = torch.zeros(w.B, w.T, w.n, dtype=self.td, device=self.dev)
        dxi = torch.zeros(w.B, w.nx, dtype=self.td, device=self.dev)
        B.tmpc_backward(self.h, self.qp, self.st, dLdx.data_ptr(), None if dLdxi is None else dLdxi.data_ptr(), mode, iters, dq.data_ptr(), dxi.data_ptr())
        return dq, dxi

    def backward_dgamma(self, dq):
        """eq. 66 after a backward() call on the same state: dL/dgamma_xi [B]."""
        out = torch.zeros(self.w.B, dtype=self.td, device=self.dev)
        B.tmpc_backward_dgamma(self.h, self.qp, self.st, dq.data_ptr(), out.data_ptr())
        return out

    def kkt_solve(self, eta):
        xt = torch.empty_like(eta)
        B.tmpc_kkt_solve(self.h, eta.data_ptr(), xt.data_ptr())
        return xt

    def state_numpy(self):
        torch.cuda.synchronize(self.dev)
        return {k: v.detach().cpu().double().numpy() for k, v in self.s.items()}

    def info_numpy(self):
        torch.cuda.synchronize(self.dev)
        return {k: v.detach().cpu().numpy() for k, v in self.info.items()}

    def launches(self) -> int:
        return B.tmpc_launch_count(self.h)

    def close(self):
        if self.h:
            torch.cuda.synchronize(self.dev)
            B.tmpc_destroy(self.h)
            self.h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass
