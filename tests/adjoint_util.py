"""Test helper: the adjoint QP of eq. 67 built with numpy from a forward solution, for the
TMPC_BWD_ADMM_REUSE_FACTOR parity tests.  Uses only the oracle's row classification and numpy."""
import copy

import numpy as np

import oracle as O


def adjoint_qp(w, cfg, state, dLdx, dLdxi=None):
    """Returns (wa, soft_rows): wa = copy of w with q <- -(dL/dx - G_s' dL/dxi_s), b <- 0, x_init <- 0, bounds lo = hi = 0 on
    active rows and +-inf on inactive rows, lambda = 0; soft_rows [B,T,ng] flags the soft-ACTIVE rows (penalty gamma, the
    gamma G_s'G_s term of eq. 65/67), the hard-active rows stay hard equalities.  Then eta_x = x^K, eta_f = y_f^K of Alg. 3 on wa,
    dL/dq = -eta_x, dL/dx_init = +eta_f[0:nx]."""
    wa = copy.copy(w)
    B, T, ng, n = w.B, w.T, w.ng, w.n
    cls = np.stack([O.classify(w, cfg, state, b) for b in range(B)])          # [B,T,ng]
    Gd = w.G_dense()
    rhs = np.array(dLdx, dtype=np.float64).reshape(B, T, n).copy()
    if dLdxi is not None:
        for b in range(B):
            G = Gd[b if Gd.shape[0] > 1 else 0]
            rhs[b] -= np.einsum("trn,tr->tn", G, np.where(cls[b] == 2, np.asarray(dLdxi)[b].reshape(T, ng), 0.0))
    wa.q = -rhs
    wa.b = np.zeros_like(w.b)
    wa.x_init = np.zeros_like(w.x_init)
    wa.lo = np.where(cls != 0, 0.0, -np.inf)
    wa.hi = np.where(cls != 0, 0.0, np.inf)
    wa.lam = 0.0
    return wa, (cls == 2).astype(np.uint8), cls
