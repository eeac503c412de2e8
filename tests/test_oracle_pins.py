"""Pins of the CPU oracle against what the paper and the mathematics fix (SURVEY.md 8(c) 'What pins each part').

Every expected value here is computed by an independent route written in this file (numpy linear algebra,
closed forms, brute force) — never by re-calling the oracle routine under test.
"""
import itertools

import numpy as np
import pytest

import oracle as O
from paper_2606_24039_b200 import workloads as W


# ----------------------------------------------------------------------------------------------- helpers
def dense_PCG(w, b=0):
    """Dense P, C, c, G of problem b straight from eq. 29-31, numpy only."""
    n, T, N, nx, ng = w.n, w.T, w.N, w.nx, w.ng
    nz, mf, mg = T * n, nx + N * nx, T * ng
    D = w.D[b if w.D.shape[0] > 1 else 0]
    E = w.E[b if w.E.shape[0] > 1 else 0]
    G3 = w.G_dense()
    G3 = G3[b if G3.shape[0] > 1 else 0]
    P = np.zeros((nz, nz)); C = np.zeros((mf, nz)); c = np.zeros(mf); G = np.zeros((mg, nz))
    for t in range(T):
        P[t * n:(t + 1) * n, t * n:(t + 1) * n] = D[t]
        G[t * ng:(t + 1) * ng, t * n:(t + 1) * n] = G3[t]
    for t in range(N):
        P[(t + 1) * n:(t + 2) * n, t * n:(t + 1) * n] = E[t]
        P[t * n:(t + 1) * n, (t + 1) * n:(t + 2) * n] = E[t].T
        C[nx + t * nx: nx + (t + 1) * nx, t * n:(t + 1) * n] = w.Am[b, t]
        C[nx + t * nx: nx + (t + 1) * nx, (t + 1) * n:(t + 2) * n] = w.Ap[b, t]
        c[nx + t * nx: nx + (t + 1) * nx] = w.b[b, t]
    C[:nx, :nx] = np.eye(nx)
    c[:nx] = w.x_init[b]
    return P, C, c, G


def small_family():
    return [
        W.random_ltv(1, 2, 5, 3, 2, [3, 4], [0, 0], implicit=True),
        W.random_ltv(2, 2, 4, 2, 1, [2, 0, 1], [0, 1, 1, 1], implicit=False, dense_g_rows=1),
        W.config2(B=2, N=6),
        W.with_dense_Ap(W.random_ltv(4, 2, 5, 3, 2, [3, 4], [0, 0], implicit=True), seed=1, scale=0.3),   # A^+ with u_{t+1} columns (Remark A1)
    ]


# ----------------------------------------------------------------------------------------------- a2: S assembly
@pytest.mark.parametrize("w", small_family(), ids=lambda w: w.name)
def test_S_equals_theta_phi_block_formulas(w):
    """Oracle S (from P, C, G) == the Theta_t / Phi_t block formulas of PAPER.md:797-801 (retyped here)."""
    cfg = O.make_cfg(w, band=0)
    n, T, N, nx = w.n, w.T, w.N, w.nx
    rf, rg, sg = w.rho_eq_scale * w.rho_bar, w.rho_bar, w.sigma
    for b in range(w.B):
        S = O.assemble_S(w, cfg, b)
        D, E = w.D[0], w.E[0]
        G3 = w.G_dense(); G3 = G3[b if G3.shape[0] > 1 else 0]
        Ainit = np.hstack([np.eye(nx), np.zeros((nx, w.nu))])
        ref = np.zeros_like(S)
        for t in range(T):
            Th = D[t] + sg * np.eye(n) + rg * G3[t].T @ G3[t]
            if t == 0:
                Th += rf * Ainit.T @ Ainit
            if t < N:
                Th += rf * w.Am[b, t].T @ w.Am[b, t]
            if t > 0:
                Th += rf * w.Ap[b, t - 1].T @ w.Ap[b, t - 1]
            ref[t * n:(t + 1) * n, t * n:(t + 1) * n] = Th
            if t < N:
                Ph = E[t] + rf * w.Ap[b, t].T @ w.Am[b, t]
                ref[(t + 1) * n:(t + 2) * n, t * n:(t + 1) * n] = Ph
                ref[t * n:(t + 1) * n, (t + 1) * n:(t + 2) * n] = Ph.T
        assert np.abs(S - ref).max() <= 1e-13 * np.abs(ref).max()


@pytest.mark.parametrize("band", [0, 1])
@pytest.mark.parametrize("w", small_family(), ids=lambda w: w.name)
def test_cholesky_solve_residual(w, band):
    """x~ = S^{-1} eta: residual against a numpy-built S and agreement with numpy.linalg.solve; dense == band."""
    cfg = O.make_cfg(w, band=band)
    P, C, c, G = dense_PCG(w, 0)
    S = P + w.sigma * np.eye(P.shape[0]) + w.rho_eq_scale * w.rho_bar * C.T @ C + w.rho_bar * G.T @ G
    eta = np.random.default_rng(0).standard_normal(P.shape[0])
    xt = O.solve_S(w, cfg, eta, 0)
    assert np.abs(S @ xt - eta).max() <= 1e-11 * np.abs(eta).max()
    assert np.abs(xt - np.linalg.solve(S, eta)).max() <= 1e-10 * np.abs(xt).max()


# ----------------------------------------------------------------------------------------------- a8: projection
def test_projection_forms_agree():
    """eq. 15a/15b == the three-case formula at PAPER.md:836 == oracle (lambda = 0); hard rows == eq. 13."""
    rng = np.random.default_rng(1)
    for _ in range(200):
        lo, hi = sorted(rng.uniform(-2, 2, 2))
        v, rho, gam = rng.uniform(-5, 5), rng.uniform(0.05, 10), rng.uniform(0.1, 20)
        pv = min(max(v, lo), hi)
        z15, xi15 = rho / (gam + rho) * v + gam / (gam + rho) * pv, rho / (gam + rho) * (pv - v)
        if v < lo:
            zc, xic = (rho * v + gam * lo) / (rho + gam), rho / (rho + gam) * (lo - v)
        elif v > hi:
            zc, xic = (rho * v + gam * hi) / (rho + gam), rho / (rho + gam) * (hi - v)
        else:
            zc, xic = v, 0.0
        z, xi = O.project(1, v, lo, hi, rho, gam, 0.0)
        assert abs(z15 - zc) < 1e-13 and abs(xi15 - xic) < 1e-13
        assert abs(z - zc) < 1e-13 and abs(xi - xic) < 1e-13
        zh, xih = O.project(0, v, lo, hi, rho, gam, 0.0)
        assert zh == pv and xih == 0.0
        zi, xii = O.project(1, v, lo, hi, rho, 1e14, 0.0)  # gamma -> inf recovers the hard projection
        assert abs(zi - pv) < 1e-9 and abs(xii) < 1e-9


def test_projection_is_the_prox_minimiser():
    """(z, xi) minimises  lam|xi| + gam/2 xi^2 + rho/2 (z - v)^2  s.t. lo <= z + xi <= hi  (eq. 52a + reading A-14): brute-force grid."""
    rng = np.random.default_rng(2)
    for _ in range(20):
        lo, hi = -0.7, 0.9
        v, rho, gam, lam = rng.uniform(-4, 4), rng.uniform(0.1, 3), rng.uniform(0.5, 4), rng.choice([0.0, 0.3, 2.0])
        z, xi = O.project(1, v, lo, hi, rho, gam, lam)
        f = lambda zz, ss: lam * np.abs(ss) + 0.5 * gam * ss ** 2 + 0.5 * rho * (zz - v) ** 2
        assert lo - 1e-12 <= z + xi <= hi + 1e-12
        zz = np.linspace(-6, 6, 2401)[:, None]; ss = np.linspace(-6, 6, 2401)[None, :]
        F = np.where((zz + ss >= lo - 1e-12) & (zz + ss <= hi + 1e-12), f(zz, ss), np.inf)
        assert f(z, xi) <= F.min() + 1e-12


# ----------------------------------------------------------------------------------------------- LQR Riccati
def riccati_rollout(w, b=0):
    """Finite-horizon affine time-varying LQR by backward Riccati recursion + forward roll-out (textbook), for
    cost sum 1/2 v'D_t v + q_t'v without stage coupling; dynamics x+ = Abar x + Bbar u + cbar with Abar = E^-1 A."""
    n, T, N, nx, nu = w.n, w.T, w.N, w.nx, w.nu
    D = w.D[0]; q = w.q[b]
    Ab, Bb, cb = [], [], []
    for t in range(N):
        Einv = np.linalg.inv(-w.Ap[b, t][:, :nx])
        Ab.append(Einv @ w.Am[b, t][:, :nx]); Bb.append(Einv @ w.Am[b, t][:, nx:]); cb.append(-Einv @ w.b[b, t])
    Pk = D[N][:nx, :nx].copy(); pk = q[N][:nx].copy()
    Ks, ks = [None] * N, [None] * N
    for t in range(N - 1, -1, -1):
        Q, R, M = D[t][:nx, :nx], D[t][nx:, nx:], D[t][:nx, nx:]
        qx, qu = q[t][:nx], q[t][nx:]
        Huu = R + Bb[t].T @ Pk @ Bb[t]
        Hux = M.T + Bb[t].T @ Pk @ Ab[t]
        hu = qu + Bb[t].T @ (Pk @ cb[t] + pk)
        Ks[t] = -np.linalg.solve(Huu, Hux); ks[t] = -np.linalg.solve(Huu, hu)
        Hxx = Q + Ab[t].T @ Pk @ Ab[t]
        hx = qx + Ab[t].T @ (Pk @ cb[t] + pk)
        Pk, pk = Hxx + Hux.T @ Ks[t], hx + Hux.T @ ks[t]
    x = w.x_init[b].copy(); out = np.zeros((T, n))
    for t in range(N):
        u = Ks[t] @ x + ks[t]
        out[t] = np.concatenate([x, u]); x = Ab[t] @ x + Bb[t] @ u + cb[t]
    out[N, :nx] = x
    out[N, nx:] = -np.linalg.solve(D[N][nx:, nx:], q[N][nx:])  # u_N is free of dynamics: minimises its own term
    return out


@pytest.mark.parametrize("mk", [lambda: W.config1(bounded=False),
                                lambda: W.random_ltv(3, 2, 12, 3, 2, [3, 4], [0, 0], bound=np.inf, implicit=True, rate=False, q_scale=0.5)],
                         ids=["cfg1_unbounded", "random_implicit"])
def test_unconstrained_admm_equals_lqr_riccati(mk):
    w = mk()
    cfg = O.make_cfg(w)
    st, info, rc = O.admm(w, cfg, iters=400)
    assert rc == 0
    for b in range(w.B):
        ref = riccati_rollout(w, b)
        assert np.abs(st["x"][b] - ref).max() <= 1e-9 * max(1.0, np.abs(ref).max())


# ----------------------------------------------------------------------------------------------- brute-force active set
def brute_force_qp(P, q, C, c, G, lo, hi):
    """Enumerate every assignment {free, at-lower, at-upper} of the inequality rows, solve the equality-constrained
    QP, keep the primal-feasible / dual-sign-correct one (unique for P > 0)."""
    nz, mf, mg = P.shape[0], C.shape[0], G.shape[0]
    best = None
    for assign in itertools.product((0, -1, 1), repeat=mg):
        act = [i for i in range(mg) if assign[i] != 0]
        rhs_a = np.array([lo[i] if assign[i] < 0 else hi[i] for i in act])
        A = np.vstack([C, G[act]]) if act else C
        K = np.block([[P, A.T], [A, np.zeros((A.shape[0], A.shape[0]))]])
        if np.linalg.matrix_rank(A) < A.shape[0]:
            continue
        sol = np.linalg.solve(K, np.concatenate([-q, c, rhs_a]))
        x, y = sol[:nz], sol[nz + mf:]
        g = G @ x
        if (g < lo - 1e-9).any() or (g > hi + 1e-9).any():
            continue
        ok = all((y[k] <= 1e-9) if assign[i] < 0 else (y[k] >= -1e-9) for k, i in enumerate(act))
        if ok:
            yg = np.zeros(mg); yg[act] = y
            best = (x, sol[nz:nz + mf], yg)
            break
    return best


@pytest.mark.parametrize("seed", [11, 12, 13, 14])
def test_tiny_qp_equals_active_set_enumeration(seed):
    """N=3, nx=2, nu=1, hard bounds on u (4 rows) and x_2 from stage 1 on: converged ADMM == brute force to 1e-8."""
    w = W.random_ltv(seed, 1, 3, 2, 1, [2, 1], [0, 0], bound=0.25, implicit=True, q_scale=1.0)
    w.lo[:, 0, 1], w.hi[:, 0, 1] = -np.inf, np.inf       # x_0 is fixed: its bound row is switched off (reading A-15)
    w.lo[:, :, 1], w.hi[:, :, 1] = np.minimum(w.lo[:, :, 1], -0.6), np.maximum(w.hi[:, :, 1], 0.6)
    w.rho_bar = 1.0
    cfg = O.make_cfg(w)
    st, info, rc = O.admm(w, cfg, iters=6000)
    P, C, c, G = dense_PCG(w, 0)
    fin = np.isfinite(w.lo[0].ravel())
    ref = brute_force_qp(P, w.q[0].ravel(), C, c, G[fin], w.lo[0].ravel()[fin], w.hi[0].ravel()[fin])
    assert ref is not None
    assert info[0, 0] < 1e-9 and info[0, 1] < 1e-9
    assert np.abs(st["x"][0].ravel() - ref[0]).max() < 1e-8
    assert np.abs(st["yg"][0].ravel()[fin] - ref[2]).max() < 1e-6
    assert (np.abs(ref[2]) > 1e-3).sum() >= 1, "instance must have an active row to be a useful pin"


# ----------------------------------------------------------------------------------------------- invariants per iteration
def test_invariants_after_every_iteration():
    """Hard rows: z_g in [lo,hi]; soft rows: z_g + xi in [lo,hi]; gamma xi + lam sgn(xi) + y_g = 0 where xi != 0;
    y_g sign complementarity; one-iteration-at-a-time resume == K iterations at once (z_f == c, w == 0 are structural)."""
    w = W.config2(B=3, N=12, soft_bound=0.5)
    w.rho_bar = 20.0
    soft = np.array(w.soft, dtype=bool)
    cfg1 = O.make_cfg(w, zg_given=1)
    st = O.new_state(w)
    st["zg"] = np.clip(st["x"][:, :, w.g_col], w.lo, w.hi)
    seen_soft = seen_dead = 0
    for k in range(40):
        st, info, rc = O.admm(w, cfg1, iters=1, state=st)
        zg, xi, yg = st["zg"], st["xi"], st["yg"]
        assert (zg[..., ~soft] >= w.lo[..., ~soft] - 1e-14).all() and (zg[..., ~soft] <= w.hi[..., ~soft] + 1e-14).all()
        assert (xi[..., ~soft] == 0).all()
        s = zg + xi
        assert (s[..., soft] >= w.lo[..., soft] - 1e-12).all() and (s[..., soft] <= w.hi[..., soft] + 1e-12).all()
        nzm = xi != 0
        assert np.abs(w.gamma * xi[nzm] + w.lam * np.sign(xi[nzm]) + yg[nzm]).max(initial=0) < 1e-9
        inter = (zg > w.lo + 1e-12) & (zg < w.hi - 1e-12) & ~nzm & ~soft
        assert np.abs(yg[inter]).max(initial=0) < 1e-12           # strictly interior hard rows carry no multiplier
        assert (yg[(zg <= w.lo) & ~soft] <= 1e-12).all() and (yg[(zg >= w.hi) & ~soft] >= -1e-12).all()
        seen_soft += int(nzm.sum()); seen_dead += int(((np.abs(yg) > 1e-9) & ~nzm & soft).sum())
    assert seen_soft > 0 and seen_dead > 0, "stress instance must exercise soft-active and L1 dead-zone rows"
    st2, _, _ = O.admm(w, O.make_cfg(w), iters=40)
    for k in st:
        assert np.abs(st[k] - st2[k]).max() < 1e-12


def test_config1_converges_below_eps():
    """Residuals (eq. 3) fall below eps_abs + eps_rel * scale (eq. 4) at K=500 on config 1; checked with numpy-built matrices."""
    w = W.config1()
    st, info, rc = O.admm(w, O.make_cfg(w))
    P, C, c, G = dense_PCG(w, 0)
    x, yf, yg, zg = st["x"][0].ravel(), st["yf"][0], st["yg"][0].ravel(), st["zg"][0].ravel()
    rp = max(np.abs(C @ x - c).max(), np.abs(G @ x - zg).max())
    rd = np.abs(P @ x + w.q[0].ravel() + C.T @ yf + G.T @ yg).max()
    assert abs(rp - info[0, 0]) < 1e-12 and abs(rd - info[0, 1]) < 1e-12
    eps = 1e-6
    assert rp <= eps + eps * max(np.abs(C @ x).max(), np.abs(G @ x).max(), np.abs(zg).max())
    assert rd <= eps + eps * max(np.abs(P @ x).max(), np.abs(C.T @ yf + G.T @ yg).max())
    assert abs(info[0, 2] - (0.5 * x @ P @ x + w.q[0].ravel() @ x)) < 1e-9
    assert (np.abs(yg) > 1e-6).sum() > 0   # bounds are active: the instance tests the projection


def test_info_slack_terms_recomputed_in_numpy():
    """r_dual's soft-row block  gamma xi + lam sgn(xi) + y_g  (eq. 3 second block with the L1 term of reading A-14) and the
    slack penalty  lam |xi| + gamma/2 xi^2  of the objective, recomputed from numpy-built matrices on the slack-stress
    instance where xi != 0.  The soft-row block is an exact identity of the prox (zero up to rounding), so the objective and
    the x-block are what move; the test also perturbs xi to show the oracle's r_dual sees that block."""
    w = W.config2(B=2, N=12, soft_bound=0.5)
    w.rho_bar = 20.0
    cfg = O.make_cfg(w)
    st, info, rc = O.admm(w, cfg, iters=60)
    assert (st["xi"] != 0).sum() > 10
    for b in range(w.B):
        P, C, c, G = dense_PCG(w, b)
        x, yf, yg, zg, xi = st["x"][b].ravel(), st["yf"][b], st["yg"][b].ravel(), st["zg"][b].ravel(), st["xi"][b].ravel()
        soft = np.tile(np.array(w.soft, dtype=bool), w.T)
        m = soft & (xi != 0)
        rd = max(np.abs(P @ x + w.q[b].ravel() + C.T @ yf + G.T @ yg).max(), np.abs(w.gamma * xi[m] + w.lam * np.sign(xi[m]) + yg[m]).max(initial=0))
        obj = 0.5 * x @ P @ x + w.q[b].ravel() @ x + (w.lam * np.abs(xi[m]) + 0.5 * w.gamma * xi[m] ** 2).sum()
        rp = max(np.abs(C @ x - c).max(), np.abs(G @ x - zg).max())
        assert abs(rp - info[b, 0]) < 1e-12 and abs(rd - info[b, 1]) < 1e-11 * max(1, rd) and abs(obj - info[b, 2]) < 1e-10 * abs(obj)
        assert (w.lam * np.abs(xi[m]) + 0.5 * w.gamma * xi[m] ** 2).sum() > 1e-3 * abs(obj)       # the penalty is visible in the objective
    # the soft-row block of r_dual: resume with zero further iterations from a state whose xi was scaled by 100 -> that block dominates
    st2 = {k: v.copy() for k, v in st.items()}
    st2["xi"] = 100.0 * st["xi"]
    _, info2, _ = O.admm(w, O.make_cfg(w, zg_given=1), iters=0, state=st2)
    for b in range(w.B):
        xi, yg = st2["xi"][b].ravel(), st2["yg"][b].ravel()
        m = np.tile(np.array(w.soft, dtype=bool), w.T) & (xi != 0)
        blk = np.abs(w.gamma * xi[m] + w.lam * np.sign(xi[m]) + yg[m]).max()
        assert blk > 2 * info[b, 1] and abs(info2[b, 1] - blk) < 1e-12 * blk


def _kkt_form_iteration(P, q, A, lo, hi, soft, sigma, rho, alpha, gamma, lam, x, z, y):
    """One iteration of Alg. 3 in the paper's ORIGINAL form: the quasi-definite KKT system eq. 7 solved
    with numpy for (x~, nu), z~ = z + rho^-1 (nu - y) (OSQP's recovery, equivalent to eq. 9), then eq. 10-16."""
    nz, m = P.shape[0], A.shape[0]
    K = np.block([[P + sigma * np.eye(nz), A.T], [A, -np.diag(1.0 / rho)]])
    sol = np.linalg.solve(K, np.concatenate([sigma * x - q, z - y / rho]))
    xt, nu = sol[:nz], sol[nz:]
    zt = z + (nu - y) / rho
    xn = alpha * xt + (1 - alpha) * x
    zh = alpha * zt + (1 - alpha) * z
    v = zh + y / rho
    pv = np.clip(v, lo, hi)
    sp = np.maximum(0.0, (rho * (v - hi) - lam) / (rho + gamma)); sm = np.maximum(0.0, (rho * (lo - v) - lam) / (rho + gamma))
    zn = np.where(soft, pv + sp - sm, pv)
    xin = np.where(soft, sm - sp, 0.0)
    yn = y + rho * (zh - zn)
    return xn, zn, yn, xin


@pytest.mark.parametrize("sigma,alpha", [(1e-6, 1.6), (0.3, 1.6), (0.3, 0.7)])
def test_iterates_equal_kkt_form_of_eq7_every_iteration(sigma, alpha):
    """Trajectory pin (not a fixed-point pin): after EVERY iteration the oracle's (x, z_g, y_f, y_g, xi) equal the iteration
    written in the paper's un-reduced form — eq. 7 with the full stacked A = [C; G], l = [c; lo], u = [c; hi] (eq. 2), i.e.
    equality rows treated like any other row (z_f is projected onto [c, c]) — with a LARGE sigma so that the relaxation of x
    (eq. 10-11) is visible in eta, and alpha != 1 so that its placement in both dual updates matters."""
    w = W.random_ltv(5, 1, 4, 3, 2, [3, 4, 0], [0, 0, 1], bound=0.3, implicit=True, dense_g_rows=1, q_scale=0.6)
    w = W.with_dense_Ap(w, seed=2, scale=0.3)                                          # general A^+ (u_{t+1} columns, Remark A1)
    w.soft = [0, 0, 1, 1]; w.lam = 0.05; w.sigma = sigma; w.alpha = alpha; w.rho_bar = 0.7; w.rho_eq_scale = 13.0
    P, C, c, G = dense_PCG(w, 0)
    A = np.vstack([C, G]); mf = C.shape[0]
    lo = np.concatenate([c, w.lo[0].ravel()]); hi = np.concatenate([c, w.hi[0].ravel()])
    soft = np.concatenate([np.zeros(mf, bool), np.tile(np.array(w.soft, bool), w.T)])
    rho = np.concatenate([np.full(mf, w.rho_eq_scale * w.rho_bar), np.full(G.shape[0], w.rho_bar)])
    rng = np.random.default_rng(3)
    st = O.new_state(w)
    st["x"] = 0.2 * rng.standard_normal(st["x"].shape); st["yf"] = 0.1 * rng.standard_normal(st["yf"].shape); st["yg"] = 0.1 * rng.standard_normal(st["yg"].shape)
    x, y = st["x"][0].ravel().copy(), np.concatenate([st["yf"][0], st["yg"][0].ravel()])
    z = np.concatenate([c, np.clip(G @ x, w.lo[0].ravel(), w.hi[0].ravel())])        # z_f == c, z_g^0 = clip(G x^0) (reading A-12)
    seen_xi = 0
    for k in range(25):
        st, info, rc = O.admm(w, O.make_cfg(w, zg_given=int(k > 0)), iters=1, state=st)
        x, z, y, xi = _kkt_form_iteration(P, w.q[0].ravel(), A, lo, hi, soft, sigma, rho, alpha, w.gamma, w.lam, x, z, y)
        assert np.abs(z[:mf] - c).max() == 0                                        # z_f == c
        for got, ref in ((st["x"][0].ravel(), x), (st["zg"][0].ravel(), z[mf:]), (st["yf"][0], y[:mf]), (st["yg"][0].ravel(), y[mf:]), (st["xi"][0].ravel(), xi[mf:])):
            assert np.abs(got - ref).max() <= 1e-10 * max(1.0, np.abs(ref).max()), k
        seen_xi += int((xi != 0).sum())
    assert seen_xi > 0


def test_equality_rows_posed_as_inequality_rows_give_the_same_iterates():
    """z_f == c / y_f pin: a two-stage problem (N = 1) is re-posed as ONE fat stage (N = 0) whose
    inequality block holds the original G rows AND the dynamics rows [A^- A^+] v = b as two-sided rows lo = hi = b.  With
    rho_eq_scale = 1 both problems have the same S, and the general row update y += rho(z^ - clip(.)) must reproduce the
    native equality update y_f += rho_f alpha (z~_f - c) after every iteration."""
    import copy
    w = W.random_ltv(8, 1, 1, 2, 1, [2, 0], [0, 1], bound=0.2, implicit=True, q_scale=0.8)
    w.rho_eq_scale = 1.0; w.rho_bar = 3.0; w.alpha = 1.7; w.sigma = 0.05
    n, nx, ng = w.n, w.nx, w.ng
    f = copy.copy(w)
    f.N, f.nx, f.nu, f.ng = 0, nx, 2 * n - nx, 2 * ng + nx
    f.D = np.zeros((1, 1, 2 * n, 2 * n)); f.D[0, 0, :n, :n] = w.D[0, 0]; f.D[0, 0, n:, n:] = w.D[0, 1]; f.D[0, 0, n:, :n] = w.E[0, 0]; f.D[0, 0, :n, n:] = w.E[0, 0].T
    f.E = np.zeros((1, 0, 2 * n, 2 * n)); f.Am = np.zeros((1, 0, nx, 2 * n)); f.Ap = np.zeros((1, 0, nx, 2 * n)); f.b = np.zeros((1, 0, nx))
    f.q = w.q.reshape(1, 1, 2 * n)
    Gd = w.G_dense()[0]
    f.G = np.zeros((1, 1, f.ng, 2 * n)); f.G[0, 0, :ng, :n] = Gd[0]; f.G[0, 0, ng:2 * ng, n:] = Gd[1]
    f.G[0, 0, 2 * ng:, :n] = w.Am[0, 0]; f.G[0, 0, 2 * ng:, n:] = w.Ap[0, 0]
    f.g_col = None
    f.lo = np.concatenate([w.lo[0, 0], w.lo[0, 1], w.b[0, 0]]).reshape(1, 1, -1); f.hi = np.concatenate([w.hi[0, 0], w.hi[0, 1], w.b[0, 0]]).reshape(1, 1, -1)
    f.soft = list(w.soft) * 2 + [0] * nx
    sw, sf = O.new_state(w), O.new_state(f)
    for k in range(30):
        sw, _, rc1 = O.admm(w, O.make_cfg(w, band=0, zg_given=int(k > 0)), iters=1, state=sw)
        sf, _, rc2 = O.admm(f, O.make_cfg(f, band=0, zg_given=int(k > 0)), iters=1, state=sf)
        assert rc1 == 0 and rc2 == 0
        assert np.abs(sw["x"].ravel() - sf["x"].ravel()).max() < 1e-12
        assert np.abs(sw["yf"][0, nx:] - sf["yg"][0, 0, 2 * ng:]).max() < 1e-12 * max(1, np.abs(sw["yf"]).max())      # dynamics multipliers
        assert np.abs(sw["yf"][0, :nx] - sf["yf"][0]).max() < 1e-12 * max(1, np.abs(sw["yf"]).max())                   # init rows stay native in both
        assert np.abs(sw["yg"].ravel() - sf["yg"][0, 0, :2 * ng]).max() < 1e-12 and np.abs(sw["xi"].ravel() - sf["xi"][0, 0, :2 * ng]).max() < 1e-12
        assert np.abs(sf["zg"][0, 0, 2 * ng:] - w.b[0, 0]).max() == 0                                                   # z_f == c
    assert np.abs(sw["yf"]).max() > 1e-2 and (sw["xi"] != 0).any()


# ----------------------------------------------------------------------------------------------- f1: adaptive rho + termination
def _eq4_quantities(w, st, b=0):
    """r_prim, r_dual (eq. 3) and the scales of eq. 4 from numpy-built matrices."""
    P, C, c, G = dense_PCG(w, b)
    x, yf, yg, zg, xi = st["x"][b].ravel(), st["yf"][b], st["yg"][b].ravel(), st["zg"][b].ravel(), st["xi"][b].ravel()
    soft = np.tile(np.array(w.soft, dtype=bool), w.T)
    m = soft & (xi != 0)
    rp = max(np.abs(C @ x - c).max(), np.abs(G @ x - zg).max())
    rd = max(np.abs(P @ x + w.q[b].ravel() + C.T @ yf + G.T @ yg).max(), np.abs(w.gamma * xi[m] + w.lam * np.sign(xi[m]) + yg[m]).max(initial=0))
    npr = max(np.abs(C @ x).max(), np.abs(c).max(), np.abs(G @ x).max(), np.abs(zg).max())
    nd = max(np.abs(P @ x).max(), np.abs(C.T @ yf + G.T @ yg).max(), np.abs(w.q[b]).max(), np.abs(w.gamma * xi[soft]).max(initial=0), np.abs(yg[soft]).max(initial=0))
    return rp, rd, npr, nd


def test_adaptive_off_equals_the_fixed_iteration_count():
    """adapt_rho = 0 and eps = 0 (never converged): exactly the K iterations of Alg. 3, whatever the check cadence."""
    w = W.config2(B=2, N=10, soft_bound=0.5)
    w.rho_bar = 20.0
    cfg = O.make_cfg(w)
    ref, _, _ = O.admm(w, cfg, iters=60)
    for every in (7, 25):
        st, info, log, rc = O.admm_adaptive(w, cfg, O.make_adaptive(60, 0.0, 0.0, check_every=every, adapt_rho=0))
        assert rc == 0 and (info[:, 4] == 60).all() and (info[:, 6] == 0).all()
        assert all((st[k] == ref[k]).all() for k in ref)


@pytest.mark.parametrize("lam,eps", [(100.0, 1e-5), (0.05, 1e-7)])
def test_adaptive_schedule_recomputed_in_numpy(lam, eps):
    """Every scheduled check of one adaptive run: the state at that iteration (obtained by capping max_iters there: the trajectory
    is deterministic) gives, through numpy-built matrices, the residuals and scales of eq. 3-4, the verdict of eq. 4, the candidate
    of eq. 17 with the clip [1e-6, 1e6] and the ratio gate 5 — all equal to what the oracle logged."""
    w = W.config2(B=1, N=10, soft_bound=0.5)
    w.lam = lam
    cfg = O.make_cfg(w)
    ad = O.make_adaptive(3000, eps, eps)
    st, info, log, rc = O.admm_adaptive(w, cfg, ad)
    nlog = int(info[0, 7])
    assert rc == 0 and info[0, 6] == 1 and nlog >= 4 and int(info[0, 4]) == int(log[0, nlog - 1, 0]) and info[0, 4] % 25 == 0
    changes = 0
    for i in range(nlog):
        k, rp_o, rd_o, np_o, nd_o, rho0, rho1, conv = log[0, i]
        assert k == 25 * (i + 1)
        sk, ik, _, _ = O.admm_adaptive(w, cfg, O.make_adaptive(int(k), eps, eps))
        rp, rd, npr, nd = _eq4_quantities(w, sk)
        for got, ref in ((rp_o, rp), (rd_o, rd), (np_o, npr), (nd_o, nd)):
            assert abs(got - ref) <= 1e-10 * max(1.0, abs(ref)), (k, got, ref)
        is_conv = rp <= eps + eps * npr and rd <= eps + eps * nd
        assert bool(conv) == is_conv and (is_conv == (i == nlog - 1))
        cand = min(max(rho0 * np.sqrt((rp / npr) / (rd / nd)), 1e-6), 1e6)
        expect = cand if (not is_conv and max(cand / rho0, rho0 / cand) > 5.0) else rho0
        assert abs(rho1 - expect) <= 1e-9 * expect, (k, rho1, expect)
        changes += int(rho1 != rho0)
        if i + 1 < nlog:
            assert log[0, i + 1, 5] == rho1                      # the next interval runs with the accepted value
    assert changes >= 1, "instance must exercise an accepted update"
    assert abs(info[0, 5] - log[0, nlog - 1, 6]) == 0


def test_adaptive_reaches_the_same_fixed_point_in_fewer_iterations():
    """The step size changes the path, not the fixed point: the adaptive run and a fixed-rho run converge to the same (x, y), and
    on the slack-stress instance (rho_bar = 0.1 makes the L1 dead zone 1000 wide, reading A-14) adaptation needs fewer iterations."""
    w = W.config2(B=2, N=10, soft_bound=0.5)
    cfg = O.make_cfg(w)
    sa, ia, _, rca = O.admm_adaptive(w, cfg, O.make_adaptive(20000, 1e-9, 1e-9))
    sf, if_, _, rcf = O.admm_adaptive(w, cfg, O.make_adaptive(20000, 1e-9, 1e-9, adapt_rho=0))
    assert rca == 0 and (ia[:, 6] == 1).all()
    assert (ia[:, 4] < if_[:, 4]).all()
    ref, info, rc = O.admm(w, O.make_cfg(w, rho_bar=20.0), iters=30000)
    assert info[:, :2].max() < 1e-10
    for k in ("x", "yf", "yg", "xi"):
        assert np.abs(sa[k] - ref[k]).max() <= 1e-6 * max(1.0, np.abs(ref[k]).max()), k


# ----------------------------------------------------------------------------------------------- backward vs finite differences
def _loss_of_solution(w, cfg, iters, xi_weight=0.0):
    st, info, rc = O.admm(w, cfg, iters=iters)
    return (st["x"] ** 2).sum(axis=(1, 2)) + xi_weight * (st["xi"] ** 2).sum(axis=(1, 2)), st, info


@pytest.mark.parametrize("soft_bound,lam,xi_weight", [(2.0, 100.0, 0.0), (0.3, 0.0, 0.0), (0.3, 0.05, 0.0), (0.4, 2.0, 0.0), (0.3, 0.0, 1.0), (0.4, 2.0, 3.0)],
                         ids=["cfg2_hard_active", "soft_active", "soft_L1", "L1_dead_zone", "soft_active_dLdxi", "L1_dead_zone_dLdxi"])
def test_backward_matches_central_finite_differences(soft_bound, lam, xi_weight):
    """dL/dq and dL/dx_init for L = ||x||^2 + xi_weight ||xi||^2 (reading A-19; the xi term exercises the right-hand side
    -G_s' Sigma_s dL/dxi_s of eq. 65) vs central differences of tightly converged solves: 1e-6 relative.
    The L1_dead_zone instances hold SOFT rows that sit on their bound with 0 < |y_g| < lambda and xi = 0: the dual-sign
    rule must class them hard-active (the slack cannot move inside the dead zone, reading A-14)."""
    import copy
    w = W.config2(B=1, N=8, soft_bound=soft_bound)
    w.lam, w.rho_bar = lam, 2.0
    w.q = w.q + 0.3 * np.random.default_rng(5).standard_normal(w.q.shape)
    cfg = O.make_cfg(w)
    iters = 30000
    L0, st, info = _loss_of_solution(w, cfg, iters, xi_weight)
    assert info[0, 0] < 1e-11 and info[0, 1] < 1e-11
    cls = O.classify(w, cfg, st, 0)
    soft = np.array(w.soft, dtype=bool)
    ya = np.abs(st["yg"][0][cls == 1]); assert ya.size == 0 or ya.min() > 1e-4      # screened instance (reading A-17)
    if soft_bound < 1.0:
        assert (cls == 2).sum() > 0
    else:
        assert (cls == 1).sum() > 0
    if lam == 2.0:                                           # dead-zone rows present, strictly inside the dead zone
        dead = np.abs(st["yg"][0][:, soft][cls[:, soft] == 1])
        assert dead.size >= 2 and dead.min() > 1e-3 and dead.max() < lam - 1e-2
        assert (st["xi"][0][:, soft][cls[:, soft] == 1] == 0).all()
    dLdxi = 2.0 * xi_weight * st["xi"] if xi_weight else None
    dq, dxi, counts, rcs = O.backward(w, cfg, st, 2.0 * st["x"], dLdxi)
    assert rcs[0] == 0
    rng = np.random.default_rng(6)
    h = 1e-5
    for trial in range(4):
        dirq = rng.standard_normal(w.q.shape)
        wp, wm = copy.copy(w), copy.copy(w)
        wp.q, wm.q = w.q + h * dirq, w.q - h * dirq
        fd = (_loss_of_solution(wp, cfg, iters, xi_weight)[0] - _loss_of_solution(wm, cfg, iters, xi_weight)[0]) / (2 * h)
        an = (dq * dirq).sum()
        assert abs(fd[0] - an) <= 1e-6 * max(1.0, abs(an))
    for i in range(w.nx):
        wp, wm = copy.copy(w), copy.copy(w)
        wp.x_init, wm.x_init = w.x_init.copy(), w.x_init.copy()
        wp.x_init[0, i] += h; wm.x_init[0, i] -= h
        fd = (_loss_of_solution(wp, cfg, iters, xi_weight)[0] - _loss_of_solution(wm, cfg, iters, xi_weight)[0]) / (2 * h)
        assert abs(fd[0] - dxi[0, i]) <= 1e-6 * max(1.0, abs(dxi[0, i]))
    if xi_weight:                                            # the xi term must matter: without it the gradient is visibly different
        dq0, _, _, _ = O.backward(w, cfg, st, 2.0 * st["x"], None)
        assert np.abs(dq0 - dq).max() > 1e-3 * np.abs(dq).max()


def test_classification_rule_hand_built_states():
    """Row classification of the backward pass (PAPER.md:878-888 with reading A-16), on hand-built (x, y_g, xi):
    dual sign first (|y| > eps_y = eps_abs + eps_rel max|y|) -> active, also for soft rows with xi = 0 (L1 dead zone);
    xi != 0 on a soft row -> soft-active; |y| <= eps_y -> active only within eps_abs + eps_rel |bound| of a bound."""
    w = W.config2(B=1, N=3, soft_bound=0.5)                 # rows: u1,u2 hard in [-1,1]; x1..x6 soft in [-0.5,0.5]
    eps_abs, eps_rel = 1e-3, 1e-2
    cfg = O.make_cfg(w, eps_abs=eps_abs, eps_rel=eps_rel)
    st = O.new_state(w)
    x, yg, xi = st["x"][0], st["yg"][0], st["xi"][0]
    expect = np.zeros((w.T, w.ng), dtype=int)
    col = w.g_col
    yg[0, 0] = 5.0; expect[0, 0] = 1                         # max|y| = 5 -> eps_y = 1e-3 + 5e-2 = 0.051
    yg[0, 1] = -0.06; expect[0, 1] = 1                       # just above eps_y: dual sign decides, whatever x is
    yg[1, 0] = 0.05; x[1, col[0]] = 0.0; expect[1, 0] = 0    # just below eps_y and far from both bounds
    x[1, col[1]] = 1.0 - 0.5 * (eps_abs + eps_rel * 1.0); expect[1, 1] = 1      # y = 0, inside the proximity band of hi = 1
    x[2, col[0]] = 1.0 - 2.0 * (eps_abs + eps_rel * 1.0); expect[2, 0] = 0      # y = 0, outside the band
    x[2, col[1]] = -1.0 + 0.5 * (eps_abs + eps_rel * 1.0); expect[2, 1] = 1     # lower bound, inside the band
    yg[0, 2] = 0.3; xi[0, 2] = 0.0; expect[0, 2] = 1         # SOFT row, xi = 0, |y| > eps_y: L1 dead zone -> hard-active
    yg[0, 3] = 0.3; xi[0, 3] = -0.2; expect[0, 3] = 2        # soft row with slack: soft-active, the slack test comes first
    xi[1, 2] = 0.5 * eps_abs; x[1, col[2]] = 0.0; expect[1, 2] = 0                # |xi| below eps_abs does not count as slack
    x[1, col[3]] = 0.5 - 0.5 * (eps_abs + eps_rel * 0.5); expect[1, 3] = 1      # soft row, y = 0, xi = 0, on its bound
    x[2, col[3]] = 0.5 - 2.0 * (eps_abs + eps_rel * 0.5); expect[2, 3] = 0      # relative part uses |bound| = 0.5
    w.lo[0, 3, 4] = -np.inf; x[3, col[4]] = -7.0; expect[3, 4] = 0               # an infinite bound is never "near"
    got = O.classify(w, cfg, st, 0)
    assert (got == expect).all(), (got, expect)


def test_adjoint_qp_of_eq67_converges_to_the_definition():
    """eq. 67: Alg. 3 on the adjoint QP (tests/adjoint_util.py, numpy) converges to the solution of the
    active-set system eq. 65 that backward() solves directly; per-row soft flags == per-type mask when they coincide."""
    from adjoint_util import adjoint_qp
    w = W.config2(B=2, N=8, soft_bound=0.4)
    w.lam, w.rho_bar = 2.0, 2.0
    w.q = w.q + 0.3 * np.random.default_rng(5).standard_normal(w.q.shape)
    cfg = O.make_cfg(w)
    st, info, rc = O.admm(w, cfg, iters=30000)
    dLdxi = 6.0 * st["xi"]
    dq, dxi, counts, rcs = O.backward(w, cfg, st, 2.0 * st["x"], dLdxi)
    assert (rcs == 0).all() and counts[:, 1].min() > 0 and counts[:, 0].min() > 0
    wa, soft_rows, cls = adjoint_qp(w, cfg, st, 2.0 * st["x"], dLdxi)
    sa, ia, rca = O.admm_rows(wa, O.make_cfg(wa), soft_rows, 60000)
    assert rca == 0
    assert np.abs(-sa["x"] - dq).max() <= 1e-8 * max(1.0, np.abs(dq).max())
    assert np.abs(sa["yf"][:, :w.nx] - dxi).max() <= 1e-8 * max(1.0, np.abs(dxi).max())
    sr = np.tile(np.array(w.soft, np.uint8), (w.B, w.T, 1))
    a, _, _ = O.admm(w, cfg, iters=40); b, _, _ = O.admm_rows(w, cfg, sr, 40)
    assert all((a[k] == b[k]).all() for k in a)


def test_backward_dgamma_matches_finite_differences():
    """dL/dgamma_xi (eq. 66) for L = |x|^2 + |xi|^2 vs central differences in gamma on a soft-active instance."""
    import copy
    w = W.config2(B=1, N=8, soft_bound=0.3)
    w.lam, w.rho_bar = 0.05, 2.0
    w.q = w.q + 0.3 * np.random.default_rng(5).standard_normal(w.q.shape)

    def loss(gam):
        ww = copy.copy(w); ww.gamma = gam
        st, info, rc = O.admm(ww, O.make_cfg(ww), iters=30000)
        assert info[0, 0] < 1e-11 and info[0, 1] < 1e-11
        return (st["x"] ** 2).sum() + (st["xi"] ** 2).sum(), st

    L0, st = loss(w.gamma)
    dq, dxi, counts, rcs, dg = O.backward(w, O.make_cfg(w), st, 2.0 * st["x"], 2.0 * st["xi"], with_dgamma=True)
    assert rcs[0] == 0 and counts[0, 1] > 0
    h = 1e-5
    fd = (loss(w.gamma + h)[0] - loss(w.gamma - h)[0]) / (2 * h)
    assert abs(fd - dg[0]) <= 1e-6 * max(1.0, abs(fd)) and abs(fd) > 1e-3


def test_backward_unconstrained_closed_form():
    """No active rows: dL/dq = -(K^-1)_xx dL/dx with K the equality KKT matrix (numpy)."""
    w = W.random_ltv(7, 1, 6, 3, 2, [3, 4], [0, 0], bound=np.inf, implicit=True, q_scale=0.5)
    cfg = O.make_cfg(w)
    st, info, rc = O.admm(w, cfg, iters=500)
    P, C, c, G = dense_PCG(w, 0)
    K = np.block([[P, C.T], [C, np.zeros((C.shape[0],) * 2)]])
    g = 2.0 * st["x"][0].ravel()
    sol = np.linalg.solve(K, np.concatenate([g, np.zeros(C.shape[0])]))
    dq, dxi, counts, rcs = O.backward(w, cfg, st, 2.0 * st["x"])
    assert counts[0, 0] == 0 and counts[0, 1] == 0
    assert np.abs(dq[0].ravel() + sol[:P.shape[0]]).max() < 1e-10 * max(1, np.abs(sol).max())
    assert np.abs(dxi[0] - sol[P.shape[0]:P.shape[0] + w.nx]).max() < 1e-10 * max(1, np.abs(sol).max())


# ----------------------------------------------------------------------------------------------- bicycle / SQP (a1, O-4)
def test_bicycle_jacobians_match_finite_differences():
    """A^-, A^+ (eq. 36) == central FD of the implicit-midpoint residual; b == eq. 37; residual == hand-typed formula."""
    w = W.config4(B=2, N=10)
    cfg = O.make_cfg(w)
    rng = np.random.default_rng(3)
    xbar = w.xbar0[1] + 0.1 * rng.standard_normal(w.xbar0[1].shape)
    Am, Ap, b, G, lo, hi = O.bicycle_linearize(w, cfg, xbar, 1)
    h = 1e-6
    for t in (0, 4, 9):
        vk, vk1 = xbar[t], xbar[t + 1]
        psi, v = 0.5 * (vk[2] + vk1[2]), 0.5 * (vk[3] + vk1[3])
        f_hand = vk[:4] + w.dt * np.array([v * np.cos(psi), v * np.sin(psi), v / w.wheelbase * np.tan(vk[5]), vk[4]]) - vk1[:4]
        f0 = O.bicycle_residual(cfg, vk, vk1)
        assert np.abs(f0 - f_hand).max() < 1e-14
        for j in range(6):
            e = np.zeros(6); e[j] = h
            dm = (O.bicycle_residual(cfg, vk + e, vk1) - O.bicycle_residual(cfg, vk - e, vk1)) / (2 * h)
            dp = (O.bicycle_residual(cfg, vk, vk1 + e) - O.bicycle_residual(cfg, vk, vk1 - e)) / (2 * h)
            assert np.abs(dm - Am[t][:, j]).max() < 1e-7 and np.abs(dp - Ap[t][:, j]).max() < 1e-7
        assert np.abs(b[t] - (Am[t] @ vk + Ap[t] @ vk1 - f0)).max() < 1e-12
    # inequality rows (eq. 38): a, delta selections; lateral error row in the reference frame, bounds shifted by G.p_ref
    ref = w.stage_ref[1]
    t = 5
    assert G[t, 0, 4] == 1 and G[t, 1, 5] == 1 and np.abs(G[t, 2, :2] - [-np.sin(ref[t, 2]), np.cos(ref[t, 2])]).max() < 1e-15
    v = xbar[t]
    e_lat = -np.sin(ref[t, 2]) * (v[0] - ref[t, 0]) + np.cos(ref[t, 2]) * (v[1] - ref[t, 1])
    assert abs((G[t, 2] @ v - lo[t, 2]) - (e_lat + 3.0)) < 1e-12 and abs((hi[t, 2] - G[t, 2] @ v) - (3.0 - e_lat)) < 1e-12
    assert (lo[t, :2] == [-6.0, -0.4]).all() and (hi[t, :2] == [3.0, 0.4]).all()


def test_sqp_driver_reduces_dynamics_residual_and_is_consistent_with_admm():
    """||f(xbar)||_inf shrinks over the fixed SQP steps (O-4); one SQP step == linearise + O-3 called by hand."""
    w = W.config4(B=2, N=30)
    cfg = O.make_cfg(w)
    st, info, rc, fnorm = O.sqp_bicycle(w, cfg, n_sqp=5, iters=200, with_fnorm=True)
    assert rc == 0 and (fnorm[:, -1] < 1e-3 * fnorm[:, 0]).all()
    st1, info1, rc1 = O.sqp_bicycle(w, cfg, n_sqp=1, iters=50)
    st3, info3, rc3 = O.sqp_bicycle(w, cfg, n_sqp=3, iters=50)
    import copy
    for b in range(w.B):
        # reading A-26 by hand, three steps: linearise at xbar -> K iterations warm-started at x^0 = xbar with y_f, y_g CARRIED
        # and z_g RE-PROJECTED (zg_given = 0: z_g^0 = clip(G xbar, lo, hi) with the NEW shifted bounds) -> full step xbar <- x^K
        s = O.new_state(w, B=1); s["x"] = w.xbar0[b:b + 1].copy()
        for step in range(3):
            Am, Ap, bb, G, lo, hi = O.bicycle_linearize(w, cfg, s["x"][0], b)
            wq = copy.copy(w)
            wq.B, wq.Am, wq.Ap, wq.b, wq.G, wq.lo, wq.hi = 1, Am[None], Ap[None], bb[None], G[None], lo[None], hi[None]
            wq.q, wq.x_init, wq.model = w.q[b:b + 1], w.x_init[b:b + 1], 0
            s, _, _ = O.admm(wq, O.make_cfg(wq), iters=50, state=s)
            if step == 0:
                assert np.abs(s["x"][0] - st1["x"][b]).max() < 1e-12
        for k in ("x", "zg", "yf", "yg", "xi"):
            assert np.abs(s[k][0] - st3[k][b]).max() < 1e-12 * max(1.0, np.abs(st3[k][b]).max()), k
        assert np.abs(st3["yf"][b]).max() > 1e-3                # the carried multipliers are not trivially zero


# ----------------------------------------------------------------------------------------------- f2: SQP with linesearch (App. D) and eq. 18
def _bicycle_f(w, x):
    """Stacked equality residual (x_0 - x_init ; implicit-midpoint bicycle residuals), numpy, for one problem x [T,6]."""
    vk, vk1 = x[:-1], x[1:]
    psi, v = 0.5 * (vk[:, 2] + vk1[:, 2]), 0.5 * (vk[:, 3] + vk1[:, 3])
    F = np.stack([v * np.cos(psi), v * np.sin(psi), v / w.wheelbase * np.tan(vk[:, 5]), vk[:, 4]], axis=1)
    return x[0, :4].copy(), vk[:, :4] + w.dt * F - vk1[:, :4]


def _merit_parts(w, b, P, q, x, xi, G, lo, hi):
    """cost l(x~) and c1 = |f|_1 + |[g - hi]_+|_1 + |[lo - g]_+|_1 (App. D) in numpy."""
    soft = np.array(w.soft, dtype=bool)
    xf = x.ravel()
    cost = 0.5 * xf @ P @ xf + q @ xf + (w.lam * np.abs(xi[:, soft]) + 0.5 * w.gamma * xi[:, soft] ** 2).sum()
    f0, fk = _bicycle_f(w, x)
    g = np.einsum("trn,tn->tr", G, x) + np.where(soft, xi, 0.0)
    viol = np.maximum(0.0, g - hi) + np.maximum(0.0, lo - g)
    return cost, np.abs(f0 - w.x_init[b]).sum() + np.abs(fk).sum() + viol.sum(), max(np.abs(f0 - w.x_init[b]).max(), np.abs(fk).max()), viol.max()


def test_sqp_linesearch_steps_recomputed_in_numpy():
    """Every SQP iteration of one run: the QP solution comes from the pinned pieces (bicycle_linearize + Alg. 3), the merit function,
    mu, D_mu, the Armijo test over alpha = 2^-j (eta = 0.4), the fallback to the smallest merit and the update of (x, xi, y) are retyped
    here from App. D; the convergence quantities of eq. 18 are recomputed with the Jacobians at the new iterate."""
    import copy
    w = W.config4(B=1, N=16, dtype="f64")
    x0 = w.xbar0.copy(); x0[:, :, :2] += np.random.default_rng(0).normal(0, 1.5, x0[:, :, :2].shape); x0[:, :, 2] += 0.3
    cfg = O.make_cfg(w)
    K, eps_c, nA, eta, nsqp = 200, 1e-3, 8, 0.4, 30
    st_all, info, log, rc = O.sqp_linesearch_bicycle(w, cfg, max_sqp=nsqp, admm_iters=K, eps_c=eps_c, n_alpha=nA, eta=eta, xbar0=x0)
    assert rc == 0
    soft = np.array(w.soft, dtype=bool)
    cur = O.new_state(w); cur["x"] = x0.copy()
    seen_backtrack = False
    for it in range(int(info[0, 0])):
        Am, Ap, bb, G, lo, hi = O.bicycle_linearize(w, cfg, cur["x"][0], 0)
        wq = copy.copy(w)
        wq.Am, wq.Ap, wq.b, wq.G, wq.lo, wq.hi, wq.model = Am[None], Ap[None], bb[None], G[None], lo[None], hi[None], 0
        s0 = {k: v.copy() for k, v in cur.items()}
        sol, _, _ = O.admm(wq, O.make_cfg(wq), iters=K, state=s0)
        P, C, c, Gd = dense_PCG(wq, 0)
        q = w.q[0].ravel()
        x, xi = cur["x"][0], cur["xi"][0]
        dx, dxi = sol["x"][0] - x, sol["xi"][0] - xi
        cost0, c1, _, _ = _merit_parts(w, 0, P, q, x, xi, G, lo, hi)
        sg = np.where(xi != 0, np.sign(xi), np.sign(dxi))
        dl = (P @ x.ravel() + q) @ dx.ravel() + ((w.lam * sg + w.gamma * xi) * dxi)[:, soft].sum()
        mu = max(0.0, dl / (0.5 * max(c1, eps_c)))
        phi0, Dmu = cost0 + mu * c1, dl - mu * c1
        phis = []
        for j in range(nA):
            a = 2.0 ** -j
            ca, c1a, _, _ = _merit_parts(w, 0, P, q, x + a * dx, xi + a * dxi, G, lo, hi)
            phis.append(ca + mu * c1a)
        ok = [j for j in range(nA) if phis[j] <= phi0 + eta * 2.0 ** -j * Dmu]
        jstar = ok[0] if ok else int(np.argmin(phis))
        alpha = 2.0 ** -jstar
        seen_backtrack |= alpha < 1.0
        assert log[0, it, 0] == alpha and bool(log[0, it, 6]) == bool(ok), (it, log[0, it], alpha)
        assert abs(log[0, it, 1] - mu) <= 1e-9 * max(1, abs(mu)) and abs(log[0, it, 2] - phi0) <= 1e-9 * abs(phi0) and abs(log[0, it, 4] - c1) <= 1e-9 * max(1, c1)
        for k in ("x", "xi", "yf", "yg"):
            cur[k] = cur[k] + alpha * (sol[k] - cur[k])
        cur["zg"] = sol["zg"]
        # eq. 18 at the new iterate
        Am, Ap, bb, G, lo, hi = O.bicycle_linearize(w, cfg, cur["x"][0], 0)
        wq.Am, wq.Ap, wq.b, wq.G, wq.lo, wq.hi = Am[None], Ap[None], bb[None], G[None], lo[None], hi[None]
        P, C, c, Gd = dense_PCG(wq, 0)
        stat = np.abs(P @ cur["x"][0].ravel() + q + C.T @ cur["yf"][0] + Gd.T @ cur["yg"][0].ravel()).max()
        _, _, finf, ginf = _merit_parts(w, 0, P, q, cur["x"][0], cur["xi"][0], G, lo, hi)
        for got, ref in ((log[0, it, 7], stat), (log[0, it, 8], finf), (log[0, it, 9], ginf)):
            assert abs(got - ref) <= 1e-9 * max(1.0, abs(ref))
        conv = stat <= eps_c and finf <= eps_c and ginf <= eps_c
        assert conv == (it == int(info[0, 0]) - 1 and bool(info[0, 1]))
    for k in ("x", "xi", "yf", "yg"):
        assert np.abs(cur[k] - st_all[k]).max() <= 1e-10 * max(1.0, np.abs(st_all[k]).max()), k
    assert info[0, 1] == 1 and info[0, 3] <= eps_c, "the run must converge by eq. 18"
    print("alphas", log[0, :int(info[0, 0]), 0], "backtracked", seen_backtrack)


# ----------------------------------------------------------------------------------------------- f3: SRB humanoid model (eq. 68-69 + RK4)
def test_srb_model_closed_forms_and_rk4_order():
    """(i) no forces, no spin: free fall p(t) = p0 + v0 t + g t^2 / 2, v(t) = v0 + g t is a quadratic and RK4 integrates it exactly (eq. 68a, 68c);
    (ii) standing reference with u_ref = m g / 2 per foot is an equilibrium (feet symmetric about the CoM: zero net torque);
    (iii) torque-free spin about a principal axis keeps omega constant and turns the yaw at that rate (eq. 68b with T(0) = I, eq. 68d);
    (iv) the one-step error against 64 sub-steps shrinks ~32x when dt is halved (local error of a 4th-order scheme)."""
    import copy
    w = W.srb_humanoid(B=1)
    cfg = O.make_cfg(w)
    x = np.array([0.1, -0.2, 0.7, 0, 0, 0, 0.3, -0.1, 0.5, 0, 0, 0.0]); u = np.zeros(6)
    xn = O.srb_step(cfg, x, u)
    g = np.array([0, 0, -9.81]); dt = w.dt
    assert np.abs(xn[:3] - (x[:3] + dt * x[6:9] + 0.5 * dt * dt * g)).max() < 1e-14 and np.abs(xn[6:9] - (x[6:9] + dt * g)).max() < 1e-14
    assert np.abs(xn[3:6]).max() == 0 and np.abs(xn[9:]).max() == 0
    xr, ur = w.stage_ref[0, 0, :12], w.stage_ref[0, 0, 12:]
    assert np.abs(O.srb_step(cfg, xr, ur) - xr).max() < 1e-14
    xs = xr.copy(); xs[11] = 0.8                                             # spin about the body z axis, upright
    xn = O.srb_step(cfg, xs, ur)
    assert abs(xn[11] - 0.8) < 1e-14 and abs(xn[5] - 0.8 * dt) < 1e-14 and np.abs(xn[3:5]).max() < 1e-14

    def fine(cfg_, x_, u_, dt_, sub=64):
        c2 = copy.copy(cfg_); c2.dt = dt_ / sub
        for _ in range(sub):
            x_ = O.srb_step(c2, x_, u_)
        return x_
    rng = np.random.default_rng(0)
    x = xr + np.concatenate([0.05 * rng.standard_normal(3), 0.2 * rng.standard_normal(3), 0.3 * rng.standard_normal(3), 0.5 * rng.standard_normal(3)])
    u = ur + 5.0 * rng.standard_normal(6)
    errs = []
    for dt_ in (0.1, 0.05):
        c1 = copy.copy(cfg); c1.dt = dt_
        errs.append(np.abs(O.srb_step(c1, x, u) - fine(cfg, x, u, dt_)).max())
    assert 20.0 < errs[0] / errs[1] < 45.0, errs


def test_srb_jacobians_match_finite_differences_and_eq37():
    """A^- = [dPhi/dx dPhi/du] (forward-mode dual numbers in the oracle) == central finite differences of the RK4 flow; A^+ = [-I 0];
    b == A^- v_k + A^+ v_{k+1} - f_k (eq. 37); the torque term: d(omega+)/d(f) has the size dt r / I (the cross product is there)."""
    w = W.srb_humanoid(B=2, N=6)
    cfg = O.make_cfg(w)
    rng = np.random.default_rng(1)
    xbar = w.xbar0[1] + np.concatenate([0.05 * rng.standard_normal((w.T, 3)), 0.2 * rng.standard_normal((w.T, 3)), 0.3 * rng.standard_normal((w.T, 6)),
                                        20.0 * rng.standard_normal((w.T, 6))], axis=1)
    Am, Ap, b = O.srb_linearize(w, cfg, xbar)
    h = 1e-6
    for t in (0, 3, 5):
        vk, vk1 = xbar[t], xbar[t + 1]
        for j in range(18):
            e = np.zeros(18); e[j] = h * max(1.0, abs(vk[j]))
            fd = (O.srb_step(cfg, (vk + e)[:12], (vk + e)[12:]) - O.srb_step(cfg, (vk - e)[:12], (vk - e)[12:])) / (2 * e[j])
            assert np.abs(fd - Am[t][:, j]).max() < 1e-7 * max(1.0, np.abs(Am[t][:, j]).max()), (t, j)
        assert np.abs(Ap[t] - np.hstack([-np.eye(12), np.zeros((12, 6))])).max() == 0
        f = O.srb_step(cfg, vk[:12], vk[12:]) - vk1[:12]
        assert np.abs(b[t] - (Am[t] @ vk + Ap[t] @ vk1 - f)).max() < 1e-11
    assert np.abs(Am[0][9:12, 12:]).max() > 1e-3            # forces torque the body


def test_srb_sqp_driver_reaches_the_reference():
    """Fixed-count SQP on the balancing OCP: the dynamics residual of the final iterate is small, the bounds on u hold, and one SQP step equals
    linearise + Alg. 3 by hand (the pieces pinned above)."""
    import copy
    w = W.srb_humanoid(B=2, N=10)
    cfg = O.make_cfg(w)
    st, info, rc = O.sqp_srb(w, cfg, n_sqp=6, iters=600)
    assert rc == 0
    for b in range(w.B):
        x = st["x"][b]
        res = max(np.abs(O.srb_step(cfg, x[t, :12], x[t, 12:]) - x[t + 1, :12]).max() for t in range(w.N))
        assert res < 1e-3
        assert (x[:, 12:] >= w.lo[b] - 1e-3).all() and (x[:, 12:] <= w.hi[b] + 1e-3).all()
    st1, _, _ = O.sqp_srb(w, cfg, n_sqp=1, iters=40)
    for b in range(w.B):
        Am, Ap, bb = O.srb_linearize(w, cfg, w.xbar0[b])
        wq = copy.copy(w)
        wq.B, wq.Am, wq.Ap, wq.b, wq.model = 1, Am[None], Ap[None], bb[None], 0
        wq.q, wq.x_init, wq.lo, wq.hi = w.q[b:b + 1], w.x_init[b:b + 1], w.lo[b:b + 1], w.hi[b:b + 1]
        s0 = O.new_state(wq); s0["x"] = w.xbar0[b:b + 1].copy()
        s, _, _ = O.admm(wq, O.make_cfg(wq), iters=40, state=s0)
        assert np.abs(s["x"][0] - st1["x"][b]).max() < 1e-12


def _srb_instance(B=1, N=10, seed=3):
    """The balancing OCP with a perturbed start and the two f_y rows (the ones that bind) made soft, so that the slack terms of the merit function act."""
    w = W.srb_humanoid(B=B, N=N)
    w.soft = [0, 1, 0, 0, 1, 0]
    w.lam, w.gamma = 0.01, 0.1
    rng = np.random.default_rng(seed)
    x0 = w.xbar0.copy()
    x0[:, :, :3] += 0.03 * rng.standard_normal(x0[:, :, :3].shape); x0[:, :, 3:6] += 0.1 * rng.standard_normal(x0[:, :, 3:6].shape)
    x0[:, :, 6:12] += 0.2 * rng.standard_normal(x0[:, :, 6:12].shape)
    return w, x0


def _merit_parts_srb(w, cfg, b, P, q, x, xi, lo, hi):
    """cost and c1 of App. D for the SRB model: f_k = Phi(x_k, u_k) - x_{k+1} with the pinned RK4 step, g = selected components (+ xi on soft rows)."""
    soft = np.array(w.soft, dtype=bool)
    xf = x.ravel()
    cost = 0.5 * xf @ P @ xf + q @ xf + (w.lam * np.abs(xi[:, soft]) + 0.5 * w.gamma * xi[:, soft] ** 2).sum()
    fk = np.stack([O.srb_step(cfg, x[t, :12], x[t, 12:]) - x[t + 1, :12] for t in range(w.N)])
    f0 = x[0, :12] - w.x_init[b]
    g = x[:, w.g_col] + np.where(soft, xi, 0.0)
    viol = np.maximum(0.0, g - hi) + np.maximum(0.0, lo - g)
    return cost, np.abs(f0).sum() + np.abs(fk).sum() + viol.sum(), max(np.abs(f0).max(), np.abs(fk).max()), viol.max()


def test_sqp_linesearch_srb_steps_recomputed_in_numpy():
    """f2 for the second model: every SQP iteration of one run of sqp_ls_srb retyped from App. D (merit, mu, D_mu, Armijo over alpha = 2^-j, fallback,
    update) around the pinned pieces (srb_linearize, srb_step, Alg. 3), and eq. 18 with the Jacobians at the new iterate.  The run backtracks, uses
    the soft row's slack and converges."""
    import copy
    w, x0 = _srb_instance()
    cfg = O.make_cfg(w)
    K, eps_c, nA, eta, nsqp = 2000, 1e-3, 8, 0.4, 25
    st_all, info, log, rc = O.sqp_linesearch_srb(w, cfg, max_sqp=nsqp, admm_iters=K, eps_c=eps_c, n_alpha=nA, eta=eta, xbar0=x0)
    assert rc == 0
    soft = np.array(w.soft, dtype=bool)
    cur = O.new_state(w); cur["x"] = x0.copy()
    seen_backtrack = seen_slack = False
    q = w.q[0].ravel(); lo, hi = w.lo[0], w.hi[0]
    for it in range(int(info[0, 0])):
        Am, Ap, bb = O.srb_linearize(w, cfg, cur["x"][0])
        wq = copy.copy(w)
        wq.Am, wq.Ap, wq.b, wq.model = Am[None], Ap[None], bb[None], 0
        s0 = {k: v.copy() for k, v in cur.items()}
        sol, _, _ = O.admm(wq, O.make_cfg(wq), iters=K, state=s0)
        P, C, c, Gd = dense_PCG(wq, 0)
        x, xi = cur["x"][0], cur["xi"][0]
        dx, dxi = sol["x"][0] - x, sol["xi"][0] - xi
        seen_slack |= bool((sol["xi"] != 0).any())
        cost0, c1, _, _ = _merit_parts_srb(w, cfg, 0, P, q, x, xi, lo, hi)
        sg = np.where(xi != 0, np.sign(xi), np.sign(dxi))
        dl = (P @ x.ravel() + q) @ dx.ravel() + ((w.lam * sg + w.gamma * xi) * dxi)[:, soft].sum()
        mu = max(0.0, dl / (0.5 * max(c1, eps_c)))
        phi0, Dmu = cost0 + mu * c1, dl - mu * c1
        phis = []
        for j in range(nA):
            a = 2.0 ** -j
            ca, c1a, _, _ = _merit_parts_srb(w, cfg, 0, P, q, x + a * dx, xi + a * dxi, lo, hi)
            phis.append(ca + mu * c1a)
        ok = [j for j in range(nA) if phis[j] <= phi0 + eta * 2.0 ** -j * Dmu]
        jstar = ok[0] if ok else int(np.argmin(phis))
        alpha = 2.0 ** -jstar
        seen_backtrack |= alpha < 1.0
        assert log[0, it, 0] == alpha and bool(log[0, it, 6]) == bool(ok), (it, log[0, it], alpha)
        assert abs(log[0, it, 1] - mu) <= 1e-8 * max(1, abs(mu)) and abs(log[0, it, 2] - phi0) <= 1e-9 * abs(phi0) and abs(log[0, it, 4] - c1) <= 1e-9 * max(1, c1)
        for k in ("x", "xi", "yf", "yg"):
            cur[k] = cur[k] + alpha * (sol[k] - cur[k])
        cur["zg"] = sol["zg"]
        Am, Ap, bb = O.srb_linearize(w, cfg, cur["x"][0])
        wq.Am, wq.Ap, wq.b = Am[None], Ap[None], bb[None]
        P, C, c, Gd = dense_PCG(wq, 0)
        stat = np.abs(P @ cur["x"][0].ravel() + q + C.T @ cur["yf"][0] + Gd.T @ cur["yg"][0].ravel()).max()
        _, _, finf, ginf = _merit_parts_srb(w, cfg, 0, P, q, cur["x"][0], cur["xi"][0], lo, hi)
        for got, ref in ((log[0, it, 7], stat), (log[0, it, 8], finf), (log[0, it, 9], ginf)):
            assert abs(got - ref) <= 1e-9 * max(1.0, abs(ref))
        conv = stat <= eps_c and finf <= eps_c and ginf <= eps_c
        assert conv == (it == int(info[0, 0]) - 1 and bool(info[0, 1]))
    for k in ("x", "xi", "yf", "yg"):
        assert np.abs(cur[k] - st_all[k]).max() <= 1e-10 * max(1.0, np.abs(st_all[k]).max()), k
    assert info[0, 1] == 1 and seen_backtrack and seen_slack, (info[0], seen_backtrack, seen_slack)
