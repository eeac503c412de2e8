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


# ----------------------------------------------------------------------------------------------- backward vs finite differences
def _loss_of_solution(w, cfg, iters):
    st, info, rc = O.admm(w, cfg, iters=iters)
    return (st["x"] ** 2).sum(axis=(1, 2)), st, info


@pytest.mark.parametrize("soft_bound,lam", [(2.0, 100.0), (0.3, 0.0), (0.3, 0.05)], ids=["cfg2_hard_active", "soft_active", "soft_L1"])
def test_backward_matches_central_finite_differences(soft_bound, lam):
    """dL/dq and dL/dx_init for L = ||x||^2 (reading A-19) vs central differences of tightly converged solves: 1e-6 relative."""
    import copy
    w = W.config2(B=1, N=8, soft_bound=soft_bound)
    w.lam, w.rho_bar = lam, 2.0
    w.q = w.q + 0.3 * np.random.default_rng(5).standard_normal(w.q.shape)
    cfg = O.make_cfg(w)
    iters = 30000
    L0, st, info = _loss_of_solution(w, cfg, iters)
    assert info[0, 0] < 1e-11 and info[0, 1] < 1e-11
    cls = O.classify(w, cfg, st, 0)
    ya = np.abs(st["yg"][0][cls == 1]); assert ya.size == 0 or ya.min() > 1e-4      # screened instance (reading A-17)
    if soft_bound < 1.0:
        assert (cls == 2).sum() > 0
    else:
        assert (cls == 1).sum() > 0
    dq, dxi, counts, rcs = O.backward(w, cfg, st, 2.0 * st["x"])
    assert rcs[0] == 0
    rng = np.random.default_rng(6)
    h = 1e-5
    for trial in range(4):
        dirq = rng.standard_normal(w.q.shape)
        wp, wm = copy.copy(w), copy.copy(w)
        wp.q, wm.q = w.q + h * dirq, w.q - h * dirq
        fd = (_loss_of_solution(wp, cfg, iters)[0] - _loss_of_solution(wm, cfg, iters)[0]) / (2 * h)
        an = (dq * dirq).sum()
        assert abs(fd[0] - an) <= 1e-6 * max(1.0, abs(an))
    for i in range(w.nx):
        wp, wm = copy.copy(w), copy.copy(w)
        wp.x_init, wm.x_init = w.x_init.copy(), w.x_init.copy()
        wp.x_init[0, i] += h; wm.x_init[0, i] -= h
        fd = (_loss_of_solution(wp, cfg, iters)[0] - _loss_of_solution(wm, cfg, iters)[0]) / (2 * h)
        assert abs(fd[0] - dxi[0, i]) <= 1e-6 * max(1.0, abs(dxi[0, i]))


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
    import copy
    for b in range(w.B):
        Am, Ap, bb, G, lo, hi = O.bicycle_linearize(w, cfg, w.xbar0[b], b)
        wq = copy.copy(w)
        wq.B, wq.Am, wq.Ap, wq.b, wq.G, wq.lo, wq.hi = 1, Am[None], Ap[None], bb[None], G[None], lo[None], hi[None]
        wq.q, wq.x_init, wq.model = w.q[b:b + 1], w.x_init[b:b + 1], 0
        s0 = O.new_state(wq); s0["x"] = w.xbar0[b:b + 1].copy()
        s, _, _ = O.admm(wq, O.make_cfg(wq), iters=50, state=s0)
        assert np.abs(s["x"][0] - st1["x"][b]).max() < 1e-12
