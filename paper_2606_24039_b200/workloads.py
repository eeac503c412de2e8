"""Seeded synthetic input generators for the five BASELINE.json configs.

This module serves BOTH the CPU oracle (``oracle/``) and the CUDA path. It holds
none of the method's arithmetic (no assembly of S, no factorisation, no ADMM, no
linearisation of the dynamics): it only draws problem data (cost blocks, dynamics
blocks, bounds, initial states, racing-track references) with a counter-based RNG
that is written out here so that every consumer sees bit-identical fp64 inputs
("Synthetic inputs"; DESIGN.md section 4 gives the recipe).

RNG: SplitMix64.  The state of stream ``p`` after ``k`` draws is ``s0_p + k*GAMMA``
(mod 2^64), so draw ``k`` of stream ``p`` is ``mix(s0_p + (k+1)*GAMMA)`` and whole
``[streams, draws]`` tables can be produced at once.  ``s0_p = (seed<<32) ^
(config_id<<24) ^ p``.  U[0,1) = (z>>11) * 2^-53.  Normals: Box-Muller, cos branch,
two uniforms per normal (u1 is mapped to (0,1] so the log is finite).

Layouts follow include/tmpc.h (problem-major, row-major blocks):
  D [Bd][T][n][n]   E [Be][N][n][n]   q [B][T][n]
  Am, Ap [B][N][nx][n]   b [B][N][nx]   x_init [B][nx]
  G [Bg][T][ng][n] or None (selection rows given by g_col)   lo, hi [B][T][ng]
with Bd/Be/Bg either B or 1 (shared by the batch).  Dynamics convention (DESIGN.md
reading A-23): E_k x_{k+1} = A_k x_k + B_k u_k + c_k  is stored as
Am=[A_k B_k], Ap=[-E_k 0], b=-c_k, i.e. Am v_k + Ap v_{k+1} = b (eq. 36).
"""
from __future__ import annotations

from dataclasses import dataclass, field
from typing import Optional

import numpy as np

_GAMMA = np.uint64(0x9E3779B97F4A7C15)
_M1 = np.uint64(0xBF58476D1CE4E5B9)
_M2 = np.uint64(0x94D049BB133111EB)


def _mix(z: np.ndarray) -> np.ndarray:
    z = (z ^ (z >> np.uint64(30))) * _M1
    z = (z ^ (z >> np.uint64(27))) * _M2
    return z ^ (z >> np.uint64(31))


class Streams:
    """One SplitMix64 stream per problem; draws are taken in a fixed order."""

    def __init__(self, seed: int, config_id: int, problem_index: np.ndarray):
        p = np.asarray(problem_index, dtype=np.uint64)
        self.s0 = (np.uint64(seed) << np.uint64(32)) ^ (np.uint64(config_id) << np.uint64(24)) ^ p
        self.k = 0  # draws consumed so far (same for every stream)

    def _raw(self, count: int) -> np.ndarray:
        ks = np.arange(self.k + 1, self.k + count + 1, dtype=np.uint64)
        self.k += count
        with np.errstate(over="ignore"):
            return _mix(self.s0[:, None] + ks[None, :] * _GAMMA)

    def uniform01(self, count: int) -> np.ndarray:
        """[streams, count] U[0,1)."""
        return (self._raw(count) >> np.uint64(11)).astype(np.float64) * (2.0 ** -53)

    def uniform(self, lo: float, hi: float, count: int) -> np.ndarray:
        return lo + (hi - lo) * self.uniform01(count)

    def normal(self, count: int) -> np.ndarray:
        """[streams, count] N(0,1); consumes 2*count uniforms per stream (u1,u2 interleaved)."""
        u = self.uniform01(2 * count)
        u1 = 1.0 - u[:, 0::2]  # (0,1]
        u2 = u[:, 1::2]
        return np.sqrt(-2.0 * np.log(u1)) * np.cos(2.0 * np.pi * u2)


@dataclass
class QPData:
    """One batch of stage-structured QPs plus the solver settings of its config."""

    name: str
    B: int
    N: int
    nx: int
    nu: int
    ng: int
    dtype: str  # "f32" | "f64": the arithmetic type the config asks for
    D: np.ndarray
    E: np.ndarray
    q: np.ndarray
    Am: Optional[np.ndarray]
    Ap: Optional[np.ndarray]
    b: Optional[np.ndarray]
    x_init: np.ndarray
    G: Optional[np.ndarray]
    lo: Optional[np.ndarray]
    hi: Optional[np.ndarray]
    g_col: Optional[list] = None  # selection rows: column index of each row of G_t
    soft: list = field(default_factory=list)  # per-row soft mask (len ng)
    sigma: float = 1e-6
    rho_bar: float = 0.1
    rho_eq_scale: float = 1e3
    alpha: float = 1.6
    gamma: float = 2.0  # gamma_xi (quadratic slack weight)
    lam: float = 0.0  # L1 slack weight [NS]
    iters: int = 100
    # nonlinear (bicycle) configs only
    model: int = 0
    stage_ref: Optional[np.ndarray] = None  # [B][T][n]  (x_ref, u_ref)
    xbar0: Optional[np.ndarray] = None  # [B][T][n]  SQP start
    g_lo: Optional[list] = None  # un-shifted bounds of g (len ng)
    g_hi: Optional[list] = None
    wheelbase: float = 2.7
    dt: float = 0.05
    sqp_iters: int = 0
    model_params: Optional[list] = None  # model 2 (SRB humanoid): mass, g[3], diag(I)[3], foot_L[3], foot_R[3]

    @property
    def n(self) -> int:
        return self.nx + self.nu

    @property
    def T(self) -> int:
        return self.N + 1

    def G_dense(self) -> np.ndarray:
        """G as a dense [Bg][T][ng][n] array (selection rows expanded)."""
        if self.G is not None:
            return self.G
        G = np.zeros((1, self.T, self.ng, self.n))
        for r, c in enumerate(self.g_col):
            G[0, :, r, c] = 1.0
        return G

    def rounded(self, np_dtype) -> "QPData":
        """Copy whose float arrays are rounded to np_dtype and widened back to fp64
        (fp32 runs: both sides consume the rounded values)."""
        import copy

        out = copy.copy(self)
        for k in ("D", "E", "q", "Am", "Ap", "b", "x_init", "G", "lo", "hi", "stage_ref", "xbar0"):
            v = getattr(self, k)
            if v is not None:
                setattr(out, k, v.astype(np_dtype).astype(np.float64))
        return out

    def subset(self, idx) -> "QPData":
        import copy

        idx = np.asarray(idx)
        out = copy.copy(self)
        out.B = len(idx)
        for k in ("D", "E", "q", "Am", "Ap", "b", "x_init", "G", "lo", "hi", "stage_ref", "xbar0"):
            v = getattr(self, k)
            if v is not None and v.shape[0] != 1:
                setattr(out, k, np.ascontiguousarray(v[idx]))
        return out


def _rate_cost_blocks(T: int, nx: int, nu: int, Q, R, S, QN=None):
    """D_t, E_t for  sum_t 1/2 x'Qx + 1/2 u'Ru  +  sum_{k=1..N} 1/2 (u_k-u_{k-1})' S (u_k-u_{k-1})
    (reading A-11: +S on the u-block of D_0 and D_N, +2S inside, -S in the u-u block of E_t)."""
    n = nx + nu
    N = T - 1
    D = np.zeros((1, T, n, n))
    E = np.zeros((1, N, n, n))
    for t in range(T):
        D[0, t, :nx, :nx] = QN if (t == N and QN is not None) else Q
        D[0, t, nx:, nx:] = R
        if S is not None:
            D[0, t, nx:, nx:] += S if (t == 0 or t == N) else 2.0 * S
    if S is not None:
        E[0, :, nx:, nx:] = -S
    return D, E


# --------------------------------------------------------------------------- config 1
def config1(seed: int = 0, bounded: bool = True) -> QPData:
    """2-D double integrator, nx=4, nu=2, dt=0.1, N=20, B=1, fp64 (BASELINE.json configs[0];
    recipe I-1).  bounded=False gives the same instance with bounds at +-inf (Riccati pin)."""
    nx, nu, N, dt, B = 4, 2, 20, 0.1, 1
    n, T = nx + nu, N + 1
    I2 = np.eye(2)
    A = np.block([[I2, dt * I2], [np.zeros((2, 2)), I2]])  # exact ZOH (A-22)
    Bm = np.vstack([0.5 * dt * dt * I2, dt * I2])
    Q = np.diag([1.0, 1.0, 0.1, 0.1])
    R = 0.01 * np.eye(2)
    D, E = _rate_cost_blocks(T, nx, nu, Q, R, None, QN=10.0 * Q)
    Am = np.zeros((B, N, nx, n))
    Ap = np.zeros((B, N, nx, n))
    Am[:, :, :, :nx] = A
    Am[:, :, :, nx:] = Bm
    Ap[:, :, :, :nx] = -np.eye(nx)
    b = np.zeros((B, N, nx))
    st = Streams(seed, 1, np.arange(B))
    pos = st.uniform(-3.0, 3.0, 2)
    vel = st.uniform(-1.0, 1.0, 2)
    x_init = np.concatenate([pos, vel], axis=1)
    g_col = [4, 5, 2, 3]  # u1, u2, vx, vy
    bnd = np.array([1.0, 1.0, 2.0, 2.0]) if bounded else np.full(4, np.inf)
    lo = np.broadcast_to(-bnd, (B, T, 4)).copy()
    hi = np.broadcast_to(bnd, (B, T, 4)).copy()
    return QPData("cfg1_double_integrator", B, N, nx, nu, 4, "f64", D, E, np.zeros((B, T, n)), Am, Ap, b,
                  x_init, None, lo, hi, g_col=g_col, soft=[0, 0, 0, 0], iters=500)


# --------------------------------------------------------------------------- config 2
def config2(seed: int = 0, B: int = 1024, N: int = 50, soft_bound: float = 2.0, dtype: str = "f32",
            first_problem: int = 0) -> QPData:
    """Random LTV QP batch with rate cost and slack (BASELINE.json configs[1]; recipe I-2).
    soft_bound=0.5 is the stress variant I-2s that actually violates soft rows."""
    nx, nu, dt = 6, 2, 0.05
    n, T = nx + nu, N + 1
    st = Streams(seed, 2, np.arange(first_problem, first_problem + B))
    per_k = nx * nx + nx * nu + nx
    nrm = st.normal(N * per_k).reshape(B, N, per_k)
    Gk = nrm[:, :, : nx * nx].reshape(B, N, nx, nx) / np.sqrt(nx)
    Bk = dt * nrm[:, :, nx * nx: nx * nx + nx * nu].reshape(B, N, nx, nu)
    ck = 0.1 * nrm[:, :, nx * nx + nx * nu:]
    x_init = st.uniform(-1.0, 1.0, nx)
    Am = np.zeros((B, N, nx, n))
    Ap = np.zeros((B, N, nx, n))
    Am[:, :, :, :nx] = np.eye(nx) + dt * Gk
    Am[:, :, :, nx:] = Bk
    Ap[:, :, :, :nx] = -np.eye(nx)
    b = -ck
    D, E = _rate_cost_blocks(T, nx, nu, np.eye(nx), 0.1 * np.eye(nu), 0.1 * np.eye(nu))
    g_col = [6, 7, 0, 1, 2, 3, 4, 5]  # u1,u2 hard; x1..x6 soft
    bnd = np.array([1.0, 1.0] + [soft_bound] * 6)
    lo = np.broadcast_to(-bnd, (B, T, 8)).copy()
    hi = np.broadcast_to(bnd, (B, T, 8)).copy()
    return QPData("cfg2_ltv_rate_slack", B, N, nx, nu, 8, dtype, D, E, np.zeros((B, T, n)), Am, Ap, b, x_init,
                  None, lo, hi, g_col=g_col, soft=[0, 0, 1, 1, 1, 1, 1, 1], gamma=2.0, lam=100.0, iters=100)


# --------------------------------------------------------------------------- config 3
def config3(seed: int = 0, B: int = 512, N: int = 32, nx: int = 64, nu: int = 24, first_problem: int = 0) -> QPData:
    """Humanoid-scale dense-block LTV QP with implicit-form dynamics, fp32
    (BASELINE.json configs[2]; recipe I-3).  Draw order per k: E, A, B, c; then x_ref, x_init."""
    n, T = nx + nu, N + 1
    st = Streams(seed, 3, np.arange(first_problem, first_problem + B))
    per_k = 2 * nx * nx + nx * nu + nx
    nrm = st.normal(N * per_k).reshape(B, N, per_k)
    o = 0
    Ek = np.eye(nx) + 0.1 * nrm[:, :, o:o + nx * nx].reshape(B, N, nx, nx) / np.sqrt(nx); o += nx * nx
    Ak = np.eye(nx) + 0.05 * nrm[:, :, o:o + nx * nx].reshape(B, N, nx, nx) / np.sqrt(nx); o += nx * nx
    Bk = 0.05 * nrm[:, :, o:o + nx * nu].reshape(B, N, nx, nu); o += nx * nu
    ck = 0.1 * nrm[:, :, o:o + nx]
    del nrm
    x_ref = np.sqrt(0.5) * st.normal(T * nx).reshape(B, T, nx)
    x_init = np.sqrt(0.5) * st.normal(nx)
    Am = np.concatenate([Ak, Bk], axis=3)
    Ap = np.concatenate([-Ek, np.zeros((B, N, nx, nu))], axis=3)
    b = -ck
    D, E = _rate_cost_blocks(T, nx, nu, np.eye(nx), 0.01 * np.eye(nu), None)
    q = np.zeros((B, T, n))
    q[:, :, :nx] = -x_ref
    g_col = list(range(nx, n))
    lo = np.full((B, T, nu), -2.0)
    hi = np.full((B, T, nu), 2.0)
    return QPData("cfg3_dense_implicit", B, N, nx, nu, nu, "f32", D, E, q, Am, Ap, b, x_init, None, lo, hi,
                  g_col=g_col, soft=[0] * nu, iters=200)


# --------------------------------------------------------------------------- configs 4, 5
def _bspline_eval(P: np.ndarray, seg: np.ndarray, u: np.ndarray):
    """Closed uniform cubic B-spline.  P [B,8,2] control points; seg/u [B,K] segment index and
    local parameter.  Returns position, first and second parameter-derivatives, each [B,K,2]."""
    nC = P.shape[1]
    b0 = (1 - u) ** 3 / 6.0
    b1 = (3 * u ** 3 - 6 * u ** 2 + 4) / 6.0
    b2 = (-3 * u ** 3 + 3 * u ** 2 + 3 * u + 1) / 6.0
    b3 = u ** 3 / 6.0
    d0 = -((1 - u) ** 2) / 2.0
    d1 = (9 * u ** 2 - 12 * u) / 6.0
    d2 = (-9 * u ** 2 + 6 * u + 3) / 6.0
    d3 = u ** 2 / 2.0
    e0 = 1 - u
    e1 = 3 * u - 2
    e2 = -3 * u + 1
    e3 = u
    rows = np.arange(P.shape[0])[:, None]
    pts = [P[rows, (seg + m) % nC] for m in range(4)]  # each [B,K,2]
    pos = sum(w[..., None] * p for w, p in zip((b0, b1, b2, b3), pts))
    d1v = sum(w[..., None] * p for w, p in zip((d0, d1, d2, d3), pts))
    d2v = sum(w[..., None] * p for w, p in zip((e0, e1, e2, e3), pts))
    return pos, d1v, d2v


def bicycle(seed: int = 0, B: int = 4096, N: int = 100, dtype: str = "f32", config_id: int = 4,
            sqp_iters: int = 5, iters: int = 50, first_problem: int = 0, chunk: int = 256) -> QPData:
    """Kinematic-bicycle racing OCP on a random closed spline (BASELINE.json configs[3] and,
    with N=8192, B=1, fp64, config_id=5, configs[4]; recipes I-4 / I-5, all 'proposed' there)."""
    nx, nu, ng = 4, 2, 3
    n, T = nx + nu, N + 1
    dt, Lwb, v_ref = 0.05, 2.7, 15.0
    samples = 2048
    stage_ref = np.zeros((B, T, n))
    x_init = np.zeros((B, nx))
    for c0 in range(0, B, chunk):
        c1 = min(B, c0 + chunk)
        nb = c1 - c0
        st = Streams(seed, config_id, np.arange(first_problem + c0, first_problem + c1))
        r = st.uniform(20.0, 60.0, 8)
        ang = 2.0 * np.pi * np.arange(8) / 8.0
        P = np.stack([r * np.cos(ang), r * np.sin(ang)], axis=2)  # [nb,8,2]
        # arc-length table: 8 segments x 2048 samples, chord lengths
        grid = np.arange(8 * samples + 1)
        seg = np.broadcast_to((grid // samples) % 8, (nb, grid.size))
        uu = np.broadcast_to((grid % samples) / samples, (nb, grid.size))
        pos, _, _ = _bspline_eval(P, seg, uu)
        ds = np.sqrt(((pos[:, 1:] - pos[:, :-1]) ** 2).sum(axis=2))
        s_tab = np.concatenate([np.zeros((nb, 1)), np.cumsum(ds, axis=1)], axis=1)
        L_track = s_tab[:, -1]
        s0 = st.uniform01(1)[:, 0] * L_track
        lat = st.uniform(-1.0, 1.0, 1)[:, 0]
        dpsi = st.uniform(-0.1, 0.1, 1)[:, 0]
        v0 = st.uniform(12.0, 18.0, 1)[:, 0]
        s_k = np.mod(s0[:, None] + np.arange(T)[None, :] * v_ref * dt, L_track[:, None])
        par = np.stack([np.interp(s_k[i], s_tab[i], grid.astype(np.float64)) for i in range(nb)])
        par = np.minimum(par, 8 * samples - 1e-9)
        segk = (par // samples).astype(np.int64) % 8
        uk = (par % samples) / samples
        pk, d1k, d2k = _bspline_eval(P, segk, uk)
        psi = np.unwrap(np.arctan2(d1k[..., 1], d1k[..., 0]), axis=1)
        kappa = (d1k[..., 0] * d2k[..., 1] - d1k[..., 1] * d2k[..., 0]) / (d1k[..., 0] ** 2 + d1k[..., 1] ** 2) ** 1.5
        stage_ref[c0:c1, :, 0] = pk[..., 0]
        stage_ref[c0:c1, :, 1] = pk[..., 1]
        stage_ref[c0:c1, :, 2] = psi
        stage_ref[c0:c1, :, 3] = v_ref
        stage_ref[c0:c1, :, 4] = 0.0
        stage_ref[c0:c1, :, 5] = np.arctan(Lwb * kappa)
        x_init[c0:c1, 0] = pk[:, 0, 0] - np.sin(psi[:, 0]) * lat
        x_init[c0:c1, 1] = pk[:, 0, 1] + np.cos(psi[:, 0]) * lat
        x_init[c0:c1, 2] = psi[:, 0] + dpsi
        x_init[c0:c1, 3] = v0
    Q = np.diag([1.0, 1.0, 10.0, 1.0])
    R = np.diag([0.01, 0.1])
    S = np.diag([0.1, 10.0])
    D, E = _rate_cost_blocks(T, nx, nu, Q, R, S)
    q = np.zeros((B, T, n))
    q[:, :, :nx] = -stage_ref[:, :, :nx] @ Q
    q[:, :, nx:] = -stage_ref[:, :, nx:] @ R
    xbar0 = stage_ref.copy()
    xbar0[:, 0, :nx] = x_init
    name = "cfg4_bicycle_sqp" if config_id == 4 else "cfg5_bicycle_long_horizon"
    return QPData(name, B, N, nx, nu, ng, dtype, D, E, q, None, None, None, x_init, None, None, None,
                  g_col=None, soft=[0, 0, 1], gamma=2.0, lam=100.0, iters=iters, model=1, stage_ref=stage_ref,
                  xbar0=xbar0, g_lo=[-6.0, -0.4, -3.0], g_hi=[3.0, 0.4, 3.0], wheelbase=Lwb, dt=dt,
                  sqp_iters=sqp_iters)


def config4(seed: int = 0, B: int = 4096, N: int = 100, dtype: str = "f32", **kw) -> QPData:
    return bicycle(seed, B, N, dtype, 4, sqp_iters=5, iters=50, **kw)


def config5(seed: int = 0, N: int = 8192, dtype: str = "f64", **kw) -> QPData:
    return bicycle(seed, 1, N, dtype, 5, sqp_iters=3, iters=100, **kw)


# --------------------------------------------------------------------------- small random QPs (tests)
def random_ltv(seed: int, B: int, N: int, nx: int, nu: int, ng_sel: list, soft: list, bound: float = 0.5,
               implicit: bool = False, rate: bool = True, dense_g_rows: int = 0, config_id: int = 9,
               q_scale: float = 0.0) -> QPData:
    """Small random LTV QP family for parity/edge tests (same structure as config 2/3, any sizes).
    dense_g_rows>0 appends that many dense inequality rows (general G path)."""
    n, T = nx + nu, N + 1
    dt = 0.1
    st = Streams(seed, config_id, np.arange(B))
    per_k = 2 * nx * nx + nx * nu + nx
    nrm = st.normal(N * per_k).reshape(B, N, per_k)
    o = 0
    Ek = np.eye(nx) + (0.1 * nrm[:, :, o:o + nx * nx].reshape(B, N, nx, nx) / np.sqrt(nx) if implicit else 0.0); o += nx * nx
    Ak = np.eye(nx) + dt * nrm[:, :, o:o + nx * nx].reshape(B, N, nx, nx) / np.sqrt(nx); o += nx * nx
    Bk = 2 * dt * nrm[:, :, o:o + nx * nu].reshape(B, N, nx, nu); o += nx * nu
    ck = 0.1 * nrm[:, :, o:o + nx]
    x_init = st.uniform(-1.0, 1.0, nx)
    qv = q_scale * st.normal(T * n).reshape(B, T, n)
    Am = np.concatenate([Ak, Bk], axis=3)
    Ap = np.concatenate([-Ek * np.ones((B, N, 1, 1)), np.zeros((B, N, nx, nu))], axis=3)
    D, E = _rate_cost_blocks(T, nx, nu, np.eye(nx), 0.1 * np.eye(nu), 0.1 * np.eye(nu) if rate else None)
    ng = len(ng_sel) + dense_g_rows
    if dense_g_rows:
        G = np.zeros((B, T, ng, n))
        for r, c in enumerate(ng_sel):
            G[:, :, r, c] = 1.0
        G[:, :, len(ng_sel):, :] = st.normal(T * dense_g_rows * n).reshape(B, T, dense_g_rows, n) / np.sqrt(n)
        g_col = None
    else:
        G, g_col = None, list(ng_sel)
    lo = np.full((B, T, ng), -bound)
    hi = np.full((B, T, ng), bound)
    return QPData(f"random_ltv_nx{nx}_nu{nu}_N{N}", B, N, nx, nu, ng, "f64", D, E, qv, Am, Ap, -ck, x_init, G,
                  lo, hi, g_col=g_col, soft=list(soft), gamma=2.0, lam=0.0, iters=100)


def with_dense_Ap(w: QPData, seed: int = 0, scale: float = 0.05) -> QPData:
    """Copy of `w` whose A_t^+ blocks also depend on u_{t+1} (implicit integrators such as the trapezoidal rule,
    PAPER.md:584-592 Remark A1 / eq. 36): the u-columns of Ap, zero in every BASELINE config, are filled with
    scale * N(0,1) from a stream of its own (config id 10), so the instances without this call are unchanged."""
    import copy

    out = copy.copy(w)
    st = Streams(seed, 10, np.arange(w.B))
    out.Ap = w.Ap.copy()
    out.Ap[:, :, :, w.nx:] = scale * st.normal(w.N * w.nx * w.nu).reshape(w.B, w.N, w.nx, w.nu)
    out.name = w.name + "_denseAp"
    return out


# --------------------------------------------------------------------------- f4: the paper's linear-system RL generator
def linear_rl(seed: int = 0, B: int = 64, N: int = 40, nx: int = 8, nu: int = 4, u_max: float = 1.0, theta: float = 1.0,
              dtype: str = "f64", first_problem: int = 0) -> QPData:
    """Linear-quadratic OCP batch of the paper's scaling study (Sec. IV-B): time-invariant
    x+ = A x + B u + b per problem with A = I + 0.1 dA, vec(dA) ~ N(0, I), eigenvalues clipped to |lambda| <= 0.99,
    vec(B) ~ N(0, I), b ~ N(0, 1e-4 I), x0 ~ N(0, 25 I); stage cost x'Qx + |u|^2 with Q = diag(theta) (all stages, u_N
    included, reading A-10), i.e. D = 2 blkdiag(Q, I) in the 1/2-convention (A-9); hard bounds |u|_inf <= u_max.
    Draw order per problem: dA (row-major), B, b, x0.  Nominal shape (B, N, nx, nu) = (64, 40, 8, 4)."""
    n, T = nx + nu, N + 1
    st = Streams(seed, 11, np.arange(first_problem, first_problem + B))
    dA = st.normal(nx * nx).reshape(B, nx, nx)
    Bm = st.normal(nx * nu).reshape(B, nx, nu)
    bv = 0.01 * st.normal(nx)
    x0 = 5.0 * st.normal(nx)
    A = np.eye(nx) + 0.1 * dA
    lam, V = np.linalg.eig(A)                                        # clip the spectrum: |lambda| in (0, 0.99]
    scale = np.minimum(1.0, 0.99 / np.maximum(np.abs(lam), 1e-300))
    A = np.real(np.einsum("bij,bj,bjk->bik", V, lam * scale, np.linalg.inv(V)))
    Am = np.zeros((B, N, nx, n))
    Ap = np.zeros((B, N, nx, n))
    Am[:, :, :, :nx] = A[:, None]
    Am[:, :, :, nx:] = Bm[:, None]
    Ap[:, :, :, :nx] = -np.eye(nx)
    b = np.broadcast_to(-bv[:, None, :], (B, N, nx)).copy()
    D, E = _rate_cost_blocks(T, nx, nu, 2.0 * theta * np.eye(nx), 2.0 * np.eye(nu), None)
    lo = np.full((B, T, nu), -u_max)
    hi = np.full((B, T, nu), u_max)
    return QPData(f"f4_linear_rl_umax{u_max:g}", B, N, nx, nu, nu, dtype, D, E, np.zeros((B, T, n)), Am, Ap, b, x0, None, lo, hi,
                  g_col=list(range(nx, n)), soft=[0] * nu, iters=100)


# --------------------------------------------------------------------------- f3: SRB humanoid balancing OCP
SRB_PARAMS = [33.34, 0.0, 0.0, -9.81, 1.2, 1.0, 0.4, 0.0, 0.1, 0.0, 0.0, -0.1, 0.0]   # m, g, diag(I) and foot positions: proposed (A-38)


def srb_humanoid(seed: int = 0, B: int = 64, N: int = 20, dtype: str = "f64", sqp_iters: int = 4, iters: int = 60, first_problem: int = 0) -> QPData:
    """Humanoid balancing OCP of the paper's imitation-learning experiment (eq. 68-70): single-rigid-body dynamics,
    x = (p, Theta, v, omega) in R^12, u = (f_L, f_R) in R^6, RK4 with dt = 0.025, N = 20, cost dx'Q dx + du'R du with Q = diag(exp(theta)),
    R = 1e-3 I, box bounds on u (eq. 70d).  The paper gives m = 33.34 kg and g; proposed here (reading A-38, the paper is silent): I = diag(1.2,
    1.0, 0.4) kg m^2, feet at (0, +-0.1, 0) m, standing reference p_ref = (0, 0, 0.6), u_ref = (0, 0, m g / 2) per foot, log-weights theta =
    log(100, 100, 100, 50, 50, 50, 1, 1, 1, 1, 1, 1), bounds f_xy in [-8, 8] N, f_z in [150, 170] N (tight enough to bind on the perturbed
    starts: the unconstrained controller asks for +-15 N and 157..173 N), and a perturbed start
    x_init = x_ref + (N(0, 0.03^2) on p, N(0, 0.08^2) on Theta, N(0, 0.2^2) on v, N(0, 0.3^2) on omega).  Draw order: the 12 normals of x_init."""
    nx, nu, n, T = 12, 6, 18, N + 1
    mp = list(SRB_PARAMS)
    mass, gz = mp[0], mp[3]
    st = Streams(seed, 12, np.arange(first_problem, first_problem + B))
    nrm = st.normal(12)
    x_ref = np.zeros(12); x_ref[2] = 0.6
    u_ref = np.array([0.0, 0.0, -mass * gz / 2.0] * 2)
    sd = np.array([0.03] * 3 + [0.08] * 3 + [0.2] * 3 + [0.3] * 3)
    x_init = x_ref[None, :] + sd[None, :] * nrm
    Q = 2.0 * np.diag([100.0] * 3 + [50.0] * 3 + [1.0] * 6)           # dx'Q dx without 1/2 -> D = 2 Q in the 1/2-convention (A-9)
    R = 2.0 * 1e-3 * np.eye(nu)
    D, E = _rate_cost_blocks(T, nx, nu, Q, R, None)
    ref = np.concatenate([x_ref, u_ref])
    q = np.broadcast_to(-(D[0, 0] @ ref), (B, T, n)).copy()
    stage_ref = np.broadcast_to(ref, (B, T, n)).copy()
    xbar0 = stage_ref.copy(); xbar0[:, 0, :nx] = x_init
    lo = np.broadcast_to(np.array([-8.0, -8.0, 150.0] * 2), (B, T, nu)).copy()
    hi = np.broadcast_to(np.array([8.0, 8.0, 170.0] * 2), (B, T, nu)).copy()
    return QPData("f3_srb_humanoid", B, N, nx, nu, nu, dtype, D, E, q, None, None, None, x_init, None, lo, hi, g_col=list(range(nx, n)),
                  soft=[0] * nu, rho_bar=0.1, iters=iters, model=2, stage_ref=stage_ref, xbar0=xbar0, dt=0.025, sqp_iters=sqp_iters, model_params=mp)
