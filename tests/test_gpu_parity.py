"""-m gpu: the CUDA path (through the C ABI) against the CPU oracle, element by element on the same seeded inputs.

Norm (reading A-27): per problem and per vector v in {x, z_g, y_f, y_g, xi}:
||v_gpu - v_oracle||_inf / max(||v_oracle||_inf, 1); the worst problem of the batch is compared with
fp64: 1e-9; fp32: 2e-3 on iterates and 1e-4 relative on the objective (north_star)."""
import numpy as np
import pytest

import oracle as O
from paper_2606_24039_b200 import workloads as W

pytestmark = pytest.mark.gpu

TOL = {"f64": 1e-9, "f32": 2e-3}
KEYS = ("x", "zg", "yf", "yg", "xi")


def rel_err(got, ref):
    B = ref.shape[0]
    g, r = got.reshape(B, -1), ref.reshape(B, -1)
    return (np.abs(g - r).max(axis=1) / np.maximum(np.abs(r).max(axis=1), 1.0)).max()


def compare_states(got, ref, tol):
    for k in KEYS:
        e = rel_err(got[k], ref[k])
        assert e <= tol, f"{k}: {e:.3e} > {tol}"


def run_pair(w, dtype, iters=None, band=None, check_obj=True):
    from paper_2606_24039_b200.solver import Solver
    wr = w.rounded(np.float32) if dtype == "f32" else w
    s = Solver(wr, dtype=dtype)
    s.solve(iters)
    got, info = s.state_numpy(), s.info_numpy()
    ref, rinfo, rc = O.admm(wr, O.make_cfg(wr, band=band), iters=iters, nthreads=8)
    assert rc == 0 and (info["status"] == 0).all()
    compare_states(got, ref, TOL[dtype])
    if check_obj:
        otol = 1e-4 if dtype == "f32" else 1e-9
        assert (np.abs(info["objective"] - rinfo[:, 2]) <= otol * np.maximum(np.abs(rinfo[:, 2]), 1.0)).all()
        rtol = 5e-3 if dtype == "f32" else 1e-7
        assert (np.abs(info["r_prim"] - rinfo[:, 0]) <= rtol * np.maximum(1.0, np.abs(ref["x"]).max())).all()
        assert (np.abs(info["r_dual"] - rinfo[:, 1]) <= rtol * np.maximum(1.0, np.abs(ref["yf"]).max())).all()
    s.close()
    return got, ref


def test_config1_fp64():
    run_pair(W.config1(), "f64")


@pytest.mark.parametrize("dtype", ["f64", "f32"])
def test_config2_subset(dtype):
    run_pair(W.config2(B=24), dtype)


@pytest.mark.parametrize("dtype", ["f64", "f32"])
def test_config2_slack_stress(dtype):
    """I-2s: soft bounds +-0.5 with rho_bar = 20 so that soft-active and L1 dead-zone rows occur (reading A-14)."""
    w = W.config2(B=16, soft_bound=0.5)
    w.rho_bar = 20.0
    got, ref = run_pair(w, dtype)
    assert (ref["xi"] != 0).sum() > 0


@pytest.mark.parametrize("dtype", ["f64", "f32"])
def test_ragged_generic_sizes(dtype):
    """n = 5 and n = 3 (no compile-time specialisation), implicit E_k, dense G rows, N not a multiple of anything."""
    run_pair(W.random_ltv(21, 5, 13, 3, 2, [3, 4], [0, 0], implicit=True, q_scale=0.3), dtype, iters=60)
    run_pair(W.random_ltv(22, 3, 7, 2, 1, [2, 0, 1], [0, 1, 1, 1], dense_g_rows=1, q_scale=0.3), dtype, iters=60)


def test_edge_cases_fp64():
    """N = 1 (shortest horizon), zero iterations (state must come back unchanged, z_g projected), unbounded rows."""
    from paper_2606_24039_b200.solver import Solver
    run_pair(W.random_ltv(23, 2, 1, 3, 2, [3, 4], [0, 0], q_scale=0.3), "f64", iters=30)
    run_pair(W.config1(bounded=False), "f64", iters=100)
    w = W.config2(B=3, N=5)
    s = Solver(w, dtype="f64")
    s.solve(0)
    st = s.state_numpy()
    assert all(np.abs(st[k]).max() == 0 for k in KEYS)
    s.close()


def test_resume_equals_single_call_fp64():
    """K1 + K2 iterations with TMPC_SOLVE_ZG_GIVEN == K1 + K2 at once (warm start = resume)."""
    from paper_2606_24039_b200.solver import Solver
    from paper_2606_24039_b200 import binding as Bd
    w = W.config2(B=4, N=20, soft_bound=0.5)
    a = Solver(w, dtype="f64"); a.solve(70); ra = a.state_numpy()
    b = Solver(w, dtype="f64"); b.solve(30); b.admm_solve(40, flags=Bd.TMPC_SOLVE_ZG_GIVEN); rb = b.state_numpy()
    compare_states(rb, ra, 1e-12)


@pytest.mark.parametrize("dtype", ["f64", "f32"])
def test_kkt_solve_matches_oracle_cholesky(dtype):
    """a2+a3+a5+a6: x~ = S^{-1} eta from the block factor vs the oracle's band Cholesky of the assembled S."""
    import torch
    from paper_2606_24039_b200.solver import Solver
    for w in (W.config2(B=4, N=17), W.random_ltv(31, 3, 9, 3, 2, [3, 4], [0, 0], implicit=True, dense_g_rows=2)):
        if len(w.soft) < w.ng:
            w.soft = w.soft + [0] * (w.ng - len(w.soft))
        wr = w.rounded(np.float32) if dtype == "f32" else w
        s = Solver(wr, dtype=dtype)
        s.factor()
        eta = np.random.default_rng(0).standard_normal((w.B, w.T, w.n))
        if dtype == "f32":
            eta = eta.astype(np.float32).astype(np.float64)
        xt = s.kkt_solve(s._up(eta)).cpu().double().numpy()
        cfg = O.make_cfg(wr)
        ref = np.stack([O.solve_S(wr, cfg, eta[b].ravel(), b).reshape(w.T, w.n) for b in range(w.B)])
        assert rel_err(xt, ref) <= (1e-10 if dtype == "f64" else 2e-3)
        s.close()
