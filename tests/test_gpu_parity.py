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


# ----------------------------------------------------------------------------------------------- a10 backward
def _backward_case(dtype, soft_bound, rho_bar, iters, B=6, N=20):
    """Oracle forward output is fed to BOTH sides (reading A-20) so the classification cannot diverge by rounding."""
    import torch
    from paper_2606_24039_b200.solver import Solver
    w = W.config2(B=B, N=N, soft_bound=soft_bound)
    w.rho_bar = rho_bar
    if soft_bound < 1.0:
        w.lam = 0.05       # lambda = 100 makes the stress instance degenerate (more rows at their bound than free directions)
    w.q = w.q + 0.3 * np.random.default_rng(5).standard_normal(w.q.shape)
    wr = w.rounded(np.float32) if dtype == "f32" else w
    eps = 1e-8 if dtype == "f64" else 1e-4
    cfg = O.make_cfg(wr, eps_abs=eps, eps_rel=eps)
    ref, info, rc = O.admm(wr, cfg, iters=iters)
    if dtype == "f32":
        ref = {k: v.astype(np.float32).astype(np.float64) for k, v in ref.items()}
    dq_o, dxi_o, counts, rcs = O.backward(wr, cfg, ref, 2.0 * ref["x"])
    ok = rcs == 0                      # degenerate active sets are skipped (reading A-18)
    assert ok.sum() >= (w.B + 1) // 2
    s = Solver(wr, dtype=dtype)
    s.set_state(ref)
    return w, s, ref, dq_o, dxi_o, counts, ok


@pytest.mark.parametrize("dtype,soft_bound", [("f64", 2.0), ("f64", 0.3), ("f32", 2.0), ("f32", 0.3)])
def test_backward_refine_matches_oracle_definition(dtype, soft_bound):
    from paper_2606_24039_b200 import binding as Bd
    w, s, ref, dq_o, dxi_o, counts, ok = _backward_case(dtype, soft_bound, 2.0, 3000)
    assert counts.sum() > 0
    dq, dxi = s.backward(2.0 * s.s["x"], mode=Bd.TMPC_BWD_REFACTOR_REFINE)
    tol = 1e-9 if dtype == "f64" else 2e-3
    assert rel_err(dq.cpu().double().numpy()[ok], dq_o[ok]) <= tol
    assert rel_err(dxi.cpu().double().numpy()[ok], dxi_o[ok]) <= tol
    s.close()


def test_backward_admm_reuse_factor_converges_to_definition():
    """eq. 67 mode: biased by its tolerance -> loose check after many iterations."""
    from paper_2606_24039_b200 import binding as Bd
    w, s, ref, dq_o, dxi_o, counts, ok = _backward_case("f64", 0.3, 2.0, 3000)
    s.factor()
    dq, dxi = s.backward(2.0 * s.s["x"], mode=Bd.TMPC_BWD_ADMM_REUSE_FACTOR, iters=4000)
    assert rel_err(dq.cpu().double().numpy()[ok], dq_o[ok]) <= 1e-5
    assert rel_err(dxi.cpu().double().numpy()[ok], dxi_o[ok]) <= 1e-5
    s.close()


# ----------------------------------------------------------------------------------------------- a1 + SQP (config 4)
@pytest.mark.parametrize("dtype", ["f64", "f32"])
def test_linearize_matches_oracle(dtype):
    from paper_2606_24039_b200.solver import Solver
    w = W.config4(B=5, N=37, dtype=dtype)
    wr = w.rounded(np.float32) if dtype == "f32" else w
    s = Solver(wr, dtype=dtype)
    s.reset_state(wr.xbar0)
    s.linearize()
    cfg = O.make_cfg(wr)
    tol = 1e-12 if dtype == "f64" else 2e-5
    for b in range(w.B):
        ref = O.bicycle_linearize(wr, cfg, wr.xbar0[b], b)
        for name, r in zip(("Am", "Ap", "b", "G", "lo", "hi"), ref):
            g = s.t[name][b].cpu().double().numpy()
            assert np.abs(g - r).max() <= tol * max(1.0, np.abs(r).max()), name
    s.close()


@pytest.mark.parametrize("dtype", ["f64", "f32"])
def test_config4_sqp_subset(dtype):
    from paper_2606_24039_b200.solver import Solver
    w = W.config4(B=12, dtype=dtype)
    wr = w.rounded(np.float32) if dtype == "f32" else w
    s = Solver(wr, dtype=dtype)
    s.reset_state(wr.xbar0)
    s.sqp()
    got = s.state_numpy()
    ref, info, rc = O.sqp_bicycle(wr, O.make_cfg(wr), nthreads=8)
    assert rc == 0
    compare_states(got, ref, TOL[dtype])
    s.close()


# ----------------------------------------------------------------------------------------------- config 3 (streamed class)
def test_config3_subset_fp32():
    w = W.config3(B=3, N=6)
    run_pair(w, "f32", iters=40, band=1)


def test_streamed_chunk_scheduling_uneven_split_fp32():
    """B = 300 is just above one wave of co-resident CTAs (2 x 148), so tmpc_admm_solve cuts the 33 iterations into 2 chunks
    of 16 and 17 and runs the 600 chunk jobs 296 per launch (a launch mixes chunk 0 and chunk 1 of different problems).
    EVERY problem must still match the oracle's uninterrupted 33 iterations."""
    w = W.config3(B=300, N=2)
    run_pair(w, "f32", iters=33, band=1)


def test_config3_shape_fp64():
    w = W.config3(B=2, N=4)
    run_pair(w, "f64", iters=25, band=1)


@pytest.mark.parametrize("dtype", ["f64", "f32"])
def test_tensor_core_factor_ragged_block_sizes(dtype):
    """factor3_kernel (DMMA tiles of 8 x 8) on block sizes that are NOT a multiple of 8 or 4: n = 37 (padded to 40, the
    synchronous staging path, 5 x 5 tiles on a 4 x 4 warp grid) with a dense G row (G' w G product), implicit E_k, and
    n = 48 (aligned: the cp.async path, nx = 40 spans a full and a ragged chunk of staged rows)."""
    run_pair(W.random_ltv(61, 3, 5, 30, 7, [30, 33, 36], [0, 0, 1, 0], implicit=True, dense_g_rows=1, q_scale=0.3), dtype, iters=40)
    run_pair(W.random_ltv(62, 2, 4, 40, 8, [40, 47], [0, 0], implicit=True, q_scale=0.3), dtype, iters=40)


# ----------------------------------------------------------------------------------------------- a11 cyclic reduction
@pytest.mark.parametrize("N", [1, 2, 4, 20, 63, 64, 100])
def test_cyclic_reduction_solve_equals_sequential_and_oracle(N):
    """T = N+1 in {2,3,5,21,64,65,101}: CR solve == oracle band Cholesky == sequential block factor (reading O-6)."""
    from paper_2606_24039_b200.solver import Solver
    from paper_2606_24039_b200 import binding as Bd
    w = W.random_ltv(40 + N, 2, N, 4, 2, [4, 5], [0, 0, 1], implicit=True, dense_g_rows=1)
    eta = np.random.default_rng(N).standard_normal((w.B, w.T, w.n))
    cfg = O.make_cfg(w)
    ref = np.stack([O.solve_S(w, cfg, eta[b].ravel(), b).reshape(w.T, w.n) for b in range(w.B)])
    for lin in (Bd.TMPC_LIN_CYCLIC_REDUCTION, Bd.TMPC_LIN_SEQUENTIAL):
        s = Solver(w, dtype="f64", linsolve=lin)
        s.factor()
        xt = s.kkt_solve(s._up(eta)).cpu().double().numpy()
        assert rel_err(xt, ref) <= 1e-10, lin
        s.close()


def test_cyclic_reduction_admm_matches_oracle():
    from paper_2606_24039_b200.solver import Solver
    from paper_2606_24039_b200 import binding as Bd
    w = W.random_ltv(51, 2, 37, 4, 2, [4, 5], [0, 0, 1], implicit=True, dense_g_rows=1, q_scale=0.3)
    s = Solver(w, dtype="f64", linsolve=Bd.TMPC_LIN_CYCLIC_REDUCTION)
    s.solve(80)
    got, info = s.state_numpy(), s.info_numpy()
    ref, rinfo, rc = O.admm(w, O.make_cfg(w), iters=80)
    compare_states(got, ref, 1e-9)
    assert (np.abs(info["objective"] - rinfo[:, 2]) <= 1e-9 * np.maximum(1, np.abs(rinfo[:, 2]))).all()
    assert (np.abs(info["r_prim"] - rinfo[:, 0]) <= 1e-9).all() and (np.abs(info["r_dual"] - rinfo[:, 1]) <= 1e-7).all()
    s.close()


@pytest.mark.parametrize("N,n_sqp,iters", [(300, 3, 100), (8192, 3, 100)])
def test_config5_long_horizon_sqp(N, n_sqp, iters):
    """BASELINE configs[4]: bicycle, B=1, fp64, cyclic reduction, 3 SQP x 100 ADMM, against the banded oracle."""
    from paper_2606_24039_b200.solver import Solver
    from paper_2606_24039_b200 import binding as Bd
    w = W.config5(N=N)
    s = Solver(w, dtype="f64", linsolve=Bd.TMPC_LIN_CYCLIC_REDUCTION)
    s.reset_state(w.xbar0)
    s.sqp(n_sqp, iters)
    got = s.state_numpy()
    ref, info, rc = O.sqp_bicycle(w, O.make_cfg(w, band=1), n_sqp=n_sqp, iters=iters)
    assert rc == 0
    compare_states(got, ref, 1e-9)
    s.close()


# ----------------------------------------------------------------------------------------------- full BASELINE sizes
# The batch sizes, horizons and iteration counts of BASELINE.json, i.e. the launch configuration bench.py times
# (CTAs per SM, problems per CTA, waves, ring depth); compared on SAMPLED problems the oracle solves one by one.
def _sample(B, k=6, seed=7):
    idx = set(range(min(3, B))) | {B - 1} | set(np.random.default_rng(seed).integers(0, B, size=k).tolist())
    return np.array(sorted(idx))


@pytest.mark.parametrize("dtype", ["f32", "f64"])
def test_config2_full_batch_sampled(dtype):
    from paper_2606_24039_b200.solver import Solver
    w = W.config2()
    assert w.B == 1024 and w.N == 50 and w.iters == 100
    wr = w.rounded(np.float32) if dtype == "f32" else w
    s = Solver(wr, dtype=dtype)
    s.solve()
    got, info = s.state_numpy(), s.info_numpy()
    assert (info["status"] == 0).all() and all(np.isfinite(got[k]).all() for k in KEYS)
    idx = _sample(w.B)
    ws = wr.subset(idx)
    ref, rinfo, rc = O.admm(ws, O.make_cfg(ws), nthreads=8)
    assert rc == 0
    compare_states({k: got[k][idx] for k in KEYS}, ref, TOL[dtype])
    otol = 1e-4 if dtype == "f32" else 1e-9
    assert (np.abs(info["objective"][idx] - rinfo[:, 2]) <= otol * np.maximum(np.abs(rinfo[:, 2]), 1.0)).all()
    s.close()


def test_config3_full_batch_sampled_fp32():
    from paper_2606_24039_b200.solver import Solver
    w = W.config3()
    assert w.B == 512 and w.N == 32 and w.n == 88 and w.iters == 200
    wr = w.rounded(np.float32)
    s = Solver(wr, dtype="f32")
    s.solve()
    got, info = s.state_numpy(), s.info_numpy()
    assert (info["status"] == 0).all() and all(np.isfinite(got[k]).all() for k in KEYS)
    idx = _sample(w.B, k=3)
    ws = wr.subset(idx)
    ref, rinfo, rc = O.admm(ws, O.make_cfg(ws, band=1), nthreads=8)
    assert rc == 0
    compare_states({k: got[k][idx] for k in KEYS}, ref, TOL["f32"])
    assert (np.abs(info["objective"][idx] - rinfo[:, 2]) <= 1e-4 * np.maximum(np.abs(rinfo[:, 2]), 1.0)).all()
    s.close()


def test_config4_full_batch_sampled_fp32():
    from paper_2606_24039_b200.solver import Solver
    w = W.config4(dtype="f32")
    assert w.B == 4096 and w.N == 100 and w.iters == 50 and w.sqp_iters == 5
    wr = w.rounded(np.float32)
    s = Solver(wr, dtype="f32")
    s.reset_state(wr.xbar0)
    s.sqp()
    got = s.state_numpy()
    assert all(np.isfinite(got[k]).all() for k in KEYS)
    idx = _sample(w.B)
    ws = wr.subset(idx)
    ref, info, rc = O.sqp_bicycle(ws, O.make_cfg(ws), nthreads=8)
    assert rc == 0
    compare_states({k: got[k][idx] for k in KEYS}, ref, TOL["f32"])
    s.close()


# ----------------------------------------------------------------------------------------------- launch-shape edge cases
@pytest.mark.parametrize("B", [1, 7])
def test_resident_odd_batch_fp32(B):
    """Odd batches leave the second problem slot of the last CTA empty (PG = 2); B = 1 takes the one-problem-per-CTA shape."""
    run_pair(W.config2(B=B, N=9), "f32", iters=40)
    run_pair(W.config2(B=B, N=10, soft_bound=0.5), "f64", iters=40)


def test_duplicate_selection_column_falls_back_fp64():
    """Two inequality rows on the same column are outside the fast path's one-row-per-column ownership: generic kernels."""
    w = W.random_ltv(77, 3, 11, 6, 2, [6, 6, 7], [0, 1, 0], q_scale=0.3)
    w.lo[..., 1] = -0.6; w.hi[..., 1] = 0.6          # a second, tighter (soft) bound on the same control
    run_pair(w, "f64", iters=60)
