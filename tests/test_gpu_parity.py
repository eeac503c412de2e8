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


def test_kkt_solve_long_horizon_variants_fp64():
    """tmpc_kkt_solve (one S^{-1} eta, no ADMM state) through the long-horizon variants of the resident kernel: cluster pair with full records
    (N = 80), one CTA with the chain's share (N = 160; and the (6, 4) block with dense G at N = 400), cluster pair with the chain's share (N = 320)."""
    from paper_2606_24039_b200.solver import Solver
    cases = [W.linear_rl(B=2, N=80, u_max=1.0), W.linear_rl(B=2, N=160, u_max=1.0), W.linear_rl(B=2, N=320, u_max=1.0),
             W.random_ltv(31, 2, 400, 4, 2, [4], [0, 1, 0], dense_g_rows=2, q_scale=0.3)]
    for w in cases:
        s = Solver(w, dtype="f64")
        s.factor()
        eta = np.random.default_rng(1).standard_normal((w.B, w.T, w.n))
        xt = s.kkt_solve(s._up(eta)).cpu().double().numpy()
        cfg = O.make_cfg(w)
        ref = np.stack([O.solve_S(w, cfg, eta[b].ravel(), b).reshape(w.T, w.n) for b in range(w.B)])
        assert rel_err(xt, ref) <= 1e-9, (w.name, rel_err(xt, ref))
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
def test_config2_full_batch_every_problem(dtype):
    from paper_2606_24039_b200.solver import Solver
    w = W.config2()
    assert w.B == 1024 and w.N == 50 and w.iters == 100
    wr = w.rounded(np.float32) if dtype == "f32" else w
    s = Solver(wr, dtype=dtype)
    s.solve()
    got, info = s.state_numpy(), s.info_numpy()
    assert (info["status"] == 0).all() and all(np.isfinite(got[k]).all() for k in KEYS)
    ref, rinfo, rc = O.admm(wr, O.make_cfg(wr), nthreads=8)      # ALL 1024 problems: the oracle needs about a second for the batch
    assert rc == 0
    compare_states(got, ref, TOL[dtype])
    otol = 1e-4 if dtype == "f32" else 1e-9
    assert (np.abs(info["objective"] - rinfo[:, 2]) <= otol * np.maximum(np.abs(rinfo[:, 2]), 1.0)).all()
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
    idx = np.unique(np.concatenate([np.arange(8), np.random.default_rng(7).choice(np.arange(8, w.B), size=8, replace=False), [w.B - 1]]))   # O-7: first 8 + 8 seeded-random (+ the last)
    assert len(idx) >= 16
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


# ----------------------------------------------------------------------------------------------- status bits (failure reporting)
@pytest.mark.parametrize("family", ["resident_n8", "generic_n5", "dmma_n37"])
def test_status_bits_indefinite_and_nan_problem(family):
    """One indefinite problem (a D block made strongly negative: non-positive pivot) and one NaN problem (NaN in q) inside a batch:
    exactly those two status words carry TMPC_ST_PIVOT / TMPC_ST_NAN — on every factor family (twisted warp-level, generic,
    DMMA) —, the caller's status buffer is overwritten (pre-filled with garbage), and the other problems still match the oracle."""
    import torch
    from paper_2606_24039_b200.solver import Solver
    from paper_2606_24039_b200 import binding as Bd
    if family == "resident_n8":
        w, iters, band = W.config2(B=8, N=10), 40, None
    elif family == "generic_n5":
        w, iters, band = W.random_ltv(91, 8, 9, 3, 2, [3, 4], [0, 0], implicit=True, q_scale=0.3), 40, None
    else:
        w, iters, band = W.random_ltv(92, 4, 4, 30, 7, [30, 33, 36], [0, 0, 1], implicit=True, q_scale=0.3), 30, 1
    bad_piv, bad_nan = 2, w.B - 1
    w.D = np.repeat(w.D, w.B, axis=0).copy() if w.D.shape[0] == 1 else w.D.copy()
    w.D[bad_piv, min(3, w.N)] = -500.0 * np.eye(w.n)
    w.q = w.q.copy(); w.q[bad_nan, 1, 0] = np.nan
    s = Solver(w, dtype="f64")
    s.info["status"].fill_(0x7f00)                      # stale garbage in the caller's buffer
    s.solve(iters)
    got, info = s.state_numpy(), s.info_numpy()
    st = info["status"]
    good = np.array([b for b in range(w.B) if b not in (bad_piv, bad_nan)])
    assert (st[good] == 0).all(), st
    assert st[bad_piv] & Bd_ST_PIVOT and st[bad_nan] & Bd_ST_NAN and not (st[bad_nan] & Bd_ST_PIVOT), st
    ws = w.subset(good)
    ref, rinfo, rc = O.admm(ws, O.make_cfg(ws, band=band), iters=iters, nthreads=4)
    assert rc == 0
    compare_states({k: got[k][good] for k in KEYS}, ref, 1e-9)
    # a second factor + solve with repaired data clears the bits (the word is rewritten by every tmpc_factor / tmpc_admm_solve)
    w2 = w.subset(np.arange(w.B)); w2.D[bad_piv] = w.D[0]; w2.q[bad_nan, 1, 0] = 0.0
    s.upload(w2); s.reset_state(); s.solve(iters)
    assert (s.info_numpy()["status"] == 0).all()
    s.close()


Bd_ST_PIVOT, Bd_ST_NAN = 1, 2


# ----------------------------------------------------------------------------------------------- general A^+ (u_{t+1} columns)
@pytest.mark.parametrize("dtype", ["f64", "f32"])
def test_dense_Ap_every_kernel_family(dtype):
    """A_t^+ with non-zero u_{t+1} columns (implicit integrators, PAPER.md:584-592 Remark A1 / eq. 36): resident fast shapes
    (8/6 and 6/4), ragged generic sizes, the DMMA factor + streamed class shape and cyclic reduction."""
    from paper_2606_24039_b200.solver import Solver
    from paper_2606_24039_b200 import binding as Bd
    run_pair(W.with_dense_Ap(W.config2(B=5, N=13, soft_bound=0.5), seed=1, scale=0.02), dtype, iters=60)
    run_pair(W.with_dense_Ap(W.random_ltv(81, 3, 11, 4, 2, [4, 5, 0], [0, 0, 1], implicit=True, q_scale=0.3), seed=2), dtype, iters=60)
    run_pair(W.with_dense_Ap(W.random_ltv(82, 3, 9, 3, 2, [3, 4], [0, 0, 1], implicit=True, dense_g_rows=1, q_scale=0.3), seed=3), dtype, iters=60)
    run_pair(W.with_dense_Ap(W.config3(B=2, N=4), seed=4, scale=0.02), dtype, iters=30, band=1)
    if dtype == "f64":
        w = W.with_dense_Ap(W.random_ltv(83, 2, 70, 4, 2, [4, 5], [0, 0, 1], implicit=True, dense_g_rows=1, q_scale=0.3), seed=5)
        s = Solver(w, dtype="f64", linsolve=Bd.TMPC_LIN_CYCLIC_REDUCTION)
        s.solve(60)
        ref, rinfo, rc = O.admm(w, O.make_cfg(w), iters=60)
        compare_states(s.state_numpy(), ref, 1e-9)
        s.close()


# ----------------------------------------------------------------------------------------------- TMPC_LIN_AUTO
def test_linsolve_auto_picks_a_path_that_exists():
    """AUTO takes cyclic reduction for a single long horizon of a supported block size (n = 6) and must fall back to the
    sequential families for a block size the cyclic-reduction kernels do not have (n = 3) instead of failing."""
    from paper_2606_24039_b200.solver import Solver
    from paper_2606_24039_b200 import binding as Bd
    for w in (W.random_ltv(84, 1, 1100, 4, 2, [4, 5], [0, 0], implicit=True, q_scale=0.3), W.random_ltv(85, 1, 1030, 2, 1, [2], [0], implicit=True, q_scale=0.3)):
        s = Solver(w, dtype="f64", linsolve=Bd.TMPC_LIN_AUTO)
        s.solve(40)
        ref, rinfo, rc = O.admm(w, O.make_cfg(w, band=1), iters=40)
        compare_states(s.state_numpy(), ref, 1e-9)
        s.close()


# ----------------------------------------------------------------------------------------------- backward: bench shape, dL/dxi, same-K reuse mode
def _gpu_backward(s, ref, dLdx, dLdxi, mode, iters=None):
    import torch
    up = lambda a: None if a is None else s._up(a)
    s.set_state(ref)
    dq, dxi = s.backward(up(dLdx), up(dLdxi), mode=mode, iters=iters)
    return dq.cpu().double().numpy(), dxi.cpu().double().numpy()


@pytest.mark.parametrize("dtype", ["f64", "f32"])
def test_backward_at_bench_shape(dtype):
    """The launch shape bench.py times (B = 1024, N = 50, config 2), fed the oracle's K = 100 state (reading A-20): REFINE mode
    against the definition on 64 sampled problems (the oracle's dense Gauss of a ~750^2 system takes ~0.3 s per problem, so the
    full batch would take minutes), and the eq. 67 mode against the oracle's Alg. 3 on the numpy-built adjoint QP at the SAME K
    on 16 of them."""
    from adjoint_util import adjoint_qp
    from paper_2606_24039_b200.solver import Solver
    from paper_2606_24039_b200 import binding as Bd
    w = W.config2()
    wr = w.rounded(np.float32) if dtype == "f32" else w
    eps = 1e-8 if dtype == "f64" else 1e-4
    cfg = O.make_cfg(wr, eps_abs=eps, eps_rel=eps)
    ref, info, rc = O.admm(wr, cfg, nthreads=8)
    if dtype == "f32":
        ref = {k: v.astype(np.float32).astype(np.float64) for k, v in ref.items()}
    s = Solver(wr, dtype=dtype)
    dq, dxi = _gpu_backward(s, ref, 2.0 * ref["x"], None, Bd.TMPC_BWD_REFACTOR_REFINE)
    assert np.isfinite(dq).all() and np.isfinite(dxi).all()
    idx = np.unique(np.concatenate([np.arange(8), np.random.default_rng(11).choice(np.arange(8, w.B), size=56, replace=False)]))
    ws = wr.subset(idx); rs = {k: v[idx] for k, v in ref.items()}
    dq_o, dxi_o, counts, rcs = O.backward(ws, cfg, rs, 2.0 * rs["x"])
    ok = rcs == 0
    assert ok.sum() >= len(idx) // 2 and counts[ok, 0].sum() > 0
    tol = 1e-9 if dtype == "f64" else 2e-3
    assert rel_err(dq[idx][ok], dq_o[ok]) <= tol and rel_err(dxi[idx][ok], dxi_o[ok]) <= tol
    # eq. 67 mode at the same K
    K = 100
    s.factor()
    dq2, dxi2 = _gpu_backward(s, ref, 2.0 * ref["x"], None, Bd.TMPC_BWD_ADMM_REUSE_FACTOR, iters=K)
    idx2 = idx[:16]
    ws2 = wr.subset(idx2); rs2 = {k: v[idx2] for k, v in ref.items()}
    wa, soft_rows, cls = adjoint_qp(ws2, cfg, rs2, 2.0 * rs2["x"])
    sa, ia, rca = O.admm_rows(wa, O.make_cfg(wa), soft_rows, K)
    assert rca == 0
    assert rel_err(dq2[idx2], -sa["x"]) <= tol and rel_err(dxi2[idx2], sa["yf"][:, :w.nx]) <= tol
    s.close()


@pytest.mark.parametrize("dtype", ["f64", "f32"])
def test_backward_with_dLdxi_and_dead_zone_rows(dtype):
    """L = |x|^2 + 3 |xi|^2 on an instance with soft-active rows AND soft rows in the L1 dead zone (classed hard-active):
    REFINE against the definition, the eq. 67 mode against the oracle's Alg. 3 on the adjoint QP at the same K (1e-9 / 2e-3)."""
    from adjoint_util import adjoint_qp
    from paper_2606_24039_b200.solver import Solver
    from paper_2606_24039_b200 import binding as Bd
    w = W.config2(B=6, N=20, soft_bound=0.4)
    w.rho_bar, w.lam = 2.0, 2.0
    w.q = w.q + 0.3 * np.random.default_rng(5).standard_normal(w.q.shape)
    wr = w.rounded(np.float32) if dtype == "f32" else w
    eps = 1e-8 if dtype == "f64" else 1e-4
    cfg = O.make_cfg(wr, eps_abs=eps, eps_rel=eps)
    ref, info, rc = O.admm(wr, cfg, iters=3000)
    if dtype == "f32":
        ref = {k: v.astype(np.float32).astype(np.float64) for k, v in ref.items()}
    dLdx, dLdxi = 2.0 * ref["x"], 6.0 * ref["xi"]
    dq_o, dxi_o, counts, rcs = O.backward(wr, cfg, ref, dLdx, dLdxi)
    ok = rcs == 0
    assert ok.sum() >= 3 and counts[ok, 1].sum() > 0
    cls = np.stack([O.classify(wr, cfg, ref, b) for b in range(w.B)])
    soft = np.array(w.soft, dtype=bool)
    assert (cls[:, :, soft] == 1).sum() > 0, "instance must hold dead-zone rows"
    dq0, _, _, _ = O.backward(wr, cfg, ref, dLdx, None)
    assert np.abs(dq0 - dq_o)[ok].max() > 1e-2 * np.abs(dq_o[ok]).max(), "the dL/dxi term must matter"
    s = Solver(wr, dtype=dtype, eps_abs=eps, eps_rel=eps)
    tol = 1e-9 if dtype == "f64" else 2e-3
    dq, dxi = _gpu_backward(s, ref, dLdx, dLdxi, Bd.TMPC_BWD_REFACTOR_REFINE)
    assert rel_err(dq[ok], dq_o[ok]) <= tol and rel_err(dxi[ok], dxi_o[ok]) <= tol
    # eq. 66: dL/dgamma_xi from the same adjoint solution
    dg_o = O.backward(wr, cfg, ref, dLdx, dLdxi, with_dgamma=True)[4]
    dg = s.backward_dgamma(s._up(dq)).cpu().double().numpy()
    assert (np.abs(dg - dg_o)[ok] <= tol * np.maximum(1.0, np.abs(dg_o[ok]))).all() and np.abs(dg_o[ok]).max() > 1e-3
    K = 300
    s.factor()
    dq2, dxi2 = _gpu_backward(s, ref, dLdx, dLdxi, Bd.TMPC_BWD_ADMM_REUSE_FACTOR, iters=K)
    wa, soft_rows, _ = adjoint_qp(wr, cfg, ref, dLdx, dLdxi)
    sa, ia, rca = O.admm_rows(wa, O.make_cfg(wa), soft_rows, K)
    assert rel_err(dq2, -sa["x"]) <= tol and rel_err(dxi2, sa["yf"][:, :w.nx]) <= tol
    s.close()


def test_backward_dense_Ap_fp64():
    """REFINE backward on a problem whose A^+ has u_{t+1} columns."""
    from paper_2606_24039_b200.solver import Solver
    from paper_2606_24039_b200 import binding as Bd
    w = W.with_dense_Ap(W.config2(B=4, N=12, soft_bound=0.4), seed=6, scale=0.02)
    w.rho_bar, w.lam = 2.0, 0.05
    w.q = w.q + 0.3 * np.random.default_rng(5).standard_normal(w.q.shape)
    cfg = O.make_cfg(w)
    ref, info, rc = O.admm(w, cfg, iters=3000)
    dq_o, dxi_o, counts, rcs = O.backward(w, cfg, ref, 2.0 * ref["x"])
    ok = rcs == 0
    assert ok.sum() >= 2
    s = Solver(w, dtype="f64")
    dq, dxi = _gpu_backward(s, ref, 2.0 * ref["x"], None, Bd.TMPC_BWD_REFACTOR_REFINE)
    assert rel_err(dq[ok], dq_o[ok]) <= 1e-9 and rel_err(dxi[ok], dxi_o[ok]) <= 1e-9
    s.close()


# ----------------------------------------------------------------------------------------------- f1: adaptive rho + termination
@pytest.mark.parametrize("shape", ["resident_n8", "resident_n6_denseG", "generic_n5"])
def test_adaptive_rho_and_termination_match_oracle_fp64(shape):
    """Alg. 3 with eq. 17 / eq. 4: per-problem iteration counts, termination flags and final rho_bar equal
    the oracle's, the final iterates agree to 1e-9, terminated problems are frozen while the others continue."""
    from paper_2606_24039_b200.solver import Solver
    if shape == "resident_n8":
        w = W.config2(B=9, N=14, soft_bound=0.5)
    elif shape == "resident_n6_denseG":
        w = W.random_ltv(95, 5, 17, 4, 2, [4, 5], [0, 0, 1], bound=0.4, implicit=True, dense_g_rows=1, q_scale=0.4)
    else:
        w = W.random_ltv(96, 4, 11, 3, 2, [3, 4], [0, 0], bound=0.3, implicit=True, q_scale=0.4)
    varied = changed = False
    for eps, kmax in ((1e-4, 600), (1e-7, 1010)):
        ad = O.make_adaptive(kmax, eps, eps)
        ref, rinfo, log, rc = O.admm_adaptive(w, O.make_cfg(w), ad)
        assert rc == 0
        s = Solver(w, dtype="f64")
        out = s.solve_adaptive(kmax, eps, eps)
        got, info = s.state_numpy(), s.info_numpy()
        assert (out["iters"] == rinfo[:, 4].astype(int)).all(), (out["iters"], rinfo[:, 4])
        assert (out["converged"] == rinfo[:, 6].astype(int)).all()
        # rho_new is a ratio of RESIDUALS, i.e. of differences of O(|.|) terms: its relative rounding error is eps |.| / r ~ 1e-16 x 1e2 / 1e-7,
        # and every later iterate inherits it through S(rho); hence 1e-6 on rho_bar and 1e-7 on the iterates here (reading A-33)
        assert (np.abs(out["rho"] - rinfo[:, 5]) <= 1e-6 * np.abs(rinfo[:, 5])).all()
        compare_states(got, ref, 1e-7)
        assert (np.abs(info["r_prim"] - rinfo[:, 0]) <= 1e-9 * np.maximum(1.0, np.abs(ref["x"]).max())).all()
        assert (np.abs(info["r_dual"] - rinfo[:, 1]) <= 1e-7 * np.maximum(1.0, np.abs(ref["yf"]).max())).all()
        assert (info["status"] == 0).all()
        s.close()
        varied |= len(set(out["iters"].tolist())) > 1
        changed |= bool((np.abs(out["rho"] - w.rho_bar) > 1e-12).any())
    assert varied, "problems should stop at different iterations in at least one of the runs"
    assert changed, "at least one accepted step-size update"


def test_adaptive_termination_only_and_fp32():
    """adapt_rho = 0 is the fixed-rho run with the eq. 4 stop; fp32: decisions are taken on fp32 residuals, so counts may differ from the
    fp64 oracle by one check interval near a threshold — where they agree the iterates must agree to the fp32 tolerance."""
    from paper_2606_24039_b200.solver import Solver
    w = W.config2(B=12, N=14, soft_bound=0.5)
    w.rho_bar = 20.0
    ad = O.make_adaptive(800, 1e-5, 1e-5, adapt_rho=0)
    ref, rinfo, log, rc = O.admm_adaptive(w, O.make_cfg(w), ad)
    s = Solver(w, dtype="f64")
    out = s.solve_adaptive(800, 1e-5, 1e-5, adapt_rho=False)
    assert (out["iters"] == rinfo[:, 4].astype(int)).all() and (np.abs(out["rho"] - 20.0) == 0).all()
    compare_states(s.state_numpy(), ref, 1e-9)
    s.close()
    # fp32: rho_new is a ratio of fp32 residuals (relative error ~ 6e-8 |.| / r, i.e. percent level), so the two runs follow different
    # paths and may stop one check apart; what is fixed is the point they converge to: with eps = 2e-4 both stop within the fp32 tolerance
    # of the same solution; every problem must terminate and at least half of the per-problem counts must equal the oracle's
    wr = W.config2(B=12, N=14).rounded(np.float32)                      # BASELINE config-2 data (hard-active control rows, well conditioned)
    ref, rinfo, log, rc = O.admm_adaptive(wr, O.make_cfg(wr), O.make_adaptive(3000, 2e-4, 2e-4))
    assert (rinfo[:, 6] == 1).all()
    s = Solver(wr, dtype="f32")
    out = s.solve_adaptive(3000, 2e-4, 2e-4)
    assert (out["converged"] == 1).all(), out
    assert (out["iters"] == rinfo[:, 4].astype(int)).sum() >= w.B // 2, (out["iters"], rinfo[:, 4])   # a diverged accept/reject decision changes the path
    compare_states(s.state_numpy(), ref, 2e-3)
    s.close()


# ----------------------------------------------------------------------------------------------- f4: the paper's linear-system RL workload
@pytest.mark.parametrize("u_max", [1.0, 10.0])
def test_f4_linear_rl_nominal_shape(u_max):
    """PAPER.md:414-416 generator at the nominal block size (nx, nu) = (8, 4), N = 40: fixed-count iterates (both dtypes), the adaptive
    run to tol 1e-5 with at most 1000 iterations (the paper's setting) and the backward pass against the oracle."""
    from paper_2606_24039_b200.solver import Solver
    from paper_2606_24039_b200 import binding as Bd
    w = W.linear_rl(B=6, N=40, u_max=u_max)
    run_pair(w, "f64", iters=100)
    run_pair(w, "f32", iters=100)
    ref, rinfo, log, rc = O.admm_adaptive(w, O.make_cfg(w), O.make_adaptive(1000, 1e-5, 1e-5))
    s = Solver(w, dtype="f64")
    out = s.solve_adaptive(1000, 1e-5, 1e-5)
    assert (out["iters"] == rinfo[:, 4].astype(int)).all() and (out["converged"] == 1).all()
    compare_states(s.state_numpy(), ref, 1e-7)
    # backward at the converged solution (tight solve first so that the active set is unambiguous)
    cfg = O.make_cfg(w)
    ref, info, rc = O.admm(w, O.make_cfg(w, rho_bar=5.0), iters=4000)
    dq_o, dxi_o, counts, rcs = O.backward(w, cfg, ref, 2.0 * ref["x"])
    ok = rcs == 0
    assert ok.sum() >= 3
    s.set_state(ref)
    dq, dxi = s.backward(s._up(2.0 * ref["x"]), mode=Bd.TMPC_BWD_REFACTOR_REFINE)
    assert rel_err(dq.cpu().double().numpy()[ok], dq_o[ok]) <= 1e-9 and rel_err(dxi.cpu().double().numpy()[ok], dxi_o[ok]) <= 1e-9
    s.close()


def test_f4_linear_rl_sweep_shapes_fp32():
    """The sweep's other block sizes: (nx, nu) = (4, 2), (16, 8) and (32, 16) at short horizons, fixed iteration count."""
    run_pair(W.linear_rl(B=5, N=12, nx=4, nu=2, u_max=1.0), "f32", iters=60)
    run_pair(W.linear_rl(B=3, N=10, nx=16, nu=8, u_max=10.0), "f32", iters=60)
    run_pair(W.linear_rl(B=2, N=8, nx=32, nu=16, u_max=1.0), "f32", iters=60, band=1)


def test_f4_linear_rl_long_horizons_chain_resident():
    """The horizon sweep's long end at the nominal block (N = 160 and 320 at (nx, nu) = (8, 4)): the records no longer fit in
    shared memory, admm3_kernel keeps only the chain's share there and reads X_t, A~_t from global memory (Rec3<.., XG>).  Fixed-count iterates
    in both dtypes, the adaptive run and the backward pass against the oracle; N = 161 is the odd-length, ragged-warp case."""
    from paper_2606_24039_b200.solver import Solver
    from paper_2606_24039_b200 import binding as Bd
    w = W.linear_rl(B=3, N=160, u_max=1.0)
    run_pair(w, "f64", iters=60)
    run_pair(w, "f32", iters=60)
    run_pair(W.linear_rl(B=2, N=161, u_max=10.0), "f64", iters=40)
    run_pair(W.linear_rl(B=2, N=320, u_max=1.0), "f32", iters=40)
    ref, rinfo, log, rc = O.admm_adaptive(w, O.make_cfg(w), O.make_adaptive(300, 1e-4, 1e-4))
    s = Solver(w, dtype="f64")
    out = s.solve_adaptive(300, 1e-4, 1e-4)
    assert (out["iters"] == rinfo[:, 4].astype(int)).all() and (out["converged"] == rinfo[:, 6].astype(int)).all()
    compare_states(s.state_numpy(), ref, 1e-7)
    cfg = O.make_cfg(w)
    ref, info, rc = O.admm(w, O.make_cfg(w, rho_bar=5.0), iters=3000)
    dq_o, dxi_o, counts, rcs = O.backward(w, cfg, ref, 2.0 * ref["x"])
    ok = rcs == 0
    assert ok.sum() >= 2
    s.set_state(ref)
    dq, dxi = s.backward(s._up(2.0 * ref["x"]), mode=Bd.TMPC_BWD_REFACTOR_REFINE)
    assert rel_err(dq.cpu().double().numpy()[ok], dq_o[ok]) <= 1e-9 and rel_err(dxi.cpu().double().numpy()[ok], dxi_o[ok]) <= 1e-9
    s.close()


def test_f4_linear_rl_cluster_pair_fp64():
    """N = 320 in fp64 (the end of the paper's horizon sweep): the chain's share of the records no longer fits one SM, the two half
    chains of the twisted factor run on a cluster of two CTAs that meet through distributed shared memory (admm3_kernel<.., CL>).  One iteration
    (every exchange exactly once), fixed counts at even and odd T, the adaptive run with per-problem termination, and the REFINE backward."""
    from paper_2606_24039_b200.solver import Solver
    from paper_2606_24039_b200 import binding as Bd
    run_pair(W.linear_rl(B=1, N=320, u_max=1.0), "f64", iters=1)
    w = W.linear_rl(B=3, N=320, u_max=1.0)
    run_pair(w, "f64", iters=40)
    run_pair(W.linear_rl(B=2, N=321, u_max=10.0), "f64", iters=40)
    # the pair with FULL records (horizons between one and two SMs' worth: N = 80 in fp64, 160 in fp32), incl. dense A^+ (remote A~^+ rows)
    run_pair(W.linear_rl(B=3, N=80, u_max=1.0), "f64", iters=60)
    run_pair(W.with_dense_Ap(W.linear_rl(B=2, N=81, u_max=10.0)), "f64", iters=40)
    run_pair(W.linear_rl(B=3, N=160, u_max=1.0), "f32", iters=60)
    run_pair(W.linear_rl(B=2, N=340, u_max=1.0), "f32", iters=40)      # fp32 on the pair with the chain's share (322 <= N <= 350)
    # a batch that fills the GPU keeps one CTA per problem (chain-resident, no cluster)
    run_pair(W.linear_rl(B=80, N=160, u_max=1.0), "f64", iters=30)
    ref, rinfo, log, rc = O.admm_adaptive(w, O.make_cfg(w), O.make_adaptive(300, 1e-4, 1e-4))
    s = Solver(w, dtype="f64")
    out = s.solve_adaptive(300, 1e-4, 1e-4)
    assert (out["iters"] == rinfo[:, 4].astype(int)).all() and (out["converged"] == rinfo[:, 6].astype(int)).all()
    assert len(set(out["iters"].tolist())) > 1            # the problems stop at different checks: pairs leave while others go on
    compare_states(s.state_numpy(), ref, 1e-7)
    cfg = O.make_cfg(w)
    ref, info, rc = O.admm(w, O.make_cfg(w, rho_bar=5.0), iters=3000)
    dq_o, dxi_o, counts, rcs = O.backward(w, cfg, ref, 2.0 * ref["x"])
    ok = rcs == 0
    assert ok.sum() >= 2
    s.set_state(ref)
    dq, dxi = s.backward(s._up(2.0 * ref["x"]), mode=Bd.TMPC_BWD_REFACTOR_REFINE)
    assert rel_err(dq.cpu().double().numpy()[ok], dq_o[ok]) <= 1e-9 and rel_err(dxi.cpu().double().numpy()[ok], dxi_o[ok]) <= 1e-9
    s.close()


def test_chain_resident_scratch_follows_the_factor_fp64():
    """The stage-minor scratch of the chain-resident variants is rebuilt only when the factor changes (full, masked, adjoint).  Call sequences on
    one handle at N = 160 (one CTA per problem) and N = 320 (cluster pair): kkt_solve before the first solve, a resumed solve that reuses the scratch,
    a REFINE backward (adjoint factor) followed by a new factor + solve, and two adaptive runs in a row — each against a fresh handle or the oracle."""
    from paper_2606_24039_b200.solver import Solver
    from paper_2606_24039_b200 import binding as Bd
    for N in (160, 320):
        w = W.linear_rl(B=3, N=N, u_max=1.0)
        cfg = O.make_cfg(w)
        ref70, _, _ = O.admm(w, cfg, iters=70)
        s = Solver(w, dtype="f64")
        s.factor()
        eta = np.random.default_rng(2).standard_normal((w.B, w.T, w.n))
        xt = s.kkt_solve(s._up(eta)).cpu().double().numpy()                 # X rows only: the next solve must still build the whole scratch
        ref = np.stack([O.solve_S(w, cfg, eta[b].ravel(), b).reshape(w.T, w.n) for b in range(w.B)])
        assert rel_err(xt, ref) <= 1e-9
        s.reset_state(); s.admm_solve(30); s.admm_solve(40, flags=Bd.TMPC_SOLVE_ZG_GIVEN)      # second call: scratch reused
        compare_states(s.state_numpy(), ref70, 1e-9)
        st = s.state_numpy()
        dq, dxi = s.backward(2.0 * s.s["x"], mode=Bd.TMPC_BWD_REFACTOR_REFINE)                 # adjoint factor takes the workspace and the scratch
        s.reset_state(); s.solve(70)                                                          # factor + solve again
        compare_states(s.state_numpy(), ref70, 1e-9)
        refa, rinfo, log, rc = O.admm_adaptive(w, cfg, O.make_adaptive(200, 1e-4, 1e-4))
        for _ in range(2):                                                                    # masked refactorisations, twice on the same handle
            s.factor(); s.reset_state()
            out = s.solve_adaptive(200, 1e-4, 1e-4)
            assert (out["iters"] == rinfo[:, 4].astype(int)).all()
            compare_states(s.state_numpy(), refa, 1e-7)
        s.close()


def test_long_horizons_chain_resident_small_blocks():
    """The same variant for the (8, 6) and (6, 4) blocks once their records outgrow shared memory (fp64: N > ~190 resp. ~330): selection G with
    soft rows (config 2's data at N = 260), dense G (config 4's bicycle QP at N = 400, G~ rows in global memory too), and the thread-cap
    variants (384 / 704 / 1024 threads per CTA)."""
    run_pair(W.config2(B=3, N=260, soft_bound=0.5), "f64", iters=60)
    run_pair(W.config2(B=2, N=420).rounded(np.float32), "f32", iters=50)
    run_pair(W.random_ltv(31, 3, 400, 4, 2, [4], [0, 1, 0], dense_g_rows=2, q_scale=0.3), "f64", iters=50)
    run_pair(W.random_ltv(32, 2, 480, 4, 2, [5], [0, 0, 1], dense_g_rows=2, q_scale=0.3), "f32", iters=50)
    from paper_2606_24039_b200.solver import Solver
    w = W.config4(B=2, N=400, dtype="f64")               # SQP on the bicycle model: linearise + factor + solve, all on the long-horizon variant
    s = Solver(w, dtype="f64")
    s.reset_state(w.xbar0)
    s.sqp()
    ref, info, rc = O.sqp_bicycle(w, O.make_cfg(w), nthreads=8)
    assert rc == 0
    compare_states(s.state_numpy(), ref, TOL["f64"])
    s.close()


# ----------------------------------------------------------------------------------------------- f2: SQP with linesearch + eq. 18
def test_sqp_linesearch_matches_oracle_fp64():
    """Alg. 1 with the App. D linesearch and the eq. 18 stop on perturbed bicycle starts: accepted
    step sizes of every iteration, per-problem iteration counts, convergence flags and the final iterates equal the oracle's."""
    from paper_2606_24039_b200.solver import Solver
    w = W.config4(B=7, N=24, dtype="f64")
    x0 = w.xbar0.copy(); x0[:, :, :2] += np.random.default_rng(0).normal(0, 1.5, x0[:, :, :2].shape); x0[:, :, 2] += 0.3
    x0[5:] = w.xbar0[5:]                                   # two problems start from the reference (first steps: smallest candidate, fallback)
    kw = dict(max_sqp=8, admm_iters=120, eps_c=1e-3, n_alpha=8, eta=0.4)
    ref, rinfo, log, rc = O.sqp_linesearch_bicycle(w, O.make_cfg(w), xbar0=x0, **kw)
    assert rc == 0
    s = Solver(w, dtype="f64")
    s.reset_state(x0)
    out = s.sqp_linesearch(**kw)
    got = s.state_numpy()
    assert (out["iters"] == rinfo[:, 0].astype(int)).all(), (out["iters"], rinfo[:, 0])
    assert (out["converged"] == rinfo[:, 1].astype(int)).all()
    for b in range(w.B):
        k = int(rinfo[b, 0])
        assert (out["alpha"][b, :k] == log[b, :k, 0]).all(), (b, out["alpha"][b, :k], log[b, :k, 0])
    assert (out["alpha"] < 1.0).any() and (out["alpha"] == 1.0).any(), "instance must exercise backtracking and full steps"
    compare_states({k: got[k] for k in ("x", "yf", "yg", "xi")} | {"zg": ref["zg"]}, ref, 1e-9)
    assert np.abs(out["kkt"] - rinfo[:, 2:5]).max() <= 1e-7
    s.close()


def test_sqp_linesearch_srb_matches_oracle_fp64():
    """f2 on the second built-in model (SRB humanoid, RK4: the merit function's equality residual is Phi(x_k, u_k) - x_{k+1}, selection rows with
    two soft rows): accepted step sizes, iteration counts, convergence flags, eq. 18 quantities and final iterates equal the oracle's."""
    from paper_2606_24039_b200.solver import Solver
    w = W.srb_humanoid(B=4, N=10)
    w.soft = [0, 1, 0, 0, 1, 0]; w.lam, w.gamma = 0.01, 0.1
    rng = np.random.default_rng(3)
    x0 = w.xbar0.copy()
    x0[:, :, :3] += 0.03 * rng.standard_normal(x0[:, :, :3].shape); x0[:, :, 3:6] += 0.1 * rng.standard_normal(x0[:, :, 3:6].shape)
    x0[:, :, 6:12] += 0.2 * rng.standard_normal(x0[:, :, 6:12].shape)
    x0[3] = w.xbar0[3]                                     # one problem starts from the reference
    kw = dict(max_sqp=20, admm_iters=2000, eps_c=1e-3, n_alpha=8, eta=0.4)
    ref, rinfo, log, rc = O.sqp_linesearch_srb(w, O.make_cfg(w), xbar0=x0, **kw)
    assert rc == 0
    s = Solver(w, dtype="f64")
    s.reset_state(x0)
    out = s.sqp_linesearch(**kw)
    got = s.state_numpy()
    assert (out["iters"] == rinfo[:, 0].astype(int)).all(), (out["iters"], rinfo[:, 0])
    assert (out["converged"] == rinfo[:, 1].astype(int)).all() and out["converged"].any()
    for b in range(w.B):
        k = int(rinfo[b, 0])
        assert (out["alpha"][b, :k] == log[b, :k, 0]).all(), (b, out["alpha"][b, :k], log[b, :k, 0])
    assert (out["alpha"] < 1.0).any() and (out["alpha"] == 1.0).any() and (ref["xi"] != 0).any()
    compare_states({k: got[k] for k in ("x", "yf", "yg", "xi")} | {"zg": ref["zg"]}, ref, 1e-8)
    assert np.abs(out["kkt"] - rinfo[:, 2:5]).max() <= 1e-6
    s.close()


def test_adaptive_on_the_streamed_class_fp64():
    """f1 on the streamed class (blocks that do not fit in shared memory: admm_stream_kernel + factor3_kernel with per-problem rho_bar,
    refactor mask and frozen terminated problems), on the f4 generator at (nx, nu) = (32, 16)."""
    from paper_2606_24039_b200.solver import Solver
    w = W.linear_rl(B=3, N=24, nx=32, nu=16, u_max=1.0)
    ref, rinfo, log, rc = O.admm_adaptive(w, O.make_cfg(w, band=1), O.make_adaptive(400, 1e-4, 1e-4))
    assert rc == 0
    s = Solver(w, dtype="f64")
    out = s.solve_adaptive(400, 1e-4, 1e-4)
    assert (out["iters"] == rinfo[:, 4].astype(int)).all(), (out["iters"], rinfo[:, 4])
    assert (out["converged"] == rinfo[:, 6].astype(int)).all()
    assert (np.abs(out["rho"] - rinfo[:, 5]) <= 1e-6 * np.abs(rinfo[:, 5])).all()
    compare_states(s.state_numpy(), ref, 1e-7)
    s.close()


# ----------------------------------------------------------------------------------------------- f3: SRB humanoid model (second built-in model)
@pytest.mark.parametrize("dtype", ["f64", "f32"])
def test_srb_linearize_matches_oracle(dtype):
    """tmpc_linearize for TMPC_MODEL_SRB_HUMANOID_RK4 (eq. 68-69 + RK4): A^- = [dPhi/dx dPhi/du], A^+ = [-I 0], b (eq. 36-37)
    element-wise against the oracle at a perturbed iterate (large angles, forces and spins so that every term of eq. 68 is active)."""
    from paper_2606_24039_b200.solver import Solver
    w = W.srb_humanoid(B=4, N=9, dtype=dtype)
    rng = np.random.default_rng(2)
    w.xbar0 = w.xbar0 + np.concatenate([0.05 * rng.standard_normal((w.B, w.T, 3)), 0.3 * rng.standard_normal((w.B, w.T, 3)),
                                        0.5 * rng.standard_normal((w.B, w.T, 6)), 30.0 * rng.standard_normal((w.B, w.T, 6))], axis=2)
    wr = w.rounded(np.float32) if dtype == "f32" else w
    s = Solver(wr, dtype=dtype)
    s.reset_state(wr.xbar0)
    s.linearize()
    cfg = O.make_cfg(wr)
    tol = 1e-12 if dtype == "f64" else 3e-5
    for b in range(w.B):
        ref = O.srb_linearize(wr, cfg, wr.xbar0[b])
        for name, r in zip(("Am", "Ap", "b"), ref):
            g = s.t[name][b].cpu().double().numpy()
            assert np.abs(g - r).max() <= tol * max(1.0, np.abs(r).max()), (name, np.abs(g - r).max())
    s.close()


@pytest.mark.parametrize("dtype", ["f64", "f32"])
def test_srb_sqp_matches_oracle(dtype):
    """The humanoid balancing OCP (eq. 70; N = 20, nx = 12, nu = 6, box bounds on the foot forces): n_sqp x (tmpc_linearize + tmpc_factor +
    tmpc_admm_solve) against the oracle's driver."""
    from paper_2606_24039_b200.solver import Solver
    w = W.srb_humanoid(B=5, dtype=dtype)
    wr = w.rounded(np.float32) if dtype == "f32" else w
    s = Solver(wr, dtype=dtype)
    s.reset_state(wr.xbar0)
    s.sqp()
    got = s.state_numpy()
    ref, info, rc = O.sqp_srb(wr, O.make_cfg(wr))
    assert rc == 0
    compare_states(got, ref, TOL[dtype])
    assert (np.abs(ref["yg"]) > 1e-3).any(), "force bounds should be active on the perturbed starts"
    s.close()
