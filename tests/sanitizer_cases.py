"""Small cases of every kernel family for `compute-sanitizer` (one tool per run, see profiles/r02_sanitizers.md):

    compute-sanitizer --tool racecheck|synccheck|memcheck --kernel-regex kns=tmpc python tests/sanitizer_cases.py

Each case is also checked against the oracle so that a sanitizer run is known to have executed the real path."""
import os
import sys

import numpy as np

sys.path.insert(0, os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
import oracle as O  # noqa: E402
from paper_2606_24039_b200 import binding as Bd  # noqa: E402
from paper_2606_24039_b200 import workloads as W  # noqa: E402
from paper_2606_24039_b200.solver import Solver  # noqa: E402


def check(got, ref, tol, what):
    for k in ("x", "zg", "yf", "yg", "xi"):
        e = np.abs(got[k].reshape(ref[k].shape) - ref[k]).max() / max(1.0, np.abs(ref[k]).max())
        assert e <= tol, (what, k, e)
    print("ok", what)


def main():
    # resident class (admm3 + factor_tw2), n = 8, two problems per CTA, fp32; backward in both modes; adaptive schedule
    w = W.config2(B=4, N=10, soft_bound=0.5).rounded(np.float32)
    s = Solver(w, dtype="f32"); s.solve(30)
    ref, _, _ = O.admm(w, O.make_cfg(w), iters=30)
    check(s.state_numpy(), ref, 2e-3, "config2 B=4 N=10 f32")
    s.backward(2.0 * s.s["x"]); s.factor(); s.backward(2.0 * s.s["x"], mode=Bd.TMPC_BWD_ADMM_REUSE_FACTOR, iters=20)
    s.reset_state(); s.solve_adaptive(100, 1e-3, 1e-3); s.close()
    # resident class, n = 6 with a dense G row, fp64, SQP on the bicycle model (linearize kernel)
    w = W.config4(B=3, N=12, dtype="f64")
    s = Solver(w, dtype="f64"); s.reset_state(w.xbar0); s.sqp(2, 20)
    ref, _, _ = O.sqp_bicycle(w, O.make_cfg(w), n_sqp=2, iters=20)
    check(s.state_numpy(), ref, 1e-9, "config4 B=3 N=12 f64"); s.close()
    # streamed class (admm_stream_kernel: mbarrier ring, producer warp) + DMMA factor
    w = W.config3(B=2, N=3).rounded(np.float32)
    s = Solver(w, dtype="f32"); s.solve(20)
    ref, _, _ = O.admm(w, O.make_cfg(w, band=1), iters=20)
    check(s.state_numpy(), ref, 2e-3, "config3 B=2 N=3 f32"); s.close()
    # generic class (n = 5)
    w = W.random_ltv(21, 3, 9, 3, 2, [3, 4], [0, 0], implicit=True, q_scale=0.3)
    s = Solver(w, dtype="f64"); s.solve(20)
    ref, _, _ = O.admm(w, O.make_cfg(w), iters=20)
    check(s.state_numpy(), ref, 1e-9, "generic n=5 f64"); s.close()
    # long-horizon forms of the resident kernel, (12, 8) block, fp64: one CTA with the chain's share (N = 160, stage-minor global operands),
    # the cluster pair with full records (N = 80) and with the chain's share (N = 320: distributed shared memory, remote mbarriers), each with
    # the adaptive schedule on top (early exit of terminated CTAs / pairs, masked multi-warp factor)
    for N in (160, 80, 320):
        w = W.linear_rl(B=2, N=N, u_max=1.0)
        s = Solver(w, dtype="f64"); s.solve(20)
        ref, _, _ = O.admm(w, O.make_cfg(w), iters=20)
        check(s.state_numpy(), ref, 1e-9, f"linear_rl B=2 N={N} f64")
        s.reset_state(); s.solve_adaptive(100, 1e-3, 1e-3); s.close()
    # cyclic reduction (grid barrier), chunked form needs T >= 256
    w = W.config5(N=300)
    s = Solver(w, dtype="f64", linsolve=Bd.TMPC_LIN_CYCLIC_REDUCTION); s.reset_state(w.xbar0); s.sqp(1, 20)
    ref, _, _ = O.sqp_bicycle(w, O.make_cfg(w, band=1), n_sqp=1, iters=20)
    check(s.state_numpy(), ref, 1e-9, "config5 N=300 f64 cyclic reduction"); s.close()


if __name__ == "__main__":
    main()
