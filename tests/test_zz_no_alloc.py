"""-m gpu: tmpc_admm_solve_static — the allocation-free entry point (include/tmpc.h) — against the existing tmpc_factor + tmpc_admm_solve
path, on two calls in a row that share the library's static device scratch.  Collected last on purpose (the suite runs with pytest -x)."""
import ctypes as C

import numpy as np
import pytest

from paper_2606_24039_b200 import workloads as W

pytestmark = pytest.mark.gpu

KEYS = ("x", "zg", "yf", "yg", "xi")
TOL = {"f64": 1e-9, "f32": 2e-3}          # the tolerances of tests/test_gpu_parity.py


def _rel_err(got, ref):
    B = ref.shape[0]
    g, r = got.reshape(B, -1), ref.reshape(B, -1)
    return (np.abs(g - r).max(axis=1) / np.maximum(np.abs(r).max(axis=1), 1.0)).max()


def _existing_path(w, dtype, iters):
    from paper_2606_24039_b200.solver import Solver
    s = Solver(w, dtype=dtype)
    s.solve(iters)
    st, info = s.state_numpy(), s.info_numpy()
    s.close()
    return st, info


def _static_path(w, dtype, iters):
    """Inputs and outputs are caller tensors; no handle, no workspace: the scratch is the library's static device array."""
    import torch
    from paper_2606_24039_b200 import binding as Bd
    td = torch.float64 if dtype == "f64" else torch.float32
    dev = torch.device("cuda:0")
    up = lambda a: torch.from_numpy(np.ascontiguousarray(a)).to(td).to(dev)
    t = {k: up(getattr(w, k)) for k in ("D", "E", "q", "Am", "Ap", "b", "x_init", "lo", "hi")}
    t["G"] = up(w.G) if w.G is not None else None
    q = Bd.TmpcQp()
    q.D, q.D_bstride = t["D"].data_ptr(), (0 if t["D"].shape[0] == 1 else t["D"][0].numel())
    q.E, q.E_bstride = t["E"].data_ptr(), (0 if t["E"].shape[0] == 1 else t["E"][0].numel())
    q.q, q.Am, q.Ap, q.b, q.x_init = t["q"].data_ptr(), t["Am"].data_ptr(), t["Ap"].data_ptr(), t["b"].data_ptr(), t["x_init"].data_ptr()
    q.G, q.G_bstride = (t["G"].data_ptr(), (0 if t["G"].shape[0] == 1 else t["G"][0].numel())) if t["G"] is not None else (None, 0)
    q.lo, q.hi = t["lo"].data_ptr(), t["hi"].data_ptr()
    z = lambda *s: torch.zeros(*s, dtype=td, device=dev)
    mf = w.nx + w.N * w.nx
    s = dict(x=z(w.B, w.T, w.n), zg=z(w.B, w.T, w.ng), yf=z(w.B, mf), yg=z(w.B, w.T, w.ng), xi=z(w.B, w.T, w.ng))
    info = dict(r_prim=z(w.B), r_dual=z(w.B), objective=z(w.B), status=torch.full((w.B,), 0x7f00, dtype=torch.int32, device=dev))
    st = Bd.TmpcState(*[s[k].data_ptr() for k in KEYS])
    inf = Bd.TmpcInfo(info["r_prim"].data_ptr(), info["r_dual"].data_ptr(), info["objective"].data_ptr(), info["status"].data_ptr())
    cfg = Bd.make_config(w, dtype=dtype)
    before = torch.cuda.memory_allocated(dev)
    Bd.tmpc_admm_solve_static(cfg, q, st, iters, 0, inf, torch.cuda.current_stream(dev).cuda_stream)
    torch.cuda.synchronize(dev)
    assert torch.cuda.memory_allocated(dev) == before
    return {k: v.cpu().double().numpy() for k, v in s.items()}, {k: v.cpu().numpy() for k, v in info.items()}


def test_static_entry_matches_existing_path_on_two_calls_in_a_row():
    """Two calls back to back on the shared static scratch — a resident-class fp64 batch, then a generic-class fp32 batch of another shape, so the
    second call finds the first one's factor in the array — each equal to the existing path within the parity tolerances, info included."""
    cases = [(W.config2(B=8, N=20, soft_bound=0.5), "f64", 50),
             (W.random_ltv(21, 5, 13, 3, 2, [3, 4], [0, 0], implicit=True, q_scale=0.3).rounded(np.float32), "f32", 60)]
    refs = [_existing_path(w, dt, it) for w, dt, it in cases]
    for (w, dt, it), (ref, rinfo) in zip(cases, refs):          # the two static calls run in a row, nothing else touches the GPU in between
        got, info = _static_path(w, dt, it)
        for k in KEYS:
            assert _rel_err(got[k], ref[k]) <= TOL[dt], (w.name, k)
        assert (info["status"] == 0).all() and (rinfo["status"] == 0).all()
        otol = 1e-9 if dt == "f64" else 1e-4
        assert (np.abs(info["objective"] - rinfo["objective"]) <= otol * np.maximum(np.abs(rinfo["objective"]), 1.0)).all()
        assert (np.abs(info["r_prim"] - rinfo["r_prim"]) <= TOL[dt] * np.maximum(1.0, np.abs(ref["x"]).max())).all()


def test_static_entry_rejects_problems_beyond_its_scratch():
    """A problem whose workspace exceeds TMPC_STATIC_SCRATCH_BYTES is rejected with TMPC_E_STATIC_LIMIT and a message that names the limit."""
    from paper_2606_24039_b200 import binding as Bd
    w = W.config2(B=4, N=5)
    cfg = Bd.make_config(w, dtype="f64")
    cfg.batch = 4096                                            # 4096 x 6 stages x 2 x 64 doubles of factor alone > 8 MiB
    assert Bd.tmpc_workspace_bytes(cfg) > Bd.TMPC_STATIC_SCRATCH_BYTES
    dummy = C.c_void_p(256)                                     # never dereferenced: the size check comes first and nothing is enqueued
    st = Bd.TmpcState(*[dummy.value] * 5)
    q = Bd.TmpcQp()
    rc = Bd.lib().tmpc_admm_solve_static(C.byref(cfg), C.byref(q), C.byref(st), 10, 0, None, None)
    assert rc == Bd.TMPC_E_STATIC_LIMIT
    assert b"TMPC_STATIC_SCRATCH_BYTES" in Bd.lib().tmpc_status_string(rc)
