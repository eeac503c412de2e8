"""-m "not gpu": the C-ABI library loads and exports every symbol include/tmpc.h declares; host-side logic
(argument checking, workspace sizing, no-CPU-fallback behaviour, input generators, sharding with gloo)."""
import ctypes as C
import os
import re
import socket

import numpy as np
import pytest
import torch

from paper_2606_24039_b200 import binding as Bd
from paper_2606_24039_b200 import sharding
from paper_2606_24039_b200 import workloads as W

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    import __graft_entry__ as g
    g.build()
    return Bd.lib()


def test_every_declared_symbol_is_exported(lib):
    hdr = open(os.path.join(ROOT, "include", "tmpc.h")).read()
    declared = sorted(set(re.findall(r"\b(tmpc_[a-z_]+)\s*\(", hdr)))
    assert set(declared) == set(Bd.EXPORTS)
    for name in declared:
        assert hasattr(lib, name), name


def test_config_struct_layout_matches_header(lib):
    w = W.config2(B=4, N=5)
    cfg = Bd.make_config(w)
    n = Bd.tmpc_workspace_bytes(cfg)          # pure host arithmetic: works without a GPU
    assert n > 0 and n % 256 == 0
    cfg64 = Bd.make_config(w, dtype="f64")
    assert Bd.tmpc_workspace_bytes(cfg64) > n
    assert Bd.tmpc_host_staging_bytes(cfg) > 0


def test_bad_arguments_are_rejected_without_side_effects(lib):
    w = W.config2(B=4, N=5)
    for field, val in (("batch", 0), ("N", 0), ("nx", 0), ("ng", 33), ("alpha", 2.5), ("sigma", 0.0), ("rho_bar", -1.0), ("dtype", 7)):
        cfg = Bd.make_config(w)
        setattr(cfg, field, val)
        nbytes = C.c_size_t()
        assert lib.tmpc_workspace_bytes(C.byref(cfg), C.byref(nbytes)) != 0, field
    cfg = Bd.make_config(w)
    h = C.c_void_p()
    assert lib.tmpc_setup(C.byref(cfg), None, 0, None, C.byref(h)) == 5          # TMPC_E_WORKSPACE
    assert lib.tmpc_factor(None, None) == 1 and lib.tmpc_admm_solve(None, None, None, 1, 0, None) == 1
    assert b"fallback" in lib.tmpc_status_string(6)


@pytest.mark.skipif(torch.cuda.is_available(), reason="checks the no-GPU behaviour")
def test_no_cpu_fallback(lib):
    from paper_2606_24039_b200.solver import Solver
    w = W.config2(B=2, N=5)
    with pytest.raises(RuntimeError):
        Solver(w)
    cfg = Bd.make_config(w)
    buf = (C.c_char * (Bd.tmpc_workspace_bytes(cfg) + 512))()
    p = (C.addressof(buf) + 255) // 256 * 256
    h = C.c_void_p()
    assert lib.tmpc_setup(C.byref(cfg), p, Bd.tmpc_workspace_bytes(cfg), None, C.byref(h)) == 6   # TMPC_E_CUDA


def test_splitmix64_reference_vector_and_determinism():
    st = W.Streams(0, 0, np.array([0]))
    assert int(st._raw(1)[0, 0]) == 0xE220A8397B1DCDAF        # published SplitMix64 output for state 0
    a, b = W.config2(B=3, N=4), W.config2(B=3, N=4)
    assert all(np.array_equal(getattr(a, k), getattr(b, k)) for k in ("Am", "b", "x_init"))
    c = W.config2(B=2, N=4, first_problem=1)
    assert np.array_equal(c.Am[0], a.Am[1]) and np.array_equal(c.x_init[1], a.x_init[2])
    nrm = W.Streams(3, 7, np.arange(4)).normal(50000)
    assert abs(nrm.mean()) < 0.02 and abs(nrm.std() - 1) < 0.02
    w4 = W.config4(B=3, N=40)
    d = np.diff(w4.stage_ref[:, :, :2], axis=1)
    assert np.abs(np.sqrt((d ** 2).sum(-1)) - 15.0 * 0.05).max() < 1e-3      # reference advances v_ref*dt of arc length per stage


def _gloo_worker(rank, world, port, out):
    import torch.distributed as dist
    dist.init_process_group("gloo", init_method=f"tcp://127.0.0.1:{port}", rank=rank, world_size=world)
    lo, hi = sharding.rank_problem_range(8, world, rank)
    w = W.config2(B=hi - lo, N=3, first_problem=lo)
    mx = sharding.max_over_ranks(10.0 + rank)
    tot = sharding.sum_over_ranks(float(hi - lo))
    first, cnt = sharding.split_batch(11, world, rank)
    out.put((rank, lo, hi, float(w.x_init[0, 0]), mx, tot, first, cnt))
    dist.destroy_process_group()


def test_sharding_two_ranks_gloo():
    import torch.multiprocessing as mp
    s = socket.socket(); s.bind(("127.0.0.1", 0)); port = s.getsockname()[1]; s.close()
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    ps = [ctx.Process(target=_gloo_worker, args=(r, 2, port, q)) for r in range(2)]
    [p.start() for p in ps]
    res = sorted(q.get(timeout=120) for _ in ps)
    [p.join(timeout=60) for p in ps]
    full = W.config2(B=16, N=3)
    assert [(r[1], r[2]) for r in res] == [(0, 8), (8, 16)]
    assert res[0][3] == full.x_init[0, 0] and res[1][3] == full.x_init[8, 0]     # disjoint, covering problem ranges
    assert all(r[4] == 11.0 and r[5] == 16.0 for r in res)                       # MAX of timings, SUM of units
    assert [(r[6], r[7]) for r in res] == [(0, 6), (6, 5)]


def test_shared_memory_plans_of_the_resident_kernel(tmp_path):
    """Host logic of tmpc_admm3.cuh: the record-stride / placement plans (plain, chain-resident, cluster pair) terminate, keep the alignments the
    kernel's vector accesses assume and cover the records they place, for every horizon 2..700 of the three fast-path blocks in both dtypes; and the
    two capacity claims of DESIGN.md 5.1 ((64,160,8,4) fp64 on one SM, (64,320,8,4) fp64 on a pair).  tests/plan_check.cu, host code only."""
    import shutil
    import subprocess
    nvcc = shutil.which("nvcc") or "/usr/local/cuda/bin/nvcc"
    here = os.path.dirname(os.path.abspath(__file__))
    exe = str(tmp_path / "plan_check")
    subprocess.run([nvcc, "-std=c++17", "-O1", "-gencode", "arch=compute_100a,code=sm_100a", "-I", os.path.join(here, "..", "include"),
                    "-o", exe, os.path.join(here, "plan_check.cu")], check=True, capture_output=True, timeout=300)
    r = subprocess.run([exe], capture_output=True, text=True, timeout=120)
    assert r.returncode == 0 and "plan_check: ok" in r.stdout, r.stdout[-2000:]
