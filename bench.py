#!/usr/bin/env python
"""bench.py — throughput of the batched ADMM-QP hot path on B200 (BASELINE.json metric: "batched QP solves/s & ADMM iters/s,
ms/solve; % of HBM/FP roofline" for the five configs).

  python bench.py --gpus N --steps K --warmup W [--config 1..5] [--dtype f32|f64] [--impl reference]

A step = one pass of the hot path over one batch of synthetic QPs: configs 1-3: tmpc_factor + tmpc_admm_solve
(fixed iteration count); configs 4-5: n_sqp x (tmpc_linearize + tmpc_factor + tmpc_admm_solve).
Without --config the run covers ALL FIVE configs and prints ONE JSON line: the headline (value, config.workload, roofline,
e2e, cpu_baseline) is config 4 (bicycle SQP, B = 4096, fp32: the largest batch, and the one that exercises linearise +
factor + solve), and `per_config` carries the same fields for configs 1, 2 (fp32 and fp64, with `backward_ms`), 3 and 5.
With --config C only that config is run (it is then the headline).
value = QP solves per second over all ranks (each rank solves its own batch: weak scaling, no collective on the
data path; NCCL only carries the barrier and the max-over-ranks reduction of the timings).
The ALU and shared-memory roofline denominators are MEASURED in the same run with tmpc_measure_peak (FMA-chain and
LDS.128 micro-benchmarks, include/tmpc.h); the HBM one comes from MEASURED_PEAKS.json.
`--impl reference` times the CPU oracle (oracle/) on the host cores on a bounded sample of the same workloads.
"""
import argparse
import json
import os
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

# algorithmic flops per problem per ADMM iteration (a4-a8, selection-type G, compact C) — SURVEY.md 8(a)/(d), DESIGN.md 6
FLOPS_PER_ITER = {1: 7.6e3, 2: 36.1e3, 3: 2.75e6, 4: 37.7e3, 5: 3.1e6}
# algorithmic HBM bytes per problem per ADMM iteration for the streamed class (config 3) — SURVEY.md 8(d)
BYTES_PER_ITER = {3: 4.33e6}
# nominal ALU peaks, used only if the micro-benchmark entry is unavailable: 148 SMs x 128 FP32 (64 FP64) FMA lanes x 2 x 1965 MHz
NOMINAL_TFLOPS = {"f32": 148 * 128 * 2 * 1.965e9 / 1e12, "f64": 148 * 64 * 2 * 1.965e9 / 1e12}
DEFAULT_DTYPE = {1: "f64", 2: "f32", 3: "f32", 4: "f32", 5: "f64"}
# dram__bytes_read.sum + dram__bytes_write.sum of the dominant kernel per tmpc_admm_solve call, from committed `ncu --set full`
# captures: (bytes, profiles/ file).  Only quoted for the exact workload the capture was taken on; None otherwise.
NCU_TRAFFIC = {
    (2, "f32", 1024): (57.05e6 + 0.38e6, "profiles/r02_ncu_full_admm3_kernel_config2_f32.md"),
    (4, "f32", 4096): (275.5e6 + 25.7e6, "profiles/r02_ncu_full_admm3_kernel_config4_f32.md (one tmpc_admm_solve = one SQP step)"),
    (5, "f64", 1): (13.38e6 + 0.003e6, "profiles/r02_ncu_full_cr2_admm_kernel_config5_f64.md"),
    # config 3: one tmpc_admm_solve = 7 chunk launches; the capture is ONE full-wave launch (296 CTAs x 50 iterations), scaled to the 2048 chunk jobs of a call
    (3, "f32", 512): ((65.42e9 + 0.572e9) * 2048 / 296, "profiles/r01_v3_ncu_full_admm_stream_kernel_config3_f32.md (kernel unchanged in round 2)"),
}
KERNEL_NAMES = {1: "admm3_kernel", 2: "admm3_kernel", 3: "admm_stream_kernel x chunk launches", 4: "admm3_kernel", 5: "cr2_admm_kernel"}
STEPS_CAP = {3: 5, 5: 10}     # per_config legs of the all-configs run: the 95 ms / 6 ms steps need fewer repetitions for a stable mean


def make_workload(cfg_id, dtype, batch=None, rank=0):
    from paper_2606_24039_b200 import workloads as W
    from paper_2606_24039_b200.sharding import rank_problem_range
    kw = {"B": batch} if batch else {}
    B = batch or {1: 1, 2: 1024, 3: 512, 4: 4096, 5: 1}[cfg_id]
    first = rank_problem_range(B, max(1, rank + 1), rank)[0]      # rank r owns problems [r*B, (r+1)*B) of the generator
    if cfg_id == 1:
        w = W.config1(seed=rank)
    elif cfg_id == 2:
        w = W.config2(dtype=dtype, first_problem=first, **kw)
    elif cfg_id == 3:
        w = W.config3(first_problem=first, **kw)
    elif cfg_id == 4:
        w = W.config4(dtype=dtype, first_problem=first, **kw)
    elif cfg_id == 5:
        w = W.config5(dtype=dtype)
    else:
        raise SystemExit("config must be 1..5")
    return w.rounded(np.float32) if dtype == "f32" else w


def workload_name(w, dtype):
    s = f"{w.name}: B={w.B} N={w.N} nx={w.nx} nu={w.nu} ng={w.ng} {dtype} iters={w.iters}"
    return s + (f" sqp={w.sqp_iters}" if w.sqp_iters else "")


def total_iters(w):
    return w.iters * max(1, w.sqp_iters)


class ClockSampler(threading.Thread):
    """Samples nvidia-smi clocks / throttle reasons during the timed region (B200_PROFILING.md clocks line)."""

    def __init__(self, index):
        super().__init__(daemon=True)
        self.index, self.rows, self.stop_flag = index, [], False

    def run(self):
        q = "clocks.sm,clocks.max.sm,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap"
        while not self.stop_flag:
            try:
                out = subprocess.run(["nvidia-smi", f"--query-gpu={q}", "--format=csv,noheader,nounits", "-i", str(self.index)],
                                     capture_output=True, text=True, timeout=5).stdout.strip()
                if out:
                    self.rows.append([c.strip() for c in out.split(",")])
            except Exception:
                pass
            time.sleep(0.1)

    def summary(self):
        self.stop_flag = True
        self.join(timeout=6)
        if not self.rows:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": []}
        sm = sorted(float(r[0]) for r in self.rows if r[0].replace(".", "").isdigit())
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        reasons = [n for i, n in enumerate(names) if any(r[2 + i].lower().startswith("active") for r in self.rows if len(r) > 2 + i)]
        return {"sm_mhz": sm[len(sm) // 2] if sm else None, "sm_max_mhz": float(self.rows[0][1]) if self.rows[0][1].replace(".", "").isdigit() else None,
                "reasons": reasons, "samples": len(self.rows)}


def oracle_rate(w, cfg_id, nthreads, budget_problems):
    """Times the oracle as it stands on a bounded sample; returns (solves/s, sample description, seconds)."""
    import oracle as O
    nb = min(w.B, budget_problems)
    ws = w.subset(np.arange(nb)) if nb < w.B else w
    cfg = O.make_cfg(ws)
    t0 = time.perf_counter()
    if w.model:
        O.sqp_bicycle(ws, cfg, nthreads=nthreads)
    else:
        O.admm(ws, cfg, nthreads=nthreads)
    dt = time.perf_counter() - t0
    return nb / dt, f"first {nb} of {w.B} problems, {total_iters(w)} ADMM iterations each, {nthreads} threads (one problem per thread)", dt


def oracle_sample_size(cfg_id):
    return {1: 1, 2: 1024, 3: 64, 4: 1024, 5: 1}[cfg_id]


def config_list(args):
    """(config id, dtype) pairs of this run, headline first."""
    if args.config is not None:
        return [(args.config, args.dtype or DEFAULT_DTYPE[args.config])]
    return [(4, "f32"), (1, "f64"), (2, "f32"), (2, "f64"), (3, "f32"), (5, "f64")]


def key_of(cfg_id, dtype):
    return f"config{cfg_id}_{dtype}"


def reference_one(cfg_id, dtype, args, cores):
    w = make_workload(cfg_id, dtype, args.batch)
    nb = oracle_sample_size(cfg_id)
    for _ in range(args.warmup if args.config is not None else 0):
        oracle_rate(w, cfg_id, cores, nb)
    t, desc = 0.0, ""
    steps = args.steps if args.config is not None else 1
    for _ in range(steps):
        r, desc, dt = oracle_rate(w, cfg_id, cores, nb)
        t += dt
    rate = min(w.B, nb) * steps / t
    return {"value": rate, "unit": "QP solves/s", "ms_per_step": 1e3 * t / steps, "dtype": "f64", "config": {"workload": workload_name(w, dtype)},
            "admm_iters_per_s": rate * total_iters(w),
            "cpu_baseline": {"value": rate, "unit": "QP solves/s", "cores": cores, "kind": "oracle", "sample": desc},
            "e2e": {"value": rate, "unit": "QP solves/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}}


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    cores = len(os.sched_getaffinity(0))
    res = [(c, d, reference_one(c, d, args, cores)) for c, d in config_list(args)]
    c0, d0, head = res[0]
    line = {"impl": "reference", "metric": "batched QP solves/s", "n_gpus": args.gpus, "steps": args.steps, "warmup": args.warmup,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "data": "synthetic"}
    line.update(head)
    if len(res) > 1:
        line["per_config"] = {key_of(c, d): r for c, d, r in res[1:]}
    print(json.dumps(line))


def measure_peaks(dev, stream):
    """FP32 / FP64 FMA and shared-memory peaks of this GPU at the clocks found, via the library's micro-benchmark entry."""
    import torch
    from paper_2606_24039_b200 import binding as Bd
    scratch = torch.zeros(64, dtype=torch.float32, device=dev)
    m = lambda what: Bd.tmpc_measure_peak(what, scratch.data_ptr(), stream.cuda_stream, 5)
    ffma2, ffma, dfma, lds = m(Bd.TMPC_PEAK_FFMA2), m(Bd.TMPC_PEAK_FFMA), m(Bd.TMPC_PEAK_DFMA), m(Bd.TMPC_PEAK_LDS)
    return {"f32_tflops": max(ffma2, ffma), "f32_ffma2_tflops": ffma2, "f32_ffma_tflops": ffma, "f64_tflops": dfma, "lds_gbs": lds,
            "how": "tmpc_measure_peak: independent FMA chains (3-register FFMA2 / FFMA / DFMA) and conflict-free LDS.128, 4 CTAs x 512 threads per SM, best of 5, CUDA events"}


def gpu_one(cfg_id, dtype, args, ctx, steps, with_cpu):
    """Times one config; returns the dict of its metrics (rank 0: complete; other ranks: None after taking part in the reductions)."""
    import torch
    import torch.distributed as dist
    from paper_2606_24039_b200 import binding as Bd
    from paper_2606_24039_b200.solver import Solver
    world, rank, local, dev, peaks = ctx["world"], ctx["rank"], ctx["local"], ctx["dev"], ctx["peaks"]
    w = make_workload(cfg_id, dtype, args.batch, rank)
    linsolve = Bd.TMPC_LIN_CYCLIC_REDUCTION if cfg_id == 5 else Bd.TMPC_LIN_SEQUENTIAL
    s = Solver(w, dtype=dtype, device=dev, linsolve=linsolve)
    flush = ctx["flush"]
    x0 = s._up(w.xbar0) if w.model else None

    def reset():
        for k, v in s.s.items():
            if k == "x" and x0 is not None:
                v.copy_(x0)
            else:
                v.zero_()

    ev = lambda: torch.cuda.Event(enable_timing=True)

    def step():
        """one pass of the hot path; returns (start, end, [(a,b) events around each tmpc_admm_solve])."""
        a, b, inner = ev(), ev(), []
        a.record()
        for _ in range(max(1, w.sqp_iters)):
            if w.model:
                s.linearize()
            s.factor()
            c, d = ev(), ev()
            c.record(); s.admm_solve(); d.record()
            inner.append((c, d))
        b.record()
        return a, b, inner

    def barrier():
        torch.cuda.synchronize(dev)
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize(dev)

    warm = max(3, args.warmup)
    for _ in range(warm):
        reset(); step()
    barrier()
    sampler = ClockSampler(local); sampler.start()
    l0 = s.launches()
    recs = []
    for _ in range(steps):
        reset(); flush.zero_()
        recs.append(step())
    barrier()
    launches = s.launches() - l0
    clocks = sampler.summary()
    step_ms = [a.elapsed_time(b) for a, b, _ in recs]
    kern_ms = [sum(c.elapsed_time(d) for c, d in inner) for _, _, inner in recs]
    n_admm_launch = sum(len(inner) for _, _, inner in recs)
    tot = torch.tensor([sum(step_ms)], dtype=torch.float64, device=dev)
    if world > 1:
        dist.all_reduce(tot, op=dist.ReduceOp.MAX)
    total_ms = float(tot.item())
    info = s.info_numpy()

    # ---- backward (config 2), separately: REFACTOR_REFINE at the state the solve left
    backward_ms = None
    if cfg_id == 2:
        dLdx = 2.0 * s.s["x"]
        ts = []
        for _ in range(3 + steps):
            s.factor(); flush.zero_()
            a, b = ev(), ev(); a.record(); s.backward(dLdx); b.record(); torch.cuda.synchronize(dev); ts.append(a.elapsed_time(b))
        backward_ms = float(np.median(ts[3:]))

    # ---- end to end through the C ABI with HOST buffers (pinned), copies inside the timed region
    e2e = None
    if not w.model and cfg_id != 5:
        hp = lambda t: t.detach().cpu().pin_memory()
        ht = {k: (hp(v) if v is not None else None) for k, v in s.t.items()}
        hs = {k: hp(torch.zeros_like(v)) for k, v in s.s.items()}
        hi = {k: hp(v) for k, v in s.info.items()}
        hq = s.make_qp(ht)
        hst = Bd.TmpcState(*[hs[k].data_ptr() for k in ("x", "zg", "yf", "yg", "xi")])
        hin = Bd.TmpcInfo(hi["r_prim"].data_ptr(), hi["r_dual"].data_ptr(), hi["objective"].data_ptr(), hi["status"].data_ptr())
        nst = Bd.tmpc_host_staging_bytes(s.cfg)
        staging = torch.empty(nst + 256, dtype=torch.uint8, device=dev)
        sp = (staging.data_ptr() + 255) // 256 * 256
        h2d = sum(v.numel() * v.element_size() for v in ht.values() if v is not None) + sum(hs[k].numel() * hs[k].element_size() for k in ("x", "yf", "yg"))
        d2h = sum(v.numel() * v.element_size() for v in hs.values()) + sum(v.numel() * v.element_size() for v in hi.values())
        ts = []
        for i in range(3 + steps):
            for v in hs.values():
                v.zero_()
            torch.cuda.synchronize(dev)
            t0 = time.perf_counter()
            Bd.tmpc_admm_solve_host(s.h, hq, hst, w.iters, 0, hin, sp, nst)
            ts.append(time.perf_counter() - t0)
        t_e2e = torch.tensor([sum(ts[3:])], dtype=torch.float64, device=dev)
        if world > 1:
            dist.all_reduce(t_e2e, op=dist.ReduceOp.MAX)
        e2e = {"value": w.B * world * steps / float(t_e2e.item()), "unit": "QP solves/s", "h2d_bytes_per_step": int(h2d), "d2h_bytes_per_step": int(d2h),
               "ms_per_step": 1e3 * float(t_e2e.item()) / steps}
        assert np.abs(hs["x"].double().numpy() - s.state_numpy()["x"]).max() < 1e-3, "host path disagrees with device path"
        del staging
    else:
        # model configs: the same public calls with pinned host inputs copied in and the result copied out every step
        hx0 = x0.cpu().pin_memory(); href = s.t["stage_ref"].cpu().pin_memory(); hq_ = s.t["q"].cpu().pin_memory(); hxi = s.t["x_init"].cpu().pin_memory()
        hout = torch.empty_like(hx0).pin_memory()
        ts = []
        for i in range(2 + steps):
            reset(); torch.cuda.synchronize(dev)
            t0 = time.perf_counter()
            s.s["x"].copy_(hx0, non_blocking=True); s.t["stage_ref"].copy_(href, non_blocking=True)
            s.t["q"].copy_(hq_, non_blocking=True); s.t["x_init"].copy_(hxi, non_blocking=True)
            step()
            hout.copy_(s.s["x"], non_blocking=True); torch.cuda.synchronize(dev)
            ts.append(time.perf_counter() - t0)
        t_e2e = torch.tensor([sum(ts[2:])], dtype=torch.float64, device=dev)
        if world > 1:
            dist.all_reduce(t_e2e, op=dist.ReduceOp.MAX)
        nb = lambda t: t.numel() * t.element_size()
        e2e = {"value": w.B * world * steps / float(t_e2e.item()), "unit": "QP solves/s", "h2d_bytes_per_step": int(nb(hx0) + nb(href) + nb(hq_) + nb(hxi)),
               "d2h_bytes_per_step": int(nb(hout)), "ms_per_step": 1e3 * float(t_e2e.item()) / steps}
    # ---- f1 (config 2): Alg. 3 as the paper runs it — adaptive step size + termination test, max 1000 iterations
    adaptive = None
    if cfg_id == 2:
        adaptive = {}
        for eps in (1e-3, 1e-5):
            ts, out = [], None
            for _ in range(3):
                reset(); torch.cuda.synchronize(dev)
                t0 = time.perf_counter(); out = s.solve_adaptive(1000, eps, eps); ts.append(time.perf_counter() - t0)
            adaptive[f"eps_{eps:g}"] = {"ms_per_batched_solve": 1e3 * min(ts), "iterations_median": float(np.median(out["iters"])), "iterations_max": int(out["iters"].max()),
                                        "converged_frac": float(out["converged"].mean()), "rho_bar_final_median": float(np.median(out["rho"])),
                                        "note": "tmpc_factor + tmpc_admm_solve_adaptive, wall clock (the call reads the live count back once per 25-iteration round)"}

    s.close()
    if rank != 0:
        return None
    ms_per_step = total_ms / steps
    value = w.B * world / (ms_per_step * 1e-3)
    iters = total_iters(w)
    kern_avg_ms = sum(kern_ms) / max(1, n_admm_launch)
    if cfg_id == 3:
        alg = BYTES_PER_ITER[3] * w.B * w.iters
        mp = ctx["measured_peaks"]
        # the kernel is timed inside a long step of back-to-back launches: the burst copy figure is the stricter denominator
        peak = mp["hbm_gbs"] if mp else 6650.0
        roof = {"bound": "hbm", "achieved": alg / (kern_avg_ms * 1e-3) / 1e9, "peak": peak, "unit": "GB/s",
                "peak_source": "measured: MEASURED_PEAKS.json hbm_gbs (copy bandwidth)" if mp else "fallback of B200_PROFILING.md"}
    else:
        alg = FLOPS_PER_ITER[cfg_id] * w.B * w.iters
        if peaks:
            peak = peaks["f64_tflops"] if dtype == "f64" else peaks["f32_tflops"]
            src = "measured: tmpc_measure_peak FMA-chain micro-benchmark in this run (" + ("DFMA" if dtype == "f64" else "max of FFMA2, FFMA") + ")"
        else:
            peak, src = NOMINAL_TFLOPS[dtype], "nominal: 148 SMs x 128 (fp32) / 64 (fp64) FMA lanes x 2 x 1965 MHz"
        roof = {"bound": "alu", "achieved": alg / (kern_avg_ms * 1e-3) / 1e12, "peak": peak, "unit": "TFLOP/s", "peak_source": src}
    roof["frac"] = roof["achieved"] / roof["peak"]
    tr = NCU_TRAFFIC.get((cfg_id, dtype, w.B))
    roof["traffic"] = tr[0] if tr else None
    if tr:
        roof["traffic_source"] = tr[1]
    roof["kernel"] = ctx["kernel_names"][cfg_id] + " (tmpc_admm_solve)"
    if cfg_id in (1, 2, 4) and peaks:
        # supplementary: the resident class reads every factor / constraint element from SHARED memory once per use, so the
        # binding on-chip resource of its stage-parallel phases is LDS bandwidth, not the FMA pipe (DESIGN.md 5.1 / 6)
        es = 8 if dtype == "f64" else 4
        lds_bytes = (2 * w.N * w.n * w.n + 2 * w.T * w.n * w.n + 4 * w.N * w.nx * w.n) * es * w.B * w.iters
        roof["lds"] = {"achieved": lds_bytes / (kern_avg_ms * 1e-3) / 1e9, "peak": peaks["lds_gbs"], "unit": "GB/s", "frac": lds_bytes / (kern_avg_ms * 1e-3) / 1e9 / peaks["lds_gbs"],
                       "peak_source": "measured: tmpc_measure_peak LDS.128 micro-benchmark in this run",
                       "note": "algorithmic shared-memory bytes (B twice, X twice, A~-/A~+ twice per iteration) / kernel time"}
    roof["kernel_ms_per_launch"] = kern_avg_ms
    roof["kernel_share_of_step"] = sum(kern_ms) / sum(step_ms)
    res = {"value": value, "unit": "QP solves/s", "steps": steps, "warmup": warm, "ms_per_step": ms_per_step, "dtype": dtype,
           "config": {"workload": workload_name(w, dtype), "l2": "256 MB flush write between timed steps",
                      "step": "tmpc_factor + tmpc_admm_solve" if not w.model else "n_sqp x (tmpc_linearize + tmpc_factor + tmpc_admm_solve)"},
           "admm_iters_per_s": value * iters, "ms_per_batched_solve": ms_per_step, "us_per_admm_iteration": 1e3 * ms_per_step / iters,
           "backward_ms": backward_ms, "adaptive": adaptive, "gpu_launches": int(launches), "clocks": clocks, "e2e": e2e, "roofline": roof,
           "parity_snapshot": {"max_r_prim": float(np.max(info["r_prim"])), "max_r_dual": float(np.max(info["r_dual"])), "status_nonzero": int((info["status"] != 0).sum())}}
    if with_cpu:
        cores = len(os.sched_getaffinity(0))
        r, desc, dt = oracle_rate(w, cfg_id, cores, oracle_sample_size(cfg_id))
        res["cpu_baseline"] = {"value": r, "unit": "QP solves/s", "cores": cores, "kind": "oracle", "sample": desc, "seconds": dt}
    return res


def f4_rows(ctx, args):
    """f4: the paper's linear-system RL workload at four shapes of its sweep x u_max in {1, 10}: time to
    tolerance 1e-3 / 1e-5 with at most 1000 ADMM iterations (the paper's setting), backward pass, and an H = 50 closed-loop roll-out of
    warm-started MPC solves at the nominal shape.  fp64 like the paper."""
    import torch
    from paper_2606_24039_b200 import binding as Bd
    from paper_2606_24039_b200 import workloads as W
    from paper_2606_24039_b200.solver import Solver
    dev = ctx["dev"]
    rows = []
    for (B, N, nx, nu) in ((64, 40, 8, 4), (1024, 40, 8, 4), (64, 160, 8, 4), (64, 40, 32, 16)):
        for u_max in (1.0, 10.0):
            w = W.linear_rl(B=B, N=N, nx=nx, nu=nu, u_max=u_max)
            s = Solver(w, dtype="f64", device=dev)
            row = {"B": B, "N": N, "nx": nx, "nu": nu, "u_max": u_max, "dtype": "f64"}
            for eps in (1e-3, 1e-5):
                ts, out, mode = [], None, "adaptive"
                for _ in range(3):
                    s.reset_state(); torch.cuda.synchronize(dev)
                    t0 = time.perf_counter()
                    try:
                        out = s.solve_adaptive(1000, eps, eps)
                    except Bd.TmpcError:                 # streamed class: fixed-count solves only
                        mode = "fixed 200 iterations (adaptive schedule not available for the streamed class)"
                        s.solve(200); torch.cuda.synchronize(dev)
                    ts.append(time.perf_counter() - t0)
                row[f"tol_{eps:g}"] = {"ms_per_batched_solve": 1e3 * min(ts), "mode": mode,
                                       "iterations_median": float(np.median(out["iters"])) if out else 200.0, "iterations_max": int(out["iters"].max()) if out else 200,
                                       "converged_frac": float(out["converged"].mean()) if out else None}
            dLdx = 2.0 * s.s["x"]
            ts = []
            for _ in range(4):
                s.factor(); torch.cuda.synchronize(dev)
                t0 = time.perf_counter(); s.backward(dLdx); torch.cuda.synchronize(dev); ts.append(time.perf_counter() - t0)
            row["backward_ms"] = 1e3 * min(ts[1:])
            if (B, N, nx, nu) == (64, 40, 8, 4):          # closed loop: H = 50 MPC solves, each warm-started from the previous solution
                A = s.t["Am"][:, 0, :, :nx]; Bm = s.t["Am"][:, 0, :, nx:]; bv = -s.t["b"][:, 0, :]
                tl = []
                for _ in range(2):                        # best of two roll-outs (the first one also pays torch's one-time einsum set-up)
                    s.reset_state(); s.t["x_init"].copy_(s._up(w.x_init)); torch.cuda.synchronize(dev)
                    t0 = time.perf_counter(); its = 0
                    for hstep in range(50):
                        out = s.solve_adaptive(1000, 1e-3, 1e-3, flags=Bd.TMPC_SOLVE_ZG_GIVEN if hstep else 0)
                        its += int(out["iters"].max())
                        u0 = s.s["x"][:, 0, nx:]
                        xn = torch.einsum("bij,bj->bi", A, s.t["x_init"]) + torch.einsum("bij,bj->bi", Bm, u0) + bv      # the environment step (not the solver)
                        s.t["x_init"].copy_(xn)
                    torch.cuda.synchronize(dev)
                    tl.append(time.perf_counter() - t0)
                row["closed_loop_H50_tol_1e-3"] = {"ms_total": 1e3 * min(tl), "max_iterations_summed": its}
            rows.append(row)
            s.close()
    return rows


def f4_sweep(ctx, args):
    """The three sweeps of the paper's Fig. 3 around the nominal (B, N, nx, nu) = (64, 40, 8, 4): batch size, horizon and block size,
    u_max in {1, 10}, tol = 1e-5 with at most 1000 ADMM iterations, fp64; forward = one batched adaptive solve (best of 3), backward = REFINE mode
    (best of 3).  One seed per point (the paper averages ten)."""
    import torch
    from paper_2606_24039_b200 import binding as Bd
    from paper_2606_24039_b200 import workloads as W
    from paper_2606_24039_b200.solver import Solver
    dev = ctx["dev"]
    pts = [("B", (B, 40, 8, 4)) for B in (1, 8, 16, 32, 64, 128, 256, 512, 1024)]
    pts += [("N", (64, N, 8, 4)) for N in (10, 20, 80, 160, 320)]
    pts += [("n", (64, 40, nx, nx // 2)) for nx in (4, 16, 32, 64)]
    rows = []
    for axis, (B, N, nx, nu) in pts:
        for u_max in (1.0, 10.0):
            row = {"sweep": axis, "B": B, "N": N, "nx": nx, "nu": nu, "u_max": u_max, "dtype": "f64"}
            try:
                w = W.linear_rl(B=B, N=N, nx=nx, nu=nu, u_max=u_max)
                s = Solver(w, dtype="f64", device=dev)
                ts, out = [], None
                for _ in range(3):
                    s.reset_state(); torch.cuda.synchronize(dev)
                    t0 = time.perf_counter(); out = s.solve_adaptive(1000, 1e-5, 1e-5); ts.append(time.perf_counter() - t0)
                row.update({"forward_ms": 1e3 * min(ts), "iterations_median": float(np.median(out["iters"])), "iterations_max": int(out["iters"].max()),
                            "converged_frac": float(out["converged"].mean())})
                dLdx = 2.0 * s.s["x"]
                ts = []
                for _ in range(4):
                    s.factor(); torch.cuda.synchronize(dev)
                    t0 = time.perf_counter(); s.backward(dLdx); torch.cuda.synchronize(dev); ts.append(time.perf_counter() - t0)
                row["backward_ms"] = 1e3 * min(ts[1:])
                s.close()
            except Bd.TmpcError as e:
                row["error"] = str(e)
            rows.append(row)
    return rows


def f3_row(ctx, args):
    """f3: the humanoid balancing OCP of the paper's imitation-learning experiment (SRB dynamics, RK4, nx = 12, nu = 6, N = 20) with
    the second built-in model: n_sqp x (tmpc_linearize + tmpc_factor + tmpc_admm_solve), fp64 like the paper, B = 1024."""
    import torch
    from paper_2606_24039_b200 import workloads as W
    from paper_2606_24039_b200.solver import Solver
    dev = ctx["dev"]
    w = W.srb_humanoid(B=1024)
    s = Solver(w, dtype="f64", device=dev)
    x0 = s._up(w.xbar0)
    ts = []
    for _ in range(6):
        for k, v in s.s.items():
            v.copy_(x0) if k == "x" else v.zero_()
        torch.cuda.synchronize(dev)
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record(); s.sqp(); b.record(); torch.cuda.synchronize(dev); ts.append(a.elapsed_time(b))
    info = s.info_numpy()
    s.close()
    ms = float(np.median(ts[2:]))
    return {"workload": workload_name(w, "f64"), "ms_per_batched_solve": ms, "qp_solves_per_s": w.B / (ms * 1e-3),
            "admm_iters_per_s": w.B * total_iters(w) / (ms * 1e-3), "max_r_prim": float(np.max(info["r_prim"])), "kernels": "srb_linearize_kernel + factor_kernel + admm_kernel (generic class, n = 18)"}


def run_gpu(args):
    import torch
    import torch.distributed as dist
    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device (no CPU fallback); use --impl reference for the oracle")
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device(f"cuda:{local}"))
    dev = torch.device(f"cuda:{local}")
    mpath = os.path.join(ROOT, "MEASURED_PEAKS.json")
    ctx = {"world": world, "rank": rank, "local": local, "dev": dev,
           "flush": torch.empty(256 * 1024 * 1024, dtype=torch.uint8, device=dev),   # > 126 MB L2
           "measured_peaks": json.load(open(mpath)) if os.path.exists(mpath) else None,
           "peaks": measure_peaks(dev, torch.cuda.current_stream(dev)),
           "kernel_names": KERNEL_NAMES}
    res = []
    for i, (c, d) in enumerate([] if (args.f4_only or args.f4_sweep) else config_list(args)):
        steps = args.steps if (args.config is not None or i == 0) else max(3, min(args.steps, STEPS_CAP.get(c, args.steps)))
        res.append((c, d, gpu_one(c, d, args, ctx, steps, world == 1 and not args.no_cpu_baseline)))
    if args.f4_sweep:
        rows = f4_sweep(ctx, args)
        if rank == 0:
            print(json.dumps({"metric": "f4 linear-system RL workload: the sweeps of PAPER.md Fig. 3 (tol 1e-5, fp64)", "rows": rows}))
        return
    f4 = f4_rows(ctx, args) if (args.config is None and world == 1 and not args.no_f4) or args.f4_only else None
    f3 = f3_row(ctx, args) if f4 is not None else None
    if args.f4_only:
        if rank == 0:
            print(json.dumps({"metric": "f4 linear-system RL workload (PAPER.md:414-416) and f3 humanoid OCP", "rows": f4, "f3_srb_humanoid": f3, "measured_peaks": ctx["peaks"]}))
        return
    if rank == 0:
        c0, d0, head = res[0]
        line = {"metric": "batched QP solves/s", "n_gpus": world, "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "data": "synthetic"}
        line.update(head)
        line["measured_peaks"] = ctx["peaks"]
        if len(res) > 1:
            line["per_config"] = {key_of(c, d): r for c, d, r in res[1:]}
            line["gpu_launches"] = int(sum(r["gpu_launches"] for _, _, r in res))
        if f4 is not None:
            line.setdefault("per_config", {})["f4_linear_rl"] = f4
            line["per_config"]["f3_srb_humanoid"] = f3
        print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="tmpc", choices=["tmpc", "reference"])
    ap.add_argument("--config", type=int, default=None, choices=[None, 1, 2, 3, 4, 5])
    ap.add_argument("--dtype", default=None, choices=[None, "f32", "f64"])
    ap.add_argument("--batch", type=int, default=None)
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-f4", action="store_true", help="skip the f4 linear-system RL rows of the all-configs run")
    ap.add_argument("--f4-only", action="store_true", help="run only the f4 linear-system RL rows")
    ap.add_argument("--f4-sweep", action="store_true", help="run only the batch / horizon / block-size sweeps of the paper's Fig. 3 on the f4 workload")
    args = ap.parse_args()
    if args.impl == "reference":
        run_reference(args)
    else:
        run_gpu(args)


if __name__ == "__main__":
    main()
