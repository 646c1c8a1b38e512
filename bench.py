#!/usr/bin/env python
"""bench.py -- BASELINE.json's metric on BASELINE.json's config, one JSON line on stdout.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--workload c4]

Metric: fp64 PCG iterations/s (and achieved HBM GB/s, % of peak) on the 256x256x512 grid
(BASELINE.json configs[3]: stretched r mesh, nu(r), s = 1e4, RHS uniform(-1,1) seed 3, 500 fixed
iterations).  A "step" is one whole solve: init + 500 iterations of {K1 fused matvec, K2 fused
vector kernel} inside one CUDA-graph WHILE loop, inputs resident in HBM.  `e2e` is the same solve
through mas_pcg_solve_host with pinned HOST buffers (H2D of b and x0, D2H of x inside the timed
region).  N > 1: replicas only (the path does not shard), one independent
solve per rank, value = all ranks' iterations / max-over-ranks time.

--impl reference times the ORACLE (oracle/mas_pcg_ref.c, as it stands, one host thread) on a
bounded sample of the same workload.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "fp64_pcg_iterations_per_s_256x256x512"
UNIT = "iterations/s"
FALLBACK_HBM_GBS = 6650.0          # /opt/skills/guides/B200_PROFILING.md fallback
REF_ITERS_PER_STEP = 4             # oracle iterations per step of --impl reference (bounded sample)
CPU_BASELINE_ITERS = 20            # oracle iterations timed for cpu_baseline (BASELINE.md sec. 5 / SURVEY 8(d): 20; about 20-30 s)


def parse():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="c4", choices=["c1", "c2", "c3", "c4", "c5", "sts", "visc", "precond"])
    ap.add_argument("--precond", type=int, default=1, choices=[1, 2],
                    help="1 = PC1 point Jacobi (default), 2 = PC2 block-Jacobi ILU(0) over phi lines (NEXT-4)")
    ap.add_argument("--mesh", default="config", choices=["config", "nonuniform", "clustered"],
                    help="configs 3-5, sts, precond: BASELINE.json's mesh (uniform theta / phi), the same shape with r, theta and "
                         "phi widths varying by +-30 %% (the kernels' general instantiations), or a paper-like mesh packed in "
                         "r and theta with a uniform nu (mas_inputs.configs.make)")
    ap.add_argument("--opt", action="append", default=[], help="name=value passed to mas_pcg_set_option (tuning)")
    ap.add_argument("--nrhs", type=int, default=1, help="right-hand sides per batched solve (1..3; NEXT-2)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--chain-steps", type=int, default=100,
                    help="--workload c5: consecutive solves timed (BASELINE.json config 5 has 100)")
    return ap.parse_args()


def workload_rhs(name, prob):
    """the config's right-hand side from prob.seed"""
    from mas_inputs import configs
    if name in ("c1", "c4"):
        return configs.rhs_uniform(prob)
    if name == "c2":
        return configs.field_manufactured(prob)   # used as a right-hand side here (bench only)
    return configs.rhs_blob(prob)


def workload(name, rank=0, mesh_kind="config"):
    """(problem, dt, b, rtol, maxit, description).  Seeds are offset by the rank for replicas."""
    from mas_inputs import configs
    import numpy as np
    prob = configs.make(name, mesh_kind=mesh_kind)
    prob.seed += 1000 * rank
    s = prob.stiffness[-1]
    dt = prob.dt_for(s)
    b = workload_rhs(name, prob)
    nr, nt, np_ = prob.mesh.shape
    rtol, maxit = (0.0, 500) if name == "c4" else (prob.rtol, prob.maxit)
    desc = (f"{name}: {nr}x{nt}x{np_} fp64, stiffness s={s:g}, rtol={rtol:g}, maxit={maxit}, "
            f"{'500 fixed PCG iterations' if name == 'c4' else 'solve to rtol'}")
    if mesh_kind != "config":
        desc += {"nonuniform": "; mesh: r, theta and phi widths varying by +-30 % (grids.random_mesh), dt from the oracle-written S1",
                 "clustered": "; mesh: packed in r and theta (grids.clustered_mesh), uniform nu, phi uniform"}[mesh_kind]
    return prob, dt, np.ascontiguousarray(b), rtol, maxit, desc


class ClockSampler:
    """nvidia-smi clocks / throttle reasons DURING the timed region (B200_PROFILING.md clocks line)."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.rows, self.proc, self.index = [], None, index

    def start(self):
        try:
            self.proc = subprocess.Popen(
                ["nvidia-smi", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits", "-lms", "100",
                 "-i", str(self.index)], stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.th = threading.Thread(target=self._read, daemon=True)
            self.th.start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append([c.strip() for c in line.split(",")])

    def stop(self):
        if not self.proc:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except Exception:
            self.proc.kill()
        self.th.join(timeout=2)
        sm, mx, reasons, pw = [], [], set(), []
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for r in self.rows:
            if len(r) < 7:
                continue
            try:
                sm.append(float(r[0])); mx.append(float(r[1])); pw.append(float(r[2]))
            except ValueError:
                continue
            for n, v in zip(names, r[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(n)
        sm.sort()
        return {"sm_mhz": sm[len(sm) // 2] if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "power_w_max": max(pw) if pw else None, "samples": len(sm), "reasons": sorted(reasons)}


def gpu_selector(torch):
    """What nvidia-smi -i should get for the current CUDA device: its UUID (robust to CUDA_VISIBLE_DEVICES)."""
    try:
        u = str(torch.cuda.get_device_properties(torch.cuda.current_device()).uuid)
        return u if u.startswith("GPU-") else "GPU-" + u
    except Exception:
        return torch.cuda.current_device()


def hbm_peak():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    try:
        with open(p) as f:
            return float(json.load(f)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    except Exception:
        return FALLBACK_HBM_GBS, "fallback (B200_PROFILING.md 6.65 TB/s)"


def ncu_traffic(kernel_key):
    """(per-launch DRAM bytes, provenance) of a kernel from the committed ncu --set full summary
    (profiles/roofline_traffic.csv; each row names the commit and the capture it was taken from)."""
    try:
        import csv
        with open(os.path.join(ROOT, "profiles", "roofline_traffic.csv")) as f:
            for row in csv.DictReader(f):
                if row["kernel"] == kernel_key:
                    return int(row["dram_bytes_per_launch"]), f"{row.get('commit', '?')} {row.get('source', '')}".strip()
    except Exception:
        pass
    return None, None


def time_oracle(prob, dt, b, iters):
    """The oracle as it stands, one host thread: seconds for `iters` PCG iterations from x0 = 0."""
    from oracle import ref
    op = ref.RefOperator(prob.mesh, dt, prob.nu_kind, prob.nu, prob.bc)
    t0 = time.perf_counter()
    st, k, _, _ = op.pcg(b, None, 0.0, iters)
    t = time.perf_counter() - t0
    op.close()
    return t, k


def reduce_over_ranks(ms, iters, launches, world, device="cuda"):
    """Replicas: time = MAX over ranks, work (iterations, launches) = SUM over ranks."""
    if world == 1:
        return ms, iters, launches
    import torch
    import torch.distributed as dist
    tmax = torch.tensor([ms], dtype=torch.float64, device=device)
    tsum = torch.tensor([iters, launches], dtype=torch.float64, device=device)
    dist.all_reduce(tmax, op=dist.ReduceOp.MAX)
    dist.all_reduce(tsum, op=dist.ReduceOp.SUM)
    return float(tmax[0]), float(tsum[0]), float(tsum[1])


def run_reference(args, rank, world):
    """Base-contract reference arm = the oracle on host cores; rank 0 only."""
    if rank != 0:
        return
    prob, dt, b, rtol, maxit, desc = workload(args.workload)
    for _ in range(min(args.warmup, 1)):
        time_oracle(prob, dt, b, 1)
    t_total, its = 0.0, 0
    for _ in range(args.steps):
        t, k = time_oracle(prob, dt, b, REF_ITERS_PER_STEP)
        t_total += t
        its += k
    value = its / t_total
    sample = (f"{args.steps} steps x {REF_ITERS_PER_STEP} PCG iterations from x0=0 (operator setup and "
              f"initial residual included), single thread, gcc -O2")
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * t_total / args.steps,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
            "data": "synthetic", "config": {"workload": desc, "sample": sample},
            "cpu_baseline": {"value": value, "unit": UNIT, "cores": 1, "kind": "oracle", "sample": sample},
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)


def run_chain(args):
    """BASELINE.json config 5, time-step proxy: 100 consecutive warm-started solves on 192x256x384, dt varying
    +-20 % per step, RHS(k+1) = x(k) + 0.05 N(0,1).  Timed per solve with CUDA events (set_dt + solve);
    RHS construction and its H2D copy are outside the timed regions.  `e2e` is the same chain
    through mas_pcg_solve_host (pinned host RHS and x; the copies are inside the timed call), run in lock-step
    with the device-resident chain so that one noise draw per step serves both."""
    import numpy as np
    import torch
    from mas_inputs import configs
    from paper_1811_02605_b200 import MasPcg
    torch.cuda.set_device(0)
    prob = configs.make("c5", mesh_kind=args.mesh)
    nsteps = max(args.chain_steps, 1)
    dt0 = prob.dt_for(prob.stiffness[-1])
    chain = configs.Chain(prob, 100)
    gpu = MasPcg(prob.mesh, dt0, prob.nu_kind, prob.nu, prob.bc)
    for kv in args.opt:
        name, val = kv.split("=")
        gpu.set_option(name, int(val))
    if args.precond == 2:
        gpu.set_preconditioner(2)
    stream = torch.cuda.current_stream()
    n = prob.mesh.ncells
    x = torch.zeros(prob.mesh.shape, dtype=torch.float64, device="cuda")
    rhs_host = torch.from_numpy(chain.state0 + chain.noise()).pin_memory()
    x_host = torch.zeros(prob.mesh.shape, dtype=torch.float64).pin_memory()
    rhs = rhs_host.cuda()
    rhs0_np = rhs_host.numpy().copy()
    # warm-up on scratch vectors (graph build, staging buffers, clocks)
    xs = torch.zeros_like(x)
    for _ in range(max(args.warmup, 3)):
        xs.zero_()
        gpu.solve(rhs, xs, prob.rtol, prob.maxit, want_hist=False)
    gpu.solve_host(rhs_host, x_host, prob.rtol, prob.maxit, want_hist=False)
    x_host.zero_()
    sampler = ClockSampler(gpu_selector(torch))
    sampler.start()
    total_ms, e2e_s, iters, launches = 0.0, 0.0, [], 0
    for step in range(nsteps):
        dt = dt0 * chain.dt_factor[step]
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        torch.cuda.synchronize()
        e0.record(stream)
        gpu.set_dt(dt)
        st, k, _ = gpu.solve(rhs, x, prob.rtol, prob.maxit, want_hist=False)      # x: warm start, in place
        e1.record(stream)
        torch.cuda.synchronize()
        total_ms += e0.elapsed_time(e1)
        iters.append(k)
        sstat = gpu.stats()
        launches += sstat["loop_launches"] + sstat["other_launches"] + 1
        if st != 0:
            raise SystemExit(f"chain step {step}: status {st}")
        t0 = time.perf_counter()                                                   # end to end: host buffers
        gpu.set_dt(dt)
        st2, k2, _ = gpu.solve_host(rhs_host, x_host, prob.rtol, prob.maxit, want_hist=False)
        e2e_s += time.perf_counter() - t0
        if (st2, k2) != (st, k):
            raise SystemExit(f"chain step {step}: host-buffer solve differs ({st2}, {k2}) vs ({st}, {k})")
        if step + 1 < nsteps:                                                      # untimed: next right-hand side
            rhs_host.copy_(x_host + torch.from_numpy(chain.noise()))
            rhs.copy_(rhs_host)
    clocks = sampler.stop()
    bpc = gpu.stats()["bytes_per_cell_iter"]
    peak, peak_src = hbm_peak()
    its = float(np.sum(iters))
    gbs = bpc * n * its / (total_ms * 1e-3) / 1e9
    line = {"metric": "pcg_solves_per_s_192x256x384_timestep_proxy" + ("" if args.mesh == "config" else f"_{args.mesh}_mesh"), "value": nsteps / (total_ms * 1e-3),
            "unit": "solves/s", "n_gpus": 1, "steps": nsteps, "warmup": max(args.warmup, 3),
            "ms_per_step": total_ms / nsteps, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": f"c5: 192x256x384 fp64, s=100 at dt0, dt +-20 %/step, warm start, rtol 1e-9, "
                                   f"{'all' if nsteps == 100 else 'first ' + str(nsteps) + ' of'} 100 chained solves",
                       "l2": "inputs larger than L2 (5 live vectors x 151 MB vs 126 MB)",
                       "mean_iters_per_solve": float(np.mean(iters)), "iters": iters, "bytes_per_cell_iter": bpc,
                       "preconditioner": {1: "PC1 point Jacobi", 2: "PC2 block-Jacobi ILU(0), phi-line domains"}[args.precond]},
            "iterations_per_s": its / (total_ms * 1e-3),
            "clocks": clocks,
            "e2e": {"value": nsteps / e2e_s, "unit": "solves/s", "h2d_bytes_per_step": 2 * 8 * n,
                    "d2h_bytes_per_step": 8 * n},
            "gpu_launches": int(launches),
            "roofline": {"bound": "hbm", "kernel": "whole solve (init + iterations + tail), model bytes = "
                                                   f"{bpc} B/cell/iteration x iterations",
                         "achieved": gbs, "peak": peak, "unit": "GB/s", "frac": gbs / peak, "traffic": None,
                         "peak_source": peak_src}}
    if not args.no_cpu_baseline:
        from oracle import ref
        op = ref.RefOperator(prob.mesh, dt0, prob.nu_kind, prob.nu, prob.bc)
        ch = configs.Chain(prob, 100)
        b, xo, t_or, k_or = rhs0_np, None, 0.0, []
        ch.noise()                                          # the draw that made rhs0
        for step in range(3):
            op.set_dt(dt0 * ch.dt_factor[step])
            t0 = time.perf_counter()
            if args.precond == 2:
                pc = op.pc2((1, 1, 0))                      # factorisation at the new dt, inside the timed region
                st_o, k_o, xo, _ = op.pcg_pc2(pc, b, xo, prob.rtol, prob.maxit)
                pc.close()
            else:
                st_o, k_o, xo, _ = op.pcg(b, xo, prob.rtol, prob.maxit)
            t_or += time.perf_counter() - t0
            k_or.append(k_o)
            b = xo + ch.noise()
        op.close()
        line["cpu_baseline"] = {"value": 3 / t_or, "unit": "solves/s", "cores": 1, "kind": "oracle",
                                "sample": f"3-solve prefix of the chain (x100/3 extrapolates to the 100 solves), "
                                          f"iterations {k_or} vs GPU {iters[:3]}, one thread of {os.cpu_count()} "
                                          f"host cores, gcc -O2"}
    print(json.dumps(line), flush=True)


def run_sts(args):
    """NEXT-1: RKL2 super time stepping of the viscosity term on the 256x256x512 mesh of config 4 (same nu),
    one super-step of 200 stages per step ("~200 sub-steps per time-step"), tau at 90 % of the
    stability limit.  Algorithmic traffic per stage: Y_{j-1}, Y_{j-2}, Y_0, M Y_0 -> Y_j = 5 doubles per cell."""
    import numpy as np
    import torch
    from mas_inputs import configs
    from paper_1811_02605_b200 import MasPcg
    torch.cuda.set_device(0)
    prob = configs.make("c4", mesh_kind=args.mesh)
    S = 200
    gpu = MasPcg(prob.mesh, 1.0, prob.nu_kind, prob.nu, prob.bc)
    for kv in args.opt:
        name, val = kv.split("=")
        gpu.set_option(name, int(val))
    tau = 0.9 * (S * S + S - 2.0) / 4.0 * 2.0 / gpu.lambda_max()
    u0 = torch.from_numpy(configs.rhs_uniform(prob)).cuda()
    u = u0.clone()
    stream = torch.cuda.current_stream()
    for _ in range(max(args.warmup, 3)):
        u.copy_(u0)
        gpu.sts_advance(u, tau, S)
    sampler = ClockSampler(gpu_selector(torch))
    sampler.start()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    torch.cuda.synchronize()
    ms = 0.0
    for _ in range(args.steps):
        u.copy_(u0)                                   # untimed reset
        torch.cuda.synchronize()
        e0.record(stream)
        gpu.sts_advance(u, tau, S)
        e1.record(stream)
        torch.cuda.synchronize()
        ms += e0.elapsed_time(e1)
    clocks = sampler.stop()
    n = prob.mesh.ncells
    stage_ms = ms / (args.steps * S)
    alg = (5.0 * (S - 1) + 3.0) / S * 8 * n            # bytes per stage, averaged (stage 1 moves 3N)
    peak, peak_src = hbm_peak()
    gbs = alg / (stage_ms * 1e-3) / 1e9
    line = {"metric": "rkl2_sts_stages_per_s_256x256x512" + ("" if args.mesh == "config" else f"_{args.mesh}_mesh"), "value": 1e3 / stage_ms, "unit": "stages/s", "n_gpus": 1,
            "steps": args.steps, "warmup": max(args.warmup, 3), "ms_per_step": ms / args.steps,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": "sts: 256x256x512 fp64, nu(r) of config 4, one RKL2 super-step of 200 stages, "
                                   "tau = 0.9 tau_max", "l2": "inputs larger than L2"},
            "clocks": clocks, "gpu_launches": args.steps * S,
            "roofline": {"bound": "hbm", "kernel": "k_stencil<EPI_STS>", "achieved": gbs, "peak": peak, "unit": "GB/s",
                         "frac": gbs / peak, "traffic": ncu_traffic("k_stencil_sts")[0],
                         "traffic_source": ncu_traffic("k_stencil_sts")[1], "peak_source": peak_src}}
    if not args.no_cpu_baseline:
        from oracle import ref
        op = ref.RefOperator(prob.mesh, 1.0, prob.nu_kind, prob.nu, prob.bc)
        ub = configs.rhs_uniform(prob)
        t0 = time.perf_counter()
        op.sts(ub, tau * 1e-3, 6)
        t = time.perf_counter() - t0
        line["cpu_baseline"] = {"value": 6 / t, "unit": "stages/s", "cores": 1, "kind": "oracle",
                                "sample": "one RKL2 super-step of 6 stages on the same mesh, one host thread, gcc -O2"}
    print(json.dumps(line), flush=True)


def run_visc(args):
    """The paper's algorithm comparison for the viscosity advance (PCG+PC1 needs ~550
    iterations, STS ~200 sub-steps, PC1+STS about 2x faster than PC1+PC1 for the whole step) on the synthetic
    256x256x512 mesh: the same dt (stiffness 1e4) advanced implicitly by the PCG solve and explicitly by RKL2."""
    import numpy as np
    import torch
    from mas_inputs import configs
    from paper_1811_02605_b200 import MasPcg
    torch.cuda.set_device(0)
    prob = configs.make("c4")
    dt = prob.dt_for(1e4)
    gpu = MasPcg(prob.mesh, dt, prob.nu_kind, prob.nu, prob.bc)
    u0 = torch.from_numpy(configs.blob(prob.mesh)
                          + 0.01 * np.random.default_rng(2).standard_normal(prob.mesh.shape)).cuda()
    x, u = torch.zeros_like(u0), u0.clone()
    S = gpu.sts_stages(dt)
    stream = torch.cuda.current_stream()

    def timed(fn):
        for _ in range(max(args.warmup, 1)):
            fn()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        torch.cuda.synchronize()
        e0.record(stream)
        for _ in range(args.steps):
            out = fn()
        e1.record(stream)
        torch.cuda.synchronize()
        return e0.elapsed_time(e1) / args.steps, out

    ms_pcg, (st, k, _) = timed(lambda: gpu.solve(u0, x.zero_(), 1e-9, 5000, want_hist=False))
    ms_sts, _ = timed(lambda: gpu.sts_advance(u.copy_(u0), dt, S))
    line = {"metric": "viscosity_advance_ms_256x256x512", "value": ms_sts, "unit": "ms", "n_gpus": 1,
            "steps": args.steps, "warmup": max(args.warmup, 1), "ms_per_step": ms_sts, "higher_is_better": False,
            "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": "visc: 256x256x512 fp64, nu(r), dt at stiffness 1e4, blob + noise field (each "
                                   "timing includes one 268 MB reset of the field)"},
            "pcg_pc1": {"ms": ms_pcg, "iterations": k, "status": st, "rtol": 1e-9},
            "sts_rkl2": {"ms": ms_sts, "stages": S},
            "sts_speedup_over_pcg": ms_pcg / ms_sts,
            "implicit_vs_explicit_max_rel_diff": float((u - x).abs().max() / u0.abs().max())}
    print(json.dumps(line), flush=True)


def run_precond(args):
    """The paper's preconditioner comparison (PC2 needs 100-200 iterations against ~550
    with PC1 but its triangular solves were left on the CPU; with cuSparse on the GPU "similar performance as using
    PC1"), on the synthetic hard viscosity solves: configs 3 and 4 (stiffness 1e4) solved to rtol 1e-9 with PC1 and
    with PC2 (block-Jacobi ILU(0) over phi-line domains), time to solution and iterations."""
    import torch
    from mas_inputs import configs
    from paper_1811_02605_b200 import MasPcg
    torch.cuda.set_device(0)
    stream = torch.cuda.current_stream()
    out = {}
    for name in ("c3", "c4"):
        prob = configs.make(name, mesh_kind=args.mesh)
        dt = prob.dt_for(1e4)
        b = torch.from_numpy(workload_rhs(name, prob)).cuda()
        x = torch.zeros_like(b)
        gpu = MasPcg(prob.mesh, dt, prob.nu_kind, prob.nu, prob.bc)
        res = {}
        for pc in (1, 2):
            gpu.set_preconditioner(pc)
            for _ in range(max(args.warmup, 1)):
                x.zero_()
                gpu.solve(b, x, 1e-9, 5000, want_hist=False)
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            ms = 0.0
            for _ in range(args.steps):
                x.zero_()
                torch.cuda.synchronize()
                e0.record(stream)
                st, k, _ = gpu.solve(b, x, 1e-9, 5000, want_hist=False)
                e1.record(stream)
                torch.cuda.synchronize()
                ms += e0.elapsed_time(e1)
            s = gpu.stats()
            res[f"pc{pc}"] = {"ms": ms / args.steps, "iterations": k, "status": st,
                              "ms_per_iteration": ms / args.steps / max(k, 1),
                              "bytes_per_cell_iter": s["bytes_per_cell_iter"],
                              "model_gbs": s["bytes_per_cell_iter"] * prob.mesh.ncells * k / (ms / args.steps * 1e-3) / 1e9}
        res["pc2_speedup"] = res["pc1"]["ms"] / res["pc2"]["ms"]
        res["iteration_ratio"] = res["pc1"]["iterations"] / res["pc2"]["iterations"]
        out[name] = res
        gpu.close()
    line = {"metric": "viscosity_solve_ms_pc2_256x256x512" + ("" if args.mesh == "config" else f"_{args.mesh}_mesh"), "value": out["c4"]["pc2"]["ms"], "unit": "ms", "n_gpus": 1,
            "steps": args.steps, "warmup": max(args.warmup, 1), "ms_per_step": out["c4"]["pc2"]["ms"],
            "higher_is_better": False, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": "precond: configs 3 (128x192x256) and 4 (256x256x512) at stiffness 1e4, solved to "
                                   "rtol 1e-9 from x0 = 0 with PC1 (point Jacobi) and PC2 (block-Jacobi ILU(0), phi-line domains)"
                                   + ("" if args.mesh == "config" else f"; mesh kind: {args.mesh} (mas_inputs.configs.make)"),
                       "note": "the PC2 / PC1 ratio depends on where the mesh puts its stiffness: the phi-line domains "
                               "contain the phi couplings only (DESIGN.md R8)"},
            "c3": out["c3"], "c4": out["c4"]}
    print(json.dumps(line), flush=True)


def main():
    args = parse()
    if args.impl == "ours" and args.workload == "visc":
        run_visc(args)
        return
    if args.impl == "ours" and args.workload == "c5":
        run_chain(args)
        return
    if args.impl == "ours" and args.workload == "precond":
        run_precond(args)
        return
    if args.impl == "ours" and args.workload == "sts":
        run_sts(args)
        return
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    if args.impl == "reference":
        run_reference(args, rank, world)
        return

    import numpy as np
    import torch
    import torch.distributed as dist
    from paper_1811_02605_b200 import MasPcg

    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the product path has no CPU fallback")
    torch.cuda.set_device(local_rank)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local_rank))

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    prob, dt, b_np, rtol, maxit, desc = workload(args.workload, rank, args.mesh)
    n = prob.mesh.ncells
    nrhs = max(1, min(3, args.nrhs))
    opts = [(kv.split("=")[0], int(kv.split("=")[1])) for kv in args.opt]
    gpu = MasPcg(prob.mesh, dt, prob.nu_kind, prob.nu, prob.bc)
    for name, val in opts:
        gpu.set_option(name, val)
    if args.precond == 2:
        gpu.set_preconditioner(2)
    # right-hand side j of a batched solve = the workload's b from seed + j (independent problems, one operator)
    b_hosts = [torch.from_numpy(b_np).pin_memory()]
    for j in range(1, nrhs):
        pj = prob
        pj.seed += 1
        b_hosts.append(torch.from_numpy(np.ascontiguousarray(workload_rhs(args.workload, pj))).pin_memory())
    x_host = torch.zeros(prob.mesh.shape, dtype=torch.float64).pin_memory()
    bs = [bh.cuda() for bh in b_hosts]
    xs = [torch.zeros_like(bs[0]) for _ in range(nrhs)]
    b, x, b_host = bs[0], xs[0], b_hosts[0]
    stream = torch.cuda.current_stream()

    def step():
        """one whole solve from x0 = 0 (the memsets are outside the solver's kernels); returns (status, iterations
        summed over the right-hand sides)"""
        for xv in xs:
            xv.zero_()
        if nrhs == 1:
            st_, k_, _ = gpu.solve(b, x, rtol, maxit, want_hist=False)
            return st_, k_
        st_, sts_, its_, _ = gpu.solve_multi(bs, xs, rtol, maxit, want_hist=False)
        return st_, int(sum(its_))

    # ---------------- device-resident timing (value) ----------------
    for _ in range(max(args.warmup, 3)):
        st, k = step()
    barrier()
    sampler = ClockSampler(gpu_selector(torch))
    if rank == 0:
        sampler.start()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    iters_done, launches = 0, 0
    barrier()
    e0.record(stream)
    for _ in range(args.steps):
        st, k = step()
        iters_done += k
        s = gpu.stats()
        launches += s["loop_launches"] + s["other_launches"]
    e1.record(stream)
    barrier()
    ms = e0.elapsed_time(e1)
    clocks = sampler.stop() if rank == 0 else None
    stats = gpu.stats()
    loop_mode = stats["loop_mode"]

    # ---------------- end to end through the C ABI with host buffers ----------------
    gpu.solve_host(b_host, x_host.zero_(), rtol, maxit, want_hist=False)          # warm (allocates staging)
    barrier()
    t0 = time.perf_counter()
    e2e_iters = 0
    for _ in range(args.steps):
        x_host.zero_()
        st2, k2, _ = gpu.solve_host(b_host, x_host, rtol, maxit, want_hist=False)
        e2e_iters += k2
    barrier()
    e2e_s = time.perf_counter() - t0

    # ---------------- per-kernel durations: CUDA events around each launch (debug library, same source + probes) ----
    from paper_1811_02605_b200.debug import MasPcgProbe
    probe = MasPcgProbe(prob.mesh, dt, prob.nu_kind, prob.nu, prob.bc, options=[o for o in opts if o[0] != "persistent"],
                        precond=args.precond)
    x.zero_()
    prof = probe.profile(b, x, 40, int(stream.cuda_stream))
    pstats = probe.stats()
    # what a trivial linear kernel with the same DRAM read/write mix sustains (context for the rooflines)
    mix = None
    if args.workload == "c4":
        mix = {"k1_mix_ms": probe.mix_probe(pstats["k1_doubles_per_cell"], 100, int(stream.cuda_stream)),
               "k2_mix_ms": probe.mix_probe(3, 100, int(stream.cuda_stream))}
    probe.close()
    barrier()

    ms, iters_all, launches_all = reduce_over_ranks(ms, float(iters_done), float(launches), world)
    e2e_ms, e2e_iters_all, _ = reduce_over_ranks(e2e_s * 1e3, float(e2e_iters), 0.0, world)

    if rank == 0:
        value = iters_all / (ms * 1e-3)
        bpc = stats["bytes_per_cell_iter"] if loop_mode != 2 else pstats["bytes_per_cell_iter"]
        peak, peak_src = hbm_peak()
        k1_bytes, k2_bytes = pstats["k1_doubles_per_cell"] * 8 * n, pstats["k2_doubles_per_cell"] * 8 * n
        k1_gbs = k1_bytes / (prof["k1_ms"] * 1e-3) / 1e9
        k2_gbs = k2_bytes / (prof["k2_ms"] * 1e-3) / 1e9
        k1_name = "k1_tma_noq" if pstats["k1_doubles_per_cell"] == 5 else ("k1_tma_zin" if args.precond == 2 else "k1_tma")
        k2_name = ("k2r_stencil_tma" if pstats["k1_doubles_per_cell"] == 5 else
                   ("k_pc2_line" if args.precond == 2 else "k2_vec"))
        dom = k1_name if prof["k1_ms"] >= prof["k2_ms"] else k2_name
        dom_gbs = k1_gbs if dom == k1_name else k2_gbs
        # the committed capture is of the uniform-phi instantiations on BASELINE.json's mesh; other meshes: not captured
        traffic, traffic_src = ncu_traffic(dom) if args.mesh == "config" else (None, None)
        it_ms = ms / (iters_all / world) if iters_all else float("nan")
        nr_, nt_, np__ = prob.mesh.shape
        line = {
            "metric": (METRIC if args.workload == "c4" else f"fp64_pcg_iterations_per_s_{nr_}x{nt_}x{np__}")
                      + ("" if args.mesh == "config" else f"_{args.mesh}_mesh"),
            "value": value, "unit": UNIT if nrhs == 1 else "rhs-iterations/s", "n_gpus": world, "steps": args.steps,
            "warmup": max(args.warmup, 3), "ms_per_step": ms / args.steps, "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": desc, "parallelism": "replicas only" if world > 1 else "1 gpu",
                       "l2": "inputs larger than L2 (%d live vectors x %.0f MB vs 126 MB)" % (4 * nrhs, 8 * n / 1e6),
                       "loop_mode": {0: "host chunks", 1: "cuda-graph while", 2: "persistent cooperative kernel"}[loop_mode],
                       "bytes_per_cell_iter": bpc, "status": st, "iters_per_step": k, "nrhs": nrhs,
                       "preconditioner": {1: "PC1 point Jacobi", 2: "PC2 block-Jacobi ILU(0), phi-line domains"}[args.precond],
                       "options": dict(opts)},
            "clocks": clocks,
            "e2e": {"value": e2e_iters_all / (e2e_ms * 1e-3), "unit": UNIT,
                    "h2d_bytes_per_step": 2 * 8 * n, "d2h_bytes_per_step": 8 * n},
            "gpu_launches": int(launches_all),
            "roofline": {"bound": "hbm", "kernel": dom, "achieved": dom_gbs, "peak": peak, "unit": "GB/s",
                         "frac": dom_gbs / peak, "traffic": traffic, "traffic_source": traffic_src,
                         "peak_source": peak_src, "frac_of_nominal_8000": dom_gbs / 8000.0},
            "kernels": {k1_name: {"ms": prof["k1_ms"], "min_ms": prof["k1_min_ms"], "alg_bytes": k1_bytes, "gbs": k1_gbs},
                        k2_name: {"ms": prof["k2_ms"], "min_ms": prof["k2_min_ms"], "alg_bytes": k2_bytes, "gbs": k2_gbs}},
            "mix_ceiling": None if mix is None else {
                "what": "trivial linear kernels with the same DRAM mix (K1: r, p, x read; p, x (, q) written; K2: 2 read + "
                        "1 written in place), best grid size, 100 back-to-back launches",
                "k1_mix_gbs": k1_bytes / (mix["k1_mix_ms"] * 1e-3) / 1e9,
                "k2_mix_gbs": k2_bytes / (mix["k2_mix_ms"] * 1e-3) / 1e9,
                "k1_frac_of_mix": mix["k1_mix_ms"] / prof["k1_ms"], "k2_frac_of_mix": mix["k2_mix_ms"] / prof["k2_ms"]},
            "iteration": {"ms": it_ms, "model_gbs": bpc * n / (it_ms * 1e-3) / 1e9,
                          "frac_of_peak": bpc * n / (it_ms * 1e-3) / 1e9 / peak,
                          "frac_of_nominal_8000": bpc * n / (it_ms * 1e-3) / 1e9 / 8000.0,
                          "kernel_sum_ms": prof["k1_ms"] + prof["k2_ms"]},
        }
        if nrhs > 1:
            line["iteration"]["note"] = "per right-hand-side iteration"
        if world == 1 and nrhs == 1 and args.workload == "c4":
            # context beside the headline: the same system solved to rtol 1e-9 with the paper's two preconditioners
            # (PAPER.md:65, 80, 98-100); one warm-up solve and one timed solve each, CUDA events on the launching stream
            tts = {}
            for pc in (1, 2):
                gpu.set_preconditioner(pc)
                for timed in (False, True):
                    x.zero_()
                    torch.cuda.synchronize()
                    e0.record(stream)
                    st_p, k_p, _ = gpu.solve(b, x, 1e-9, 5000, want_hist=False)
                    e1.record(stream)
                    torch.cuda.synchronize()
                tts[f"pc{pc}"] = {"ms": e0.elapsed_time(e1), "iterations": k_p, "status": st_p}
            gpu.set_preconditioner(args.precond)
            tts["pc2_speedup"] = tts["pc1"]["ms"] / tts["pc2"]["ms"]
            tts["what"] = ("the same system solved to rtol 1e-9 from x0 = 0: PC1 point Jacobi vs PC2 block-Jacobi ILU(0) "
                           "over phi-line domains (not part of `value`)")
            line["time_to_solution_rtol_1e-9"] = tts
        if world == 1 and not args.no_cpu_baseline and args.workload == "c3":
            from oracle import ref                      # config 3 = the oracle's FULL solve
            op = ref.RefOperator(prob.mesh, dt, prob.nu_kind, prob.nu, prob.bc)
            t0 = time.perf_counter()
            st_o, k_o, _, _ = op.pcg(b_np, None, rtol, maxit)
            t_o = time.perf_counter() - t0
            op.close()
            line["cpu_baseline"] = {
                "value": k_o / t_o, "unit": UNIT, "cores": 1, "kind": "oracle",
                "sample": f"full solve of the same workload: {k_o} iterations (GPU {k}) in {t_o:.1f} s including setup "
                          f"and the initial residual, one thread of {os.cpu_count()} host cores, gcc -O2"}
        elif world == 1 and not args.no_cpu_baseline:
            nit = CPU_BASELINE_ITERS if args.workload in ("c4", "c5") else 40
            t_a, _ = time_oracle(prob, dt, b_np, 2)
            t_b, _ = time_oracle(prob, dt, b_np, 2 + nit)
            line["cpu_baseline"] = {
                "value": nit / max(t_b - t_a, 1e-9), "unit": UNIT, "cores": 1, "kind": "oracle",
                "sample": f"{nit} steady-state PCG iterations of the same workload (time of {2 + nit} "
                          f"iterations minus time of 2), one thread of {os.cpu_count()} host cores, gcc -O2"}
        print(json.dumps(line), flush=True)
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
