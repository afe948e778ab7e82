#!/usr/bin/env python
"""bench.py -- one JSON line for the Soft-DTW barycenter hot path on B200 (contract: see DESIGN.md section 8).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--config 4]

A "step" is one pass of the whole hot path over one batch of synthetic input: forward wavefront, checkpointing,
reverse wavefront + gradient contraction, reduction over pairs and the descent update -- i.e. one barycenter
iteration on BASELINE.json's configs[3] ("Full-length robot cycles", N = 100 cycles of 27-33k samples against
m = 30000, gamma = 0.01), the configuration the metric ("... at Nx30k") is quoted on.  value = DP cells/s
(sum_k n_k * m per step, counted once however much is recomputed), whole job, inputs resident in HBM.

N > 1 (torchrun, one rank per GPU): weak scaling -- every rank owns its own 100 cycles (seed + rank), Z is
replicated, and the only exchange is one NCCL all-reduce of the m*d gradient per step (dist.py).

--impl reference times the float64 CPU oracle (oracle/) on the box's host cores on a bounded sample of the same
workload; it is a deliberately plain program, reported as a baseline, not a target.
"""
from __future__ import annotations

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

from paper_2404_12134_b200 import synth  # noqa: E402

METRIC = "sdtw_fwd_bwd_dp_cells_per_s"
UNIT = "cells/s"
# roofline constants: MUFU (ex2/lg2/rcp) results per clock per SM on sm_100, SM count, max clock
MUFU_PER_CLK_PER_SM = 16
ALGO_MUFU_FWD, ALGO_MUFU_BWD = 3, 3          # algorithmic special-function evaluations per cell (2 ex2 + lg2; 3 ex2)
# dram__bytes_read.sum + dram__bytes_write.sum of ONE launch of the named kernel at the named config, from the
# ncu --set full capture summarised in profiles/ (null for workloads without a capture)
NCU_TRAFFIC_BYTES_PER_LAUNCH = {("forward_kernel", 4): 2563222000 + 36700025000}   # profiles/r1e_forward_kernel_cfg4_full.txt


def workload_string(cfg):
    return (f"configs[{cfg.index - 1}] {cfg.name}: N={cfg.N} cycles/GPU, n_k~U[{cfg.n_lo},{cfg.n_hi}], m={cfg.m}, d={cfg.d}, "
            f"gamma={cfg.gamma}, fixed-step GD step={cfg.step}")


# ---------------------------------------------------------------------------------------------- clocks sampling
class ClockSampler:
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.index, self.proc, self.lines = index, None, []

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", f"--id={self.index}", f"--query-gpu={self.Q}",
                                          "--format=csv,noheader,nounits", "-lms", "200"], stdout=subprocess.PIPE, text=True)
            threading.Thread(target=self._pump, daemon=True).start()
        except OSError:
            self.proc = None

    def _pump(self):
        for line in self.proc.stdout:
            self.lines.append(line.strip())

    def stop(self):
        if not self.proc:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        self.proc.terminate()
        sm, mx, reasons = [], [], set()
        if not self.lines:                      # timed region shorter than the sampling period: one sample right after it
            try:
                out = subprocess.run(["nvidia-smi", f"--id={self.index}", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits"],
                                     capture_output=True, text=True, timeout=20).stdout
                self.lines = [l.strip() for l in out.splitlines() if l.strip()]
            except (OSError, subprocess.SubprocessError):
                pass
        for ln in self.lines:
            f = [x.strip() for x in ln.split(",")]
            if len(f) < 7:
                continue
            try:
                sm.append(float(f[0])); mx.append(float(f[1]))
            except ValueError:
                continue
            for name, v in zip(("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"), f[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(name)
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "reasons": sorted(reasons), "samples": len(sm)}


# ---------------------------------------------------------------------------------------------- oracle legs
def oracle_sample(data, cores):
    """Bounded sample of the workload for the CPU legs: the first 2*cores cycles cut to their first 6000 samples,
    against the first 6000 points of Z0 (same generator, same gamma; ~3.6e7 cells per pair)."""
    cfg = data["cfg"]
    P = min(cfg.N, 2 * cores)
    L = min(6000, cfg.m)
    chunks = [data["X"][data["offsets"][k]:data["offsets"][k] + min(L, data["lengths"][k])] for k in range(P)]
    off = np.zeros(P + 1, np.int64)
    np.cumsum([c.shape[0] for c in chunks], out=off[1:])
    X = np.ascontiguousarray(np.concatenate(chunks))
    Z = np.ascontiguousarray(data["Z0"][:L])
    return Z, X, off, int(off[-1]) * L, f"first {P} cycles cut to {L} samples vs Z0[:{L}], value+gradient, float64"


def time_oracle(data, reps=1):
    import oracle
    cores = os.cpu_count() or 1
    Z, X, off, ncells, what = oracle_sample(data, cores)
    best = None
    for _ in range(reps):
        t = time.perf_counter()
        oracle.value_grad(Z, X, off, data["cfg"].gamma, mode="checkpointed", nthreads=cores)
        dt = time.perf_counter() - t
        best = dt if best is None else min(best, dt)
    return {"value": ncells / best, "unit": UNIT, "cores": min(cores, oracle.num_threads()), "kind": "oracle",
            "sample": what, "seconds": best}


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    data = synth.make(args.config)
    cfg = data["cfg"]
    import oracle
    cores = os.cpu_count() or 1
    Z, X, off, ncells, what = oracle_sample(data, cores)
    for _ in range(args.warmup):
        oracle.value_grad(Z, X, off, cfg.gamma, mode="checkpointed", nthreads=cores)
    t = time.perf_counter()
    for _ in range(args.steps):
        oracle.value_grad(Z, X, off, cfg.gamma, mode="checkpointed", nthreads=cores)
    dt = (time.perf_counter() - t) / max(args.steps, 1)
    val = ncells / dt
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": dt * 1e3, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f64", "data": "synthetic", "config": {"workload": workload_string(cfg), "sample_per_step": what},
        "cpu_baseline": {"value": val, "unit": UNIT, "cores": min(cores, oracle.num_threads()), "kind": "oracle", "sample": what},
        "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }))


# ---------------------------------------------------------------------------------------------- our arm
def run_ours(args):
    import torch
    import torch.distributed as dist
    from paper_2404_12134_b200 import binding as B
    from paper_2404_12134_b200.dist import allreduce_sum_

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: there is no CPU fallback (use --impl reference for the oracle)")
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    dev = torch.device("cuda", local)

    base = synth.CONFIGS[args.config]
    data = synth.make(base, seed=synth.BASE_SEED + base.index + 1000 * rank)     # rank 0 == the canonical draw
    cfg = data["cfg"]
    ncells_local = synth.cells(data)
    Z0 = torch.from_numpy(data["Z0"]).to(dev)
    X = torch.from_numpy(data["X"]).to(dev)
    offsets = data["offsets"]
    forward_only = cfg.iters == 0
    ws_bytes = B.sdtw_workspace_bytes(cfg.m, cfg.d, offsets, not forward_only)

    Z = Z0.clone()
    G = torch.empty_like(Z)
    vals = torch.empty(cfg.N, dtype=torch.float32, device=dev)
    obj = torch.zeros(1, dtype=torch.float32, device=dev)

    def step():
        if forward_only:
            B.sdtw_value_grad(Z, X, offsets, cfg.gamma, out_values=vals, want_grad=False)
        elif world == 1:
            B.sdtw_barycenter(Z, X, offsets, cfg.gamma, 1, cfg.step, out_values=vals, out_objective=obj)
        else:
            B.sdtw_value_grad(Z, X, offsets, cfg.gamma, out_values=vals, out_grad=G)
            allreduce_sum_(G)
            B.sdtw_gd_update(Z, G, cfg.step)

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    for _ in range(args.warmup):
        step()
    barrier()
    Z.copy_(Z0)                                    # time the first K iterations of the configured descent
    B.sdtw_profile_enable(True)
    B.sdtw_profile_read()
    sampler = ClockSampler(local)
    sampler.start()
    launches0 = B.sdtw_launch_count()
    barrier()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    for _ in range(args.steps):
        step()
    e1.record()
    barrier()
    ms_total = e0.elapsed_time(e1)
    launches = B.sdtw_launch_count() - launches0
    prof = B.sdtw_profile_read()
    B.sdtw_profile_enable(False)
    clocks = sampler.stop()
    t = torch.tensor([ms_total], dtype=torch.float64, device=dev)
    if world > 1:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
    ms_total = float(t.item())
    cells_total = torch.tensor([float(ncells_local)], dtype=torch.float64, device=dev)
    if world > 1:
        dist.all_reduce(cells_total, op=dist.ReduceOp.SUM)
    cells_job = float(cells_total.item())
    ms_step = ms_total / args.steps
    value = cells_job / (ms_step * 1e-3)

    # ---- end to end: HOST buffers in, HOST results out, every step (C-ABI host entry point at N = 1)
    e2e = None
    if not args.skip_e2e:
        Xh = torch.from_numpy(data["X"]).pin_memory()
        Zh = torch.from_numpy(data["Z0"].copy()).pin_memory()
        objh = torch.zeros(1, dtype=torch.float32).pin_memory()
        valh = torch.zeros(cfg.N, dtype=torch.float32).pin_memory()
        e2e_steps = max(1, min(args.steps, 3))

        def e2e_step():
            if world == 1 and not forward_only:
                B.sdtw_barycenter_host(Zh, Xh, offsets, cfg.gamma, 1, cfg.step, valh, objh,
                                       stream=torch.cuda.current_stream().cuda_stream)
            elif world == 1:
                B.sdtw_value_grad_host(Zh, Xh, offsets, cfg.gamma, valh, None, stream=torch.cuda.current_stream().cuda_stream)
            else:
                X.copy_(Xh, non_blocking=True)
                Z.copy_(Zh, non_blocking=True)
                step()
                Zh.copy_(Z, non_blocking=True)
                valh.copy_(vals, non_blocking=True)
                torch.cuda.synchronize()

        e2e_step()
        barrier()
        t0 = time.perf_counter()
        for _ in range(e2e_steps):
            e2e_step()
        barrier()
        t_e2e = torch.tensor([(time.perf_counter() - t0) / e2e_steps], dtype=torch.float64, device=dev)
        if world > 1:
            dist.all_reduce(t_e2e, op=dist.ReduceOp.MAX)
        e2e_val = cells_job / float(t_e2e.item())
        h2d = int(Xh.numel() * 4 + Zh.numel() * 4)
        d2h = int(valh.numel() * 4 + (0 if forward_only else Zh.numel() * 4 + 4))
        e2e = {"value": e2e_val, "unit": UNIT, "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h,
               "steps": e2e_steps, "api": "sdtw_barycenter_host" if world == 1 and not forward_only else
               ("sdtw_value_grad_host" if world == 1 else "pinned copies + sdtw_value_grad + all_reduce + sdtw_gd_update")}

    # ---- measured special-function issue rate of this device (the roofline denominator)
    mufu = {}
    if rank == 0:
        for kind, name in ((0, "ex2"), (1, "lg2"), (2, "rcp")):
            mufu[name], _ = B.sdtw_measure_mufu_peak(kind)

    if rank == 0:
        sm_max_hz = (clocks.get("sm_max_mhz") or 1965.0) * 1e6
        sms = torch.cuda.get_device_properties(local).multi_processor_count
        mufu_peak = MUFU_PER_CLK_PER_SM * sms * sm_max_hz
        n_eval = max(prof["evaluations"], 1)
        t_fwd, t_bwd = prof["ms_forward"] / n_eval * 1e-3, prof["ms_backward"] / n_eval * 1e-3
        # the dominant kernel is the one with the longest measured duration (the reverse kernel skips chunks whose
        # incoming E flow is +0, so it usually is the forward kernel)
        if forward_only or t_bwd <= t_fwd:
            dom, t_dom, algo = "forward_kernel", t_fwd, ALGO_MUFU_FWD
        else:
            dom, t_dom, algo = "backward_kernel", t_bwd, ALGO_MUFU_BWD
        achieved = algo * ncells_local / t_dom
        algo_total = ALGO_MUFU_FWD + (0 if forward_only else ALGO_MUFU_BWD)
        roofline = {
            "bound": "alu", "kernel": dom, "achieved": achieved / 1e9, "peak": mufu_peak / 1e9, "unit": "GMUFU-op/s",
            "frac": achieved / mufu_peak,
            "traffic": NCU_TRAFFIC_BYTES_PER_LAUNCH.get((dom, args.config)) if world == 1 else None,
            "algorithmic_bytes": None if forward_only else int(ncells_local * 0.375 + ncells_local * 4 / 128),
            "peak_source": f"derived: {MUFU_PER_CLK_PER_SM} MUFU results/clk/SM x {sms} SMs x {sm_max_hz / 1e6:.0f} MHz (clocks.max.sm); "
                           "MEASURED_PEAKS.json holds no ALU figure (DESIGN.md section 8)",
            "mufu_measured_gops": {k: v / 1e9 for k, v in mufu.items()},
            "algorithmic_per_cell": {"forward": ALGO_MUFU_FWD, "reverse": ALGO_MUFU_BWD},
            "note": "achieved counts the special-function evaluations the method needs (3 per forward cell); the forward "
                    "kernel issues 2.625 of them on the MUFU pipe and evaluates 3 in 8 of the second exponentials with "
                    "an FMA-pipe polynomial, so frac can exceed the MUFU-only bound (DESIGN.md 5.2)",
            "kernel_ms": {"forward": t_fwd * 1e3, "reverse": t_bwd * 1e3, "other": prof["ms_other"] / n_eval},
            "forward_frac": (ALGO_MUFU_FWD * ncells_local / t_fwd) / mufu_peak if t_fwd > 0 else None,
            "step_frac_of_cell_rate_roofline": (value / world) / (mufu_peak / algo_total),
            "checkpoint_hbm_gbs": None if forward_only else
                (2 * ws_bytes) / max(t_fwd + t_bwd, 1e-9) / 1e9,
        }
        cpu = None if args.skip_cpu else time_oracle(data)
        out = {
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
            "ms_per_step": ms_step, "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f32",
            "data": "synthetic",
            "config": {"workload": workload_string(cfg), "cells_per_step": cells_job, "workspace_gb": ws_bytes / 1e9,
                       "l2": ("no flush: every step streams its checkpoints (workspace) through HBM, far above the 126 MB L2"
                              if ws_bytes > 4 * 126e6 else
                              "no flush: small configuration, the working set fits in the 126 MB L2 (latency-bound; not a roofline case)"),
                       "parallelism": f"pairs sharded over {world} GPU(s); all-reduce of m*d gradient" if world > 1 else "single GPU",
                       "tile": B.sdtw_tile_info()},
            "barycenter_iter_s": ms_step * 1e-3,
            "roofline": roofline, "cpu_baseline": cpu,
            "e2e": e2e,
            "gpu_launches": int(launches), "clocks": clocks,
        }
        print(json.dumps(out))
    if world > 1:
        dist.barrier()
        dist.destroy_process_group()


# ---------------------------------------------------------------------------------------------- Step-3 scoring arm
def run_score(args):
    """--op score: sdtw_dtw_score (eq. 8: DTW, |pi|, d_score) over one batch; default workload = configs[4], the scoring
    sweep.  Extra to the headline line; same JSON shape.  Bound: instruction issue (no special functions): the method
    needs 8 thread-instructions per cell at d = 1 (x - z, square, min of three, add, two compares, select, increment)."""
    import torch
    from paper_2404_12134_b200 import binding as B
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if world > 1 and rank != 0:
        return                                     # replicas only: pairs are independent, nothing to exchange
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: there is no CPU fallback")
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    data = synth.make(args.config)
    cfg = data["cfg"]
    cells = synth.cells(data)
    Z = torch.from_numpy(data["Z0"]).to(dev)
    X = torch.from_numpy(data["X"]).to(dev)
    for _ in range(args.warmup):
        B.sdtw_dtw_score(Z, X, data["offsets"])
    torch.cuda.synchronize()
    sampler = ClockSampler(local)
    sampler.start()
    n0 = B.sdtw_launch_count()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    for _ in range(args.steps):
        out = B.sdtw_dtw_score(Z, X, data["offsets"])
    e1.record()
    torch.cuda.synchronize()
    ms = e0.elapsed_time(e1) / args.steps
    launches = B.sdtw_launch_count() - n0
    clocks = sampler.stop()
    # end to end: pinned host inputs -> device -> results back on the host, every step
    Xh, Zh = torch.from_numpy(data["X"]).pin_memory(), torch.from_numpy(data["Z0"]).pin_memory()
    t0 = time.perf_counter()
    nrep = max(1, min(args.steps, 3))
    for _ in range(nrep):
        X.copy_(Xh, non_blocking=True); Z.copy_(Zh, non_blocking=True)
        res = [t.cpu() for t in B.sdtw_dtw_score(Z, X, data["offsets"])]
    t_e2e = (time.perf_counter() - t0) / nrep
    sm_max_hz = (clocks.get("sm_max_mhz") or 1965.0) * 1e6
    sms = torch.cuda.get_device_properties(local).multi_processor_count
    algo = 6 + 2 * cfg.d                            # thread-instructions per cell the recurrence needs
    peak = 128.0 * sms * sm_max_hz
    import oracle
    cores = os.cpu_count() or 1
    Zs, Xs, off, ncs, what = oracle_sample(data, cores)
    t = time.perf_counter()
    oracle.dtw_score(Zs, Xs, off, nthreads=cores)
    t_cpu = time.perf_counter() - t
    print(json.dumps({
        "metric": "dtw_score_dp_cells_per_s", "value": cells / (ms * 1e-3), "unit": UNIT, "n_gpus": 1, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": ms, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f32", "data": "synthetic",
        "config": {"workload": workload_string(cfg) + "; op = sdtw_dtw_score (eq. 8)", "cells_per_step": cells,
                   "l2": "no flush: inputs + strip-boundary columns exceed the 126 MB L2" if cells > 1e10 else "no flush (small)"},
        "roofline": {"bound": "alu", "kernel": "dtw_kernel", "achieved": algo * cells / (ms * 1e-3) / 1e9, "peak": peak / 1e9,
                     "unit": "Gthread-instr/s", "frac": algo * cells / (ms * 1e-3) / peak, "traffic": None,
                     "peak_source": f"derived: 128 thread-instructions/clk/SM (4 schedulers x 32 lanes) x {sms} SMs x {sm_max_hz / 1e6:.0f} MHz",
                     "algorithmic_per_cell": algo},
        "cpu_baseline": {"value": ncs / t_cpu, "unit": UNIT, "cores": min(cores, oracle.num_threads()), "kind": "oracle",
                         "sample": what.replace("value+gradient, float64", "DTW + path length, float32 decisions")},
        "e2e": {"value": cells / t_e2e, "unit": UNIT, "h2d_bytes_per_step": int(Xh.numel() * 4 + Zh.numel() * 4),
                "d2h_bytes_per_step": int(cfg.N * 12), "steps": nrep, "api": "pinned copies + sdtw_dtw_score + .cpu()"},
        "gpu_launches": int(launches), "clocks": clocks,
    }))


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", choices=["ours", "reference"], default="ours")
    ap.add_argument("--config", type=int, default=4, choices=[1, 2, 3, 4, 5])
    ap.add_argument("--op", choices=["barycenter", "score"], default="barycenter",
                    help="score = the Step-3 d_score kernel (extra; the headline is barycenter)")
    ap.add_argument("--skip-e2e", action="store_true", help="profiling runs only: leave out the host-buffer leg")
    ap.add_argument("--skip-cpu", action="store_true", help="profiling runs only: leave out the timed oracle leg")
    args = ap.parse_args()
    if args.impl == "reference":
        run_reference(args)
    elif args.op == "score":
        run_score(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
