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

from paper_2404_12134_b200 import paper_setup, synth  # noqa: E402

METRIC = "sdtw_fwd_bwd_dp_cells_per_s"
UNIT = "cells/s"
# roofline constants: MUFU (ex2/lg2/rcp) results per clock per SM on sm_100, SM count, max clock
MUFU_PER_CLK_PER_SM = 16
ALGO_MUFU_FWD, ALGO_MUFU_BWD = 3, 3          # algorithmic special-function evaluations per cell (2 ex2 + lg2; 3 ex2)
PROFILE_ROUNDS = ("r3", "r2", "r1e")          # newest first: profiles/<round>_<kernel>_cfg<idx>[_<variant>]_full.txt
STALE_TOL = 0.05                              # a capture whose kernel time differs from this run's by more is not used


def ncu_traffic(kernel, cfg_index, variant="", kernel_ms=None):
    """dram__bytes_read.sum + dram__bytes_write.sum of ONE launch of `kernel` on config `cfg_index`, read from the
    header of the committed `ncu --set full` summary under profiles/ (the "# raw:" lines).  The capture is tied to the
    kernel that was timed by its own gpu__time_duration: if that differs from this run's CUDA-event time of the kernel
    (`kernel_ms`) by more than STALE_TOL, the kernel has changed since the capture and the file is refused.
    Returns (bytes or None, path or None, note)."""
    note = "no committed capture of this kernel / workload"
    for rnd in PROFILE_ROUNDS:
        path = os.path.join(ROOT, "profiles", f"{rnd}_{kernel}_cfg{cfg_index}{'_' + variant if variant else ''}_full.txt")
        if not os.path.exists(path):
            continue
        tot, seen, dur, commit = 0.0, 0, None, None
        for ln in open(path):
            f = ln.split()
            if len(f) == 5 and f[:2] == ["#", "raw:"] and f[2] in ("dram__bytes_read.sum", "dram__bytes_write.sum"):
                tot += float(f[4]) * {"Gbyte": 1e9, "Mbyte": 1e6, "Kbyte": 1e3, "byte": 1.0}[f[3]]
                seen += 1
            if len(f) == 5 and f[:3] == ["#", "raw:", "gpu__time_duration.sum"]:
                dur = float(f[4]) * {"s": 1e3, "ms": 1.0, "us": 1e-3, "ns": 1e-6}.get(f[3], float("nan"))
            if len(f) >= 3 and f[:2] == ["#", "commit:"]:
                commit = f[2]
        rel = os.path.relpath(path, ROOT)
        if seen != 2:
            continue
        if kernel_ms is not None and dur is not None and abs(dur - kernel_ms) > STALE_TOL * kernel_ms:
            note = f"{rel} refused: its launch took {dur:.2f} ms, this run's {kernel_ms:.2f} ms (kernel changed since the capture)"
            continue
        return int(tot), rel, (f"capture at commit {commit}, " if commit else "") + (
            f"launch {dur:.2f} ms under ncu vs {kernel_ms:.2f} ms here" if dur is not None and kernel_ms is not None else "duration not recorded")
    return None, None, note


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
    P = min(len(data["lengths"]), 2 * cores)
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
    out = {"value": ncells / best, "unit": UNIT, "cores": min(cores, oracle.num_threads()), "kind": "oracle",
           "sample": what, "seconds": best}
    # the same oracle at FULL length (row-checkpointed mode, the one the full-size references are made with): one
    # whole cycle per core against the whole Z0, forward recurrence only (value), so that the leg stays near 30 s
    cfg = data["cfg"]
    if cfg.m >= 20000:
        P = min(len(data["lengths"]), cores)
        off = data["offsets"]
        t = time.perf_counter()
        oracle.value_grad(data["Z0"], data["X"][:off[P]], off[:P + 1], cfg.gamma, want_grad=False, mode="checkpointed",
                          nthreads=cores)
        dt = time.perf_counter() - t
        out["full_length"] = {"value": float(off[P]) * cfg.m / dt, "unit": "forward cells/s", "seconds": dt,
                              "sample": f"first {P} whole cycles vs the whole Z0 (m = {cfg.m}), value only, float64"}
    return out


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


# ---------------------------------------------------------------------------------------------- secondary workloads
def measure_secondary(B, torch, dev, data4, mufu_peak, sms, sm_max_hz):
    """The other workloads BASELINE.md section 5 quotes, measured in this process after the headline region (device-
    resident inputs, CUDA events, one warm-up pass each; kernel times from the library's own event brackets):
    cfg 5 forward-only scoring sweep, cfg 3 descent, cfg 4 with the dense reverse pass, cfg 5 d_score."""
    def timed(fn, reps):
        fn()                                                    # warm-up (first call of a shape also uploads its plan)
        torch.cuda.synchronize()
        B.sdtw_profile_enable(True)
        B.sdtw_profile_read()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        for _ in range(reps):
            fn()
        e1.record()
        torch.cuda.synchronize()
        prof = B.sdtw_profile_read()
        B.sdtw_profile_enable(False)
        n = max(prof["evaluations"], 1)
        return e0.elapsed_time(e1) / reps, {"forward": prof["ms_forward"] / n, "reverse": prof["ms_backward"] / n,
                                            "other": prof["ms_other"] / n}

    def up(a):
        return torch.from_numpy(a).to(dev)

    out = {"note": "measured after the headline region in the same process; 1 warm-up + the stated repetitions; "
                   "frac = algorithmic special functions (3 per forward cell, 3 per reverse cell) / kernel time / MUFU peak"}
    # cfg 5: forward-only scoring sweep (rings)
    d5 = synth.make(5)
    c5, cells5 = d5["cfg"], synth.cells(d5)
    Z5, X5 = up(d5["Z0"]), up(d5["X"])
    v5 = torch.empty(c5.N, dtype=torch.float32, device=dev)
    ms, k = timed(lambda: B.sdtw_value_grad(Z5, X5, d5["offsets"], c5.gamma, out_values=v5, want_grad=False), 2)
    out["cfg5_forward_only"] = {"workload": workload_string(c5), "reps": 2, "ms_per_step": ms, "value": cells5 / (ms * 1e-3),
                                "unit": UNIT, "kernel_ms": k, "forward_frac": ALGO_MUFU_FWD * cells5 / (k["forward"] * 1e-3) / mufu_peak,
                                "workspace_gb": B.sdtw_workspace_bytes(c5.m, c5.d, d5["offsets"], False) / 1e9,
                                "finite": bool(torch.isfinite(v5).all().item())}
    # cfg 5: d_score (eq. 8), the DTW kernel; bound = instruction issue
    ms, _ = timed(lambda: B.sdtw_dtw_score(Z5, X5, d5["offsets"]), 2)
    algo = 6 + 2 * c5.d
    out["cfg5_dtw_score"] = {"workload": workload_string(c5) + "; op = sdtw_dtw_score (eq. 8)", "reps": 2, "ms_per_step": ms,
                             "value": cells5 / (ms * 1e-3), "unit": UNIT,
                             "frac": algo * cells5 / (ms * 1e-3) / (128.0 * sms * sm_max_hz),
                             "frac_note": f"{algo} thread-instructions per cell the recurrence needs / (128 per clk per SM x {sms} SMs x "
                                          f"{sm_max_hz / 1e6:.0f} MHz)"}
    del Z5, X5
    # cfg 3: the configured descent (10 iterations, d = 4)
    d3 = synth.make(3)
    c3, cells3 = d3["cfg"], synth.cells(d3)
    Z30, X3 = up(d3["Z0"]), up(d3["X"])
    Z3 = Z30.clone()

    def cfg3_descent():
        Z3.copy_(Z30)
        B.sdtw_barycenter(Z3, X3, d3["offsets"], c3.gamma, c3.iters, c3.step)
    ms, k = timed(cfg3_descent, 2)
    out["cfg3"] = {"workload": workload_string(c3), "reps": 2, "ms_per_step": ms / c3.iters, "value": cells3 / (ms / c3.iters * 1e-3),
                   "unit": UNIT, "kernel_ms": k, "forward_frac": ALGO_MUFU_FWD * cells3 / (k["forward"] * 1e-3) / mufu_peak,
                   "finite": bool(torch.isfinite(Z3).all().item()),
                   "note": "few pairs (32) of 10k: a latency chain per pair, not a throughput case (DESIGN.md 5.4)"}
    # cfg 4 with the dense reverse pass (every reverse cell visited: backward_kernel)
    c4, cells4 = data4["cfg"], synth.cells(data4)
    Z40, X4 = up(data4["Z0"]), up(data4["X"])
    Z4 = Z40.clone()
    B.sdtw_set_reverse_mode(True)
    try:
        def cfg4_dense():
            Z4.copy_(Z40)
            B.sdtw_barycenter(Z4, X4, data4["offsets"], c4.gamma, 1, c4.step)
        ms, k = timed(cfg4_dense, 2)
    finally:
        B.sdtw_set_reverse_mode(False)
    out["cfg4_reverse_dense"] = {"workload": workload_string(c4) + "; reverse pass visits every cell", "reps": 2, "ms_per_step": ms,
                                 "value": cells4 / (ms * 1e-3), "unit": UNIT, "kernel_ms": k,
                                 "forward_frac": ALGO_MUFU_FWD * cells4 / (k["forward"] * 1e-3) / mufu_peak,
                                 "reverse_frac": ALGO_MUFU_BWD * cells4 / (k["reverse"] * 1e-3) / mufu_peak,
                                 "step_frac": (ALGO_MUFU_FWD + ALGO_MUFU_BWD) * cells4 / (ms * 1e-3) / mufu_peak}
    return out


# ---------------------------------------------------------------------------------------------- our arm
def table3_config(pairs):
    """The shape of the paper's Table 3 (Table 1): `pairs` univariate cycles of
    up to 18385 samples against a barycenter of 18385 points, gamma = 1, Sakoe-Chiba band 0.6, eq. 7 weights."""
    from dataclasses import replace
    return replace(synth.CONFIGS[4], name=f"table3_N{pairs}", N=pairs, n_lo=16500, n_hi=18385, m=18385, gamma=1.0,
                   iters=1, step=0.0)


def run_ours(args):
    import torch
    import torch.distributed as dist
    from dataclasses import replace
    from paper_2404_12134_b200 import binding as B
    from paper_2404_12134_b200 import dist as D

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: there is no CPU fallback (use --impl reference for the oracle)")
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    dev = torch.device("cuda", local)

    table3 = args.shape == "table3"
    base = table3_config(args.pairs) if table3 else synth.CONFIGS[args.config]
    if args.gamma is not None:
        base = replace(base, gamma=float(args.gamma))
    strong = args.scaling == "strong" and world > 1
    # weak scaling: every rank draws its own cycles (rank 0 = the canonical draw); strong scaling: ONE problem (the
    # canonical draw), its pairs partitioned over the ranks by dist.partition_pairs
    data = synth.make(base, seed=synth.BASE_SEED + base.index + (0 if strong else 1000 * rank))
    cfg = data["cfg"]
    if strong:
        mine = D.partition_pairs(data["lengths"], world)[rank]
        Xl, offl = D.take_pairs(data["X"], data["offsets"], mine)
        data = dict(data, X=Xl, offsets=offl, lengths=data["lengths"][mine])
    ncells_local = synth.cells(data)
    Z0 = torch.from_numpy(data["Z0"]).to(dev)
    X = torch.from_numpy(data["X"]).to(dev)
    offsets = data["offsets"]
    Nl = len(offsets) - 1
    forward_only = cfg.iters == 0
    iters_cfg = max(cfg.iters, 1)
    ws_bytes = B.sdtw_workspace_bytes(cfg.m, cfg.d, offsets, not forward_only)
    dense = args.reverse == "dense"
    B.sdtw_set_reverse_mode(dense)
    if table3:
        weights = paper_setup.eq7_weights(data["lengths"])
        band = paper_setup.table1_band(cfg.m, data["lengths"])

    Z = Z0.clone()
    G = torch.empty_like(Z)
    vals = torch.empty(Nl, dtype=torch.float32, device=dev)
    obj_hist = torch.zeros(max(args.steps, args.warmup, 1), dtype=torch.float32, device=dev)

    def run_steps(count):
        """`count` steps.  A step = one pass of the hot path; for the descent configs the steps are the iterations of
        the CONFIGURED descent (cfg.iters iterations from Z0 at cfg.step), restarted from Z0 when it is complete."""
        done = 0
        while done < count:
            if forward_only:
                B.sdtw_value_grad(Z, X, offsets, cfg.gamma, out_values=vals, want_grad=False)
                k = 1
            elif table3:
                B.sdtw_value_grad_ex(Z, X, offsets, cfg.gamma, weights=weights, band=band, out_values=vals, out_grad=G)
                k = 1
            else:
                k = min(iters_cfg, count - done)
                Z.copy_(Z0)
                if world == 1:
                    B.sdtw_barycenter(Z, X, offsets, cfg.gamma, k, cfg.step, out_values=vals, out_objective=obj_hist[done:done + k])
                else:
                    for _ in range(k):
                        B.sdtw_value_grad(Z, X, offsets, cfg.gamma, out_values=vals, out_grad=G)
                        D.allreduce_sum_(G)
                        B.sdtw_gd_update(Z, G, cfg.step)
            done += k

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    run_steps(args.warmup)
    barrier()
    B.sdtw_profile_enable(True)
    B.sdtw_profile_read()
    sampler = ClockSampler(local)
    sampler.start()
    launches0 = B.sdtw_launch_count()
    barrier()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    run_steps(args.steps)
    e1.record()
    barrier()
    ms_total = e0.elapsed_time(e1)
    launches = B.sdtw_launch_count() - launches0
    prof = B.sdtw_profile_read()
    rev_chunks, rev_skipped = B.sdtw_reverse_stats() if not forward_only else (0, 0)
    B.sdtw_profile_enable(False)
    clocks = sampler.stop()
    # what was timed stayed finite (the step passed the contractivity check of tests/golden/make_fullsize_refs.py)
    finite = bool(torch.isfinite(Z).all().item() and torch.isfinite(vals).all().item())
    if not finite:
        raise SystemExit("bench.py: non-finite barycenter or values after the timed steps")
    objective = obj_hist[:min(args.steps, iters_cfg)].cpu().tolist() if not (forward_only or table3 or world > 1) else None
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
        Gh = torch.zeros_like(Zh).pin_memory()
        objh = torch.zeros(1, dtype=torch.float32).pin_memory()
        valh = torch.zeros(Nl, dtype=torch.float32).pin_memory()
        e2e_steps = max(1, args.steps)
        cur = torch.cuda.current_stream().cuda_stream

        def e2e_step(i):
            if world == 1 and not forward_only and not table3:
                if i % iters_cfg == 0:
                    Zh.copy_(torch.from_numpy(data["Z0"]))
                B.sdtw_barycenter_host(Zh, Xh, offsets, cfg.gamma, 1, cfg.step, valh, objh, stream=cur)
            elif world == 1 and forward_only:
                B.sdtw_value_grad_host(Zh, Xh, offsets, cfg.gamma, valh, None, stream=cur)
            else:
                X.copy_(Xh, non_blocking=True)
                Z.copy_(Zh, non_blocking=True)
                if table3:
                    run_steps(1)
                    Gh.copy_(G, non_blocking=True)
                else:
                    B.sdtw_value_grad(Z, X, offsets, cfg.gamma, out_values=vals, out_grad=G)
                    D.allreduce_sum_(G)
                    B.sdtw_gd_update(Z, G, cfg.step)
                    Zh.copy_(Z, non_blocking=True)
                valh.copy_(vals, non_blocking=True)
                torch.cuda.synchronize()

        e2e_step(0)
        barrier()
        t0 = time.perf_counter()
        for i in range(e2e_steps):
            e2e_step(i)
        barrier()
        t_e2e = torch.tensor([(time.perf_counter() - t0) / e2e_steps], dtype=torch.float64, device=dev)
        if world > 1:
            dist.all_reduce(t_e2e, op=dist.ReduceOp.MAX)
        e2e_val = cells_job / float(t_e2e.item())
        h2d = int(Xh.numel() * 4 + Zh.numel() * 4)
        d2h = int(valh.numel() * 4 + (0 if forward_only else Zh.numel() * 4 + 4))
        e2e = {"value": e2e_val, "unit": UNIT, "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h,
               "steps": e2e_steps, "api": "sdtw_barycenter_host" if world == 1 and not forward_only and not table3 else
               ("sdtw_value_grad_host" if world == 1 and forward_only else
                "pinned copies + sdtw_value_grad(_ex) (+ all_reduce + sdtw_gd_update)")}

    # ---- measured special-function issue rate of this device (the roofline denominator)
    mufu = {}
    if rank == 0:
        for kind, name in ((0, "ex2"), (1, "lg2"), (2, "rcp")):
            mufu[name], _ = B.sdtw_measure_mufu_peak(kind)

    if rank == 0:
        sm_max_hz = (clocks.get("sm_max_mhz") or 1965.0) * 1e6
        sms = torch.cuda.get_device_properties(local).multi_processor_count
        mufu_derived = MUFU_PER_CLK_PER_SM * sms * sm_max_hz
        mufu_peak = min(mufu.values())                 # live: dependent ex2 / lg2 / rcp chains on every SM (mufu_peak.cu)
        n_eval = max(prof["evaluations"], 1)
        t_fwd, t_bwd = prof["ms_forward"] / n_eval * 1e-3, prof["ms_backward"] / n_eval * 1e-3
        # reverse pass: cells it visited (a visited (strip, chunk) unit = 32 steps x 32 lanes x 2 x 4 cells; the other
        # units carry E = +0 exactly and are skipped)
        tile = B.sdtw_tile_info()
        cells_per_chunk = tile["chunk_steps"] * 32 * tile["rows_per_step"] * tile["cols_per_thread"]
        visited_cells = (rev_chunks - rev_skipped) * cells_per_chunk
        reverse = None
        if not forward_only:
            reverse = {"mode": args.reverse, "units": int(rev_chunks), "skipped_frac": (rev_skipped / rev_chunks) if rev_chunks else None,
                       "visited_cells": int(visited_cells), "visited_frac_of_cells": visited_cells / ncells_local,
                       "ms": t_bwd * 1e3,
                       "frac_on_visited": (ALGO_MUFU_BWD * visited_cells / t_bwd) / mufu_peak if t_bwd > 0 else None,
                       "note": "algorithmic 3 ex2 per VISITED cell / reverse kernel time / MUFU peak; with the exact +0 skip "
                               "the pass is a per-pair latency chain, not a throughput kernel"}
        # the dominant kernel is the one with the longest measured duration
        if forward_only or t_bwd <= t_fwd:
            dom, t_dom, achieved = "forward_kernel", t_fwd, ALGO_MUFU_FWD * ncells_local / t_fwd
        else:
            dom, t_dom, achieved = "backward_kernel", t_bwd, ALGO_MUFU_BWD * visited_cells / t_bwd
        variant = ("dense" if dense else "") if not args.gamma else f"gamma{args.gamma:g}"
        traffic, traffic_src, traffic_note = ((None, None, "not read for this run") if (world > 1 or table3) else
                                              ncu_traffic(dom, cfg.index, variant, t_dom * 1e3))
        algo_total = ALGO_MUFU_FWD + (0 if forward_only else ALGO_MUFU_BWD)
        # SURVEY.md 8(d), "HBM (algorithmic bytes)": inputs 4 d (n_k + m) per pair + strips 8/T per cell (T = strip
        # width; written by the forward pass, read back by the reverse pass) + per-pair gradient partials 4 m d
        T_strip = tile["strip_cols"]
        rows_local = int(data["lengths"].sum())
        algo_bytes = {"inputs": 4 * cfg.d * (rows_local + Nl * cfg.m),
                      "strips": 0 if forward_only else int(8 * ncells_local / T_strip),
                      "partials": 0 if forward_only else 4 * Nl * cfg.m * cfg.d}
        algo_bytes_total = int(sum(algo_bytes.values()))
        own_work = ALGO_MUFU_FWD * ncells_local + (0 if forward_only else ALGO_MUFU_BWD * visited_cells)
        roofline = {
            "bound": "alu", "kernel": dom, "achieved": achieved / 1e9, "peak": mufu_peak / 1e9, "unit": "GMUFU-op/s",
            "frac": achieved / mufu_peak,
            "traffic": traffic, "traffic_source": traffic_src, "traffic_note": traffic_note,
            "algorithmic_bytes": algo_bytes_total, "algorithmic_bytes_parts": algo_bytes,
            "algorithmic_bytes_note": f"SURVEY.md 8(d): inputs 4 d (sum n_k + N m) + strips 8/T B per cell at the built strip width "
                                      f"T = {T_strip} + gradient partials 4 N m d, per evaluation",
            "traffic_ratio": (traffic / algo_bytes_total) if traffic else None,
            "design_checkpoint_bytes": None if forward_only else int(ncells_local * 0.375 + ncells_local * 4 / 128),
            "design_checkpoint_bytes_note": "what THIS design's forward launch writes: warp-state records every 8 steps (0.375 B/cell) "
                                            "+ strip-boundary column (4/128 B/cell), DESIGN.md 5.5; the reverse pass reads back only "
                                            "the records of the chunks it visits",
            "step_frac_own_work": (own_work / (ms_step * 1e-3) / mufu_peak) if world == 1 else None,
            "step_frac_own_work_note": "whole step: (3 special functions per forward cell + 3 per VISITED reverse cell) / step "
                                       "time / MUFU peak",
            "peak_source": "measured live: dependent ex2 / lg2 / rcp chains on every SM (sdtw_measure_mufu_peak), the slowest "
                           "of the three; MEASURED_PEAKS.json holds no ALU figure (DESIGN.md section 8)",
            "peak_derived": mufu_derived / 1e9,
            "peak_derived_source": f"{MUFU_PER_CLK_PER_SM} MUFU results/clk/SM x {sms} SMs x {sm_max_hz / 1e6:.0f} MHz (clocks.max.sm)",
            "mufu_measured_gops": {k: v / 1e9 for k, v in mufu.items()},
            "algorithmic_per_cell": {"forward": ALGO_MUFU_FWD, "reverse": ALGO_MUFU_BWD},
            "note": "achieved counts the special-function evaluations the method needs (3 per forward cell, 3 per visited "
                    "reverse cell); the forward kernel issues 2.625 per cell on the MUFU pipe and evaluates 3 in 8 of the "
                    "second exponentials with an FMA-pipe polynomial, so the MUFU-only fraction can pass 1 (DESIGN.md 5.2)",
            "kernel_ms": {"forward": t_fwd * 1e3, "reverse": t_bwd * 1e3, "other": prof["ms_other"] / n_eval},
            "forward_frac": (ALGO_MUFU_FWD * ncells_local / t_fwd) / mufu_peak if t_fwd > 0 else None,
            "reverse": reverse,
            "cells_per_s_rel_dense_bound": (value / world) / (mufu_peak / algo_total),
            "cells_per_s_rel_dense_bound_note": "whole-step cells/s relative to the dense bound of 6 special functions per "
                "cell (3 forward + 3 reverse); NOT a roofline fraction when the reverse pass skips cells: see reverse.visited_frac_of_cells",
            "checkpoint_hbm_gbs": None if forward_only else (2 * ws_bytes) / max(t_fwd + t_bwd, 1e-9) / 1e9,
        }
        secondary = None
        if (world == 1 and not args.skip_secondary and args.config == 4 and not table3 and args.gamma is None and not dense):
            secondary = measure_secondary(B, torch, dev, data, mufu_peak, sms, sm_max_hz)
        cpu = None if args.skip_cpu else time_oracle(data)
        out = {
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
            "ms_per_step": ms_step, "higher_is_better": True, "scaling": "strong" if strong else "weak", "vs_baseline": None,
            "dtype": "f32", "data": "synthetic",
            "config": {"workload": workload_string(cfg) + ("; eq. 7 weights, Sakoe-Chiba band 0.6; step = one value+gradient evaluation" if table3 else ""),
                       "cells_per_step": cells_job, "workspace_gb": ws_bytes / 1e9,
                       "descent": None if (forward_only or table3) else
                           f"steps are the iterations of the configured descent ({iters_cfg} iterations from Z0 at step {cfg.step:g}), "
                           f"restarted from Z0 every {iters_cfg} steps (one 120 KB device copy inside the timed region)",
                       "reverse_mode": None if forward_only else args.reverse,
                       "l2": ("no flush: every step streams its checkpoints (workspace) through HBM, far above the 126 MB L2"
                              if ws_bytes > 4 * 126e6 else
                              "no flush: small configuration, the working set fits in the 126 MB L2 (latency-bound; not a roofline case)"),
                       "parallelism": (f"pairs of ONE problem partitioned over {world} GPUs (LPT on n_k); " if strong else
                                       f"every GPU its own {cfg.N} pairs; ") + "all-reduce of the m*d gradient per step"
                                      if world > 1 else "single GPU",
                       "tile": tile},
            "barycenter_iter_s": ms_step * 1e-3,
            "objective": objective, "finite": finite,
            "roofline": roofline, "secondary": secondary, "cpu_baseline": cpu,
            "e2e": e2e,
            "gpu_launches": int(launches), "clocks": clocks,
        }
        print(json.dumps(out))
    B.sdtw_set_reverse_mode(False)
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
                   "workspace_gb": B.sdtw_dtw_workspace_bytes(cfg.m, cfg.d, data["offsets"]) / 1e9,
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


def run_table3(args):
    """--op table3: the paper's Table 3 experiment end to end (setup Table 1): the
    Soft-DTW barycenter of --pairs univariate cycles of <= 18385 samples by L-BFGS (max 40 iterations, max 200 function
    evaluations), gamma = 1, Sakoe-Chiba band 0.6, eq. 7 weights, initialised with the resampled Euclidean mean --
    sdtw_barycenter_lbfgs, seconds for the whole optimisation.  Synthetic cycles of that shape; the paper's own figures
    (40.3 / 64 / 128 min for 5 / 10 / 25 cycles on an A10G with host round trips) are context, not a target."""
    import torch
    from paper_2404_12134_b200 import binding as B
    if int(os.environ.get("RANK", "0")) != 0:
        return
    torch.cuda.set_device(int(os.environ.get("LOCAL_RANK", "0")))
    cfg = table3_config(args.pairs)
    data = synth.make(cfg)
    Z0 = torch.from_numpy(data["Z0"]).cuda()
    X = torch.from_numpy(data["X"]).cuda()
    w = paper_setup.eq7_weights(data["lengths"])
    band = paper_setup.table1_band(cfg.m, data["lengths"])
    step0 = 1.0 / float(np.sum(w))                      # first trial step of the steepest-descent iteration
    def optimise():
        Z = Z0.clone()
        n0 = B.sdtw_launch_count()
        torch.cuda.synchronize()
        t = time.perf_counter()
        Z, vals, obj, steps, trials = B.sdtw_barycenter_lbfgs(Z, X, data["offsets"], cfg.gamma, 40, 10, step0, weights=w,
                                                              band=band, max_trials=5)
        torch.cuda.synchronize()
        return time.perf_counter() - t, obj, steps, trials, B.sdtw_launch_count() - n0, Z
    optimise()
    dt, obj, steps, trials, launches, Z = optimise()
    evals = int(trials.sum()) + 1
    its = int((steps > 0).sum())
    print(json.dumps({
        "metric": "table3_barycenter_seconds", "value": dt, "unit": "s", "n_gpus": 1, "steps": 1, "warmup": 1,
        "ms_per_step": dt * 1e3, "higher_is_better": False, "scaling": "weak", "vs_baseline": None, "dtype": "f32",
        "data": "synthetic",
        "config": {"workload": workload_string(cfg) + "; L-BFGS (hist 10, <= 40 iterations, Armijo backtracking), band 0.6, eq. 7 weights",
                   "iterations": its, "function_evaluations": evals, "cells_per_evaluation": synth.cells(data)},
        "objective_first_last": [float(obj[0]), float(obj[-1])], "finite": bool(torch.isfinite(Z).all().item()),
        "paper_minutes": {5: 40.3, 10: 64.0, 25: 128.0}.get(args.pairs),
        "paper_hardware": "1x NVIDIA A10G, chunks round-trip through host memory; TSLearn on CPU: 777 / 1217 / 3933 min",
        "gpu_launches": int(launches),
    }))


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", choices=["ours", "reference"], default="ours")
    ap.add_argument("--config", type=int, default=4, choices=[1, 2, 3, 4, 5])
    ap.add_argument("--op", choices=["barycenter", "score", "table3"], default="barycenter",
                    help="score = the Step-3 d_score kernel; table3 = the paper's Table 3 experiment (L-BFGS barycenter of "
                         "--pairs cycles) end to end (extras; the headline is barycenter)")
    ap.add_argument("--reverse", choices=["skip", "dense"], default="skip",
                    help="dense = the reverse kernel visits every cell (no exact-zero skip): the throughput measurement")
    ap.add_argument("--gamma", type=float, default=None, help="override the config's gamma (1.0 = the paper's default, Table 1)")
    ap.add_argument("--shape", choices=["config", "table3"], default="config",
                    help="table3 = the paper's Table 3 shape (--pairs cycles of <= 18385 samples, gamma 1, band 0.6, eq. 7 weights)")
    ap.add_argument("--pairs", type=int, default=5, help="number of cycles for --shape table3 (the paper: 5, 10, 25)")
    ap.add_argument("--scaling", choices=["weak", "strong"], default="weak",
                    help="N > 1: weak = every rank its own pairs; strong = one problem partitioned by dist.partition_pairs")
    ap.add_argument("--skip-e2e", action="store_true", help="profiling runs only: leave out the host-buffer leg")
    ap.add_argument("--skip-cpu", action="store_true", help="profiling runs only: leave out the timed oracle leg")
    ap.add_argument("--skip-secondary", action="store_true",
                    help="leave out the secondary workloads (cfg 5 scoring / d_score, cfg 3, dense reverse) of the default line")
    args = ap.parse_args()
    if args.impl == "reference":
        run_reference(args)
    elif args.op == "score":
        run_score(args)
    elif args.op == "table3":
        run_table3(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
