#!/usr/bin/env python
"""Writes the full-size reference outputs of tests/golden/ (fullsize_cfg3.npz, fullsize_cfg4.npz, fullsize_cfg5.npz,
fullsize_refs.json).  Calls ONLY the float64 oracle (oracle/) and the seeded input generator (synth) -- never the
CUDA path.  Hours of CPU time for cfg 4; resumable (every oracle evaluation is cached under --state-dir).

    python tests/golden/make_fullsize_refs.py [--cfg 3 4 5] [--cfg5-all | --cfg5-pairs P] [--threads T] [--state-dir DIR] [--only base|pert]

What is stored (BASELINE.json north_star: "summed Soft-DTW value+gradient and the barycenter matching the float64
oracle ... on all five configs"; cfg 1-2 are computed live by the tests, cfg 3-5 come from here):
  cfg 3, cfg 4   values[N] and the summed gradient G (eq. 6) at Z0 over ALL pairs;
                 the objective history, the last evaluated per-pair values and the iterate Z after the configured
                 iterations of Z <- Z - step G (eq. 7; Z kept in float64 between iterations, reading C14)
                 at the step frozen in synth.CONFIGS (reading C12), after the contractivity check below has passed.
  cfg 5          Soft-DTW values of all 1000 pairs (--cfg5-all), else of 64 seeded pairs, 16 of them anomalous
                 (--cfg5-pairs P: a seeded superset of P pairs with every anomalous cycle).
Contractivity check (reading C13): the same descent is run from Z0 (1 + 1e-6 xi), xi ~ N(0, 1) seeded.
If the two final iterates differ by more than 1e-4 (relative L2), i.e. the map amplifies a perturbation more than
100 x, parity of the iterated map would measure chaos, not correctness: the step is halved and the check repeated;
the step that passes is recorded and must equal synth.CONFIGS[idx].step (the test checks it).
Every file carries the SHA-256 of the input bytes it was computed from and of oracle/sdtw_oracle.c.
"""
from __future__ import annotations

import argparse
import hashlib
import json
import os
import sys
import time
from pathlib import Path

import numpy as np

HERE = Path(__file__).resolve().parent
ROOT = HERE.parent.parent
sys.path.insert(0, str(ROOT))

import oracle  # noqa: E402
from paper_2404_12134_b200 import synth  # noqa: E402  (input generator only: holds none of the method's arithmetic)

PERTURB = 1e-6          # relative size of the perturbation of Z0 (C13)
CONTRACT_TOL = 1e-4     # largest accepted relative difference of the two final iterates
CFG5_PAIRS, CFG5_ANOMALOUS = 64, 16


def sha256_inputs(data) -> str:
    h = hashlib.sha256()
    for a in (data["Z0"], data["X"], data["offsets"]):
        h.update(np.ascontiguousarray(a).tobytes())
    return h.hexdigest()


def sha256_oracle() -> str:
    return hashlib.sha256((ROOT / "oracle" / "sdtw_oracle.c").read_bytes()).hexdigest()


def rel_l2(a, b) -> float:
    return float(np.linalg.norm(a - b) / np.linalg.norm(b))


class Evaluator:
    """oracle.value_grad_f64z with an on-disk cache keyed by the bytes of Z (resumable)."""

    def __init__(self, data, state_dir: Path, threads: int, tag: str):
        self.data, self.dir, self.threads, self.tag = data, state_dir, threads, tag
        self.dir.mkdir(parents=True, exist_ok=True)
        self.key0 = sha256_inputs(data)[:16] + sha256_oracle()[:16]

    def __call__(self, Z):
        key = hashlib.sha256(self.key0.encode() + np.ascontiguousarray(Z, np.float64).tobytes()).hexdigest()[:24]
        f = self.dir / f"{self.tag}_{key}.npz"
        if f.exists():
            z = np.load(f)
            return z["values"], z["grad"], float(z["objective"])
        cfg = self.data["cfg"]
        t = time.time()
        values, grad, obj = oracle.value_grad_f64z(Z, self.data["X"], self.data["offsets"], cfg.gamma,
                                                   mode="checkpointed", nthreads=self.threads)
        print(f"  [{self.tag}] evaluation {key[:8]}: objective {obj:.6f}  ({time.time() - t:.0f} s)", flush=True)
        tmp = f.with_suffix(".tmp.npz")
        np.savez(tmp, values=values, grad=grad, objective=obj)
        os.replace(tmp, f)
        return values, grad, obj


def descent(ev, Z0, iters, step, kind):
    """PAPER.md:185 / eq. 7 with fixed step, Z in float64 throughout (the loop of oracle_barycenter_ex_f32, driven
    one evaluation at a time).  Returns (Z after `iters` updates, objective history, last evaluated values, G at Z0).
    The finished descent is cached as a whole (`kind` = "base" / "pert"), so that the two descents of the
    contractivity check may be computed by two runs of this script (--only), even on two machines."""
    f = ev.dir / f"{ev.tag}_descent_{kind}_{step:.6e}_{iters}.npz"
    if f.exists():
        z = np.load(f)
        if np.array_equal(z["Z0"], Z0):
            return z["Z"], z["hist"], z["values"], z["G0"]
    Z = np.array(Z0, np.float64)
    hist, values, G0 = [], None, None
    for it in range(iters):
        values, G, obj = ev(Z)
        if it == 0:
            G0 = G
        hist.append(obj)
        Z = Z - step * G
    tmp = f.with_suffix(".tmp.npz")
    np.savez(tmp, Z0=Z0, Z=Z, hist=np.array(hist), values=values, G0=G0)
    os.replace(tmp, f)
    return Z, np.array(hist), values, G0


def make_descent_config(idx, args):
    data = synth.make(idx)
    cfg = data["cfg"]
    ev = Evaluator(data, Path(args.state_dir), args.threads, f"cfg{idx}")
    Z0 = data["Z0"].astype(np.float64)
    xi = np.random.Generator(np.random.PCG64(13000 + idx)).standard_normal(Z0.shape)
    Zp0 = Z0 * (1.0 + PERTURB * xi)
    rel_in = rel_l2(Zp0, Z0)
    step = cfg.step
    tried = []
    while True:
        print(f"cfg {idx}: descent with step {step:g}, {cfg.iters} iterations", flush=True)
        if args.only == "pert":                      # this run only contributes the perturbed descent to the state dir
            descent(ev, Zp0, cfg.iters, step, "pert")
            return None
        Z, hist, values_last, G0 = descent(ev, Z0, cfg.iters, step, "base")
        if args.only == "base":
            return None
        Zp, hist_p, _, _ = descent(ev, Zp0, cfg.iters, step, "pert")
        rel_out = rel_l2(Zp, Z)
        tried.append({"step": step, "rel_in": rel_in, "rel_out": rel_out, "amplification": rel_out / rel_in,
                      "objective": hist.tolist(), "objective_perturbed": hist_p.tolist()})
        print(f"cfg {idx}: step {step:g}: perturbation {rel_in:.3e} -> {rel_out:.3e} (x {rel_out / rel_in:.2f}); "
              f"objective {hist[0]:.4f} -> {hist[-1]:.4f}", flush=True)
        if rel_out <= CONTRACT_TOL and np.all(np.isfinite(Z)):
            break
        step *= 0.5
    values0, _, obj0 = ev(Z0)
    np.savez(HERE / f"fullsize_cfg{idx}.npz", values0=values0, grad0=G0.astype(np.float32), Z_final=Z,
             values_last=values_last, objective=hist, step=np.float64(step), iters=np.int64(cfg.iters))
    return {"inputs_sha256": sha256_inputs(data), "step": step, "iters": cfg.iters, "contractivity": tried,
            "moved_rel": rel_l2(Z, Z0), "grad0_l2": float(np.linalg.norm(G0)), "grad0_max": float(np.abs(G0).max())}


def cfg5_sample(data, pairs=CFG5_PAIRS):
    """64 seeded pair indices, 16 of them anomalous (ascending).  With pairs > 64 (--cfg5-pairs) a superset of those:
    every remaining anomalous cycle, then seeded normal ones up to `pairs`."""
    rng = np.random.Generator(np.random.PCG64(13005))
    anom = np.flatnonzero(data["anomalous"])
    norm = np.flatnonzero(~data["anomalous"])
    ks = np.concatenate([rng.choice(anom, CFG5_ANOMALOUS, replace=False),
                         rng.choice(norm, CFG5_PAIRS - CFG5_ANOMALOUS, replace=False)])
    if pairs > CFG5_PAIRS:
        more_anom = np.setdiff1d(anom, ks)
        more_norm = np.random.Generator(np.random.PCG64(13006)).choice(
            np.setdiff1d(norm, ks), pairs - CFG5_PAIRS - len(more_anom), replace=False)
        ks = np.concatenate([ks, more_anom, more_norm])
    return np.sort(ks)


def make_cfg5(args):
    """--cfg5-all: all 1000 values of the scoring sweep ("all 1000 values if the cache exists"; about
    15 core-hours), else the 64-pair sample.  Computed in batches of pairs cached under --state-dir (resumable); the
    output file is written only when every batch is there."""
    data = synth.make(5)
    cfg = data["cfg"]
    ks = np.arange(cfg.N) if args.cfg5_all else cfg5_sample(data, args.cfg5_pairs)
    off = data["offsets"]
    state = Path(args.state_dir)
    state.mkdir(parents=True, exist_ok=True)
    key0 = sha256_inputs(data)[:16] + sha256_oracle()[:16]
    batch = max(8 * args.threads, 8)
    values = np.zeros(len(ks), np.float64)
    t = time.time()
    for b0 in range(0, len(ks), batch):
        kb = ks[b0:b0 + batch]
        f = state / f"cfg5_{key0}_{int(kb[0])}_{int(kb[-1])}_{len(kb)}.npy"
        if f.exists():
            values[b0:b0 + len(kb)] = np.load(f)
            continue
        chunks = [data["X"][off[k]:off[k + 1]] for k in kb]
        o = np.zeros(len(kb) + 1, np.int64)
        np.cumsum([len(c) for c in chunks], out=o[1:])
        v, _ = oracle.value_grad(data["Z0"], np.concatenate(chunks), o, cfg.gamma, want_grad=False, mode="checkpointed",
                                 nthreads=args.threads)
        tmp = f.with_suffix(".tmp.npy")
        np.save(tmp, v)
        os.replace(tmp, f)
        values[b0:b0 + len(kb)] = v
        print(f"cfg 5: pairs {b0 + len(kb)} of {len(ks)} ({time.time() - t:.0f} s)", flush=True)
    np.savez(HERE / "fullsize_cfg5.npz", pairs=ks, values=values, anomalous=data["anomalous"][ks])
    return {"inputs_sha256": sha256_inputs(data), "pairs": int(len(ks)), "anomalous": int(data["anomalous"][ks].sum())}


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--cfg", type=int, nargs="+", default=[3, 5, 4])
    ap.add_argument("--threads", type=int, default=os.cpu_count() or 1)
    ap.add_argument("--state-dir", default="/tmp/sdtw_fullsize_refs")
    ap.add_argument("--only", choices=["base", "pert"], default=None,
                    help="compute only one of the two descents of a config into --state-dir (no output file is written)")
    ap.add_argument("--cfg5-all", action="store_true", help="cfg 5: all N values instead of the 64-pair sample")
    ap.add_argument("--cfg5-pairs", type=int, default=CFG5_PAIRS,
                    help="cfg 5: size of the seeded sample (a superset of the 64-pair one; every anomalous cycle from 98 up)")
    args = ap.parse_args()
    oracle.build()
    meta_path = HERE / "fullsize_refs.json"
    meta = json.loads(meta_path.read_text()) if meta_path.exists() else {}
    for idx in args.cfg:
        t = time.time()
        entry = make_cfg5(args) if idx == 5 else make_descent_config(idx, args)
        if entry is None:
            continue
        entry["oracle_sha256"] = sha256_oracle()
        entry["seconds"] = round(time.time() - t)
        entry["threads"] = args.threads
        meta[f"cfg{idx}"] = entry
        meta_path.write_text(json.dumps(meta, indent=1, sort_keys=True) + "\n")


if __name__ == "__main__":
    main()
