"""CPU-side checks: libsdtw.so loads and exports every symbol include/sdtw.h declares (no compute calls), the
host planner's argument handling, and the seeded input generator."""
import ctypes
import os
import re

import numpy as np
import pytest

from paper_2404_12134_b200 import synth

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def binding():
    from paper_2404_12134_b200 import build
    build.build()
    from paper_2404_12134_b200 import binding as b
    return b


def test_library_exports_every_declared_symbol(binding):
    """Every prototype of include/*.h (sdtw.h: the product boundary; sdtw_debug.h: instrumentation / tuning hooks) is
    exported by libsdtw.so and bound under the same name."""
    declared = {}
    for name in ("sdtw.h", "sdtw_debug.h"):
        hdr = open(os.path.join(ROOT, "include", name)).read()
        hdr = re.sub(r"/\*.*?\*/", "", hdr, flags=re.S)
        declared[name] = set(re.findall(r"\b(sdtw_[a-z_]+)\s*\(", hdr))
    assert {"sdtw_value_grad", "sdtw_barycenter", "sdtw_workspace_bytes", "sdtw_set_workspace"} <= declared["sdtw.h"]
    # the product header carries no measurement or tuning switches
    assert not any(("profile" in n or "schedule" in n or "stats" in n or "measure" in n) for n in declared["sdtw.h"])
    assert not (declared["sdtw.h"] & declared["sdtw_debug.h"])
    both = declared["sdtw.h"] | declared["sdtw_debug.h"]
    lib = ctypes.CDLL(os.path.join(ROOT, "paper_2404_12134_b200", "libsdtw.so"))
    for name in both:
        assert hasattr(lib, name), name
    assert both == set(binding.SYMBOLS), both ^ set(binding.SYMBOLS)


def test_paper_setup_helpers_eq7_weights_table1_band_default_length(binding):
    """paper_setup.eq7_weights / table1_band / default_barycenter_length against numbers written out by hand from eq. 7
    (lambda_i / m_i, lambda = 1 by default), Table 1 (bandwidth = 0.6 x the
    longest signal length) and "by default m_b = max m_i".  They live outside binding.py, which only
    marshals arguments and does not import them."""
    from paper_2404_12134_b200 import paper_setup
    assert not any(hasattr(binding, n) for n in ("eq7_weights", "table1_band", "segment_cycles", "paper_setup"))
    assert paper_setup.default_barycenter_length([27000, 33000, 31000]) == 33000
    assert paper_setup.default_barycenter_length(np.array([5])) == 5
    w = paper_setup.eq7_weights([4, 8, 5])
    assert w.dtype == np.float32 and np.array_equal(w, np.array([0.25, 0.125, 0.2], np.float32))
    w = paper_setup.eq7_weights([4, 8, 5], lam=[2.0, 1.0, 0.5])
    assert np.array_equal(w, np.array([0.5, 0.125, 0.1], np.float32))
    assert paper_setup.table1_band(30000, [27000, 33000, 31000]) == 19800         # 0.6 x 33000
    assert paper_setup.table1_band(30000, [27000, 28000]) == 18000                # the barycenter is the longest: 0.6 x 30000
    assert paper_setup.table1_band(18385, [18385] * 5) == 11031                   # Table 3's length: floor(11031.0)
    assert paper_setup.table1_band(1001, [1001], 0.25) == 250                     # floor(250.25)
    assert paper_setup.table1_band(10, [10], 1.0) == 10


def test_status_strings_and_tile_info(binding):
    assert binding.status_string(0) == "ok"
    for code in (-1, -2, -3, -4):
        assert binding.status_string(code) not in ("ok", "unknown status")
    assert binding.status_string(-99) == "unknown status"
    ti = binding.sdtw_tile_info()
    assert ti["strip_cols"] == 32 * ti["cols_per_thread"] and ti["chunk_steps"] % ti["ckpt_steps"] == 0


def test_workspace_bytes_planner(binding):
    off = np.array([0, 30000, 57000, 90000])
    full = binding.sdtw_workspace_bytes(30000, 1, off, True)
    fwd = binding.sdtw_workspace_bytes(30000, 1, off, False)
    assert 0 < fwd < full
    ti = binding.sdtw_tile_info()
    # checkpoints dominate: (W + R) floats per thread per ckpt_steps (W columns x R rows per step)
    #   => 4 (W + R) / (W R ckpt_steps) bytes per cell
    cells = 90000 * 30000
    Wc, Rr = ti["cols_per_thread"], ti["rows_per_step"]
    per_cell = 4 * (Wc + Rr) / (Wc * Rr * ti["ckpt_steps"])
    assert 0.9 * per_cell * cells < full < 1.3 * per_cell * cells
    # invalid arguments -> 0
    assert binding.sdtw_workspace_bytes(0, 1, off, True) == 0
    assert binding.sdtw_workspace_bytes(10, 0, off, True) == 0
    assert binding.sdtw_workspace_bytes(10, 1, np.array([0, 5, 5]), True) == 0       # empty cycle
    assert binding.sdtw_workspace_bytes(10, 1, np.array([1, 5, 9]), True) == 0       # offsets[0] != 0
    assert binding.sdtw_workspace_bytes(10, 5, off, True) == 0                        # d above compiled maximum
    # size is monotone in the problem
    assert binding.sdtw_workspace_bytes(30000, 1, off[:3], True) < full
    # forward-only sweeps keep O(chunks) boundary state per resident strip and one column per unit of strips (SURVEY.md
    # 8(a) a3): the scoring sweep of configs[4] (1000 cycles of 20-40k against m = 30000) needs about 1 GB, not a column
    # per strip (28 GB, what a banded forward-only call of the same shape still takes); the DTW kernels likewise
    off5 = synth.make(5)["offsets"]
    assert binding.sdtw_workspace_bytes(30000, 1, off5, False) < 1.1e9
    assert binding.sdtw_workspace_bytes_ex(30000, 1, off5, False, 25000) > 25e9
    assert binding.sdtw_dtw_workspace_bytes(30000, 1, off5) < 2.2e9


def test_synth_is_deterministic_and_shaped():
    a, b = synth.make(2), synth.make(2)
    assert np.array_equal(a["X"], b["X"]) and np.array_equal(a["Z0"], b["Z0"]) and np.array_equal(a["offsets"], b["offsets"])
    cfg = a["cfg"]
    assert a["X"].dtype == np.float32 and a["Z0"].dtype == np.float32 and a["offsets"].dtype == np.int64
    assert a["Z0"].shape == (cfg.m, cfg.d) and len(a["lengths"]) == cfg.N
    assert a["lengths"].min() >= cfg.n_lo and a["lengths"].max() <= cfg.n_hi
    assert a["offsets"][0] == 0 and a["offsets"][-1] == a["X"].shape[0]
    c = synth.make(2, seed=7)
    assert not np.array_equal(a["lengths"], c["lengths"])


def test_synth_configs_match_baseline_json():
    c = synth.CONFIGS
    assert (c[1].N, c[1].n_lo, c[1].n_hi, c[1].m, c[1].gamma, c[1].iters, c[1].step) == (8, 48, 64, 56, 1.0, 10, 0.01)
    assert (c[2].N, c[2].m, c[2].gamma, c[2].iters) == (64, 1000, 0.1, 20)
    assert (c[3].N, c[3].d, c[3].m, c[3].gamma, c[3].iters) == (32, 4, 10000, 0.1, 10)
    assert (c[4].N, c[4].n_lo, c[4].n_hi, c[4].m, c[4].gamma, c[4].iters) == (100, 27000, 33000, 30000, 0.01, 5)
    assert (c[5].N, c[5].n_lo, c[5].n_hi, c[5].m, c[5].iters, c[5].anomaly_frac) == (1000, 20000, 40000, 30000, 0, 0.05)


def test_synth_scoring_sweep_small():
    cfg = synth.scaled(synth.CONFIGS[5], 0.01, N=40)
    d = synth.make(cfg)
    assert d["anomalous"].sum() == 2 and d["Z0"].shape == (cfg.m, 1)
    # multichannel cycles share one warp: plateaus (zero slope) coincide across channels up to the noise
    d3 = synth.make(synth.scaled(synth.CONFIGS[3], 0.05, N=3))
    assert d3["X"].shape[1] == 4


def test_bench_reference_arm_prints_the_contract_line():
    """bench.py --impl reference (the oracle timed on the host cores; needs no GPU): one JSON line with the keys the
    driver reads.  Config 1 keeps it to a fraction of a second."""
    import json
    import subprocess
    import sys
    out = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--config", "1",
                          "--steps", "1", "--warmup", "0"], capture_output=True, text=True, timeout=300, cwd=ROOT)
    assert out.returncode == 0, out.stderr[-2000:]
    lines = [l for l in out.stdout.splitlines() if l.strip()]
    assert len(lines) == 1
    d = json.loads(lines[0])
    for key in ("impl", "metric", "value", "unit", "n_gpus", "steps", "warmup", "ms_per_step", "higher_is_better",
                "scaling", "vs_baseline", "dtype", "data", "config", "cpu_baseline", "e2e", "gpu_launches"):
        assert key in d, key
    assert d["impl"] == "reference" and d["value"] > 0 and d["unit"] == "cells/s" and d["dtype"] == "f64"
    assert d["cpu_baseline"]["kind"] == "oracle" and d["cpu_baseline"]["cores"] >= 1 and d["cpu_baseline"]["value"] == d["value"]
    assert d["e2e"]["h2d_bytes_per_step"] == 0 and d["e2e"]["d2h_bytes_per_step"] == 0 and d["e2e"]["value"] == d["value"]
    assert "workload" in d["config"]
