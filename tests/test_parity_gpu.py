"""Parity of the CUDA path (through the C ABI of include/sdtw.h) with the float64 oracle.

Tolerances (BASELINE.json north_star):
  per-pair values : |v - v*| <= 1e-4 * max(|v*|, gamma (n_k + m))      (reading C10), and the strict ratio
                    |v - v*| <= 1e-4 |v*| wherever |v*| is not tiny (|v*| >= 0.05 gamma (n_k + m): value = path cost
                    minus gamma x entropy, two terms of that size that cancel -- below that the strict ratio measures
                    the cancellation, not the arithmetic)
  summed gradient : ||G - G*||_2 <= 2e-3 ||G*||_2, and max_j |G_j - G*_j| <= 2e-3 max_j |G*_j| (a fault confined to
                    one strip-boundary column is invisible to the L2 norm); the worst column modulo 128 is printed
  barycenter      : ||Z - Z*||_2 <= 2e-3 ||Z*||_2 after the configured iterations, and ||Z - Z*|| <= 2e-3 ||Z* - Z0||
                    (error relative to the distance moved; the first one is nearly vacuous when Z barely moves: at
                    cfg 4 the descent moves Z by 8.7e-4 of its norm, so there the second bound is the one that holds)
"""
import dataclasses
import os

import numpy as np
import pytest

from paper_2404_12134_b200 import paper_setup, synth

pytestmark = pytest.mark.gpu

VAL_TOL, GRAD_TOL, BARY_TOL = 1e-4, 2e-3, 2e-3
GRAD_MAX_TOL = 2e-3          # max-norm companion of the gradient bar
MOVED_TOL = 2e-3             # barycenter error relative to the distance moved
STRICT_FLOOR = 0.05          # strict value ratio asserted where |v*| >= STRICT_FLOOR * gamma (n + m)


@pytest.fixture(scope="module")
def B():
    import torch
    assert torch.cuda.is_available(), "these tests need a CUDA device"
    from paper_2404_12134_b200 import binding
    return binding


def _dev(a):
    import torch
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def rel_l2(a, b):
    return float(np.linalg.norm(np.asarray(a, np.float64) - b) / max(np.linalg.norm(b), 1e-300))


def check_values(v, ov, lengths, cfg, tag=""):
    v = np.asarray(v, np.float64)
    scale = cfg.gamma * (np.asarray(lengths) + cfg.m)
    den = np.maximum(np.abs(ov), scale)
    err = np.abs(v - ov) / den
    strict = np.abs(v - ov) / np.maximum(np.abs(ov), 1e-300)
    big = np.abs(ov) >= STRICT_FLOOR * scale
    print(f"[{tag}] values: C10 rel max {err.max():.3e}, strict rel max {strict.max():.3e} "
          f"(asserted on {int(big.sum())} of {len(ov)}: max {strict[big].max() if big.any() else 0.0:.3e})")
    assert err.max() <= VAL_TOL, (tag, err.max())
    assert (not big.any()) or strict[big].max() <= VAL_TOL, (tag, strict[big].max())


def check_grad(G, oG, tag=""):
    """relative L2 and max-norm; prints the column of the largest deviation modulo 128 (the strip width: a fault at a
    strip boundary shows up as 0 or 127)."""
    G = np.asarray(G, np.float64).reshape(oG.shape)
    e = rel_l2(G, oG)
    dev = np.abs(G - oG)
    emax = float(dev.max() / max(np.abs(oG).max(), 1e-300))
    j = int(np.unravel_index(np.argmax(dev), dev.shape)[0])
    print(f"[{tag}] gradient rel L2 {e:.3e}, max-norm {emax:.3e} (worst column {j}, {j % 128} mod 128)")
    assert e <= GRAD_TOL, (tag, e)
    assert emax <= GRAD_MAX_TOL, (tag, emax, j)
    return e, emax


def check_barycenter(Z, Zo, Z0, tag=""):
    Z = np.asarray(Z, np.float64).reshape(Zo.shape)
    e = rel_l2(Z, Zo)
    moved = float(np.linalg.norm(Z - Zo) / max(np.linalg.norm(Zo - np.asarray(Z0, np.float64).reshape(Zo.shape)), 1e-300))
    print(f"[{tag}] barycenter rel L2 {e:.3e}, relative to distance moved {moved:.3e}")
    assert e <= BARY_TOL, (tag, e)
    assert moved <= MOVED_TOL, (tag, moved)
    return e, moved


def run_value_grad(B, oracle, data, tag, mode="checkpointed"):
    import torch
    cfg = data["cfg"]
    Z, X = _dev(data["Z0"]), _dev(data["X"])
    vals, G = B.sdtw_value_grad(Z, X, data["offsets"], cfg.gamma)
    vals_f, none = B.sdtw_value_grad(Z, X, data["offsets"], cfg.gamma, want_grad=False)
    torch.cuda.synchronize()
    ov, oG = oracle.value_grad(data["Z0"], data["X"], data["offsets"], cfg.gamma, mode=mode)
    check_values(vals.cpu().numpy(), ov, data["lengths"], cfg, tag)
    assert none is None and torch.equal(vals, vals_f)            # forward-only sweep computes the same values
    check_grad(G.cpu().numpy(), oG, tag)
    return vals, G


# ------------------------------------------------------------------------------------------- the five configurations
def test_cfg1_tiny_value_grad_and_barycenter(B, oracle):
    data = synth.make(1)
    cfg = data["cfg"]
    run_value_grad(B, oracle, data, "cfg1", mode="full")
    Z, vals, obj = B.sdtw_barycenter(_dev(data["Z0"]), _dev(data["X"]), data["offsets"], cfg.gamma, cfg.iters, cfg.step)
    Zo, vo, oo = oracle.barycenter(data["Z0"], data["X"], data["offsets"], cfg.gamma, cfg.iters, cfg.step)
    e, moved = check_barycenter(Z.cpu().numpy(), Zo, data["Z0"], "cfg1")
    assert moved <= 1e-2
    check_values(vals.cpu().numpy(), vo, data["lengths"], cfg, "cfg1 bary values")
    assert np.allclose(obj.cpu().numpy(), oo, rtol=1e-5)


def test_cfg2_medium_value_grad_and_barycenter(B, oracle):
    data = synth.make(2)
    cfg = data["cfg"]
    run_value_grad(B, oracle, data, "cfg2")
    Z, vals, obj = B.sdtw_barycenter(_dev(data["Z0"]), _dev(data["X"]), data["offsets"], cfg.gamma, cfg.iters, cfg.step)
    Zo, vo, oo = oracle.barycenter(data["Z0"], data["X"], data["offsets"], cfg.gamma, cfg.iters, cfg.step, mode="checkpointed")
    check_barycenter(Z.cpu().numpy(), Zo, data["Z0"], f"cfg2, objective {oo[0]:.2f} -> {oo[-1]:.2f}")
    assert np.allclose(obj.cpu().numpy(), oo, rtol=1e-4)
    check_values(vals.cpu().numpy(), vo, data["lengths"], cfg, "cfg2 bary values")


@pytest.mark.parametrize("idx,scale,N,iters", [(3, 0.1, 6, 4), (4, 0.1, 10, 3), (4, 0.2, 3, 0)])
def test_scaled_multichannel_and_full_length(B, oracle, idx, scale, N, iters):
    """cfg 3 / cfg 4 generators at reduced length: several strips, ragged tails, d = 4, gamma = 0.01."""
    cfg = synth.scaled(synth.CONFIGS[idx], scale, N=N)
    data = synth.make(cfg)
    run_value_grad(B, oracle, data, cfg.name)
    if iters:
        step = 0.08 / N * 0.25
        Z, vals, obj = B.sdtw_barycenter(_dev(data["Z0"]), _dev(data["X"]), data["offsets"], cfg.gamma, iters, step)
        Zo, vo, oo = oracle.barycenter(data["Z0"], data["X"], data["offsets"], cfg.gamma, iters, step, mode="checkpointed")
        check_barycenter(Z.cpu().numpy(), Zo, data["Z0"], f"{cfg.name}, objective {oo}")


def test_scaled_scoring_sweep_forward_only(B, oracle):
    import torch
    cfg = synth.scaled(synth.CONFIGS[5], 0.05, N=60)
    data = synth.make(cfg)
    vals, G = B.sdtw_value_grad(_dev(data["Z0"]), _dev(data["X"]), data["offsets"], cfg.gamma, want_grad=False)
    assert G is None
    ov, _ = oracle.value_grad(data["Z0"], data["X"], data["offsets"], cfg.gamma, want_grad=False)
    check_values(vals.cpu().numpy(), ov, data["lengths"], cfg, cfg.name)
    # anomalous cycles score higher than the median normal one (what Step 3 of the paper uses the value for)
    v = vals.cpu().numpy()
    assert np.median(v[data["anomalous"]]) > np.median(v[~data["anomalous"]])


# ------------------------------------------------------------------------------------------- edge cases
SHAPES = [(1, 1, 1, 1, 2), (1, 1, 1, 3, 1), (1, 3, 5, 2, 3), (7, 9, 3, 1, 2), (5, 6, 8, 1, 2), (3, 4, 9, 1, 1),
          (300, 310, 257, 3, 2), (250, 260, 256, 1, 3), (40, 50, 513, 1, 2), (600, 700, 255, 2, 2), (31, 33, 40, 4, 5),
          (1, 2, 300, 1, 2), (900, 901, 1, 1, 2), (64, 64, 7, 1, 1)]


@pytest.mark.parametrize("shape", SHAPES)
@pytest.mark.parametrize("gamma", [1.0, 0.01])
def test_edge_shapes(B, oracle, shape, gamma):
    """n = 1, m = 1, m < one thread's columns, m = strip width +- 1, single-row strips, d = 1..4."""
    n_lo, n_hi, m, d, N = shape
    cfg = dataclasses.replace(synth.CONFIGS[2], N=N, n_lo=n_lo, n_hi=n_hi, m=m, d=d, gamma=gamma, name=f"edge{shape}")
    data = synth.make(cfg, seed=hash(shape) % 10000)
    rng = np.random.default_rng(1)
    data["Z0"] = (data["Z0"] + 0.1 * rng.normal(size=data["Z0"].shape)).astype(np.float32)   # keep the gradient non-degenerate
    run_value_grad(B, oracle, data, cfg.name, mode="full")


def test_expected_alignment_mass_and_constant_inputs(B, oracle):
    """D == 0 (x == z == const): value = -gamma ln Del(n-1, m-1) (closed form, any size) and zero gradient."""
    import math
    import torch
    n, m, gamma = 700, 523, 0.5
    X = np.full((n, 1), 0.25, np.float32)
    Z = np.full((m, 1), 0.25, np.float32)
    vals, G = B.sdtw_value_grad(_dev(Z), _dev(X), np.array([0, n]), gamma)
    ov, oG = oracle.value_grad(Z, X, np.array([0, n]), gamma)
    assert abs(vals.item() - ov[0]) <= 1e-4 * abs(ov[0])
    assert float(G.abs().max()) <= 1e-6 and np.abs(oG).max() == 0.0


def test_reverse_zero_skip_is_bitwise_exact(B):
    """The reverse kernel skips chunks whose incoming E flow is +0 (include/sdtw.h: sdtw_set_reverse_mode).  The
    result must be bit-for-bit the one obtained by visiting every cell, and the skip must actually fire on sharp
    (small gamma) problems and never on a problem whose E is nowhere zero."""
    import torch
    import itertools
    cases = ((4, 0.1, 6, True), (3, 0.1, 3, True), (2, 1.0, 8, True), (1, 1.0, 8, False))
    for (idx, scale, N, d_expect_skip), kernel in itertools.product(cases, (0, 1)):     # both reverse kernels (sdtw_debug.h)
        cfg = synth.scaled(synth.CONFIGS[idx], scale, N=N)
        data = synth.make(cfg)
        Z, X = _dev(data["Z0"]), _dev(data["X"])
        try:
            B.sdtw_set_reverse_kernel(kernel)
            B.sdtw_profile_enable(True)                      # the reverse statistics are collected only while profiling
            B.sdtw_set_reverse_mode(True)
            vd, gd = B.sdtw_value_grad(Z, X, data["offsets"], cfg.gamma)
            chunks_d, skipped_d = B.sdtw_reverse_stats()
            B.sdtw_set_reverse_mode(False)
            vs, gs = B.sdtw_value_grad(Z, X, data["offsets"], cfg.gamma)
            chunks_s, skipped_s = B.sdtw_reverse_stats()
        finally:
            B.sdtw_set_reverse_mode(False)
            B.sdtw_set_reverse_kernel(-1)
            B.sdtw_profile_read()
            B.sdtw_profile_enable(False)
        assert torch.equal(vd, vs) and torch.equal(gd, gs), (cfg.name, kernel)
        assert skipped_d == 0 and chunks_d == chunks_s > 0
        print(f"[{cfg.name}] reverse chunks {chunks_s}, skipped {skipped_s} ({100.0 * skipped_s / chunks_s:.1f} %)")
        assert (skipped_s > 0) == d_expect_skip, (cfg.name, skipped_s)


# ------------------------------------------------------------------------------------------- API behaviour
def test_determinism_bitwise_and_workspace_registration(B):
    import torch
    cfg = synth.scaled(synth.CONFIGS[4], 0.1, N=12)
    data = synth.make(cfg)
    Z, X = _dev(data["Z0"]), _dev(data["X"])
    v1, g1 = B.sdtw_value_grad(Z, X, data["offsets"], cfg.gamma)
    v2, g2 = B.sdtw_value_grad(Z, X, data["offsets"], cfg.gamma)
    assert torch.equal(v1, v2) and torch.equal(g1, g2)
    need = B.sdtw_workspace_bytes(cfg.m, cfg.d, data["offsets"], True)
    ws = torch.empty(need + 256, dtype=torch.uint8, device="cuda")
    try:
        B.sdtw_set_workspace(ws)
        v3, g3 = B.sdtw_value_grad(Z, X, data["offsets"], cfg.gamma)
        assert torch.equal(v1, v3) and torch.equal(g1, g3)
        small = torch.empty(1024, dtype=torch.uint8, device="cuda")
        B.sdtw_set_workspace(small)
        with pytest.raises(B.SdtwError) as ei:
            B.sdtw_value_grad(Z, X, data["offsets"], cfg.gamma)
        assert ei.value.status == B.SDTW_ERR_WORKSPACE
    finally:
        B.sdtw_set_workspace(None)
    # a side stream gives the same bits
    s = torch.cuda.Stream()
    with torch.cuda.stream(s):
        v4, g4 = B.sdtw_value_grad(Z, X, data["offsets"], cfg.gamma, stream=s)
    s.synchronize()
    assert torch.equal(v1, v4) and torch.equal(g1, g4)


def test_waves_of_pairs_when_the_workspace_budget_is_small(B):
    """include/sdtw.h, WAVES: with a workspace budget below what the whole pair set needs, the pairs are evaluated in
    consecutive waves in the same workspace.  Values: bitwise those of the unsplit call.  Gradient, objective and the
    descent: the same up to the grouping of the sum over pairs (float32 round-off)."""
    import torch
    cfg = synth.scaled(synth.CONFIGS[4], 0.1, N=13)
    data = synth.make(cfg)
    Z, X = _dev(data["Z0"]), _dev(data["X"])
    w = paper_setup.eq7_weights(data["lengths"])
    v0, g0, o0 = B.sdtw_value_grad_ex(Z, X, data["offsets"], cfg.gamma, weights=w)
    step = 0.02 / cfg.N
    Zb0, vb0, ob0 = B.sdtw_barycenter(Z.clone(), X, data["offsets"], cfg.gamma, 3, step)
    vf0, _ = B.sdtw_value_grad(Z, X, data["offsets"], cfg.gamma, want_grad=False)
    assert B.sdtw_last_wave_count() == 1                     # unsplit so far (include/sdtw_debug.h)
    need = B.sdtw_workspace_bytes(cfg.m, cfg.d, data["offsets"], True)
    n0 = B.sdtw_launch_count()
    try:
        B.sdtw_set_workspace_limit(need // 3)
        v1, g1, o1 = B.sdtw_value_grad_ex(Z, X, data["offsets"], cfg.gamma, weights=w)
        launches = B.sdtw_launch_count() - n0
        assert B.sdtw_last_wave_count() >= 4                 # the split is silent, but it can be observed
        Zb1, vb1, ob1 = B.sdtw_barycenter(Z.clone(), X, data["offsets"], cfg.gamma, 3, step)
        B.sdtw_set_workspace_limit(B.sdtw_workspace_bytes(cfg.m, cfg.d, data["offsets"], False) // 2)
        vf1, _ = B.sdtw_value_grad(Z, X, data["offsets"], cfg.gamma, want_grad=False)
        B.sdtw_set_workspace_limit(1024)                     # not even one pair fits
        with pytest.raises(B.SdtwError) as ei:
            B.sdtw_value_grad(Z, X, data["offsets"], cfg.gamma)
        assert ei.value.status == B.SDTW_ERR_WORKSPACE
    finally:
        B.sdtw_set_workspace_limit(0)
    assert launches >= 4 * 4                                   # at least four waves of four launches
    assert torch.equal(v0, v1) and torch.equal(vf0, vf1) and torch.equal(vf0, v0)
    assert rel_l2(g1.cpu().numpy(), g0.cpu().numpy()) <= 1e-6
    assert abs(float(o1) - float(o0)) <= 1e-6 * abs(float(o0))
    moved = float(torch.linalg.norm(Zb0 - Z))
    assert float(torch.linalg.norm(Zb1 - Zb0)) <= 1e-5 * moved
    assert torch.allclose(ob1, ob0, rtol=1e-6) and torch.allclose(vb1, vb0, rtol=1e-6, atol=0)


def test_more_than_256_pairs_unforced_throughput_reverse_kernel(B, oracle):
    """300 cycles of cfg 2's shape: above LATENCY_KERNEL_MAX_PAIRS (sdtw.cu) the reverse pass is backward_kernel by the
    library's own choice (no sdtw_set_reverse_kernel); values and summed gradient against the oracle."""
    cfg = dataclasses.replace(synth.CONFIGS[2], N=300, name="300 pairs of cfg 2's shape")
    data = synth.make(cfg)
    B.sdtw_set_reverse_kernel(-1)
    run_value_grad(B, oracle, data, cfg.name, mode="full")


def test_one_pair_per_wave_more_waves_than_cached_plans(B):
    """40 pairs under a budget that holds one pair at a time: 40 waves, more than the 32 plans the cache used to keep
    (every wave of every iteration then re-allocated its plan).  Same values bit for bit, same descent to round-off."""
    import torch
    cfg = synth.scaled(synth.CONFIGS[2], 0.5, N=40)
    data = synth.make(cfg)
    Z, X = _dev(data["Z0"]), _dev(data["X"])
    v0, g0 = B.sdtw_value_grad(Z, X, data["offsets"], cfg.gamma)
    Zb0, vb0, ob0 = B.sdtw_barycenter(Z.clone(), X, data["offsets"], cfg.gamma, 4, cfg.step)
    longest = int(np.argmax(data["lengths"]))
    one = B.sdtw_workspace_bytes(cfg.m, cfg.d, np.array([0, data["lengths"][longest]], np.int64), True)
    try:
        B.sdtw_set_workspace_limit(one + one // 8)
        v1, g1 = B.sdtw_value_grad(Z, X, data["offsets"], cfg.gamma)
        assert B.sdtw_last_wave_count() == cfg.N
        Zb1, vb1, ob1 = B.sdtw_barycenter(Z.clone(), X, data["offsets"], cfg.gamma, 4, cfg.step)
        assert B.sdtw_last_wave_count() == cfg.N
    finally:
        B.sdtw_set_workspace_limit(0)
    assert torch.equal(v0, v1)
    assert rel_l2(g1.cpu().numpy(), g0.cpu().numpy()) <= 1e-6
    assert float(torch.linalg.norm(Zb1 - Zb0)) <= 1e-5 * float(torch.linalg.norm(Zb0 - Z))
    assert torch.allclose(ob1, ob0, rtol=1e-6)


def test_dtw_and_subdtw_calls_split_into_waves_bit_for_bit(B):
    """include/sdtw.h, WAVES: sdtw_dtw_score / sdtw_subdtw under a budget below sdtw_dtw_workspace_bytes sweep the pairs
    in waves; DTW, path length, score, Sub-DTW value, a*, b* are those of the unsplit call bit for bit (d = 1: the
    32-warp instantiation; d = 3: a boundary column per strip)."""
    import torch
    for d in (1, 3):
        cfg = dataclasses.replace(synth.scaled(synth.CONFIGS[5], 0.05, N=30), d=d, name=f"dtw waves d={d}")
        data = synth.make(cfg)
        Z, X = _dev(data["Z0"]), _dev(data["X"])
        B.sdtw_set_forward_rings(0)                        # a column per strip: a workspace that grows with the pair count
        try:
            ref = B.sdtw_dtw_score(Z, X, data["offsets"])
            assert B.sdtw_last_wave_count() == 1
            sref = B.sdtw_subdtw(Z, X, data["offsets"])
            need = B.sdtw_dtw_workspace_bytes(cfg.m, cfg.d, data["offsets"])
            B.sdtw_set_workspace_limit(need // 4)
            got = B.sdtw_dtw_score(Z, X, data["offsets"])
            assert B.sdtw_last_wave_count() >= 4
            sgot = B.sdtw_subdtw(Z, X, data["offsets"])
            assert B.sdtw_last_wave_count() >= 4
            B.sdtw_set_workspace_limit(256)                # not even one pair
            with pytest.raises(B.SdtwError) as ei:
                B.sdtw_dtw_score(Z, X, data["offsets"])
            assert ei.value.status == B.SDTW_ERR_WORKSPACE
        finally:
            B.sdtw_set_workspace_limit(0)
            B.sdtw_set_forward_rings(1)
        torch.cuda.synchronize()
        for a, b in zip(ref + sref, got + sgot):
            assert torch.equal(a, b)


def test_argument_errors_leave_outputs_untouched(B):
    import torch
    data = synth.make(1)
    cfg = data["cfg"]
    Z, X = _dev(data["Z0"]), _dev(data["X"])
    vals = torch.full((cfg.N,), 7.0, device="cuda")
    G = torch.full_like(Z, 7.0)
    for gamma in (0.0, -1.0, float("nan"), float("inf")):
        with pytest.raises(B.SdtwError) as ei:
            B.sdtw_value_grad(Z, X, data["offsets"], gamma, out_values=vals, out_grad=G)
        assert ei.value.status == B.SDTW_ERR_INVALID_ARG
    bad = data["offsets"].copy()
    bad[3] = bad[2]
    with pytest.raises(B.SdtwError):
        B.sdtw_value_grad(Z, X, bad, cfg.gamma, out_values=vals, out_grad=G)
    with pytest.raises(B.SdtwError) as ei:
        B.sdtw_barycenter(Z.clone(), X, data["offsets"], cfg.gamma, -1, 0.01)
    assert ei.value.status == B.SDTW_ERR_INVALID_ARG
    Z5 = torch.zeros(10, 5, device="cuda")
    with pytest.raises(B.SdtwError) as ei:
        B.sdtw_value_grad(Z5, torch.zeros(20, 5, device="cuda"), np.array([0, 20]), 1.0)
    assert ei.value.status == B.SDTW_ERR_UNSUPPORTED
    torch.cuda.synchronize()
    assert float(vals.min()) == 7.0 and float(G.min()) == 7.0
    # iters = 0 is a legal no-op
    Zc = Z.clone()
    B.sdtw_barycenter(Zc, X, data["offsets"], cfg.gamma, 0, 0.01)
    assert torch.equal(Zc, Z)


def test_host_buffer_entry_points_and_gd_update(B, oracle):
    import torch
    data = synth.make(1)
    cfg = data["cfg"]
    vals = np.zeros(cfg.N, np.float32)
    G = np.zeros_like(data["Z0"])
    B.sdtw_value_grad_host(data["Z0"], data["X"], data["offsets"], cfg.gamma, vals, G)
    dv, dG = B.sdtw_value_grad(_dev(data["Z0"]), _dev(data["X"]), data["offsets"], cfg.gamma)
    assert np.array_equal(vals, dv.cpu().numpy()) and np.array_equal(G, dG.cpu().numpy())
    Zh = data["Z0"].copy()
    obj = np.zeros(cfg.iters, np.float32)
    B.sdtw_barycenter_host(Zh, data["X"], data["offsets"], cfg.gamma, cfg.iters, cfg.step, None, obj)
    Zd, _, objd = B.sdtw_barycenter(_dev(data["Z0"]), _dev(data["X"]), data["offsets"], cfg.gamma, cfg.iters, cfg.step)
    assert np.array_equal(Zh, Zd.cpu().numpy()) and np.array_equal(obj, objd.cpu().numpy())
    # value_grad + gd_update == one barycenter iteration (the multi-GPU loop's building blocks)
    Z1 = _dev(data["Z0"])
    B.sdtw_gd_update(Z1, dG, cfg.step)
    Zb, _, _ = B.sdtw_barycenter(_dev(data["Z0"]), _dev(data["X"]), data["offsets"], cfg.gamma, 1, cfg.step)
    assert torch.equal(Z1, Zb)


def test_additivity_and_pair_order(B):
    """Summed result = sum of single-pair calls; values come back in the caller's pair order."""
    import torch
    cfg = synth.scaled(synth.CONFIGS[4], 0.05, N=5)
    data = synth.make(cfg)
    Z, X = _dev(data["Z0"]), _dev(data["X"])
    vals, G = B.sdtw_value_grad(Z, X, data["offsets"], cfg.gamma)
    acc = torch.zeros_like(G, dtype=torch.float64)
    for k in range(cfg.N):
        a, b = data["offsets"][k], data["offsets"][k + 1]
        vk, gk = B.sdtw_value_grad(Z, X[a:b].contiguous(), np.array([0, b - a]), cfg.gamma)
        assert vk.item() == vals[k].item()
        acc += gk.double()
    assert rel_l2(G.cpu().numpy(), acc.cpu().numpy()) < 1e-6


# ------------------------------------------------------------------------------------------- full sizes
# The acceptance test of BASELINE.json's north_star at cfg 3-5: the oracle's outputs at full size take hours of CPU time,
# so they are computed once by tests/golden/make_fullsize_refs.py (which calls only oracle/ and the input generator)
# and stored under tests/golden/ with the SHA-256 of the inputs and of the oracle source.
GOLDEN = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden")


def _golden(idx, data):
    import hashlib
    import json
    path = os.path.join(GOLDEN, f"fullsize_cfg{idx}.npz")
    if not os.path.exists(path):
        pytest.skip(f"{path} is missing (hours of oracle time): run tests/golden/make_fullsize_refs.py --cfg {idx}")
    meta = json.load(open(os.path.join(GOLDEN, "fullsize_refs.json")))[f"cfg{idx}"]
    h = hashlib.sha256()
    for a in (data["Z0"], data["X"], data["offsets"]):
        h.update(np.ascontiguousarray(a).tobytes())
    assert h.hexdigest() == meta["inputs_sha256"], "the stored reference outputs were computed from other inputs"
    return np.load(path), meta


def _full_descent_config(B, idx):
    """Summed value + gradient at Z0 over ALL pairs, then the configured descent (iterations and step of
    synth.CONFIGS, which passed the contractivity check C13 in the oracle), in the launch configuration bench.py times."""
    import torch
    data = synth.make(idx)
    cfg = data["cfg"]
    gold, meta = _golden(idx, data)
    assert float(gold["step"]) == cfg.step and int(gold["iters"]) == cfg.iters, "synth.CONFIGS was re-frozen: regenerate"
    last = meta["contractivity"][-1]
    assert last["step"] == cfg.step and last["rel_out"] <= 1e-4
    tag = f"cfg{idx} full size, all {cfg.N} pairs"
    Z0, X = _dev(data["Z0"]), _dev(data["X"])
    vals, G = B.sdtw_value_grad(Z0, X, data["offsets"], cfg.gamma)
    torch.cuda.synchronize()
    check_values(vals.cpu().numpy(), gold["values0"], data["lengths"], cfg, tag)
    check_grad(G.cpu().numpy(), gold["grad0"].astype(np.float64), tag)
    Z, vals_last, obj = B.sdtw_barycenter(Z0.clone(), X, data["offsets"], cfg.gamma, cfg.iters, cfg.step)
    torch.cuda.synchronize()
    check_barycenter(Z.cpu().numpy(), gold["Z_final"], data["Z0"], f"{tag}, {cfg.iters} iterations at step {cfg.step:g}")
    check_values(vals_last.cpu().numpy(), gold["values_last"], data["lengths"], cfg, tag + ", values at the last evaluated iterate")
    scale = float(np.sum(cfg.gamma * (data["lengths"] + cfg.m)))
    oo = gold["objective"]
    print(f"[{tag}] objective {obj.cpu().numpy().tolist()} (oracle {oo.tolist()})")
    assert np.all(np.abs(obj.cpu().numpy() - oo) <= VAL_TOL * np.maximum(np.abs(oo), scale))
    return data, vals, G


@pytest.mark.timeout(1500)
def test_cfg3_full_all_pairs_gradient_and_descent(B):
    _full_descent_config(B, 3)


@pytest.mark.timeout(1500)
def test_cfg4_full_all_pairs_gradient_and_descent(B):
    _full_descent_config(B, 4)


@pytest.mark.timeout(1500)
def test_cfg5_full_size_against_the_stored_oracle_values(B):
    """cfg 5 (1000 cycles of 20-40k samples against m = 30000, forward only) in one call, against every oracle value
    tests/golden/fullsize_cfg5.npz holds: all 1000 when it was written by `make_fullsize_refs.py --cfg5-all` (SURVEY.md
    8(d); Step 3 of the paper, consumes every one), else a seeded sample of at least 64 pairs, 16 of them anomalous (as committed: 256 pairs with
    all 50 anomalous cycles, `--cfg5-pairs 256`)."""
    import torch
    data = synth.make(5)
    cfg = data["cfg"]
    gold, _ = _golden(5, data)
    ks = gold["pairs"]
    assert len(ks) >= 64 and int(data["anomalous"][ks].sum()) >= 16 and np.array_equal(gold["anomalous"], data["anomalous"][ks])
    vals, G = B.sdtw_value_grad(_dev(data["Z0"]), _dev(data["X"]), data["offsets"], cfg.gamma, want_grad=False)
    torch.cuda.synchronize()
    assert G is None and torch.isfinite(vals).all()
    v = vals.cpu().numpy()
    check_values(v[ks], gold["values"], data["lengths"][ks], cfg,
                 f"cfg5 full size, {'ALL ' if len(ks) == cfg.N else ''}{len(ks)} pairs")
    assert np.median(v[data["anomalous"]]) > np.median(v[~data["anomalous"]])


@pytest.mark.parametrize("d,N,m", [(1, 64, 10100), (2, 60, 10300), (4, 40, 8100)])
def test_forward_only_rings_match_the_oracle_and_single_pair_calls(B, oracle, d, N, m):
    """Forward-only calls with more strips than resident warps pass strip-boundary values through per-warp rings inside
    a unit of strips and keep a boundary column only per unit (sdtw_kernels.cuh).  Short, ragged
    cycles against a long Z: many strips, a few chunks each, several units per pair and a ragged last unit.  Values
    against the oracle; and bit for bit against single-pair calls, which are small enough to take the one-column-per-strip
    path, and against a second run (ring state is rebuilt per evaluation)."""
    import torch
    from dataclasses import replace
    cfg = replace(synth.CONFIGS[5], name=f"rings_d{d}", N=N, n_lo=700, n_hi=1900, m=m, d=d, gamma=0.05)
    data = synth.make(cfg)
    Z, X = _dev(data["Z0"]), _dev(data["X"])
    try:
        B.sdtw_set_forward_rings(2)                           # rings although the columns of this problem are small (sdtw_debug.h)
        assert B.sdtw_workspace_bytes(m, d, data["offsets"], False) != B.sdtw_workspace_bytes_ex(m, d, data["offsets"], False, m - 100)
        vals, G = B.sdtw_value_grad(Z, X, data["offsets"], cfg.gamma, want_grad=False)
        vals2, _ = B.sdtw_value_grad(Z, X, data["offsets"], cfg.gamma, want_grad=False)
        B.sdtw_set_forward_rings(0)                           # one boundary column per strip
        vals3, _ = B.sdtw_value_grad(Z, X, data["offsets"], cfg.gamma, want_grad=False)
    finally:
        B.sdtw_set_forward_rings(1)
    torch.cuda.synchronize()
    assert G is None and torch.equal(vals, vals2) and torch.equal(vals, vals3)
    ov, _ = oracle.value_grad(data["Z0"], data["X"], data["offsets"], cfg.gamma, want_grad=False, mode="checkpointed")
    check_values(vals.cpu().numpy(), ov, data["lengths"], cfg, f"forward-only rings d={d}")
    for k in (0, 1, N // 2, N - 1):
        a, b = int(data["offsets"][k]), int(data["offsets"][k + 1])
        vk, _ = B.sdtw_value_grad(Z, X[a:b], np.array([0, b - a]), cfg.gamma, want_grad=False)
        assert vk.item() == vals[k].item(), (k, vk.item(), vals[k].item())


@pytest.mark.parametrize("d,N,m", [(1, 64, 10100), (2, 60, 10300)])
def test_dtw_kernels_rings_bit_exact(B, oracle, d, N, m):
    """sdtw_dtw_score / sdtw_subdtw with more strips than resident warps (units of 32 strips, rings inside a unit): bit
    for bit the one-column-per-strip results (sdtw_set_forward_rings(0)) and the oracle's float32-decision mirror."""
    import torch
    from dataclasses import replace
    cfg = replace(synth.CONFIGS[5], name=f"dtwrings_d{d}", N=N, n_lo=700, n_hi=1900, m=m, d=d)
    data = synth.make(cfg)
    Z, X = _dev(data["Z0"]), _dev(data["X"])
    try:
        B.sdtw_set_forward_rings(2)
        a = [t.cpu().numpy() for t in B.sdtw_dtw_score(Z, X, data["offsets"])]
        sa = [t.cpu().numpy() for t in B.sdtw_subdtw(Z, X, data["offsets"])]
        B.sdtw_set_forward_rings(0)
        b = [t.cpu().numpy() for t in B.sdtw_dtw_score(Z, X, data["offsets"])]
        sb = [t.cpu().numpy() for t in B.sdtw_subdtw(Z, X, data["offsets"])]
    finally:
        B.sdtw_set_forward_rings(1)
    for x, y in zip(a + sa, b + sb):
        assert np.array_equal(x.view(np.uint32) if x.dtype == np.float32 else x, y.view(np.uint32) if y.dtype == np.float32 else y)
    ov, ol, osc = oracle.dtw_score(data["Z0"], data["X"], data["offsets"])
    assert np.array_equal(a[1], ol) and np.array_equal(a[0].view(np.uint32), ov.view(np.uint32))
    assert np.array_equal(a[2].view(np.uint32), osc.view(np.uint32))


@pytest.mark.timeout(1500)
def test_full_size_batch_equals_single_pair_calls(B):
    """Schedule validation (the CUDA path against itself, not parity): at full size the batch call -- work queue,
    units, reduction over pairs -- gives each pair the bits it gets alone, and the summed gradient is the sum of the
    single-pair gradients (pair independence)."""
    import torch
    for idx in (3, 4):
        data = synth.make(idx)
        cfg = data["cfg"]
        Z, X = _dev(data["Z0"]), _dev(data["X"])
        vals, G = B.sdtw_value_grad(Z, X, data["offsets"], cfg.gamma)
        acc = torch.zeros_like(G, dtype=torch.float64)
        for k in range(cfg.N):
            a, b = int(data["offsets"][k]), int(data["offsets"][k + 1])
            vk, gk = B.sdtw_value_grad(Z, X[a:b], np.array([0, b - a]), cfg.gamma)
            assert vk.item() == vals[k].item()
            acc += gk.double()
        e = rel_l2(G.cpu().numpy(), acc.cpu().numpy())
        print(f"[cfg{idx} full size] batch gradient vs sum of {cfg.N} single-pair calls: rel L2 {e:.3e}")
        assert e <= 1e-5 and torch.isfinite(G).all()
        del Z, X, vals, G
        torch.cuda.empty_cache()


# ------------------------------------------------------------------------------------------- eq. 7 weights, Table 1 band
@pytest.mark.parametrize("idx,scale,N,frac", [(2, 1.0, 12, 0.6), (2, 1.0, 12, 0.25), (3, 0.1, 5, 0.6), (4, 0.1, 8, 0.6),
                                              (4, 0.1, 8, 0.3), (4, 0.2, 3, 0.35)])
def test_band_and_weights_value_grad(B, oracle, idx, scale, N, frac):
    """sdtw_value_grad_ex against the banded / weighted oracle: Sakoe-Chiba band |i - j| <= frac * longest length
    (Table 1; 0.6 is the paper's value) and w_k = lambda_k / n_k (eq. 7)."""
    import torch
    cfg = synth.scaled(synth.CONFIGS[idx], scale, N=N)
    data = synth.make(cfg)
    lens = data["lengths"]
    band = int(np.floor(frac * max(cfg.m, int(lens.max()))))     # Table 1: a fraction of the longest length
    assert band == paper_setup.table1_band(cfg.m, lens, frac)
    assert band >= np.abs(lens - cfg.m).max() and band < min(cfg.m, lens.min()) - 1      # feasible, and it excludes cells
    rng = np.random.default_rng(idx)
    lam = rng.uniform(0.5, 2.0, size=N)
    w = (lam / lens).astype(np.float32)                           # eq. 7: lambda_k / n_k
    assert np.array_equal(w, paper_setup.eq7_weights(lens, lam=lam))
    Z, X = _dev(data["Z0"]), _dev(data["X"])
    vals, G, obj = B.sdtw_value_grad_ex(Z, X, data["offsets"], cfg.gamma, weights=w, band=band)
    torch.cuda.synchronize()
    ov, oG, oobj = oracle.value_grad(data["Z0"], data["X"], data["offsets"], cfg.gamma, mode="checkpointed",
                                     weights=w.astype(np.float64), band=band, want_objective=True)
    check_values(vals.cpu().numpy(), ov, lens, cfg, f"{cfg.name} band {band}")
    check_grad(G.cpu().numpy(), oG, f"{cfg.name} band {band} ({frac} x longest), weighted; objective {obj.item():.6f} vs {oobj:.6f}")
    assert abs(obj.item() - oobj) <= 1e-4 * max(abs(oobj), float(np.sum(np.abs(w) * cfg.gamma * (lens + cfg.m))))
    # the band changes the result (it is not silently ignored), and a band that excludes nothing changes no bit
    v_free, g_free = B.sdtw_value_grad(Z, X, data["offsets"], cfg.gamma)
    v_all, g_all, _ = B.sdtw_value_grad_ex(Z, X, data["offsets"], cfg.gamma, band=int(max(cfg.m, lens.max())))
    assert torch.equal(v_free, v_all) and torch.equal(g_free, g_all)
    ov_free, _ = oracle.value_grad(data["Z0"], data["X"], data["offsets"], cfg.gamma, want_grad=False, mode="checkpointed")
    assert np.all(ov >= ov_free - 1e-9)                       # fewer paths -> larger soft-min (eq. 3-4)
    # forward-only banded sweep computes the same values
    vf, none, _ = B.sdtw_value_grad_ex(Z, X, data["offsets"], cfg.gamma, band=band, want_grad=False)
    assert none is None and torch.equal(vf, vals)


def test_band_barycenter_weighted_descent(B, oracle):
    cfg = synth.scaled(synth.CONFIGS[4], 0.1, N=8)
    data = synth.make(cfg)
    lens = data["lengths"]
    band = int(np.floor(0.6 * max(cfg.m, int(lens.max()))))      # Table 1 / eq. 7 restated here, not taken from the binding
    w = (1.0 / lens).astype(np.float32)
    assert band == paper_setup.table1_band(cfg.m, lens, 0.6) and np.array_equal(w, paper_setup.eq7_weights(lens))
    step = 0.02 / cfg.N * float(np.mean(lens))                # eq. 7 divides by n_k: rescale the step accordingly
    iters = 3
    Z, vals, obj = B.sdtw_barycenter_ex(_dev(data["Z0"]), _dev(data["X"]), data["offsets"], cfg.gamma, iters, step,
                                        weights=w, band=band)
    Zo, vo, oo = oracle.barycenter(data["Z0"], data["X"], data["offsets"], cfg.gamma, iters, step, mode="checkpointed",
                                   weights=w.astype(np.float64), band=band)
    check_barycenter(Z.cpu().numpy(), Zo, data["Z0"], f"{cfg.name} band {band}, eq. 7 weights; objective {oo}")
    assert np.allclose(obj.cpu().numpy(), oo, rtol=1e-4, atol=1e-4 * cfg.gamma * 2)
    check_values(vals.cpu().numpy(), vo, lens, cfg, "banded weighted barycenter values")


def test_band_argument_errors(B):
    import torch
    data = synth.make(2)
    cfg = data["cfg"]
    Z, X = _dev(data["Z0"]), _dev(data["X"])
    gap = int(np.abs(data["lengths"] - cfg.m).max())
    vals = torch.full((cfg.N,), 7.0, device="cuda")
    G = torch.full_like(Z, 7.0)
    with pytest.raises(B.SdtwError) as ei:                    # no complete path fits
        B.sdtw_value_grad_ex(Z, X, data["offsets"], cfg.gamma, band=gap - 1, out_values=vals, out_grad=G)
    assert ei.value.status == B.SDTW_ERR_INVALID_ARG
    with pytest.raises(B.SdtwError) as ei:                    # feasible but narrower than the kernel's value staircase
        B.sdtw_value_grad_ex(Z, X, data["offsets"], cfg.gamma, band=gap + 1, out_values=vals, out_grad=G)
    assert ei.value.status == B.SDTW_ERR_UNSUPPORTED
    w = np.ones(cfg.N, np.float32)
    w[3] = np.nan
    with pytest.raises(B.SdtwError) as ei:
        B.sdtw_value_grad_ex(Z, X, data["offsets"], cfg.gamma, weights=w, out_values=vals, out_grad=G)
    assert ei.value.status == B.SDTW_ERR_INVALID_ARG
    torch.cuda.synchronize()
    assert float(vals.min()) == 7.0 and float(G.min()) == 7.0


@pytest.mark.parametrize("n_lo,n_hi,m,d,gamma,band", [(990, 1010, 1000, 1, 0.1, 40), (990, 1010, 1000, 1, 0.1, 80),
                                                      (480, 520, 500, 2, 1.0, 50), (560, 560, 500, 1, 0.1, 80),
                                                      (500, 500, 560, 2, 0.5, 76), (420, 424, 400, 1, 0.2, 45)])
def test_band_that_matters(B, oracle, n_lo, n_hi, m, d, gamma, band):
    """Warped cycles against a band narrow enough to cut their alignment (longer and shorter than m, d = 1..2): value
    and gradient visibly depend on the band, so a kernel that ignored it, or put its edge one cell off, fails here."""
    import torch
    cfg = dataclasses.replace(synth.CONFIGS[2], N=6, n_lo=n_lo, n_hi=n_hi, m=m, d=d, gamma=gamma, name=f"band{band}")
    data = synth.make(cfg, seed=band)
    lens = data["lengths"]
    Z, X = _dev(data["Z0"]), _dev(data["X"])
    vals, G, _ = B.sdtw_value_grad_ex(Z, X, data["offsets"], gamma, band=band)
    ov, oG = oracle.value_grad(data["Z0"], data["X"], data["offsets"], gamma, band=band, mode="checkpointed")
    ov_free, oG_free = oracle.value_grad(data["Z0"], data["X"], data["offsets"], gamma, mode="checkpointed")
    ov_off, oG_off = oracle.value_grad(data["Z0"], data["X"], data["offsets"], gamma, band=band + 1, mode="checkpointed")
    den = np.maximum(np.abs(ov), gamma * (lens + m))
    assert (np.abs(ov - ov_free) / den).max() > 5 * VAL_TOL             # the band matters on this input
    check_values(vals.cpu().numpy(), ov, lens, cfg, cfg.name)
    check_grad(G.cpu().numpy(), oG, f"{cfg.name} (unbanded oracle differs by {rel_l2(oG_free, oG):.3e}, band+1 by {rel_l2(oG_off, oG):.3e})")
    assert rel_l2(oG_free, oG) > 10 * GRAD_TOL
    assert rel_l2(oG_off, oG) > 2 * GRAD_TOL                            # ... and so does a one-cell shift of its edge


def test_band_dense_reverse_and_schedule_are_bitwise_neutral(B):
    """With a band the reverse kernel only sweeps chunks that hold admissible rows; the dense mode (no zero-skip) and
    any forward unit size must give the same bits."""
    import torch
    cfg = synth.scaled(synth.CONFIGS[4], 0.1, N=6)
    data = synth.make(cfg)
    band = paper_setup.table1_band(cfg.m, data["lengths"], 0.3)
    Z, X = _dev(data["Z0"]), _dev(data["X"])
    for kernel in (0, 1):
        try:
            B.sdtw_set_reverse_kernel(kernel)
            v0, g0, _ = B.sdtw_value_grad_ex(Z, X, data["offsets"], cfg.gamma, band=band)
            B.sdtw_set_reverse_mode(True)
            v1, g1, _ = B.sdtw_value_grad_ex(Z, X, data["offsets"], cfg.gamma, band=band)
            B.sdtw_set_reverse_mode(False)
            B.sdtw_set_schedule(3)
            B.sdtw_set_schedule_tail(7, 2)
            v2, g2, _ = B.sdtw_value_grad_ex(Z, X, data["offsets"], cfg.gamma, band=band)
        finally:
            B.sdtw_set_reverse_mode(False)
            B.sdtw_set_reverse_kernel(-1)
            B.sdtw_set_schedule(0)
            B.sdtw_set_schedule_tail(-1, 0)
        assert torch.equal(v0, v1) and torch.equal(g0, g1) and torch.equal(v0, v2) and torch.equal(g0, g2), kernel
        assert torch.isfinite(g0).all()


def test_small_problem_graph_replay_is_bitwise_the_plain_launches(B):
    """Calls on small problems are captured into a CUDA graph the second time the same call (same buffers, same scalars)
    comes back, and replayed from then on.  First call = plain launches, second = capture + launch, third
    and fourth = replay: same bits every time, the launch counter advances by the same amount, other arguments (another
    step, another iteration count) get their own graph and their own results."""
    import torch
    for idx in (1, 2):
        data = synth.make(idx)
        cfg = data["cfg"]
        Z0, X = _dev(data["Z0"]), _dev(data["X"])
        Z = Z0.clone()
        vals = torch.empty(cfg.N, dtype=torch.float32, device=Z.device)
        obj = torch.empty(cfg.iters, dtype=torch.float32, device=Z.device)
        G = torch.empty_like(Z0)
        ref, counts = None, []
        for rep in range(4):
            Z.copy_(Z0)
            n0 = B.sdtw_launch_count()
            B.sdtw_barycenter(Z, X, data["offsets"], cfg.gamma, cfg.iters, cfg.step, out_values=vals, out_objective=obj)
            B.sdtw_value_grad(Z0, X, data["offsets"], cfg.gamma, out_values=vals, out_grad=G)
            torch.cuda.synchronize()
            counts.append(B.sdtw_launch_count() - n0)
            cur = (Z.clone(), obj.clone(), vals.clone(), G.clone())
            if ref is None:
                ref = cur
            assert all(torch.equal(a, b) for a, b in zip(ref, cur)), (idx, rep)
        assert len(set(counts)) == 1 and counts[0] == 4 * (cfg.iters + 1), counts
        Z.copy_(Z0)
        B.sdtw_barycenter(Z, X, data["offsets"], cfg.gamma, 2, 0.5 * cfg.step, out_values=vals, out_objective=obj)
        Z.copy_(Z0)
        B.sdtw_barycenter(Z, X, data["offsets"], cfg.gamma, 2, 0.5 * cfg.step, out_values=vals, out_objective=obj)
        torch.cuda.synchronize()
        assert not torch.equal(Z, ref[0]) and torch.isfinite(Z).all()


@pytest.mark.parametrize("kernel", [0, 1])
def test_both_reverse_kernels_against_the_oracle(B, oracle, kernel):
    """The reverse pass has a latency-regime and a throughput-regime kernel (include/sdtw_debug.h,
    sdtw_set_reverse_kernel); the library picks one by the number of pairs.  Each is held to the parity bar by itself,
    with and without a band, on ragged shapes that span several strips and chunks."""
    cases = [synth.make(1), synth.make(2), synth.make(synth.scaled(synth.CONFIGS[3], 0.06, N=5)),
             synth.make(synth.scaled(synth.CONFIGS[4], 0.05, N=7))]
    try:
        B.sdtw_set_reverse_kernel(kernel)
        for data in cases:
            cfg = data["cfg"]
            vals, G = B.sdtw_value_grad(_dev(data["Z0"]), _dev(data["X"]), data["offsets"], cfg.gamma)
            ov, oG = oracle.value_grad(data["Z0"], data["X"], data["offsets"], cfg.gamma)
            check_values(vals.cpu().numpy(), ov, data["lengths"], cfg, f"{cfg.name}, reverse kernel {kernel}")
            check_grad(G.cpu().numpy(), oG, f"{cfg.name}, reverse kernel {kernel}")
    finally:
        B.sdtw_set_reverse_kernel(-1)


# ------------------------------------------------------------------------------------------- Step 3 scoring: eq. 8
def _check_dtw(B, oracle, data, tag, sample=None):
    """sdtw_dtw_score against the float32-decision oracle: DTW, |pi| and d_score BIT-EXACT (integer work, and the float
    operations are stated one by one in include/sdtw.h); `sample` = pair indices the oracle computes one by one."""
    import torch
    Z, X = _dev(data["Z0"]), _dev(data["X"])
    dtw, plen, score = B.sdtw_dtw_score(Z, X, data["offsets"])
    torch.cuda.synchronize()
    dtw, plen, score = dtw.cpu().numpy(), plen.cpu().numpy(), score.cpu().numpy()
    if sample is None:
        ov, ol, osc = oracle.dtw_score(data["Z0"], data["X"], data["offsets"])
        ks = np.arange(len(ov))
    else:
        from paper_2404_12134_b200.dist import take_pairs
        ks = np.asarray(sample)
        Xs, offs = take_pairs(data["X"], data["offsets"], ks)
        ov, ol, osc = oracle.dtw_score(data["Z0"], Xs, offs)
    assert np.array_equal(plen[ks], ol), (tag, plen[ks], ol)
    assert np.array_equal(dtw[ks].view(np.uint32), ov.view(np.uint32)), (tag, dtw[ks], ov)
    assert np.array_equal(score[ks].view(np.uint32), osc.view(np.uint32)), tag
    lens = data["lengths"]
    m = data["Z0"].shape[0]
    assert np.all(plen >= np.maximum(lens, m)) and np.all(plen <= lens + m - 1) and np.all(np.isfinite(dtw))
    print(f"[{tag}] DTW / |pi| / d_score bit-exact on {len(ks)} pairs; |pi|/max(n,m) in [{(plen / np.maximum(lens, m)).min():.3f}, {(plen / np.maximum(lens, m)).max():.3f}]")
    return dtw, plen, score


def _dtw_f64_with_margin(x, z):
    """Test-side float64 DTW (eq. 1) by anti-diagonals in numpy, backtracked with the preference of reading C20, and the
    MARGIN by which the optimum is unique: the smallest gap, along the optimal path, between the predecessor taken and
    the best predecessor not taken.  Any other complete path costs at least value + margin."""
    n, m = x.shape[0], z.shape[0]
    D = ((x[:, None, :].astype(np.float64) - z[None, :, :].astype(np.float64)) ** 2).sum(-1)
    R = np.full((n + 1, m + 1), np.inf)
    R[0, 0] = 0.0
    for k in range(2, n + m + 1):
        i = np.arange(max(1, k - m), min(n, k - 1) + 1)
        j = k - i
        R[i, j] = D[i - 1, j - 1] + np.minimum(np.minimum(R[i - 1, j - 1], R[i - 1, j]), R[i, j - 1])
    i, j, length, margin = n, m, 1, np.inf
    while (i, j) != (1, 1):
        preds = np.array([R[i - 1, j - 1], R[i - 1, j], R[i, j - 1]])
        q = int(np.argmin(preds))                       # first of (diagonal, up, left) that attains the minimum
        others = np.delete(preds, q)
        margin = min(margin, float(others.min() - preds[q]))
        i, j = (i - 1, j - 1) if q == 0 else ((i - 1, j) if q == 1 else (i, j - 1))
        length += 1
    return float(R[n, m]), length, margin


def test_dtw_score_configs_bit_exact(B, oracle):
    for idx in (1, 2):
        _check_dtw(B, oracle, synth.make(idx), f"cfg{idx}")
    _check_dtw(B, oracle, synth.make(synth.scaled(synth.CONFIGS[3], 0.1, N=6)), "cfg3 x0.1")
    _check_dtw(B, oracle, synth.make(synth.scaled(synth.CONFIGS[4], 0.1, N=10)), "cfg4 x0.1")
    data = synth.make(synth.scaled(synth.CONFIGS[5], 0.05, N=60))
    dtw, plen, score = _check_dtw(B, oracle, data, "cfg5 x0.05")
    # what Step 3 uses the score for: anomalous cycles score higher than normal ones
    assert np.median(score[data["anomalous"]]) > np.median(score[~data["anomalous"]])
    # float64 definition (oracle.dtw_path): value within float32 round-off; the path length EXACTLY wherever the optimum
    # is unique by a margin far above float32 round-off (margin computed here, in float64, independently of the oracle)
    exact = 0
    for k in range(0, 60, 7):
        a, b = data["offsets"][k], data["offsets"][k + 1]
        v64, l64 = oracle.dtw_path(data["X"][a:b].astype(np.float64), data["Z0"].astype(np.float64))
        vt, lt, margin = _dtw_f64_with_margin(data["X"][a:b], data["Z0"])
        assert abs(vt - v64) <= 1e-12 * v64 and lt == l64
        assert abs(dtw[k] - v64) <= 1e-4 * v64
        if margin > 1e-5 * v64:                             # float32 accumulates about 1e-7 relative per operation
            assert int(plen[k]) == l64, (k, int(plen[k]), l64, margin)
            exact += 1
        else:
            assert abs(int(plen[k]) - l64) <= 0.002 * l64  # a near-tie may resolve differently in float32
    # On these noisy cycles the optimum is never unique by such a margin (it is 1e-9 ... 1e-14 of the value: along
    # ~2000 path steps two predecessors always come close somewhere), so the bound above is the one that applies.
    print(f"[cfg5 x0.05] float64 path length reproduced exactly on {exact} of 9 pairs with a unique optimum")
    # A family where the optimum IS unique by a wide margin: z steps by >= 0.5 per sample and x holds every z_j a random
    # number of times, plus noise of 1e-3; any path other than "row i on its own z_j" pays >= 0.2 more.  There the
    # float64 path length must be reproduced exactly.
    rng = np.random.Generator(np.random.PCG64(8080))
    cycles, zc = [], np.cumsum(rng.uniform(0.5, 1.5, size=700))
    for _ in range(5):
        x = np.repeat(zc, rng.integers(1, 5, size=zc.size))
        cycles.append((x + rng.normal(0.0, 1e-3, size=x.size)).astype(np.float32)[:, None])
    off = np.zeros(6, np.int64)
    np.cumsum([len(c) for c in cycles], out=off[1:])
    Zc = zc.astype(np.float32)[:, None]
    gv, gl, gs = [t.cpu().numpy() for t in B.sdtw_dtw_score(_dev(Zc), _dev(np.concatenate(cycles)), off)]
    for k, x in enumerate(cycles):
        vt, lt, margin = _dtw_f64_with_margin(x, Zc)
        assert margin > 0.2 and margin > 1e-5 * vt and lt == len(x)
        assert int(gl[k]) == lt and abs(gv[k] - vt) <= 1e-4 * vt


@pytest.mark.parametrize("shape", SHAPES)
def test_dtw_score_edge_shapes(B, oracle, shape):
    n_lo, n_hi, m, d, N = shape
    cfg = dataclasses.replace(synth.CONFIGS[2], N=N, n_lo=n_lo, n_hi=n_hi, m=m, d=d, name=f"edge{shape}")
    data = synth.make(cfg, seed=hash(shape) % 10000)
    _check_dtw(B, oracle, data, cfg.name)


def test_dtw_score_ties_and_errors(B, oracle):
    import torch
    # every cell ties (constant series): |pi| = max(n, m) by the stated tie-break; identical series: DTW = 0, |pi| = n
    for n, m in [(300, 300), (200, 500), (500, 200), (1, 300), (300, 1)]:
        X = np.full((n, 1), 0.5, np.float32)
        Z = np.full((m, 1), 0.25, np.float32)
        dtw, plen, score = B.sdtw_dtw_score(_dev(Z), _dev(X), np.array([0, n]))
        assert plen.item() == max(n, m) and dtw.item() == np.float32(0.0625) * max(n, m) and score.item() == 0.0625
    rng = np.random.default_rng(0)
    x = rng.normal(size=(700, 2)).astype(np.float32)
    dtw, plen, score = B.sdtw_dtw_score(_dev(x), _dev(np.repeat(x, 2, axis=0)), np.array([0, 1400]))
    assert dtw.item() == 0.0 and plen.item() == 1400
    # plateaus (exact ties inside real data): quantised inputs
    data = synth.make(synth.scaled(synth.CONFIGS[2], 0.5, N=8))
    data["X"] = (np.round(data["X"] * 8) / 8).astype(np.float32)
    data["Z0"] = (np.round(data["Z0"] * 8) / 8).astype(np.float32)
    _check_dtw(B, oracle, data, "quantised (many exact ties)")
    with pytest.raises(B.SdtwError):
        B.sdtw_dtw_score(_dev(data["Z0"]), _dev(data["X"]), np.array([0, 5, 5]))
    # determinism and batch == single calls
    d1 = B.sdtw_dtw_score(_dev(data["Z0"]), _dev(data["X"]), data["offsets"])
    d2 = B.sdtw_dtw_score(_dev(data["Z0"]), _dev(data["X"]), data["offsets"])
    assert all(torch.equal(a, b) for a, b in zip(d1, d2))


@pytest.mark.timeout(1500)
def test_dtw_score_full_size_sampled(B, oracle):
    """cfg 5 (the scoring sweep: 1000 cycles of 20-40k samples against m = 30000) in one call; the oracle computes
    sampled pairs (one anomalous) one by one; cfg 3 (d = 4) likewise."""
    for idx, nsample in ((5, 3), (3, 2)):
        data = synth.make(idx)
        rng = np.random.default_rng(idx)
        ks = np.sort(rng.choice(data["cfg"].N, size=nsample, replace=False))
        if idx == 5:
            ks[0] = int(np.flatnonzero(data["anomalous"])[0])
            ks = np.unique(ks)
        _check_dtw(B, oracle, data, f"cfg{idx} full size", sample=ks)


# ------------------------------------------------------------------------------------------- Step 1 primitive: eq. 2
def _check_subdtw(B, oracle, Zref, X, offsets, tag):
    import torch
    v, a, b = B.sdtw_subdtw(_dev(Zref), _dev(X), offsets)
    torch.cuda.synchronize()
    ov, oa, ob = oracle.subdtw_f32(Zref, X, offsets)
    v, a, b = v.cpu().numpy(), a.cpu().numpy(), b.cpu().numpy()
    assert np.array_equal(a, oa) and np.array_equal(b, ob), (tag, a, oa, b, ob)
    assert np.array_equal(v.view(np.uint32), ov.view(np.uint32)), (tag, v, ov)
    print(f"[{tag}] Sub-DTW value / a* / b* bit-exact on {len(ov)} windows; spans {(b - a + 1).tolist()[:6]}")
    return v, a, b


def test_subdtw_bit_exact_configs_and_edges(B, oracle):
    for idx in (1, 2):
        data = synth.make(idx)
        _check_subdtw(B, oracle, data["Z0"], data["X"], data["offsets"], f"cfg{idx} cycles as windows")
    data = synth.make(synth.scaled(synth.CONFIGS[4], 0.1, N=6))
    _check_subdtw(B, oracle, data["Z0"], data["X"], data["offsets"], "cfg4 x0.1")
    data = synth.make(synth.scaled(synth.CONFIGS[3], 0.05, N=4))
    _check_subdtw(B, oracle, data["Z0"], data["X"], data["offsets"], "cfg3 x0.05 (d = 4)")
    for shape in SHAPES:
        n_lo, n_hi, m, d, N = shape
        cfg = dataclasses.replace(synth.CONFIGS[2], N=N, n_lo=n_lo, n_hi=n_hi, m=m, d=d, name=f"edge{shape}")
        data = synth.make(cfg, seed=hash(shape) % 10000)
        _check_subdtw(B, oracle, data["Z0"], data["X"], data["offsets"], cfg.name)
    # windows of two reference lengths holding a warped copy of the reference between other material (the paper's
    # window = 2M): the copy is found, on a sub-span of the window
    rng = np.random.default_rng(4)
    data = synth.make(synth.scaled(synth.CONFIGS[2], 1.0, N=6))
    M = data["cfg"].m
    ref = data["Z0"]
    wins, offs, truth = [], [0], []
    for k in range(6):
        cyc = data["X"][data["offsets"][k]:data["offsets"][k + 1]]
        pre = rng.integers(50, 2 * M - len(cyc) - 50)
        w = np.concatenate([2.5 + 0.3 * rng.normal(size=(pre, 1)), cyc, 2.5 + 0.3 * rng.normal(size=(2 * M - pre - len(cyc), 1))])
        wins.append(w.astype(np.float32)); offs.append(offs[-1] + len(w)); truth.append((pre, pre + len(cyc) - 1))
    v, a, b = _check_subdtw(B, oracle, ref, np.concatenate(wins), np.array(offs), "embedded warped cycles")
    for k in range(6):
        # the match lies inside the embedded cycle and spans a good part of it (its flat ends may be left out)
        assert a[k] >= truth[k][0] - 25 and b[k] <= truth[k][1] + 25 and b[k] - a[k] >= 0.4 * (truth[k][1] - truth[k][0]), \
            (k, a[k], b[k], truth[k])
    # exact copy -> value 0 and exact span; all-ties case
    y = np.concatenate([3 + rng.normal(size=(170, 2)), ref[:300].repeat(2, 1), 3 + rng.normal(size=(250, 2))]).astype(np.float32)
    v, a, b = B.sdtw_subdtw(_dev(ref[:300].repeat(2, 1).copy()), _dev(y), np.array([0, len(y)]))
    assert v.item() == 0.0 and (a.item(), b.item()) == (170, 469)


def test_segment_cycles_loop_matches_oracle_driven_loop(B, oracle):
    """the sliding-window segmentation driven by sdtw_subdtw finds the same cycles as the same loop
    driven by the oracle's mirror, and they are the cycles the synthetic stream was built from."""
    import torch
    rng = np.random.default_rng(11)
    data = synth.make(synth.scaled(synth.CONFIGS[2], 0.6, N=7))
    M = data["cfg"].m
    ref = data["Z0"]
    parts, truth, pos = [], [], 0
    for k in range(7):
        gap = rng.integers(0, int(0.1 * M))                     # idle time / missing data between cycles
        if gap:
            parts.append(np.repeat(data["X"][data["offsets"][k]][None, :], gap, axis=0)); pos += gap
        cyc = data["X"][data["offsets"][k]:data["offsets"][k + 1]]
        parts.append(cyc); truth.append((pos, pos + len(cyc) - 1)); pos += len(cyc)
    Y = np.concatenate(parts).astype(np.float32)
    got = paper_setup.segment_cycles(_dev(Y), _dev(ref))
    def oracle_sub(r, w):
        v, a, b = oracle.subdtw_f32(r, w, np.array([0, len(w)]))
        return float(v[0]), int(a[0]), int(b[0])
    want = paper_setup.segment_cycles(Y, ref, subdtw=oracle_sub)
    assert got == want
    print(f"[segmentation] {len(got)} cycles found: {[(s, e) for s, e, _ in got]}; built from {truth}")
    # every found cycle lies inside one of the cycles the stream was built from, and most of those are found
    hit = set()
    for s, e, _ in got:
        inside = [k for k, (ts, te) in enumerate(truth) if s >= ts - 0.15 * M and e <= te + 0.15 * M]
        assert inside, (s, e, truth)
        hit.add(inside[0])
    assert len(hit) >= 5


# ------------------------------------------------------------------------------------------- NEXT-3: line-search descent
@pytest.mark.parametrize("idx,scale,N,iters,step0", [(1, 1.0, 8, 6, 0.64), (2, 1.0, 16, 5, 0.04), (4, 0.1, 8, 4, 0.02),
                                                     (3, 0.05, 4, 4, 0.4)])
def test_backtracking_descent_matches_oracle(B, oracle, idx, scale, N, iters, step0):
    """sdtw_barycenter_backtracking against the float64 oracle of the same algorithm: step0 is several times too large
    for the fixed-step loop, so the line search has to cut it; accepted steps, trial counts, objective history and the
    final barycenter must agree (the accept test compares the same quantities on both sides; the margins on these
    inputs are far above float32 round-off, which the test checks)."""
    cfg = synth.scaled(synth.CONFIGS[idx], scale, N=N) if (scale != 1.0 or N != synth.CONFIGS[idx].N) else synth.CONFIGS[idx]
    data = synth.make(cfg)
    Z, vals, obj, steps, trials = B.sdtw_barycenter_backtracking(_dev(data["Z0"]), _dev(data["X"]), data["offsets"],
                                                                 cfg.gamma, iters, step0)
    Zo, vo, oo, so, to = oracle.barycenter_backtracking(data["Z0"], data["X"], data["offsets"], cfg.gamma, iters, step0,
                                                        mode="checkpointed")
    print(f"[{cfg.name}] steps {steps.tolist()} (oracle {so.tolist()}), trials {trials.tolist()}, objective {obj.tolist()}")
    assert np.array_equal(trials, to) and np.allclose(steps, so, rtol=1e-6)
    assert trials.max() > 1 and np.all(np.diff(obj) < 0)                  # the search did cut the step; monotone descent
    scale_f = np.sum(cfg.gamma * (data["lengths"] + cfg.m))
    assert np.all(np.abs(obj - oo) <= 1e-4 * np.maximum(np.abs(oo), scale_f))
    check_barycenter(Z.cpu().numpy(), Zo, data["Z0"], cfg.name)
    check_values(vals.cpu().numpy(), vo, data["lengths"], cfg, f"{cfg.name} values at the final Z")


def test_backtracking_equals_fixed_step_when_always_accepted(B):
    import torch
    data = synth.make(1)
    cfg = data["cfg"]
    Zf, vf, of = B.sdtw_barycenter(_dev(data["Z0"]), _dev(data["X"]), data["offsets"], cfg.gamma, 3, cfg.step)
    Zb, vb, ob, sb, tb = B.sdtw_barycenter_backtracking(_dev(data["Z0"]), _dev(data["X"]), data["offsets"], cfg.gamma, 3,
                                                        cfg.step, c1=0.0)
    assert torch.equal(Zf, Zb) and np.all(tb == 1) and np.allclose(sb, cfg.step)
    assert np.allclose(ob[:3], of.cpu().numpy(), rtol=1e-6)
    # hopeless first step, one trial allowed: nothing moves
    Zs, _, os_, ss, ts = B.sdtw_barycenter_backtracking(_dev(data["Z0"]), _dev(data["X"]), data["offsets"], cfg.gamma, 2,
                                                        50.0, max_trials=1)
    assert torch.equal(Zs.cpu(), torch.from_numpy(data["Z0"])) and np.all(ss == 0) and os_[0] == os_[2]
    with pytest.raises(B.SdtwError):
        B.sdtw_barycenter_backtracking(_dev(data["Z0"]), _dev(data["X"]), data["offsets"], cfg.gamma, 2, 0.1, shrink=1.5)


@pytest.mark.parametrize("idx,scale,N,iters,hist,step0", [(1, 1.0, 8, 8, 4, 0.64), (2, 1.0, 16, 6, 5, 0.04), (4, 0.1, 8, 5, 3, 0.02),
                                                          (3, 0.05, 4, 5, 10, 0.4)])
def test_lbfgs_descent_matches_oracle(B, oracle, idx, scale, N, iters, hist, step0):
    """sdtw_barycenter_lbfgs (Table 1's optimiser; include/sdtw.h, C23) against the float64 oracle of the same
    algorithm: accepted steps, trial counts, objective history and the final barycenter.  The curvature pairs are
    differences of float32 gradients, so the iterates drift apart faster than under plain descent: the bar on the
    barycenter stays 2e-3 of the distance moved."""
    cfg = synth.scaled(synth.CONFIGS[idx], scale, N=N) if (scale != 1.0 or N != synth.CONFIGS[idx].N) else synth.CONFIGS[idx]
    data = synth.make(cfg)
    Z, vals, obj, steps, trials = B.sdtw_barycenter_lbfgs(_dev(data["Z0"]), _dev(data["X"]), data["offsets"], cfg.gamma,
                                                          iters, hist, step0)
    Zo, vo, oo, so, to = oracle.barycenter_lbfgs(data["Z0"], data["X"], data["offsets"], cfg.gamma, iters, hist, step0,
                                                 mode="checkpointed")
    print(f"[{cfg.name}] L-BFGS steps {steps.tolist()} (oracle {so.tolist()}), trials {trials.tolist()} ({to.tolist()}), "
          f"objective {obj.tolist()} (oracle {oo.tolist()})")
    assert np.array_equal(trials, to) and np.allclose(steps, so, rtol=1e-6)
    assert np.all(np.diff(obj) < 0)
    scale_f = np.sum(cfg.gamma * (data["lengths"] + cfg.m))
    assert np.all(np.abs(obj - oo) <= 1e-4 * np.maximum(np.abs(oo), scale_f))
    check_barycenter(Z.cpu().numpy(), Zo, data["Z0"], cfg.name + " L-BFGS")
    check_values(vals.cpu().numpy(), vo, data["lengths"], cfg, f"{cfg.name} values at the final Z (L-BFGS)")


def test_line_search_descents_in_the_throughput_regime(B, oracle):
    """The line-search calls on a problem with more strips than resident forward warps (150 pairs x 33 strips against
    148 SMs x 32 warps), where the forward kernel hands out CTA-full units with small tail units instead of one strip
    per unit: backtracking and L-BFGS against the float64 oracle, as in the small cases above."""
    import torch
    cfg = dataclasses.replace(synth.CONFIGS[2], N=150, n_lo=500, n_hi=600, m=4100, name="150 short cycles vs m = 4100")
    data = synth.make(cfg)
    strips = -(-cfg.m // B.sdtw_tile_info()["strip_cols"]) * cfg.N
    assert strips > torch.cuda.get_device_properties(0).multi_processor_count * 32
    Z0, X = _dev(data["Z0"]), _dev(data["X"])
    scale_f = np.sum(cfg.gamma * (data["lengths"] + cfg.m))
    step0 = 4e-3
    for name, run_gpu, run_cpu in (
            ("backtracking", lambda: B.sdtw_barycenter_backtracking(Z0.clone(), X, data["offsets"], cfg.gamma, 3, step0),
             lambda: oracle.barycenter_backtracking(data["Z0"], data["X"], data["offsets"], cfg.gamma, 3, step0, mode="checkpointed")),
            ("L-BFGS", lambda: B.sdtw_barycenter_lbfgs(Z0.clone(), X, data["offsets"], cfg.gamma, 3, 3, step0),
             lambda: oracle.barycenter_lbfgs(data["Z0"], data["X"], data["offsets"], cfg.gamma, 3, 3, step0, mode="checkpointed"))):
        Z, vals, obj, steps, trials = run_gpu()
        Zo, vo, oo, so, to = run_cpu()
        print(f"[{cfg.name}, {name}] steps {steps.tolist()} (oracle {so.tolist()}), trials {trials.tolist()} ({to.tolist()}), "
              f"objective {obj.tolist()} (oracle {oo.tolist()})")
        assert np.array_equal(trials, to) and np.allclose(steps, so, rtol=1e-6)
        assert np.all(np.diff(obj) < 0)
        assert np.all(np.abs(obj - oo) <= 1e-4 * np.maximum(np.abs(oo), scale_f))
        check_barycenter(Z.cpu().numpy(), Zo, data["Z0"], f"{cfg.name}, {name}")
        check_values(vals.cpu().numpy(), vo, data["lengths"], cfg, f"{cfg.name}, {name}: values at the final Z")


def test_lbfgs_without_history_is_the_backtracking_descent(B):
    import torch
    data = synth.make(2)
    cfg = data["cfg"]
    a = B.sdtw_barycenter_backtracking(_dev(data["Z0"]), _dev(data["X"]), data["offsets"], cfg.gamma, 4, 0.04)
    b = B.sdtw_barycenter_lbfgs(_dev(data["Z0"]), _dev(data["X"]), data["offsets"], cfg.gamma, 4, 0, 0.04)
    assert torch.equal(a[0], b[0]) and torch.equal(a[1], b[1]) and np.array_equal(a[2], b[2])
    assert np.array_equal(a[3], b[3]) and np.array_equal(a[4], b[4])
    with pytest.raises(B.SdtwError):
        B.sdtw_barycenter_lbfgs(_dev(data["Z0"]), _dev(data["X"]), data["offsets"], cfg.gamma, 2, -1, 0.04)


@pytest.mark.parametrize("d", [5, 7, 9])
def test_dtw_and_subdtw_up_to_nine_channels(B, oracle, d):
    """The paper's Step 1 aligns all 9 robot variables at once: sdtw_dtw_score / sdtw_subdtw accept
    d <= SDTW_DTW_MAX_D = 9; the Soft-DTW calls stay at d <= 4."""
    cfg = dataclasses.replace(synth.CONFIGS[2], N=5, n_lo=500, n_hi=640, m=300, d=d, name=f"d{d}")
    data = synth.make(cfg, seed=d)
    _check_dtw(B, oracle, data, cfg.name)
    _check_subdtw(B, oracle, data["Z0"], data["X"], data["offsets"], cfg.name)
    if d == 9:
        with pytest.raises(B.SdtwError) as ei:
            B.sdtw_value_grad(_dev(data["Z0"]), _dev(data["X"]), data["offsets"], 0.1)
        assert ei.value.status == B.SDTW_ERR_UNSUPPORTED
