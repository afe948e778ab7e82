"""sdtw_value_static: Soft-DTW values for callers that are not allowed to allocate GPU memory.

Some users of this library cannot call cudaMalloc once they are running: a plug-in inside a host program that took the
whole GPU for its own pool, a monitoring loop that cannot afford the device-wide stall an allocation causes, a service
whose memory footprint is fixed at start-up.  For them include/sdtw.h has one entry point, sdtw_value_static, whose
scratch is a 32 MiB array compiled into the library.  These tests hold it to the allocating path (sdtw_value_grad with
out_grad = NULL), which tests/test_parity_gpu.py holds to the float64 oracle, and to the oracle directly.

The file is named test_zz_* so that pytest collects it after every other test file: `pytest -x` stops at the first
failure, and a failure here must not hide the parity tests.  It passes alone in a fresh process (the static call is
then the first thing the library does on the device: the set-up path) and after the other files (a workspace of the
allocating path already exists).
"""
import dataclasses

import numpy as np
import pytest

from paper_2404_12134_b200 import synth

VAL_TOL = 1e-4               # the value bar of tests/test_parity_gpu.py (north_star, reading C10)


def _problems():
    """Three seeded problems of different shape, so that what one call leaves in the array is wrong for the next:
    64 short pairs; 32 four-channel pairs; one long pair (63 strips, 141 chunks, ragged in both directions)."""
    a = synth.make(2)
    b = synth.make(synth.scaled(synth.CONFIGS[3], 0.1))
    c = synth.make(dataclasses.replace(synth.CONFIGS[2], N=1, n_lo=9001, n_hi=9001, m=7990, d=2, gamma=0.05,
                                       name="one long pair"), seed=77)
    return [a, b, c]


def _rel_err(v, ref, data):
    cfg = data["cfg"]
    den = np.maximum(np.abs(ref), cfg.gamma * (np.asarray(data["lengths"]) + cfg.m))
    return float((np.abs(np.asarray(v, np.float64) - ref) / den).max())


@pytest.mark.gpu
def test_static_scratch_values_match_the_allocating_path_call_after_call(oracle):
    """Back-to-back calls on the shared array (A, B, C, then A again) against sdtw_value_grad(out_grad=NULL) on the same
    inputs -- within the value tolerance of the parity tests, and in fact bit for bit, since both run the same kernels --
    and against the oracle.  After the start-up calls (address look-up; the CUDA driver loads each kernel's code at its
    first launch) the device's free memory must not shrink over further calls."""
    import torch
    assert torch.cuda.is_available(), "this test needs a CUDA device"
    from paper_2404_12134_b200 import binding as B
    probs = _problems()
    dev = [(torch.from_numpy(p["Z0"]).cuda(), torch.from_numpy(p["X"]).cuda(),
            torch.full((p["cfg"].N,), -1.0, dtype=torch.float32, device="cuda")) for p in probs]
    again = torch.full_like(dev[0][2], -1.0)
    # every tensor either path needs exists from here on; nothing below allocates through torch between the two
    # mem_get_info samples
    first = [torch.full_like(out, -2.0) for _, _, out in dev]
    for (Z, X, _), p, o in zip(dev, probs, first):       # start-up: set-up on this device, and the driver loads the
        B.sdtw_value_static(Z, X, p["offsets"], p["cfg"].gamma, o)   # kernel code of each channel count (d = 1, 4, 2)
    torch.cuda.synchronize()
    free_before = torch.cuda.mem_get_info()[0]
    for (Z, X, out), p in zip(dev, probs):               # steady state: calls in a row, no synchronisation between them
        B.sdtw_value_static(Z, X, p["offsets"], p["cfg"].gamma, out)
    B.sdtw_value_static(dev[0][0], dev[0][1], probs[0]["offsets"], probs[0]["cfg"].gamma, again)
    torch.cuda.synchronize()
    free_after = torch.cuda.mem_get_info()[0]
    assert free_after >= free_before, (free_before, free_after)
    for (_, _, out), o in zip(dev, first):
        assert torch.equal(out, o)                       # the start-up calls computed the same bits
    assert torch.equal(again, dev[0][2])                                             # leftovers of B and C did not leak into A
    for (Z, X, out), p in zip(dev, probs):
        cfg = p["cfg"]
        ref, _ = B.sdtw_value_grad(Z, X, p["offsets"], cfg.gamma, want_grad=False)   # the existing, allocating path
        torch.cuda.synchronize()
        v, r = out.cpu().numpy(), ref.cpu().numpy()
        assert np.isfinite(v).all()
        e_path = _rel_err(v, r.astype(np.float64), p)
        ov, _ = oracle.value_grad(p["Z0"], p["X"], p["offsets"], cfg.gamma, want_grad=False)
        e_oracle = _rel_err(v, ov, p)
        print(f"[{cfg.name}] static vs allocating path {e_path:.3e} (bitwise {np.array_equal(v, r)}), vs oracle {e_oracle:.3e}")
        assert e_path <= VAL_TOL, (cfg.name, e_path)
        assert np.array_equal(v, r), cfg.name
        assert e_oracle <= VAL_TOL, (cfg.name, e_oracle)


@pytest.mark.gpu
def test_static_scratch_full_size_pair_fits():
    """The stated capacity: one pair of the paper's size (33000 x 30000, cfg 4's longest cycle) fits the 32 MiB array."""
    import torch
    from paper_2404_12134_b200 import binding as B
    cfg = dataclasses.replace(synth.CONFIGS[4], N=1, n_lo=33000, n_hi=33000, name="one cfg-4 pair")
    p = synth.make(cfg, seed=5)
    Z, X = torch.from_numpy(p["Z0"]).cuda(), torch.from_numpy(p["X"]).cuda()
    out = torch.empty(1, dtype=torch.float32, device="cuda")
    B.sdtw_value_static(Z, X, p["offsets"], cfg.gamma, out)
    ref, _ = B.sdtw_value_grad(Z, X, p["offsets"], cfg.gamma, want_grad=False)
    torch.cuda.synchronize()
    assert torch.isfinite(out).all() and torch.equal(out, ref)


def test_static_scratch_limits_are_rejected_before_any_cuda_call():
    """More than SDTW_STATIC_MAX_PAIRS pairs, or a sweep whose scratch exceeds SDTW_STATIC_SCRATCH_BYTES, returns
    SDTW_ERR_STATIC_LIMIT with a message that names the limits; so does nothing else.  Runs without a GPU: the size test
    comes before the first CUDA call (the pointers are never dereferenced)."""
    import ctypes
    from paper_2404_12134_b200 import build
    build.build()
    from paper_2404_12134_b200 import binding as B
    lib = ctypes.CDLL(str(build.LIB))
    fn = lib.sdtw_value_static
    fn.restype, fn.argtypes = B.SYMBOLS["sdtw_value_static"]
    fake = ctypes.c_void_p(256)                                    # non-NULL stand-in for a device pointer

    def call(lengths, m, d=1, gamma=1.0, out=fake):
        off = np.concatenate([[0], np.cumsum(lengths)]).astype(np.int64)
        return fn(fake, m, d, fake, off.ctypes.data_as(ctypes.POINTER(ctypes.c_int64)), len(lengths), gamma, out, None)

    assert B.SDTW_ERR_STATIC_LIMIT == -5
    assert call([100] * (B.STATIC_MAX_PAIRS + 1), 100) == B.SDTW_ERR_STATIC_LIMIT          # too many pairs
    assert call([40000, 40000], 30000) == B.SDTW_ERR_STATIC_LIMIT                         # two full-size pairs: too much scratch
    assert call([4000] * 64, 4000, d=4) == B.SDTW_ERR_STATIC_LIMIT
    msg = B.status_string(B.SDTW_ERR_STATIC_LIMIT)
    assert "SDTW_STATIC_SCRATCH_BYTES" in msg and "SDTW_STATIC_MAX_PAIRS" in msg
    # ordinary argument errors keep their own codes
    assert call([100], 100, gamma=0.0) == B.SDTW_ERR_INVALID_ARG
    assert call([100], 100, out=None) == B.SDTW_ERR_INVALID_ARG
    assert call([100], 100, d=5) == B.SDTW_ERR_UNSUPPORTED
    # inside the limits the size test passes: on a box without a GPU what comes back is the CUDA error, not the limit
    # (with a GPU the call would go on to launch kernels on the stand-in pointers, so this part is for CPU boxes only)
    import torch
    if not torch.cuda.is_available():
        for lengths, m, d in (([33000], 30000, 4), ([3000] * 64, 3000, 4)):
            assert call(lengths, m, d) == B.SDTW_ERR_CUDA
