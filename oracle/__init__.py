"""float64 CPU oracle for the Soft-DTW value / gradient / barycenter path (TEST INFRASTRUCTURE).

Only ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s ``cpu_baseline`` /
``--impl reference`` legs may import this package.  The product
(``paper_2404_12134_b200``) never imports it and it never imports the product.

The arithmetic lives in ``sdtw_oracle.c`` (plain C, IEEE double, OpenMP over pairs only);
this module only compiles it with gcc and marshals numpy arrays through ctypes.
Citations (PAPER.md line numbers) are in the C file's header.
"""
from __future__ import annotations

import ctypes
import os
import subprocess
from pathlib import Path

import numpy as np

_HERE = Path(__file__).resolve().parent
_SRC = _HERE / "sdtw_oracle.c"
_LIB = _HERE / "libsdtw_oracle.so"
_lib = None

_c_double_p = ctypes.POINTER(ctypes.c_double)
_c_float_p = ctypes.POINTER(ctypes.c_float)
_c_i64_p = ctypes.POINTER(ctypes.c_int64)


def build(force: bool = False) -> Path:
    """Compile sdtw_oracle.c + sdtw_oracle_lbfgs.c -> libsdtw_oracle.so (no-op when up to date)."""
    srcs = [_SRC, _SRC.with_name("sdtw_oracle_lbfgs.c")]
    if force or (not _LIB.exists()) or any(_LIB.stat().st_mtime < p.stat().st_mtime for p in srcs):
        tmp = _LIB.with_suffix(f".tmp{os.getpid()}.so")
        cmd = ["gcc", "-O2", "-ffp-contract=off", "-fno-fast-math", "-std=c11", "-fPIC", "-shared", "-fopenmp",
               "-o", str(tmp)] + [str(p) for p in srcs] + ["-lm"]
        subprocess.run(cmd, check=True)
        os.replace(tmp, _LIB)
    return _LIB


def _load():
    global _lib
    if _lib is None:
        build()
        _lib = ctypes.CDLL(str(_LIB))
        _lib.oracle_num_threads.restype = ctypes.c_int
    return _lib


def _d(a):
    return a.ctypes.data_as(_c_double_p)


def _chk(rc):
    if rc != 0:
        raise RuntimeError(f"oracle returned {rc}")


def num_threads() -> int:
    return int(_load().oracle_num_threads())


def cost_matrix(x, z):
    """Def. 3 with squared-Euclidean delta: (n, m) float64."""
    x = _as2d(x)
    z = _as2d(z)
    n, d = x.shape
    m = z.shape[0]
    D = np.empty((n, m), np.float64)
    _chk(_load().oracle_cost_matrix(_d(x), ctypes.c_int64(n), _d(z), ctypes.c_int64(m), ctypes.c_int(d), _d(D)))
    return D


def _as2d(a):
    a = np.asarray(a, np.float64)
    if a.ndim == 1:
        a = a[:, None]
    return np.ascontiguousarray(a)


def forward_R(D, gamma):
    """eq. 5 on a given cost matrix; returns the (n+2, m+2) bordered R (rows/cols 0..n / 0..m valid)."""
    D = np.ascontiguousarray(D, np.float64)
    n, m = D.shape
    R = np.full((n + 2, m + 2), np.nan, np.float64)
    _chk(_load().oracle_forward_R(_d(D), ctypes.c_int64(n), ctypes.c_int64(m), ctypes.c_double(gamma), _d(R)))
    return R


def pair(x, z, gamma, want_grad=True, want_E=False, want_R=False, mode="full", band=-1):
    """One (x, z) pair.  Returns dict(value, grad (m,d) or None, E (n,m) or None, R or None).
    band >= 0: Sakoe-Chiba band |i - j| <= band (Table 1); band < 0: none."""
    x = _as2d(x)
    z = _as2d(z)
    n, d = x.shape
    m = z.shape[0]
    assert z.shape[1] == d
    value = ctypes.c_double(0.0)
    grad = np.zeros((m, d), np.float64) if want_grad else None
    lib = _load()
    if mode == "checkpointed":
        assert not want_E and not want_R
        _chk(lib.oracle_pair_checkpointed_banded(_d(x), ctypes.c_int64(n), _d(z), ctypes.c_int64(m), ctypes.c_int(d),
                                                 ctypes.c_double(gamma), ctypes.c_int64(band), ctypes.byref(value),
                                                 _d(grad) if want_grad else None))
        return dict(value=value.value, grad=grad, E=None, R=None)
    E = np.empty((n, m), np.float64) if want_E else None
    R = np.empty((n + 2, m + 2), np.float64) if want_R else None
    _chk(lib.oracle_pair_full_banded(_d(x), ctypes.c_int64(n), _d(z), ctypes.c_int64(m), ctypes.c_int(d),
                                     ctypes.c_double(gamma), ctypes.c_int64(band), ctypes.byref(value),
                                     _d(grad) if want_grad else None, _d(E) if want_E else None,
                                     _d(R) if want_R else None))
    return dict(value=value.value, grad=grad, E=E, R=R)


def backward_E_normalised(D, R, gamma):
    """The probability-flow form of the reverse DP (self-check of the textbook form)."""
    D = np.ascontiguousarray(D, np.float64)
    R = np.ascontiguousarray(R, np.float64)
    n, m = D.shape
    assert R.shape == (n + 2, m + 2)
    E = np.empty((n, m), np.float64)
    _chk(_load().oracle_backward_E_normalised(_d(D), ctypes.c_int64(n), ctypes.c_int64(m), ctypes.c_double(gamma),
                                              _d(R), _d(E)))
    return E


def dtw(x, z):
    """eq. 1 (classic DTW, squared-Euclidean delta)."""
    x = _as2d(x)
    z = _as2d(z)
    v = ctypes.c_double(0.0)
    _chk(_load().oracle_dtw(_d(x), ctypes.c_int64(x.shape[0]), _d(z), ctypes.c_int64(z.shape[0]),
                            ctypes.c_int(x.shape[1]), ctypes.byref(v)))
    return v.value


def dtw_path(x, z, want_path=False):
    """eq. 1 + eq. 8's |pi| in float64: (DTW value, path length[, path as (len, 2) 1-based (i, j)])."""
    x = _as2d(x)
    z = _as2d(z)
    n, m = x.shape[0], z.shape[0]
    v = ctypes.c_double(0.0)
    ln = ctypes.c_int64(0)
    path = np.zeros((n + m, 2), np.int64) if want_path else None
    _chk(_load().oracle_dtw_path(_d(x), ctypes.c_int64(n), _d(z), ctypes.c_int64(m), ctypes.c_int(x.shape[1]),
                                 ctypes.byref(v), ctypes.byref(ln), path.ctypes.data_as(_c_i64_p) if want_path else None))
    if want_path:
        return v.value, ln.value, path[:ln.value]
    return v.value, ln.value


def dtw_score(Z, X_concat, offsets, nthreads=0):
    """Mirror of the C-ABI sdtw_dtw_score (eq. 8), decisions in float32: (DTW (N,) f32, |pi| (N,) i32, score (N,) f32)."""
    Z, X, off = _f32_inputs(Z, X_concat, offsets)
    m, d = Z.shape
    N = len(off) - 1
    values = np.zeros(N, np.float32)
    plen = np.zeros(N, np.int32)
    score = np.zeros(N, np.float32)
    _chk(_load().oracle_dtw_score_f32(Z.ctypes.data_as(_c_float_p), ctypes.c_int64(m), ctypes.c_int(d),
                                      X.ctypes.data_as(_c_float_p), off.ctypes.data_as(_c_i64_p), ctypes.c_int(N),
                                      values.ctypes.data_as(_c_float_p), plen.ctypes.data_as(ctypes.POINTER(ctypes.c_int32)),
                                      score.ctypes.data_as(_c_float_p), ctypes.c_int(nthreads)))
    return values, plen, score


def subdtw(y, z):
    """eq. 2 in float64: reference z against the best subsequence of window y -> (value, a*, b*) 0-based inclusive."""
    y = _as2d(y)
    z = _as2d(z)
    v = ctypes.c_double(0.0)
    a, b = ctypes.c_int64(0), ctypes.c_int64(0)
    _chk(_load().oracle_subdtw(_d(y), ctypes.c_int64(y.shape[0]), _d(z), ctypes.c_int64(z.shape[0]),
                               ctypes.c_int(y.shape[1]), ctypes.byref(v), ctypes.byref(a), ctypes.byref(b)))
    return v.value, a.value, b.value


def subdtw_f32(Z, X_concat, offsets, nthreads=0):
    """Mirror of the C-ABI sdtw_subdtw, decisions in float32: (value (N,) f32, a* (N,) i32, b* (N,) i32)."""
    Z, X, off = _f32_inputs(Z, X_concat, offsets)
    m, d = Z.shape
    N = len(off) - 1
    values = np.zeros(N, np.float32)
    a = np.zeros(N, np.int32)
    b = np.zeros(N, np.int32)
    i32p = ctypes.POINTER(ctypes.c_int32)
    _chk(_load().oracle_subdtw_f32(Z.ctypes.data_as(_c_float_p), ctypes.c_int64(m), ctypes.c_int(d),
                                   X.ctypes.data_as(_c_float_p), off.ctypes.data_as(_c_i64_p), ctypes.c_int(N),
                                   values.ctypes.data_as(_c_float_p), a.ctypes.data_as(i32p), b.ctypes.data_as(i32p),
                                   ctypes.c_int(nthreads)))
    return values, a, b


def _f32_inputs(Z, X_concat, offsets):
    Z = np.ascontiguousarray(Z, np.float32)
    if Z.ndim == 1:
        Z = Z[:, None]
    X = np.ascontiguousarray(X_concat, np.float32)
    if X.ndim == 1:
        X = X[:, None]
    off = np.ascontiguousarray(offsets, np.int64)
    assert X.shape[1] == Z.shape[1] and off[0] == 0 and off[-1] == X.shape[0]
    return Z, X, off


def _weights(weights, N):
    if weights is None:
        return None, None
    w = np.ascontiguousarray(weights, np.float64)
    assert w.shape == (N,)
    return w, _d(w)


def value_grad(Z, X_concat, offsets, gamma, want_grad=True, mode="full", nthreads=0, weights=None, band=-1,
               want_objective=False):
    """Mirror of the C-ABI sdtw_value_grad / sdtw_value_grad_ex: fp32 inputs promoted to float64.
    Returns (values (N,) float64, grad (m, d) float64 or None) [+ objective if want_objective];
    grad = sum_k w_k grad_k, objective = sum_k w_k values[k] (weights None = 1), band < 0 = none."""
    Z, X, off = _f32_inputs(Z, X_concat, offsets)
    m, d = Z.shape
    N = len(off) - 1
    values = np.zeros(N, np.float64)
    grad = np.zeros((m, d), np.float64) if want_grad else None
    w, wp = _weights(weights, N)
    obj = ctypes.c_double(0.0)
    _chk(_load().oracle_value_grad_ex_f32(Z.ctypes.data_as(_c_float_p), ctypes.c_int64(m), ctypes.c_int(d),
                                          X.ctypes.data_as(_c_float_p), off.ctypes.data_as(_c_i64_p), ctypes.c_int(N),
                                          ctypes.c_double(gamma), wp, ctypes.c_int64(band), _d(values),
                                          _d(grad) if want_grad else None, ctypes.byref(obj),
                                          ctypes.c_int(1 if mode == "checkpointed" else 0), ctypes.c_int(nthreads)))
    if want_objective:
        return values, grad, obj.value
    return values, grad


def value_grad_f64z(Z, X_concat, offsets, gamma, want_grad=True, mode="full", nthreads=0, weights=None, band=-1):
    """value_grad at a barycenter given in float64 (an iterate of the descent, which keeps Z in float64 between
    iterations -- reading C14).  X_concat stays the float32 input.  Returns (values, grad or None, objective)."""
    Z = np.ascontiguousarray(Z, np.float64)
    if Z.ndim == 1:
        Z = Z[:, None]
    X = np.ascontiguousarray(X_concat, np.float32)
    if X.ndim == 1:
        X = X[:, None]
    off = np.ascontiguousarray(offsets, np.int64)
    assert X.shape[1] == Z.shape[1] and off[0] == 0 and off[-1] == X.shape[0]
    m, d = Z.shape
    N = len(off) - 1
    values = np.zeros(N, np.float64)
    grad = np.zeros((m, d), np.float64) if want_grad else None
    w, wp = _weights(weights, N)
    obj = ctypes.c_double(0.0)
    _chk(_load().oracle_value_grad_ex_f64z(_d(Z), ctypes.c_int64(m), ctypes.c_int(d), X.ctypes.data_as(_c_float_p),
                                           off.ctypes.data_as(_c_i64_p), ctypes.c_int(N), ctypes.c_double(gamma), wp,
                                           ctypes.c_int64(band), _d(values), _d(grad) if want_grad else None,
                                           ctypes.byref(obj), ctypes.c_int(1 if mode == "checkpointed" else 0),
                                           ctypes.c_int(nthreads)))
    return values, grad, obj.value


def barycenter(Z0, X_concat, offsets, gamma, iters, step, mode="full", nthreads=0, weights=None, band=-1):
    """Mirror of sdtw_barycenter / sdtw_barycenter_ex: fixed-step GD in float64 on sum_k w_k value_k.
    Returns (Z (m,d) float64, values (N,) at the last evaluated iterate, objective (iters,))."""
    Z0, X, off = _f32_inputs(Z0, X_concat, offsets)
    m, d = Z0.shape
    N = len(off) - 1
    Z = np.zeros((m, d), np.float64)
    values = np.zeros(N, np.float64)
    obj = np.zeros(max(iters, 1), np.float64)
    w, wp = _weights(weights, N)
    _chk(_load().oracle_barycenter_ex_f32(Z0.ctypes.data_as(_c_float_p), ctypes.c_int64(m), ctypes.c_int(d),
                                          X.ctypes.data_as(_c_float_p), off.ctypes.data_as(_c_i64_p), ctypes.c_int(N),
                                          ctypes.c_double(gamma), wp, ctypes.c_int64(band), ctypes.c_int(iters),
                                          ctypes.c_double(step), _d(Z), _d(values), _d(obj),
                                          ctypes.c_int(1 if mode == "checkpointed" else 0), ctypes.c_int(nthreads)))
    return Z, values, obj[:iters]


def lbfgs_direction(S, Y, g):
    """r = H g by the two-loop recursion over the stored pairs (rows of S, Y: oldest first); float64."""
    g = np.ascontiguousarray(g, np.float64).reshape(-1)
    S = np.ascontiguousarray(S, np.float64).reshape(-1, g.size) if len(S) else np.zeros((0, g.size))
    Y = np.ascontiguousarray(Y, np.float64).reshape(-1, g.size) if len(Y) else np.zeros((0, g.size))
    r = np.zeros_like(g)
    _chk(_load().oracle_lbfgs_direction(_d(S) if len(S) else None, _d(Y) if len(Y) else None, ctypes.c_int(len(S)),
                                        ctypes.c_int64(g.size), _d(g), _d(r)))
    return r


def barycenter_lbfgs(Z0, X_concat, offsets, gamma, iters, hist, step0, shrink=0.5, c1=1e-4, max_trials=20, mode="full",
                     nthreads=0, weights=None, band=-1):
    """Mirror of sdtw_barycenter_lbfgs (Table 1's optimiser: two-loop L-BFGS + Armijo backtracking), float64.
    Returns (Z (m,d), values (N,) at the final Z, objective (iters+1,), steps (iters,), trials (iters,))."""
    Z0, X, off = _f32_inputs(Z0, X_concat, offsets)
    m, d = Z0.shape
    N = len(off) - 1
    Z = np.zeros((m, d), np.float64)
    values = np.zeros(N, np.float64)
    obj = np.zeros(iters + 1, np.float64)
    steps = np.zeros(max(iters, 1), np.float64)
    trials = np.zeros(max(iters, 1), np.int32)
    w, wp = _weights(weights, N)
    _chk(_load().oracle_barycenter_lbfgs_f32(
        Z0.ctypes.data_as(_c_float_p), ctypes.c_int64(m), ctypes.c_int(d), X.ctypes.data_as(_c_float_p),
        off.ctypes.data_as(_c_i64_p), ctypes.c_int(N), ctypes.c_double(gamma), wp, ctypes.c_int64(band),
        ctypes.c_int(iters), ctypes.c_int(hist), ctypes.c_double(step0), ctypes.c_double(shrink), ctypes.c_double(c1),
        ctypes.c_int(max_trials), _d(Z), _d(values), _d(obj), _d(steps),
        trials.ctypes.data_as(ctypes.POINTER(ctypes.c_int32)), ctypes.c_int(1 if mode == "checkpointed" else 0),
        ctypes.c_int(nthreads)))
    return Z, values, obj, steps[:iters], trials[:iters]


def barycenter_backtracking(Z0, X_concat, offsets, gamma, iters, step0, shrink=0.5, c1=1e-4, max_trials=20, mode="full",
                            nthreads=0, weights=None, band=-1):
    """Mirror of sdtw_barycenter_backtracking: descent with an Armijo backtracking line search, float64.
    Returns (Z (m,d), values (N,) at the final Z, objective (iters+1,), steps (iters,), trials (iters,))."""
    Z0, X, off = _f32_inputs(Z0, X_concat, offsets)
    m, d = Z0.shape
    N = len(off) - 1
    Z = np.zeros((m, d), np.float64)
    values = np.zeros(N, np.float64)
    obj = np.zeros(iters + 1, np.float64)
    steps = np.zeros(max(iters, 1), np.float64)
    trials = np.zeros(max(iters, 1), np.int32)
    w, wp = _weights(weights, N)
    _chk(_load().oracle_barycenter_backtracking_f32(
        Z0.ctypes.data_as(_c_float_p), ctypes.c_int64(m), ctypes.c_int(d), X.ctypes.data_as(_c_float_p),
        off.ctypes.data_as(_c_i64_p), ctypes.c_int(N), ctypes.c_double(gamma), wp, ctypes.c_int64(band),
        ctypes.c_int(iters), ctypes.c_double(step0), ctypes.c_double(shrink), ctypes.c_double(c1),
        ctypes.c_int(max_trials), _d(Z), _d(values), _d(obj), _d(steps),
        trials.ctypes.data_as(ctypes.POINTER(ctypes.c_int32)), ctypes.c_int(1 if mode == "checkpointed" else 0),
        ctypes.c_int(nthreads)))
    return Z, values, obj, steps[:iters], trials[:iters]
