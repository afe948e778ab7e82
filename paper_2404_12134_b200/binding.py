"""Thin ctypes binding of libsdtw.so (include/sdtw.h): argument marshalling only.

Every step of the path runs in the CUDA kernels of csrc/; this module converts torch tensors /
numpy arrays to raw pointers and raises on a non-zero status.  There is no CPU fallback: if
libsdtw.so has not been built, importing this module raises.
"""
from __future__ import annotations

import ctypes
from pathlib import Path

import numpy as np

_LIBPATH = Path(__file__).resolve().parent / "libsdtw.so"
if not _LIBPATH.exists():
    raise ImportError(f"{_LIBPATH} is missing: build it with `python -m paper_2404_12134_b200.build` "
                      "(there is no CPU fallback)")
_lib = ctypes.CDLL(str(_LIBPATH))

_vp, _i64, _i32, _f32 = ctypes.c_void_p, ctypes.c_int64, ctypes.c_int32, ctypes.c_float
_i64p = ctypes.POINTER(ctypes.c_int64)

SYMBOLS = {
    "sdtw_value_grad": (ctypes.c_int, [_vp, _i64, _i32, _vp, _i64p, _i32, _f32, _vp, _vp, _vp]),
    "sdtw_barycenter": (ctypes.c_int, [_vp, _i64, _i32, _vp, _i64p, _i32, _f32, _i32, _f32, _vp, _vp, _vp]),
    "sdtw_value_grad_ex": (ctypes.c_int, [_vp, _i64, _i32, _vp, _i64p, _i32, _f32, _vp, _i64, _vp, _vp, _vp, _vp]),
    "sdtw_barycenter_ex": (ctypes.c_int, [_vp, _i64, _i32, _vp, _i64p, _i32, _f32, _vp, _i64, _i32, _f32, _vp, _vp, _vp]),
    "sdtw_barycenter_backtracking": (ctypes.c_int, [_vp, _i64, _i32, _vp, _i64p, _i32, _f32, _vp, _i64, _i32, _f32, _f32,
                                                    _f32, _i32, _vp, _vp, _vp, _vp, _vp]),
    "sdtw_barycenter_lbfgs": (ctypes.c_int, [_vp, _i64, _i32, _vp, _i64p, _i32, _f32, _vp, _i64, _i32, _i32, _f32, _f32,
                                             _f32, _i32, _vp, _vp, _vp, _vp, _vp]),
    "sdtw_dtw_score": (ctypes.c_int, [_vp, _i64, _i32, _vp, _i64p, _i32, _vp, _vp, _vp, _vp]),
    "sdtw_subdtw": (ctypes.c_int, [_vp, _i64, _i32, _vp, _i64p, _i32, _vp, _vp, _vp, _vp]),
    "sdtw_gd_update": (ctypes.c_int, [_vp, _vp, _i64, _f32, _vp]),
    "sdtw_value_static": (ctypes.c_int, [_vp, _i64, _i32, _vp, _i64p, _i32, _f32, _vp, _vp]),
    "sdtw_value_grad_host": (ctypes.c_int, [_vp, _i64, _i32, _vp, _i64p, _i32, _f32, _vp, _vp, _vp]),
    "sdtw_barycenter_host": (ctypes.c_int, [_vp, _i64, _i32, _vp, _i64p, _i32, _f32, _i32, _f32, _vp, _vp, _vp]),
    "sdtw_workspace_bytes": (ctypes.c_size_t, [_i64, _i32, _i64p, _i32, ctypes.c_int]),
    "sdtw_workspace_bytes_ex": (ctypes.c_size_t, [_i64, _i32, _i64p, _i32, ctypes.c_int, _i64]),
    "sdtw_dtw_workspace_bytes": (ctypes.c_size_t, [_i64, _i32, _i64p, _i32]),
    "sdtw_set_workspace": (ctypes.c_int, [_vp, ctypes.c_size_t]),
    "sdtw_set_workspace_limit": (ctypes.c_int, [ctypes.c_size_t]),
    "sdtw_status_string": (ctypes.c_char_p, [ctypes.c_int]),
    "sdtw_last_cuda_error": (ctypes.c_int, []),
    "sdtw_launch_count": (ctypes.c_uint64, []),
    "sdtw_last_wave_count": (ctypes.c_int, []),
    "sdtw_profile_enable": (ctypes.c_int, [ctypes.c_int]),
    "sdtw_profile_read": (ctypes.c_int, [ctypes.POINTER(ctypes.c_double)] * 3 + [_i64p]),
    "sdtw_tile_info": (ctypes.c_int, [ctypes.POINTER(ctypes.c_int32)] * 5),
    "sdtw_set_reverse_mode": (ctypes.c_int, [ctypes.c_int]),
    "sdtw_set_reverse_kernel": (ctypes.c_int, [ctypes.c_int]),
    "sdtw_set_forward_rings": (ctypes.c_int, [ctypes.c_int]),
    "sdtw_set_schedule": (ctypes.c_int, [ctypes.c_int]),
    "sdtw_set_schedule_tail": (ctypes.c_int, [ctypes.c_int, ctypes.c_int]),
    "sdtw_reverse_stats": (ctypes.c_int, [ctypes.POINTER(ctypes.c_uint64)] * 2),
    "sdtw_measure_mufu_peak": (ctypes.c_int, [_i32, ctypes.POINTER(ctypes.c_double), ctypes.POINTER(ctypes.c_int32)]),
}
for _name, (_res, _args) in SYMBOLS.items():
    _fn = getattr(_lib, _name)          # AttributeError here = the library does not export what sdtw.h declares
    _fn.restype, _fn.argtypes = _res, _args

SDTW_OK, SDTW_ERR_INVALID_ARG, SDTW_ERR_UNSUPPORTED, SDTW_ERR_WORKSPACE, SDTW_ERR_CUDA = 0, -1, -2, -3, -4
SDTW_ERR_STATIC_LIMIT = -5
STATIC_SCRATCH_BYTES, STATIC_MAX_PAIRS = 32 << 20, 64     # sdtw_value_static (include/sdtw.h)


class SdtwError(RuntimeError):
    def __init__(self, status):
        self.status = status
        msg = _lib.sdtw_status_string(status).decode()
        if status == SDTW_ERR_CUDA:
            msg += f" [cudaError {_lib.sdtw_last_cuda_error()}]"
        super().__init__(f"libsdtw status {status}: {msg}")


def _check(status):
    if status != SDTW_OK:
        raise SdtwError(status)


def status_string(status: int) -> str:
    return _lib.sdtw_status_string(status).decode()


def _offsets(offsets):
    off = np.ascontiguousarray(np.asarray(offsets, dtype=np.int64))
    return off, off.ctypes.data_as(_i64p), len(off) - 1


def _ptr(t):
    return None if t is None else ctypes.c_void_p(t.data_ptr())


def _stream(stream):
    if stream is None:
        import torch
        return ctypes.c_void_p(torch.cuda.current_stream().cuda_stream)
    return ctypes.c_void_p(stream if isinstance(stream, int) else stream.cuda_stream)


def _dims(Z):
    if Z.dim() == 1:
        return Z.shape[0], 1
    return Z.shape[0], Z.shape[1]


def _dev_f32(t, name):
    import torch
    if not (isinstance(t, torch.Tensor) and t.is_cuda and t.dtype == torch.float32 and t.is_contiguous()):
        raise TypeError(f"{name} must be a contiguous float32 CUDA tensor")
    return t


def sdtw_value_grad(Z, X_concat, offsets, gamma, out_values=None, out_grad=None, want_grad=True, stream=None):
    """values[k] = Soft-DTW^gamma(x_k, Z); grad = sum_k d value_k / d Z (include/sdtw.h).  Device tensors in,
    device tensors out (allocated here unless given).  want_grad=False runs the forward-only scoring sweep."""
    import torch
    Z = _dev_f32(Z, "Z")
    X = _dev_f32(X_concat, "X_concat")
    m, d = _dims(Z)
    off, offp, N = _offsets(offsets)
    if out_values is None:
        out_values = torch.empty(N, dtype=torch.float32, device=Z.device)
    if want_grad and out_grad is None:
        out_grad = torch.empty_like(Z)
    with torch.cuda.device(Z.device):
        _check(_lib.sdtw_value_grad(_ptr(Z), m, d, _ptr(X), offp, N, float(gamma), _ptr(out_values),
                                    _ptr(out_grad) if want_grad else None, _stream(stream)))
    return out_values, (out_grad if want_grad else None)


def sdtw_value_static(Z, X_concat, offsets, gamma, out_values, stream=None):
    """Soft-DTW values of every pair, for callers that must not allocate device memory (a guest inside another
    program's memory pool, a latency-bound loop, a fixed-footprint service): the library call behind this uses only its
    built-in 32 MiB scratch array and the tensors passed in.  So `out_values` (float32, CUDA, one entry per pair) is
    REQUIRED here -- this wrapper, too, allocates nothing on the device.  Problems beyond the array or beyond 64 pairs
    raise SdtwError(SDTW_ERR_STATIC_LIMIT).  Calls on one GPU share the array: keep them stream-ordered.  Returns
    out_values (bitwise what sdtw_value_grad(..., want_grad=False) computes)."""
    Z = _dev_f32(Z, "Z")
    X = _dev_f32(X_concat, "X_concat")
    out_values = _dev_f32(out_values, "out_values")
    m, d = _dims(Z)
    off, offp, N = _offsets(offsets)
    if out_values.numel() != N:
        raise ValueError("out_values must have one entry per pair")
    import torch
    with torch.cuda.device(Z.device):
        _check(_lib.sdtw_value_static(_ptr(Z), m, d, _ptr(X), offp, N, float(gamma), _ptr(out_values), _stream(stream)))
    return out_values


def sdtw_barycenter(Z_inout, X_concat, offsets, gamma, iters, step, out_values=None, out_objective=None, stream=None):
    """iters fixed-step gradient-descent iterations, in place on Z_inout.  Returns (Z_inout, values, objective)."""
    import torch
    Z = _dev_f32(Z_inout, "Z_inout")
    X = _dev_f32(X_concat, "X_concat")
    m, d = _dims(Z)
    off, offp, N = _offsets(offsets)
    if out_values is None:
        out_values = torch.zeros(N, dtype=torch.float32, device=Z.device)
    if out_objective is None:
        out_objective = torch.zeros(max(int(iters), 0), dtype=torch.float32, device=Z.device)
    with torch.cuda.device(Z.device):
        _check(_lib.sdtw_barycenter(_ptr(Z), m, d, _ptr(X), offp, N, float(gamma), int(iters), float(step),
                                    _ptr(out_values), _ptr(out_objective) if iters > 0 else None, _stream(stream)))
    return Z, out_values, out_objective


def _weights(weights, N):
    if weights is None:
        return None, None
    w = np.ascontiguousarray(np.asarray(weights, dtype=np.float32))
    if w.shape != (N,):
        raise ValueError("weights must have one entry per pair")
    return w, ctypes.c_void_p(w.ctypes.data)


def sdtw_value_grad_ex(Z, X_concat, offsets, gamma, weights=None, band=-1, out_values=None, out_grad=None,
                       out_objective=None, want_grad=True, stream=None):
    """sdtw_value_grad with eq. 7 weights (host array, one per pair) and a Sakoe-Chiba band (include/sdtw.h).
    Returns (values, grad or None, objective[1])."""
    import torch
    Z = _dev_f32(Z, "Z")
    X = _dev_f32(X_concat, "X_concat")
    m, d = _dims(Z)
    off, offp, N = _offsets(offsets)
    w, wp = _weights(weights, N)
    if out_values is None:
        out_values = torch.empty(N, dtype=torch.float32, device=Z.device)
    if want_grad and out_grad is None:
        out_grad = torch.empty_like(Z)
    if out_objective is None:
        out_objective = torch.zeros(1, dtype=torch.float32, device=Z.device)
    with torch.cuda.device(Z.device):
        _check(_lib.sdtw_value_grad_ex(_ptr(Z), m, d, _ptr(X), offp, N, float(gamma), wp, int(band), _ptr(out_values),
                                       _ptr(out_grad) if want_grad else None, _ptr(out_objective), _stream(stream)))
    return out_values, (out_grad if want_grad else None), out_objective


def sdtw_barycenter_ex(Z_inout, X_concat, offsets, gamma, iters, step, weights=None, band=-1, out_values=None,
                       out_objective=None, stream=None):
    """sdtw_barycenter on eq. 7's weighted objective with an optional band.  Returns (Z_inout, values, objective)."""
    import torch
    Z = _dev_f32(Z_inout, "Z_inout")
    X = _dev_f32(X_concat, "X_concat")
    m, d = _dims(Z)
    off, offp, N = _offsets(offsets)
    w, wp = _weights(weights, N)
    if out_values is None:
        out_values = torch.zeros(N, dtype=torch.float32, device=Z.device)
    if out_objective is None:
        out_objective = torch.zeros(max(int(iters), 0), dtype=torch.float32, device=Z.device)
    with torch.cuda.device(Z.device):
        _check(_lib.sdtw_barycenter_ex(_ptr(Z), m, d, _ptr(X), offp, N, float(gamma), wp, int(band), int(iters),
                                       float(step), _ptr(out_values), _ptr(out_objective) if iters > 0 else None,
                                       _stream(stream)))
    return Z, out_values, out_objective


def sdtw_barycenter_backtracking(Z_inout, X_concat, offsets, gamma, iters, step0, shrink=0.5, c1=1e-4, max_trials=20,
                                 weights=None, band=-1, out_values=None, stream=None):
    """Descent with an Armijo backtracking line search, in place on Z_inout (include/sdtw.h; blocks).
    Returns (Z_inout, values (dev, N), objective (iters + 1,) f64, steps (iters,) f32, trials (iters,) i32)."""
    import torch
    Z = _dev_f32(Z_inout, "Z_inout")
    X = _dev_f32(X_concat, "X_concat")
    m, d = _dims(Z)
    off, offp, N = _offsets(offsets)
    w, wp = _weights(weights, N)
    if out_values is None:
        out_values = torch.zeros(N, dtype=torch.float32, device=Z.device)
    obj = np.zeros(int(iters) + 1, np.float64)
    steps = np.zeros(max(int(iters), 1), np.float32)
    trials = np.zeros(max(int(iters), 1), np.int32)
    with torch.cuda.device(Z.device):
        _check(_lib.sdtw_barycenter_backtracking(_ptr(Z), m, d, _ptr(X), offp, N, float(gamma), wp, int(band), int(iters),
                                                 float(step0), float(shrink), float(c1), int(max_trials), _ptr(out_values),
                                                 ctypes.c_void_p(obj.ctypes.data), ctypes.c_void_p(steps.ctypes.data),
                                                 ctypes.c_void_p(trials.ctypes.data), _stream(stream)))
    return Z, out_values, obj, steps[:iters], trials[:iters]


def sdtw_barycenter_lbfgs(Z_inout, X_concat, offsets, gamma, iters, hist, step0, shrink=0.5, c1=1e-4, max_trials=20,
                          weights=None, band=-1, out_values=None, stream=None):
    """L-BFGS (Table 1's optimiser) with an Armijo backtracking line search, in place on Z_inout (include/sdtw.h; blocks).
    Returns (Z_inout, values (dev, N), objective (iters + 1,) f64, steps (iters,) f32, trials (iters,) i32)."""
    import torch
    Z = _dev_f32(Z_inout, "Z_inout")
    X = _dev_f32(X_concat, "X_concat")
    m, d = _dims(Z)
    off, offp, N = _offsets(offsets)
    w, wp = _weights(weights, N)
    if out_values is None:
        out_values = torch.zeros(N, dtype=torch.float32, device=Z.device)
    obj = np.zeros(int(iters) + 1, np.float64)
    steps = np.zeros(max(int(iters), 1), np.float32)
    trials = np.zeros(max(int(iters), 1), np.int32)
    with torch.cuda.device(Z.device):
        _check(_lib.sdtw_barycenter_lbfgs(_ptr(Z), m, d, _ptr(X), offp, N, float(gamma), wp, int(band), int(iters), int(hist),
                                          float(step0), float(shrink), float(c1), int(max_trials), _ptr(out_values),
                                          ctypes.c_void_p(obj.ctypes.data), ctypes.c_void_p(steps.ctypes.data),
                                          ctypes.c_void_p(trials.ctypes.data), _stream(stream)))
    return Z, out_values, obj, steps[:iters], trials[:iters]


def sdtw_dtw_score(Z, X_concat, offsets, stream=None):
    """eq. 8: (DTW [N] f32, |pi| [N] i32, d_score [N] f32) of every cycle against the prototype Z (include/sdtw.h)."""
    import torch
    Z = _dev_f32(Z, "Z")
    X = _dev_f32(X_concat, "X_concat")
    m, d = _dims(Z)
    off, offp, N = _offsets(offsets)
    dtw = torch.empty(N, dtype=torch.float32, device=Z.device)
    plen = torch.empty(N, dtype=torch.int32, device=Z.device)
    score = torch.empty(N, dtype=torch.float32, device=Z.device)
    with torch.cuda.device(Z.device):
        _check(_lib.sdtw_dtw_score(_ptr(Z), m, d, _ptr(X), offp, N, _ptr(dtw), _ptr(plen), _ptr(score), _stream(stream)))
    return dtw, plen, score


def sdtw_subdtw(Z_ref, X_windows, offsets, stream=None):
    """eq. 2: (Sub-DTW value [N] f32, a* [N] i32, b* [N] i32) of the reference Z_ref against each window (sdtw.h)."""
    import torch
    Z = _dev_f32(Z_ref, "Z_ref")
    X = _dev_f32(X_windows, "X_windows")
    m, d = _dims(Z)
    off, offp, N = _offsets(offsets)
    val = torch.empty(N, dtype=torch.float32, device=Z.device)
    a = torch.empty(N, dtype=torch.int32, device=Z.device)
    b = torch.empty(N, dtype=torch.int32, device=Z.device)
    with torch.cuda.device(Z.device):
        _check(_lib.sdtw_subdtw(_ptr(Z), m, d, _ptr(X), offp, N, _ptr(val), _ptr(a), _ptr(b), _stream(stream)))
    return val, a, b


def sdtw_gd_update(Z_inout, G, step, stream=None):
    import torch
    Z = _dev_f32(Z_inout, "Z_inout")
    G = _dev_f32(G, "G")
    assert G.numel() == Z.numel()
    with torch.cuda.device(Z.device):
        _check(_lib.sdtw_gd_update(_ptr(Z), _ptr(G), Z.numel(), float(step), _stream(stream)))
    return Z


def _host_f32(a, name):
    """numpy float32 C-contiguous array or CPU torch tensor (pinned or not) -> (keepalive, pointer)."""
    if a is None:
        return None, None
    if isinstance(a, np.ndarray):
        if a.dtype != np.float32 or not a.flags.c_contiguous:
            raise TypeError(f"{name} must be C-contiguous float32")
        return a, ctypes.c_void_p(a.ctypes.data)
    import torch
    if isinstance(a, torch.Tensor) and (not a.is_cuda) and a.dtype == torch.float32 and a.is_contiguous():
        return a, ctypes.c_void_p(a.data_ptr())
    raise TypeError(f"{name} must be a float32 numpy array or CPU tensor")


def sdtw_value_grad_host(Z, X_concat, offsets, gamma, out_values, out_grad, stream=0):
    """Host-buffer variant: H2D copies, the device path, D2H copies and a stream sync inside one C call."""
    kz, pz = _host_f32(Z, "Z")
    kx, px = _host_f32(X_concat, "X_concat")
    kv, pv = _host_f32(out_values, "out_values")
    kg, pg = _host_f32(out_grad, "out_grad")
    m = Z.shape[0]
    d = 1 if len(Z.shape) == 1 else Z.shape[1]
    off, offp, N = _offsets(offsets)
    _check(_lib.sdtw_value_grad_host(pz, m, d, px, offp, N, float(gamma), pv, pg,
                                     ctypes.c_void_p(stream if isinstance(stream, int) else stream.cuda_stream)))
    return out_values, out_grad


def sdtw_barycenter_host(Z_inout, X_concat, offsets, gamma, iters, step, out_values=None, out_objective=None, stream=0):
    kz, pz = _host_f32(Z_inout, "Z_inout")
    kx, px = _host_f32(X_concat, "X_concat")
    kv, pv = _host_f32(out_values, "out_values")
    ko, po = _host_f32(out_objective, "out_objective")
    m = Z_inout.shape[0]
    d = 1 if len(Z_inout.shape) == 1 else Z_inout.shape[1]
    off, offp, N = _offsets(offsets)
    _check(_lib.sdtw_barycenter_host(pz, m, d, px, offp, N, float(gamma), int(iters), float(step), pv, po,
                                     ctypes.c_void_p(stream if isinstance(stream, int) else stream.cuda_stream)))
    return Z_inout, out_values, out_objective


def sdtw_workspace_bytes(m, d, offsets, want_grad=True) -> int:
    off, offp, N = _offsets(offsets)
    return int(_lib.sdtw_workspace_bytes(int(m), int(d), offp, N, 1 if want_grad else 0))


def sdtw_workspace_bytes_ex(m, d, offsets, want_grad=True, band=-1) -> int:
    offp, N = _offsets(offsets)[1:]
    return int(_lib.sdtw_workspace_bytes_ex(int(m), int(d), offp, N, 1 if want_grad else 0, int(band)))


def sdtw_dtw_workspace_bytes(m, d, offsets) -> int:
    offp, N = _offsets(offsets)[1:]
    return int(_lib.sdtw_dtw_workspace_bytes(int(m), int(d), offp, N))


def sdtw_set_workspace(tensor_or_none):
    """Register a device byte buffer (torch uint8 CUDA tensor, kept alive by the caller) or None to unregister."""
    if tensor_or_none is None:
        _check(_lib.sdtw_set_workspace(None, 0))
    else:
        t = tensor_or_none
        _check(_lib.sdtw_set_workspace(ctypes.c_void_p(t.data_ptr()), t.numel() * t.element_size()))


def sdtw_set_workspace_limit(nbytes: int = 0):
    """Workspace budget of the calls that follow (0 = unset): beyond it the pair set is evaluated in waves (sdtw.h)."""
    _check(_lib.sdtw_set_workspace_limit(int(nbytes)))


def sdtw_launch_count() -> int:
    return int(_lib.sdtw_launch_count())


def sdtw_last_wave_count() -> int:
    """Waves of pairs this thread's last value_grad / barycenter call was split into (1 = unsplit)."""
    return int(_lib.sdtw_last_wave_count())


def sdtw_profile_enable(on: bool):
    _check(_lib.sdtw_profile_enable(1 if on else 0))


def sdtw_profile_read():
    f, b, o = ctypes.c_double(0), ctypes.c_double(0), ctypes.c_double(0)
    n = ctypes.c_int64(0)
    _check(_lib.sdtw_profile_read(ctypes.byref(f), ctypes.byref(b), ctypes.byref(o), ctypes.byref(n)))
    return dict(ms_forward=f.value, ms_backward=b.value, ms_other=o.value, evaluations=n.value)


def sdtw_tile_info():
    v = [ctypes.c_int32(0) for _ in range(5)]
    _check(_lib.sdtw_tile_info(*[ctypes.byref(x) for x in v]))
    return dict(cols_per_thread=v[0].value, strip_cols=v[1].value, ckpt_steps=v[2].value, chunk_steps=v[3].value,
                rows_per_step=v[4].value)


def sdtw_measure_mufu_peak(kind: int = 0):
    """Measured special-function results per second on the current device (0 = ex2, 1 = lg2, 2 = rcp) and SM count."""
    r, n = ctypes.c_double(0), ctypes.c_int32(0)
    _check(_lib.sdtw_measure_mufu_peak(int(kind), ctypes.byref(r), ctypes.byref(n)))
    return r.value, n.value


def sdtw_set_reverse_mode(dense: bool):
    """dense=True visits every cell in the reverse pass; False (default) skips chunks whose incoming flow is +0."""
    _check(_lib.sdtw_set_reverse_mode(1 if dense else 0))


def sdtw_set_reverse_kernel(which: int = -1):
    """-1 automatic, 0 one warp per strip (throughput regime), 1 one CTA per strip (latency regime).  Same arithmetic."""
    _check(_lib.sdtw_set_reverse_kernel(int(which)))


def sdtw_set_forward_rings(mode=1):
    """0 / False: a boundary column per strip; 1 / True (default): rings when the columns would be large; 2: rings whenever
    the problem has more strips than resident warps (include/sdtw_debug.h).  Same values."""
    _check(_lib.sdtw_set_forward_rings(int(mode)))


def sdtw_set_schedule(unit_strips: int = 0):
    """Forward schedule tuning: adjacent strips of one pair per unit (0 = automatic).  Results do not change."""
    _check(_lib.sdtw_set_schedule(int(unit_strips)))


def sdtw_set_schedule_tail(tail_strips: int = -1, tail_unit: int = 0):
    """Forward schedule tuning: size of the small units at the end of the queue (-1 = automatic)."""
    _check(_lib.sdtw_set_schedule_tail(int(tail_strips), int(tail_unit)))


def sdtw_reverse_stats():
    """(strip-chunk units, units skipped) of the last reverse pass; synchronises the device."""
    a, b = ctypes.c_uint64(0), ctypes.c_uint64(0)
    _check(_lib.sdtw_reverse_stats(ctypes.byref(a), ctypes.byref(b)))
    return a.value, b.value
