"""The paper's set-up arithmetic around the C ABI calls: what a user computes on the host BEFORE or BETWEEN calls of
include/sdtw.h when following the paper's recipe.  None of it is on the hot path, and none of it is in binding.py,
which only marshals arguments.

  eq7_weights                 eq. 7's lambda_k / n_k
  default_barycenter_length   "by default m_b = max m_i"
  table1_band                 Table 1's Sakoe-Chiba bandwidth, 0.6 x the longest length (C18)
  segment_cycles              the sliding-window loop of Step 1                       (C21)
"""
from __future__ import annotations

import numpy as np


def eq7_weights(lengths, lam=None):
    """w_k = lambda_k / n_k of eq. 7; lambda defaults to 1."""
    n = np.asarray(lengths, np.float64)
    return ((1.0 if lam is None else np.asarray(lam, np.float64)) / n).astype(np.float32)


def table1_band(m, lengths, fraction=0.6):
    """Table 1's Sakoe-Chiba bandwidth: a fraction of the longest signal length, in cells."""
    return int(np.floor(fraction * max(int(m), int(np.max(lengths)))))


def default_barycenter_length(lengths) -> int:
    """The barycenter length the paper uses when none is given: m_b = max_i m_i, the longest cycle."""
    return int(np.max(np.asarray(lengths)))


def segment_cycles(Y, X_ref, alpha_frac=-0.15, subdtw=None):
    """The sliding-window loop of PAPER.md:135-145 (Step 1).  Y: the stream [T][d], X_ref: the reference quasi-period
    [M][d] (device float32 tensors when `subdtw` is None).  Window [ws, ws + 2M); Sub-DTW gives a*, b*; the cycle
    Y[ws + a* .. ws + b*] is recorded; the next window starts at ws + b* + 1 + alpha_frac * M.  Reading C21: the
    extracted text prints "ws = b* alpha" with alpha = 0.15 M "to ensure that missing data between two cycles does not
    interfere"; the default steps BACK by alpha so that the start of the next cycle stays inside the next window
    (a positive alpha_frac gives the other reading, a skipped gap).  The paper leaves termination open (its ws < N
    never fails when stepping back): the loop advances by at least M/4 per window and stops when fewer than M/2
    samples remain.  `subdtw(ref, window) -> (value, a, b)` replaces the CUDA call (the tests pass the oracle's mirror:
    this loop holds none of the method's arithmetic).  Returns a list of (start, end, value), end inclusive."""
    M = X_ref.shape[0]
    T = Y.shape[0]
    alpha = int(alpha_frac * M)
    if subdtw is None:
        from . import binding                      # the CUDA call; imported here so that the helpers above need no library
        def subdtw(ref, win):
            v, a, b = binding.sdtw_subdtw(ref, win.contiguous(), np.array([0, win.shape[0]], np.int64))
            return float(v.item()), int(a.item()), int(b.item())
    cycles = []
    ws = 0
    while T - ws >= max(1, M // 2):
        we = min(T, ws + 2 * M)
        v, a, b = subdtw(X_ref, Y[ws:we])
        cycles.append((ws + a, ws + b, v))
        ws = max(ws + b + 1 + alpha, ws + max(1, M // 4))
    return cycles
