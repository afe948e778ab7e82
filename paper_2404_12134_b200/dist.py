"""Sharding of the pair set over ranks (one process per GPU) -- DESIGN.md section 9.

Pairs are independent ("completely independent for each pair"), so each rank
evaluates its own subset with the single-GPU library call and the only exchange is one
all-reduce (sum) of the m*d gradient per evaluation / descent step.  This module holds the
host-side logic only (partition, all-reduce, the distributed descent loop); the evaluation
itself is passed in as a callable so that the same code drives the CUDA binding on GPUs
(NCCL) and, in the CPU tests, a stand-in evaluator over gloo.
"""
from __future__ import annotations

import numpy as np


def partition_pairs(lengths, world_size: int):
    """Longest-processing-time partition of pairs by n_k.  Returns a list (per rank) of sorted
    pair-index arrays.  Deterministic: ties broken by pair index, ranks filled lowest-load first."""
    lengths = np.asarray(lengths, dtype=np.int64)
    order = sorted(range(len(lengths)), key=lambda k: (-int(lengths[k]), k))
    loads = [0] * world_size
    parts = [[] for _ in range(world_size)]
    for k in order:
        r = min(range(world_size), key=lambda q: (loads[q], q))
        parts[r].append(k)
        loads[r] += int(lengths[k])
    return [np.array(sorted(p), dtype=np.int64) for p in parts]


def take_pairs(X_concat, offsets, idx):
    """Gather the cycles idx (host arrays) into a new (X_concat, offsets)."""
    offsets = np.asarray(offsets, dtype=np.int64)
    if len(idx) == 0:
        return X_concat[:0].copy(), np.zeros(1, np.int64)
    chunks = [X_concat[offsets[k]:offsets[k + 1]] for k in idx]
    lens = np.array([c.shape[0] for c in chunks], dtype=np.int64)
    off = np.zeros(len(idx) + 1, np.int64)
    np.cumsum(lens, out=off[1:])
    return np.ascontiguousarray(np.concatenate(chunks, axis=0)), off


def allreduce_sum_(tensor, group=None):
    """In-place sum over ranks (NCCL on GPUs, gloo on CPU); a no-op without an initialised process group.

    Bitwise reproducible and identical on every rank, whatever algorithm the collective library picks (SURVEY.md
    8(e)): the partials are ALL-GATHERED and every rank adds them itself in rank order 0, 1, ..., R-1 (a fixed
    left-to-right chain in the tensor's dtype), instead of trusting the reduction order of all_reduce.  The exchange
    is m*d floats per rank (120 KB at m = 30000): latency bound either way."""
    import torch
    import torch.distributed as dist
    if dist.is_available() and dist.is_initialized() and dist.get_world_size(group) > 1:
        world = dist.get_world_size(group)
        flat = tensor.contiguous().view(-1)
        gathered = torch.empty(world * flat.numel(), dtype=flat.dtype, device=flat.device)
        dist.all_gather_into_tensor(gathered, flat, group=group)
        parts = gathered.view(world, flat.numel())
        acc = parts[0].clone()
        for r in range(1, world):
            acc += parts[r]
        tensor.copy_(acc.view_as(tensor))
    return tensor


def distributed_descent(Z, local_value_grad, update, iters: int, step: float, group=None):
    """Fixed-step descent with the gradient summed over ranks.

    local_value_grad(Z) -> (values_local, grad_local) for this rank's pairs (grad_local is a torch tensor on the
    device the collective runs on); update(Z, G, step) applies Z <- Z - step * G in place.  Every rank holds the
    same Z throughout because every rank applies the same reduced gradient.  Returns (Z, last local values,
    list of global objectives)."""
    import torch
    objective = []
    values = None
    for _ in range(iters):
        values, G = local_value_grad(Z)
        obj = values.double().sum().reshape(1).to(G.device)
        allreduce_sum_(G, group)
        allreduce_sum_(obj, group)
        objective.append(float(obj.item()))
        update(Z, G, step)
    return Z, values, objective
