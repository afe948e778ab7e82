"""world_size-2 gloo test of the multi-rank path's host logic (partition, all-reduce, descent loop).

No GPU here: the per-rank evaluator is the float64 oracle standing in for the CUDA call, which is what lets the
result be compared with the single-process oracle.  The collective and the loop are the product's (dist.py)."""
import os
import socket

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_2404_12134_b200 import synth
from paper_2404_12134_b200.dist import partition_pairs, take_pairs, distributed_descent, allreduce_sum_


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def _worker(rank, world, port, out_dir):
    import oracle
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    data = synth.make(1)
    cfg = data["cfg"]
    parts = partition_pairs(data["lengths"], world)
    Xl, offl = take_pairs(data["X"], data["offsets"], parts[rank])

    def local_value_grad(Z):
        v, g = oracle.value_grad(Z.numpy().astype(np.float32), Xl, offl, cfg.gamma, nthreads=1)
        return torch.from_numpy(v), torch.from_numpy(g)

    def update(Z, G, step):
        Z -= step * G

    Z = torch.from_numpy(data["Z0"].astype(np.float64))
    # one summed evaluation
    v, g = local_value_grad(Z)
    allreduce_sum_(g)
    Zf, _, obj = distributed_descent(Z.clone(), local_value_grad, update, 3, cfg.step)
    if rank == 0:
        np.save(os.path.join(out_dir, "g.npy"), g.numpy())
        np.save(os.path.join(out_dir, "Z.npy"), Zf.numpy())
        np.save(os.path.join(out_dir, "obj.npy"), np.array(obj))
    dist.barrier()
    dist.destroy_process_group()


def test_partition_is_balanced_and_complete():
    rng = np.random.default_rng(0)
    lengths = rng.integers(27000, 33001, size=100)
    for world in (1, 2, 4, 8):
        parts = partition_pairs(lengths, world)
        allk = np.sort(np.concatenate(parts))
        assert np.array_equal(allk, np.arange(100))
        loads = np.array([lengths[p].sum() for p in parts])
        assert loads.max() - loads.min() <= lengths.max()
    assert [p.tolist() for p in partition_pairs([5, 5, 5], 2)] == [[0, 2], [1]]


def test_take_pairs_roundtrip():
    data = synth.make(1)
    idx = np.array([1, 4, 6])
    X, off = take_pairs(data["X"], data["offsets"], idx)
    for q, k in enumerate(idx):
        assert np.array_equal(X[off[q]:off[q + 1]], data["X"][data["offsets"][k]:data["offsets"][k + 1]])


@pytest.mark.timeout(300)
def test_two_rank_gloo_matches_single_process(tmp_path, oracle):
    port = _free_port()
    mp.spawn(_worker, args=(2, port, str(tmp_path)), nprocs=2, join=True)
    data = synth.make(1)
    cfg = data["cfg"]
    _, G = oracle.value_grad(data["Z0"], data["X"], data["offsets"], cfg.gamma)
    g2 = np.load(tmp_path / "g.npy")
    assert np.abs(g2 - G).max() <= 1e-12 * np.abs(G).max()
    # the 2-rank loop rounds Z to fp32 when it hands it to the evaluator; mirror that in the single-process loop
    Z = data["Z0"].astype(np.float64)
    objs = []
    for _ in range(3):
        v, g = oracle.value_grad(Z.astype(np.float32), data["X"], data["offsets"], cfg.gamma)
        objs.append(v.sum())
        Z = Z - cfg.step * g
    assert np.abs(np.load(tmp_path / "Z.npy") - Z).max() <= 1e-12
    assert np.allclose(np.load(tmp_path / "obj.npy"), objs, rtol=1e-12)


def _reduce_worker(rank, world, port, out_dir):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    rng = np.random.Generator(np.random.PCG64(77 + rank))
    # magnitudes spread over 12 decades: the float32 sum depends on the order of the additions
    x = torch.from_numpy((rng.standard_normal((1000, 3)) * 10.0 ** rng.uniform(-6, 6, size=(1000, 3))).astype(np.float32))
    np.save(os.path.join(out_dir, f"part{rank}.npy"), x.numpy())
    y = allreduce_sum_(x.clone())
    np.save(os.path.join(out_dir, f"sum{rank}.npy"), y.numpy())
    dist.barrier()
    dist.destroy_process_group()


@pytest.mark.timeout(300)
def test_allreduce_is_the_rank_ordered_chain_bit_for_bit(tmp_path):
    """the reduction over ranks is an all-gather plus a fixed chain 0 + 1 + ... + R-1 in the tensor's
    dtype, so every rank holds the same bits whatever the collective library does."""
    world = 3
    mp.spawn(_reduce_worker, args=(world, _free_port(), str(tmp_path)), nprocs=world, join=True)
    parts = [np.load(tmp_path / f"part{r}.npy") for r in range(world)]
    expect = parts[0].copy()
    for r in range(1, world):
        expect = (expect + parts[r]).astype(np.float32)
    for r in range(world):
        assert np.array_equal(np.load(tmp_path / f"sum{r}.npy"), expect)
