"""Multi-rank CUDA test of SURVEY.md 8(e): pairs partitioned over the GPUs of one node (dist.partition_pairs), one
sdtw_value_grad per rank, the rank-ordered reduction over NCCL, sdtw_gd_update -- against the single-GPU call on the
union.  Collected only where at least two GPUs are visible (the development pool has one)."""
import os
import socket

import numpy as np
import pytest

from paper_2404_12134_b200 import synth

pytestmark = pytest.mark.gpu


def _ngpu():
    try:
        import torch
        return torch.cuda.device_count()
    except Exception:
        return 0


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def _worker(rank, world, port, out_dir):
    import torch
    import torch.distributed as dist
    from paper_2404_12134_b200 import binding as B
    from paper_2404_12134_b200 import dist as D
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    torch.cuda.set_device(rank)
    dist.init_process_group("nccl", rank=rank, world_size=world, device_id=torch.device("cuda", rank))
    cfg = synth.scaled(synth.CONFIGS[4], 0.1, N=12)
    data = synth.make(cfg)
    mine = D.partition_pairs(data["lengths"], world)[rank]
    Xl, offl = D.take_pairs(data["X"], data["offsets"], mine)
    Z = torch.from_numpy(data["Z0"]).cuda()
    X = torch.from_numpy(Xl).cuda()
    step = 0.02 / cfg.N
    objs = []
    for _ in range(3):
        vals, G = B.sdtw_value_grad(Z, X, offl, cfg.gamma)
        D.allreduce_sum_(G)
        o = vals.double().sum()
        dist.all_reduce(o)
        objs.append(float(o))
        B.sdtw_gd_update(Z, G, step)
    torch.cuda.synchronize()
    np.save(os.path.join(out_dir, f"Z{rank}.npy"), Z.cpu().numpy())
    if rank == 0:
        np.save(os.path.join(out_dir, "obj.npy"), np.array(objs))
    dist.barrier()
    dist.destroy_process_group()


@pytest.mark.skipif(_ngpu() < 2, reason="needs at least two GPUs on the node")
@pytest.mark.timeout(600)
def test_partitioned_descent_matches_single_gpu(tmp_path):
    import torch
    import torch.multiprocessing as mp
    from paper_2404_12134_b200 import binding as B
    world = 2
    mp.spawn(_worker, args=(world, _free_port(), str(tmp_path)), nprocs=world, join=True)
    cfg = synth.scaled(synth.CONFIGS[4], 0.1, N=12)
    data = synth.make(cfg)
    Z = torch.from_numpy(data["Z0"]).cuda()
    X = torch.from_numpy(data["X"]).cuda()
    Zs, _, obj = B.sdtw_barycenter(Z.clone(), X, data["offsets"], cfg.gamma, 3, 0.02 / cfg.N)
    Z0, Z1 = np.load(tmp_path / "Z0.npy"), np.load(tmp_path / "Z1.npy")
    assert np.array_equal(Z0, Z1), "every rank must hold the same barycenter bits"
    ref = Zs.cpu().numpy()
    moved = np.linalg.norm(ref - data["Z0"])
    assert np.linalg.norm(Z0 - ref) <= 1e-4 * moved          # only the order of the sum over pairs differs
    assert np.allclose(np.load(tmp_path / "obj.npy"), obj.cpu().numpy(), rtol=1e-5)
