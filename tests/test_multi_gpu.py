"""World-size-2 CUDA test of the sharded render: one process per GPU, NCCL.  Each rank
renders its range of the global point ids with cfs_render on its own device and the images are combined by
cfs.allreduce_image on DEVICE tensors (sum; for DEPTH the unsigned min carried by a sign-flipped int64 MIN) -- the
exchange step bench.py --gpus N times.  The reduced image must equal the single-GPU render of all points bit for bit
(HIST, DEPTH; RGBA with integer-valued colours below 2^24).  Skipped on a box with fewer than two GPUs (the round's
GPU boxes have one; tests/test_multi_rank_cpu.py covers the same host logic over gloo)."""
from __future__ import annotations

import os
import socket
import sys

import numpy as np
import pytest

pytestmark = pytest.mark.gpu
ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _free_port() -> int:
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    port = s.getsockname()[1]
    s.close()
    return port


def _worker(rank: int, world: int, port: int, cfg: int, n_points: int, out_dir: str):
    if ROOT not in sys.path:
        sys.path.insert(0, ROOT)
    import torch
    import torch.distributed as dist
    from paper_2606_02226_b200 import cfs, workloads as W

    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    torch.cuda.set_device(rank)
    dist.init_process_group("nccl", rank=rank, world_size=world, device_id=torch.device("cuda", rank))
    w = W.config(cfg).scaled(n_points=n_points, iterations=60, width=320, height=180)
    sysh = cfs.cfs_create(w.system)
    img = cfs.new_image(w.render, device=f"cuda:{rank}")
    ctr = torch.zeros(2, dtype=torch.int64, device=f"cuda:{rank}")
    cfs.render_sharded(sysh, w.render, img, rank, world, d_counters=ctr, variant="direct")
    dist.all_reduce(ctr, op=dist.ReduceOp.SUM)
    torch.cuda.synchronize()
    if rank == 0:
        whole = cfs.new_image(w.render, device="cuda:0")
        wc = torch.zeros(2, dtype=torch.int64, device="cuda:0")
        cfs.cfs_render(sysh, cfs.make_args(w.render, d_image=whole, d_counters=wc, variant="direct"))
        torch.cuda.synchronize()
        np.save(os.path.join(out_dir, f"ok_{cfg}.npy"), np.array([int(torch.equal(img, whole)), int(torch.equal(ctr, wc))]))
    sysh.close()
    dist.barrier()
    dist.destroy_process_group()


@pytest.mark.parametrize("cfg", [0, 1, 4])
def test_two_gpus_reduce_to_the_single_gpu_render(tmp_path, cfg):
    import torch
    if torch.cuda.device_count() < 2:
        pytest.skip("needs two GPUs")
    import torch.multiprocessing as mp
    mp.spawn(_worker, args=(2, _free_port(), cfg, 20001, str(tmp_path)), nprocs=2, join=True)
    ok = np.load(tmp_path / f"ok_{cfg}.npy")
    assert ok[0] == 1 and ok[1] == 1
