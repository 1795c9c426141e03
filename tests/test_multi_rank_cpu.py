"""World-size-2 `gloo` test of the multi-GPU plan on the CPU.

Points are independent units keyed by their GLOBAL id, so rank r renders the sub-range
`cfs.shard_points(P, r, world)` into a private image and ONE exchange step follows: an
all-reduce of the image (sum for HIST / RGBA, min on the int64 view of the depth||colour keys).
Here each rank's renderer is the oracle (no GPU in this container); what is under test is the
host logic that bench.py --gpus N uses: the sharding arithmetic, the reduce operators and
that the reduced image equals the single-process render bit for bit.
"""
from __future__ import annotations

import os
import socket
import sys

import numpy as np
import pytest

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
    from oracle import cfs_oracle
    from paper_2606_02226_b200 import cfs, workloads as W

    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    w = W.config(cfg).scaled(n_points=n_points, iterations=60, width=96, height=64)
    off, n = cfs.shard_points(n_points, rank, world)
    img, ctr = cfs_oracle.render(w.system, w.render, n_points=n, point_offset=off)
    # the binding's exchange step (cfs.allreduce_image), on CPU tensors in the library's layout
    if w.render.out_mode == "hist_u32":
        t = torch.from_numpy(img.astype(np.uint32).view(np.int32).copy())
        red = cfs.allreduce_image(t, "hist_u32").numpy().view(np.uint32)
    elif w.render.out_mode == "rgba_f32":
        t = torch.from_numpy(np.ascontiguousarray(img, dtype=np.float64))
        red = cfs.allreduce_image(t, "rgba_f32").numpy()
    else:
        # depth keys are < 2^63 unless empty (all ones = -1 as int64): the helper flips the sign bit so that
        # the signed MIN of the int64 view orders like the unsigned keys (what ncclMin on int64 needs too)
        t = torch.from_numpy(img.view(np.int64).copy())
        red = cfs.allreduce_image(t, "depth_u64").numpy().view(np.uint64)
    c = torch.from_numpy(np.asarray(ctr, dtype=np.int64).copy())
    dist.all_reduce(c, op=dist.ReduceOp.SUM)
    if rank == 0:
        np.save(os.path.join(out_dir, f"img_{cfg}.npy"), red)
        np.save(os.path.join(out_dir, f"ctr_{cfg}.npy"), c.numpy())
    dist.barrier()
    dist.destroy_process_group()


@pytest.mark.parametrize("cfg", [0, 1, 4])
def test_two_ranks_reduce_to_single_render(oracle, tmp_path, cfg):
    import torch.multiprocessing as mp
    from paper_2606_02226_b200 import workloads as W

    n_points, world = 1001, 2          # odd: the ranges are ragged
    mp.spawn(_worker, args=(world, _free_port(), cfg, n_points, str(tmp_path)), nprocs=world, join=True)
    w = W.config(cfg).scaled(n_points=n_points, iterations=60, width=96, height=64)
    want, wc = oracle.render(w.system, w.render)
    got = np.load(tmp_path / f"img_{cfg}.npy")
    gc = np.load(tmp_path / f"ctr_{cfg}.npy")
    assert int(gc[0]) == int(wc[0]) and int(gc[1]) == int(wc[1])
    if cfg == 1:
        # integer-valued colours (DESIGN R9): sums are exact in double, so equality is exact too
        assert np.array_equal(got, want)
    else:
        assert np.array_equal(got, want)


def test_shard_points_partition():
    from paper_2606_02226_b200 import cfs
    for n in (0, 1, 7, 1 << 20, (1 << 26) + 3):
        for world in (1, 2, 3, 8):
            parts = [cfs.shard_points(n, r, world) for r in range(world)]
            assert parts[0][0] == 0
            assert sum(c for _, c in parts) == n
            for (o0, c0), (o1, _) in zip(parts, parts[1:]):
                assert o0 + c0 == o1
            assert max(c for _, c in parts) - min(c for _, c in parts) <= 1
