"""Helpers of the GPU parity tests: run one workload through the C ABI (CUDA) and through the
oracle on the same seeded inputs."""
from __future__ import annotations

import numpy as np


def gpu_render(cfs, w, t=None, cloud=None, variant="auto", n_points=None, point_offset=None, image=None,
               want_counters=True, flags=0, scratch_bytes=None):
    """cfs_render through the binding. Returns (numpy image, counters[2])."""
    import torch
    sysh = cfs.cfs_create(w.system)
    img = cfs.new_image(w.render) if image is None else image
    ctr = torch.zeros(2, dtype=torch.int64, device="cuda") if want_counters else None
    d_cloud = cfs.cloud_to_device(cloud) if cloud is not None else None
    args = cfs.make_args(w.render, d_image=img, d_cloud=d_cloud, d_counters=ctr, t=t, variant=variant,
                         n_points=n_points, point_offset=point_offset, flags=flags)
    if variant == "binned" or scratch_bytes is not None:       # scratch of the tile-binned variant
        nbytes = cfs.cfs_binned_scratch_bytes(sysh, args) if scratch_bytes is None else scratch_bytes
        scratch = torch.empty(max(int(nbytes), 1), dtype=torch.uint8, device="cuda")
        args = cfs.make_args(w.render, d_image=img, d_cloud=d_cloud, d_counters=ctr, t=t, variant=variant,
                             n_points=n_points, point_offset=point_offset, flags=flags, d_scratch=scratch)
    cfs.cfs_render(sysh, args)
    torch.cuda.synchronize()
    out = cfs.image_to_numpy(img, w.render.out_mode)
    c = ctr.cpu().numpy().astype(np.uint64) if want_counters else None
    sysh.close()
    return out, c


def gpu_trace(cfs, w, t=None, cloud=None, n_points=None, point_offset=None, flags=0):
    import torch
    n = int(w.render.n_points if n_points is None else n_points)
    I = int(w.render.iterations)
    sysh = cfs.cfs_create(w.system)
    picks = torch.zeros((n, I), dtype=torch.uint8, device="cuda")
    fg = torch.zeros((n, 3), dtype=torch.float32, device="cuda")
    fq = torch.zeros((n, 3), dtype=torch.float32, device="cuda")
    al = torch.zeros(n, dtype=torch.uint8, device="cuda")
    d_cloud = cfs.cloud_to_device(cloud) if cloud is not None else None
    args = cfs.make_args(w.render, d_cloud=d_cloud, t=t, n_points=n_points, point_offset=point_offset, flags=flags)
    cfs.cfs_trace(sysh, args, picks, fg, fq, al)
    torch.cuda.synchronize()
    sysh.close()
    return picks.cpu().numpy(), fg.cpu().numpy(), fq.cpu().numpy(), al.cpu().numpy()


def density_l1(a, b):
    """Normalised-density L1 distance sum |a/sum a - b/sum b| (SURVEY 8(c) S10 iv)."""
    a = np.asarray(a, dtype=np.float64).ravel()
    b = np.asarray(b, dtype=np.float64).ravel()
    sa, sb = a.sum(), b.sum()
    if sa == 0 and sb == 0:
        return 0.0
    return float(np.abs(a / sa - b / sb).sum())
