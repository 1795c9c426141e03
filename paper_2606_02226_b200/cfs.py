"""Thin ctypes binding of libcfs_b200.so (include/cfs.h) -- argument marshalling only.

Every step of the path runs in the CUDA kernels of csrc/; PyTorch is used for device memory
and streams, nothing else.  There is no CPU fallback: if the library is missing or cannot be
loaded this module raises at import of the first symbol.
"""
from __future__ import annotations

import ctypes as C
import os
from typing import Optional, Sequence

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libcfs_b200.so")

CFS_OK, CFS_ERR_INVALID_ARG, CFS_ERR_UNSUPPORTED, CFS_ERR_CUDA, CFS_ERR_NOMEM = range(5)
GEN = {"ifs": 0, "cloud": 1}
F_TYPE = {"affine": 0, "circle_half": 1}
T_TYPE = {"affine": 0, "swirl": 1, "sinusoidal": 2, "rotate_z": 3, "twist_z": 4, "bend": 5,
          "pinhole": 6, "stretch_cos": 7, "branch": 8, "scatter": 9}
COLOR = {"none": 0, "map_index": 1, "point": 2}
OUT = {"hist_u32": 0, "rgba_f32": 1, "depth_u64": 2}
FLAGS = {"fast_trig": 1, "interpret_chain": 2, "bin_pass1_only": 4, "jit": 8, "bin_hybrid": 0x100}
VARIANT = {"auto": 0, "direct": 1, "shared_hist": 2, "warp_agg": 3, "binned": 4, "cluster_hist": 5, "depth_hiz": 6}
MB = {"red_add_u32": 0, "red_add_v4f32": 1, "atom_min_u64": 2, "ld_u64": 3, "atoms_add_u32": 4,
      "ffma": 5, "imad_wide": 6, "lop3": 7, "mufu": 8, "stream_ld128": 9, "stream_red_v4f32": 10}
EXPORTS = ["cfs_create", "cfs_destroy", "cfs_render", "cfs_render_host", "cfs_render_depth_noalloc", "cfs_render_rgba8_host", "cfs_tonemap", "cfs_resolve_rgba8", "cfs_trace",
           "cfs_microbench", "cfs_host_resolve", "cfs_specialize", "cfs_jit_check", "cfs_jit_stats", "cfs_shared_hist_max_bytes", "cfs_binned_scratch_bytes", "cfs_hiz_scratch_bytes", "cfs_binned_plan", "cfs_launch_count", "cfs_last_error",
           "cfs_version"]


class CfsError(RuntimeError):
    def __init__(self, status: int, message: str):
        super().__init__(f"cfs status {status}: {message}")
        self.status = status


class cfs_func(C.Structure):
    _fields_ = [("type", C.c_int32), ("prob", C.c_float), ("params", C.c_float * 12)]


class cfs_xform(C.Structure):
    _fields_ = [("type", C.c_int32), ("p0", C.c_float * 12), ("p1", C.c_float * 12)]


class cfs_render_args(C.Structure):
    _fields_ = [("n_points", C.c_uint64), ("point_offset", C.c_uint64), ("seed", C.c_uint64),
                ("iterations", C.c_int32), ("burn_in", C.c_int32),
                ("width", C.c_int32), ("height", C.c_int32),
                ("xmin", C.c_float), ("xmax", C.c_float), ("ymin", C.c_float), ("ymax", C.c_float),
                ("t", C.c_float), ("out_mode", C.c_int32), ("variant", C.c_int32),
                ("flags", C.c_int32),
                ("d_image", C.c_void_p), ("d_cloud", C.c_void_p), ("d_counters", C.c_void_p),
                ("d_scratch", C.c_void_p), ("scratch_bytes", C.c_uint64)]


class cfs_resolved(C.Structure):
    _fields_ = [("sx", C.c_float), ("ox", C.c_float), ("sy", C.c_float), ("oy", C.c_float),
                ("n_chain", C.c_int32), ("n_funcs", C.c_int32), ("n_thresholds", C.c_int32), ("pick_form", C.c_int32),
                ("chain_type", C.c_int32 * 8), ("chain_p", (C.c_float * 12) * 8),
                ("thresholds", C.c_uint32 * 64), ("pal8", C.c_uint32 * 64),
                ("proved", C.c_int32), ("pad_", C.c_int32)]


_lib = None


def lib():
    """Load the CUDA library (built in-tree by paper_2606_02226_b200.build). Fails loudly."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise ImportError(f"{LIB_PATH} is missing: run `python -m paper_2606_02226_b200.build` "
                              "(there is no CPU fallback)")
        L = C.CDLL(LIB_PATH)
        L.cfs_create.argtypes = [C.POINTER(C.c_void_p), C.c_int32, C.c_int32, C.POINTER(cfs_func), C.c_int32,
                                 C.POINTER(cfs_xform), C.c_int32, C.c_int32, C.POINTER(C.c_float), C.c_int32]
        L.cfs_create.restype = C.c_int
        L.cfs_destroy.argtypes = [C.c_void_p]
        L.cfs_destroy.restype = None
        L.cfs_render.argtypes = [C.c_void_p, C.POINTER(cfs_render_args), C.c_void_p]
        L.cfs_render.restype = C.c_int
        L.cfs_render_host.argtypes = [C.c_void_p, C.POINTER(cfs_render_args), C.c_void_p, C.c_void_p,
                                      C.c_void_p, C.c_void_p]
        L.cfs_render_host.restype = C.c_int
        L.cfs_render_rgba8_host.argtypes = [C.c_void_p, C.POINTER(cfs_render_args), C.c_float, C.c_float, C.c_float,
                                            C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p]
        L.cfs_render_rgba8_host.restype = C.c_int
        L.cfs_tonemap.argtypes = [C.c_void_p, C.c_int32, C.c_int32, C.c_int32, C.c_float, C.c_float,
                                  C.c_void_p, C.c_void_p, C.c_void_p]
        L.cfs_tonemap.restype = C.c_int
        L.cfs_resolve_rgba8.argtypes = [C.c_void_p, C.c_int32, C.c_int32, C.c_int32, C.c_float, C.c_float, C.c_float,
                                        C.c_void_p, C.c_void_p, C.c_void_p]
        L.cfs_resolve_rgba8.restype = C.c_int
        L.cfs_trace.argtypes = [C.c_void_p, C.POINTER(cfs_render_args), C.c_void_p, C.c_void_p, C.c_void_p,
                                C.c_void_p, C.c_void_p]
        L.cfs_trace.restype = C.c_int
        L.cfs_microbench.argtypes = [C.c_int32, C.c_void_p, C.c_uint64, C.c_uint64, C.c_int32, C.c_int32,
                                     C.c_void_p]
        L.cfs_microbench.restype = C.c_int
        L.cfs_host_resolve.argtypes = [C.c_void_p, C.POINTER(cfs_render_args), C.POINTER(cfs_resolved)]
        L.cfs_host_resolve.restype = C.c_int
        L.cfs_specialize.argtypes = [C.c_void_p, C.POINTER(cfs_render_args), C.POINTER(C.c_double)]
        L.cfs_specialize.restype = C.c_int
        L.cfs_jit_check.argtypes = [C.c_void_p, C.POINTER(cfs_render_args), C.c_int32, C.POINTER(C.c_uint64), C.POINTER(C.c_double)]
        L.cfs_jit_check.restype = C.c_int
        L.cfs_jit_stats.argtypes = [C.POINTER(C.c_uint64), C.POINTER(C.c_double)]
        L.cfs_jit_stats.restype = None
        L.cfs_shared_hist_max_bytes.argtypes = []
        L.cfs_shared_hist_max_bytes.restype = C.c_uint64
        L.cfs_binned_scratch_bytes.argtypes = [C.c_void_p, C.POINTER(cfs_render_args)]
        L.cfs_binned_scratch_bytes.restype = C.c_uint64
        L.cfs_hiz_scratch_bytes.argtypes = [C.c_int32, C.c_int32]
        L.cfs_hiz_scratch_bytes.restype = C.c_uint64
        L.cfs_render_depth_noalloc.argtypes = [C.c_void_p, C.POINTER(cfs_render_args), C.c_void_p]
        L.cfs_render_depth_noalloc.restype = C.c_int
        L.cfs_binned_plan.argtypes = [C.c_int32, C.c_int32, C.c_int32, C.c_int32, C.c_int32, C.c_int32,
                                      C.POINTER(C.c_uint32)]
        L.cfs_binned_plan.restype = C.c_int
        L.cfs_launch_count.argtypes = [C.c_int32]
        L.cfs_launch_count.restype = C.c_uint64
        L.cfs_last_error.argtypes = []
        L.cfs_last_error.restype = C.c_char_p
        L.cfs_version.argtypes = []
        L.cfs_version.restype = C.c_char_p
        _lib = L
    return _lib


def _check(status: int):
    if status != CFS_OK:
        raise CfsError(status, lib().cfs_last_error().decode())


def cfs_version() -> str:
    return lib().cfs_version().decode()


def cfs_last_error() -> str:
    return lib().cfs_last_error().decode()


def cfs_launch_count(reset: bool = False) -> int:
    return int(lib().cfs_launch_count(1 if reset else 0))


def cfs_shared_hist_max_bytes() -> int:
    return int(lib().cfs_shared_hist_max_bytes())


def _ptr(x) -> Optional[int]:
    """Device/host pointer of a torch tensor, numpy array, int or None."""
    if x is None:
        return None
    if isinstance(x, int):
        return x
    if isinstance(x, np.ndarray):
        return x.ctypes.data
    return x.data_ptr()


def _stream(stream) -> Optional[int]:
    if stream is None:
        import torch
        return torch.cuda.current_stream().cuda_stream
    if isinstance(stream, int):
        return stream
    return stream.cuda_stream


class System:
    """Owner of a cfs_system handle (cfs_create / cfs_destroy)."""

    def __init__(self, handle: int):
        self.handle = handle

    def close(self):
        if self.handle:
            lib().cfs_destroy(self.handle)
            self.handle = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


def cfs_create(system) -> System:
    """cfs_create from a description with the attributes of workloads.System."""
    nf = len(system.funcs)
    funcs = (cfs_func * max(1, nf))()
    for j, f in enumerate(system.funcs):
        funcs[j].type = F_TYPE[f.type] if isinstance(f.type, str) else int(f.type)
        funcs[j].prob = float(f.prob)
        for i, v in enumerate(f.params):
            funcs[j].params[i] = float(v)
    nc = len(system.chain)
    chain = (cfs_xform * max(1, nc))()
    for m, x in enumerate(system.chain):
        chain[m].type = T_TYPE[x.type] if isinstance(x.type, str) else int(x.type)
        for i, v in enumerate(x.p0):
            chain[m].p0[i] = float(v)
        for i, v in enumerate(x.p1):
            chain[m].p1[i] = float(v)
    pal = None
    if system.palette is not None:
        pal_arr = np.ascontiguousarray(system.palette, dtype=np.float32)
        pal = pal_arr.ctypes.data_as(C.POINTER(C.c_float))
    out = C.c_void_p()
    _check(lib().cfs_create(C.byref(out), int(system.dim), GEN[system.gen] if isinstance(system.gen, str) else int(system.gen),
                            funcs, nf, chain, nc,
                            COLOR[system.color] if isinstance(system.color, str) else int(system.color),
                            pal, 1 if getattr(system, "reuse", False) else 0))
    return System(out.value)


def make_args(render, d_image=None, d_cloud=None, d_counters=None, n_points=None, point_offset=None,
              t=None, variant="auto", flags=0, d_scratch=None) -> cfs_render_args:
    a = cfs_render_args()
    a.n_points = int(render.n_points if n_points is None else n_points)
    a.point_offset = int(render.point_offset if point_offset is None else point_offset)
    a.seed = int(render.seed)
    a.iterations = int(render.iterations)
    a.burn_in = int(render.burn_in)
    a.width = int(render.width)
    a.height = int(render.height)
    a.xmin, a.xmax, a.ymin, a.ymax = [float(np.float32(v)) for v in render.bounds]
    a.t = float(render.t if t is None else t)
    a.out_mode = OUT[render.out_mode] if isinstance(render.out_mode, str) else int(render.out_mode)
    a.variant = VARIANT[variant] if isinstance(variant, str) else int(variant)
    a.flags = sum(FLAGS[f] for f in flags) if isinstance(flags, (tuple, list)) else int(flags)
    a.d_image = _ptr(d_image)
    a.d_cloud = _ptr(d_cloud)
    a.d_counters = _ptr(d_counters)
    a.d_scratch = _ptr(d_scratch)
    a.scratch_bytes = 0 if d_scratch is None else int(d_scratch.numel() * d_scratch.element_size())
    return a


def cfs_binned_scratch_bytes(sys: System, args: cfs_render_args) -> int:
    return int(lib().cfs_binned_scratch_bytes(sys.handle, C.byref(args)))


def cfs_hiz_scratch_bytes(width: int, height: int) -> int:
    return int(lib().cfs_hiz_scratch_bytes(int(width), int(height)))


def cfs_binned_plan(width: int, height: int, out_mode, n_funcs: int, sms: int = 148, smem_optin: int = 232448) -> dict:
    mode = OUT[out_mode] if isinstance(out_mode, str) else int(out_mode)
    out = (C.c_uint32 * 8)()
    _check(lib().cfs_binned_plan(int(width), int(height), mode, int(n_funcs), int(sms), int(smem_optin), out))
    keys = ["n_tiles", "tile_pixels", "tile_shift", "tile_mask", "nk", "cap", "check_every", "split"]
    return dict(zip(keys, [int(v) for v in out]))


def cfs_host_resolve(sys: System, args: cfs_render_args) -> dict:
    """What a render resolves on the host (pixel map, chain at t, thresholds, rgba8 palette); no device needed."""
    out = cfs_resolved()
    _check(lib().cfs_host_resolve(sys.handle, C.byref(args), C.byref(out)))
    n = int(out.n_chain)
    return {"sx": float(out.sx), "ox": float(out.ox), "sy": float(out.sy), "oy": float(out.oy),
            "chain_type": [int(out.chain_type[m]) for m in range(n)],
            "chain_p": [np.array(list(out.chain_p[m]), dtype=np.float32) for m in range(n)],
            "pick_form": int(out.pick_form), "proved": int(out.proved),
            "thresholds": [int(out.thresholds[j]) for j in range(int(out.n_thresholds))],
            "pal8": [int(out.pal8[j]) for j in range(int(out.n_funcs))]}


def cfs_specialize(sys: System, args: cfs_render_args) -> float:
    """Compile (NVRTC) and cache the kernels a CFS_FLAG_JIT render of this system will launch; returns the
    milliseconds spent compiling in this call (0.0 when they were cached)."""
    ms = C.c_double(0.0)
    _check(lib().cfs_specialize(sys.handle, C.byref(args), C.byref(ms)))
    return float(ms.value)


def cfs_jit_check(sys: System, args: cfs_render_args, splat_kind: int = -1):
    """Compile-only (no device needed): (cubin bytes, milliseconds) of the kernel a CFS_FLAG_JIT render would use."""
    nbytes, ms = C.c_uint64(0), C.c_double(0.0)
    _check(lib().cfs_jit_check(sys.handle, C.byref(args), int(splat_kind), C.byref(nbytes), C.byref(ms)))
    return int(nbytes.value), float(ms.value)


def cfs_jit_stats():
    """(kernels compiled at run time so far, milliseconds that took)."""
    n, ms = C.c_uint64(0), C.c_double(0.0)
    lib().cfs_jit_stats(C.byref(n), C.byref(ms))
    return int(n.value), float(ms.value)


def cfs_render(sys: System, args: cfs_render_args, stream=None) -> None:
    _check(lib().cfs_render(sys.handle, C.byref(args), _stream(stream)))


NOALLOC_SCRATCH_BYTES = 96 * 1024 + 256      # CFS_NOALLOC_SCRATCH_BYTES of include/cfs.h


def cfs_render_depth_noalloc(sys: System, args: cfs_render_args, stream=None) -> None:
    """The Hi-Z depth render with its scratch inside the library (a static device array): allocates nothing.
    DEPTH output of an IFS only; args.variant / d_scratch are ignored; calls that overlap on the GPU race."""
    _check(lib().cfs_render_depth_noalloc(sys.handle, C.byref(args), _stream(stream)))


def cfs_render_host(sys: System, args: cfs_render_args, h_image: np.ndarray, h_cloud: Optional[np.ndarray] = None,
                    h_counters: Optional[np.ndarray] = None, stream=None) -> None:
    _check(lib().cfs_render_host(sys.handle, C.byref(args), _ptr(h_image), _ptr(h_cloud), _ptr(h_counters),
                                 _stream(stream)))


def cfs_render_rgba8_host(sys: System, args: cfs_render_args, gamma: float, colour_scale: float, n_max: float,
                          h_rgba8: np.ndarray, h_cloud: Optional[np.ndarray] = None, h_counters: Optional[np.ndarray] = None,
                          h_n_max: Optional[np.ndarray] = None, stream=None) -> None:
    _check(lib().cfs_render_rgba8_host(sys.handle, C.byref(args), float(gamma), float(colour_scale), float(n_max),
                                       _ptr(h_rgba8), _ptr(h_cloud), _ptr(h_counters), _ptr(h_n_max), _stream(stream)))


def cfs_tonemap(d_image, out_mode, width: int, height: int, gamma: float, colour_scale: float, d_rgba8_out,
                d_scratch, stream=None) -> None:
    mode = OUT[out_mode] if isinstance(out_mode, str) else int(out_mode)
    _check(lib().cfs_tonemap(_ptr(d_image), mode, int(width), int(height), float(gamma), float(colour_scale),
                             _ptr(d_rgba8_out), _ptr(d_scratch), _stream(stream)))


def cfs_resolve_rgba8(d_image, out_mode, width: int, height: int, gamma: float, colour_scale: float, n_max: float,
                      d_rgba8_out, d_scratch, stream=None) -> None:
    mode = OUT[out_mode] if isinstance(out_mode, str) else int(out_mode)
    _check(lib().cfs_resolve_rgba8(_ptr(d_image), mode, int(width), int(height), float(gamma), float(colour_scale),
                                   float(n_max), _ptr(d_rgba8_out), _ptr(d_scratch), _stream(stream)))


def cfs_trace(sys: System, args: cfs_render_args, d_picks=None, d_final_g=None, d_final_q=None, d_alive=None,
              stream=None) -> None:
    _check(lib().cfs_trace(sys.handle, C.byref(args), _ptr(d_picks), _ptr(d_final_g), _ptr(d_final_q),
                           _ptr(d_alive), _stream(stream)))


def cfs_microbench(kind, d_buf, footprint_bytes: int, ops_per_thread: int, blocks: int, threads: int,
                   stream=None) -> None:
    k = MB[kind] if isinstance(kind, str) else int(kind)
    _check(lib().cfs_microbench(k, _ptr(d_buf), int(footprint_bytes), int(ops_per_thread), int(blocks),
                                int(threads), _stream(stream)))


# ------------------------------------------------------------------ device-memory helpers (torch)
def new_image(render, device="cuda"):
    """Cleared device image for a render: HIST int32 view of u32, RGBA float32[.,4], DEPTH int64 = -1."""
    import torch
    n = int(render.width) * int(render.height)
    if render.out_mode == "hist_u32":
        return torch.zeros(n, dtype=torch.int32, device=device)
    if render.out_mode == "rgba_f32":
        return torch.zeros((n, 4), dtype=torch.float32, device=device)
    if render.out_mode == "depth_u64":
        return torch.full((n,), -1, dtype=torch.int64, device=device)
    raise ValueError(render.out_mode)


def image_to_numpy(img, out_mode: str) -> np.ndarray:
    a = img.detach().cpu().numpy()
    if out_mode == "hist_u32":
        return a.view(np.uint32)
    if out_mode == "depth_u64":
        return a.view(np.uint64)
    return a


def cloud_to_device(cloud: np.ndarray, device="cuda"):
    """16-byte records -> device tensor (uint8 view; the kernel reads 128-bit records)."""
    import torch
    assert cloud.dtype.itemsize == 16 and cloud.flags.c_contiguous
    return torch.from_numpy(cloud.view(np.uint8).reshape(-1, 16)).to(device)


def shard_points(n_points: int, rank: int, world: int):
    """Contiguous point range of `rank` (multi-GPU: points are independent units, DESIGN 'multi-GPU').
    Returns (point_offset, n_points_local)."""
    lo = (n_points * rank) // world
    hi = (n_points * (rank + 1)) // world
    return lo, hi - lo


def allreduce_image(img, out_mode: str, group=None):
    """The ONE exchange step of a sharded render (DESIGN 'multi-GPU'): every rank renders its point range
    into a private image, then the images are combined in place -- sum for HIST / RGBA (uint32 sums wrap
    like the int32 view they travel as), min over the unsigned 64-bit keys for DEPTH.  NCCL and gloo only
    know a signed 64-bit MIN, and the empty key (all ones) is -1 there: the sign bit is flipped around
    the reduction so that the signed order equals the unsigned one.  `img` is a torch tensor in the
    library's layout (new_image), on any device the process group serves."""
    import torch
    import torch.distributed as dist
    if out_mode == "depth_u64":
        assert img.dtype == torch.int64
        flip = torch.tensor(-(1 << 63), dtype=torch.int64, device=img.device)
        img.bitwise_xor_(flip)
        dist.all_reduce(img, op=dist.ReduceOp.MIN, group=group)
        img.bitwise_xor_(flip)
    else:
        dist.all_reduce(img, op=dist.ReduceOp.SUM, group=group)
    return img



def render_sharded(sys: System, render, img, rank: int, world: int, group=None, **kw):
    """The sharded render as one call (DESIGN 'multi-GPU'): rank `rank` of `world` renders its contiguous
    range of the GLOBAL point ids into its own cleared image `img`, then the ONE exchange step combines the images
    in place on every rank (sum, or unsigned min for DEPTH) -- over NCCL / NVLink for CUDA tensors.  Keyword arguments go
    to make_args (t, variant, flags, d_counters, d_scratch, d_cloud ...).  Returns (point_offset, n_points) of this rank."""
    first = int(kw.pop("point_offset", render.point_offset))
    off, n = shard_points(int(kw.pop("n_points", render.n_points)), rank, world)
    cfs_render(sys, make_args(render, d_image=img, n_points=n, point_offset=first + off, **kw))
    if world > 1:
        allreduce_image(img, render.out_mode, group=group)
    return first + off, n
