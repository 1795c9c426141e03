"""ctypes binding of the CPU oracle -- TEST INFRASTRUCTURE, NOT THE PRODUCT.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference
legs may import this module.  It imports nothing from paper_2606_02226_b200/: system
and render descriptions are duck-typed (any object with the attribute names of
`paper_2606_02226_b200.workloads.System` / `.Render`, the neutral input module).

All arithmetic lives in cfs_oracle.c; this file only marshals arguments and, for the
multi-threaded driver, splits a render into disjoint point ranges (points are
independent units) and merges the partial images by sum / 64-bit min.
"""
from __future__ import annotations

import ctypes as C
import os
from concurrent.futures import ThreadPoolExecutor

import numpy as np

from . import build as _build

_F_TYPES = {"affine": 0, "circle_half": 1}
_T_TYPES = {"affine": 0, "swirl": 1, "sinusoidal": 2, "rotate_z": 3, "twist_z": 4, "bend": 5,
            "pinhole": 6, "stretch_cos": 7, "branch": 8, "scatter": 9}
_COLORS = {"none": 0, "map_index": 1, "point": 2}
_OUTS = {"hist_u32": 0, "rgba_f32": 1, "depth_u64": 2}
_GENS = {"ifs": 0, "cloud": 1}

CLOUD_DTYPE = np.dtype([("x", "<f4"), ("y", "<f4"), ("z", "<f4"), ("rgba8", "<u4")])
DEPTH_EMPTY = np.uint64(0xFFFFFFFFFFFFFFFF)


class _Func(C.Structure):
    _fields_ = [("type", C.c_int32), ("prob", C.c_float), ("params", C.c_float * 12)]


class _Xform(C.Structure):
    _fields_ = [("type", C.c_int32), ("p0", C.c_float * 12), ("p1", C.c_float * 12)]


class _System(C.Structure):
    _fields_ = [("dim", C.c_int32), ("gen_kind", C.c_int32), ("n_funcs", C.c_int32),
                ("n_chain", C.c_int32), ("color_rule", C.c_int32), ("reuse", C.c_int32),
                ("funcs", C.POINTER(_Func)), ("chain", C.POINTER(_Xform)),
                ("palette", C.POINTER(C.c_float))]


class _Args(C.Structure):
    _fields_ = [("n_points", C.c_uint64), ("point_offset", C.c_uint64), ("seed", C.c_uint64),
                ("iterations", C.c_int32), ("burn_in", C.c_int32),
                ("width", C.c_int32), ("height", C.c_int32),
                ("xmin", C.c_float), ("xmax", C.c_float), ("ymin", C.c_float), ("ymax", C.c_float),
                ("t", C.c_float), ("out_mode", C.c_int32), ("pad_", C.c_int32),
                ("image", C.c_void_p), ("cloud", C.c_void_p), ("counters", C.c_void_p)]


_lib = None


def lib():
    global _lib
    if _lib is None:
        L = C.CDLL(_build.build())
        L.orc_philox4x32_10.argtypes = [C.POINTER(C.c_uint32)] * 3
        L.orc_philox4x32_10.restype = None
        L.orc_thresholds.argtypes = [C.POINTER(C.c_float), C.c_int, C.POINTER(C.c_uint64)]
        L.orc_thresholds.restype = C.c_int
        L.orc_pick.argtypes = [C.c_uint32, C.POINTER(C.c_uint64), C.c_int]
        L.orc_pick.restype = C.c_int
        L.orc_pick_word.argtypes = [C.c_uint64, C.c_uint64, C.c_uint32]
        L.orc_pick_word.restype = C.c_uint32
        L.orc_init_point.argtypes = [C.c_uint64, C.c_uint64, C.c_int, C.POINTER(C.c_float)]
        L.orc_init_point.restype = None
        L.orc_apply_func.argtypes = [C.POINTER(_Func), C.c_int, C.POINTER(C.c_float)]
        L.orc_apply_func.restype = None
        L.orc_apply_xform.argtypes = [C.c_int, C.POINTER(C.c_float), C.c_int, C.POINTER(C.c_float)]
        L.orc_apply_xform.restype = C.c_int
        L.orc_resolve_xform.argtypes = [C.POINTER(_Xform), C.c_int, C.c_float, C.c_int, C.c_int,
                                        C.POINTER(C.c_int), C.POINTER(C.c_float)]
        L.orc_resolve_xform.restype = None
        L.orc_pixel.argtypes = [C.c_float] * 6 + [C.c_int, C.c_int]
        L.orc_pixel.restype = C.c_int64
        L.orc_render.argtypes = [C.POINTER(_System), C.POINTER(_Args)]
        L.orc_render.restype = C.c_int
        L.orc_trace.argtypes = [C.POINTER(_System), C.POINTER(_Args), C.c_void_p, C.c_void_p,
                                C.c_void_p, C.c_void_p]
        L.orc_trace.restype = C.c_int
        L.orc_tonemap.argtypes = [C.c_void_p, C.c_int, C.c_int, C.c_int, C.c_float, C.c_float,
                                  C.c_void_p]
        L.orc_tonemap.restype = C.c_int
        _lib = L
    return _lib


# --------------------------------------------------------------------------- small pieces
def philox4x32_10(ctr, key):
    c = (C.c_uint32 * 4)(*[int(v) & 0xFFFFFFFF for v in ctr])
    k = (C.c_uint32 * 2)(*[int(v) & 0xFFFFFFFF for v in key])
    o = (C.c_uint32 * 4)()
    lib().orc_philox4x32_10(c, k, o)
    return [int(v) for v in o]


def thresholds(probs):
    n = len(probs)
    p = (C.c_float * n)(*[float(v) for v in probs])
    T = (C.c_uint64 * n)()
    if lib().orc_thresholds(p, n, T) != 0:
        raise ValueError("invalid probabilities")
    return [int(v) for v in T]


def pick(u, T):
    n = len(T)
    return int(lib().orc_pick(int(u) & 0xFFFFFFFF, (C.c_uint64 * n)(*T), n))


def pick_word(seed, p, it):
    return int(lib().orc_pick_word(int(seed), int(p), int(it)))


def init_point(seed, p, dim):
    g = (C.c_float * 3)()
    lib().orc_init_point(int(seed), int(p), int(dim), g)
    return np.array(list(g), dtype=np.float32)


def _mk_func(f):
    out = _Func()
    out.type = _F_TYPES[f.type]
    out.prob = float(f.prob)
    for i, v in enumerate(f.params):
        out.params[i] = float(v)
    return out


def _mk_xform(x):
    out = _Xform()
    out.type = _T_TYPES[x.type]
    for i, v in enumerate(x.p0):
        out.p0[i] = float(v)
    for i, v in enumerate(x.p1):
        out.p1[i] = float(v)
    return out


def apply_func(f, dim, g):
    v = (C.c_float * 3)(*[float(c) for c in g])
    ff = _mk_func(f)
    lib().orc_apply_func(C.byref(ff), int(dim), v)
    return np.array(list(v), dtype=np.float32)


def resolve_xform(x, dim, t, width, height):
    xf = _mk_xform(x)
    ty = C.c_int()
    prm = (C.c_float * 12)()
    lib().orc_resolve_xform(C.byref(xf), int(dim), float(t), int(width), int(height), C.byref(ty), prm)
    return int(ty.value), np.array(list(prm), dtype=np.float32)


def apply_xform(x, dim, q, t=0.0, width=1, height=1):
    """One chain step on one point. Returns (q', alive)."""
    ty, prm = resolve_xform(x, dim, t, width, height)
    v = (C.c_float * 3)(*[float(c) for c in q])
    p = (C.c_float * 12)(*[float(c) for c in prm])
    alive = lib().orc_apply_xform(ty, p, int(dim), v)
    return np.array(list(v), dtype=np.float32), bool(alive)


def pixel(x, y, bounds, W, H):
    return int(lib().orc_pixel(float(x), float(y), float(bounds[0]), float(bounds[1]),
                               float(bounds[2]), float(bounds[3]), int(W), int(H)))


# --------------------------------------------------------------------------- whole path
class _Packed:
    """Keeps the ctypes arrays alive for the lifetime of one call."""

    def __init__(self, system):
        self.funcs = (_Func * max(1, len(system.funcs)))(*[_mk_func(f) for f in system.funcs])
        self.chain = (_Xform * max(1, len(system.chain)))(*[_mk_xform(x) for x in system.chain])
        self.pal = None
        s = _System()
        s.dim = int(system.dim)
        s.gen_kind = _GENS[system.gen]
        s.n_funcs = len(system.funcs)
        s.n_chain = len(system.chain)
        s.color_rule = _COLORS[system.color]
        s.reuse = 1 if getattr(system, "reuse", False) else 0
        s.funcs = C.cast(self.funcs, C.POINTER(_Func))
        s.chain = C.cast(self.chain, C.POINTER(_Xform))
        if system.palette is not None:
            self.pal = np.ascontiguousarray(system.palette, dtype=np.float32)
            s.palette = self.pal.ctypes.data_as(C.POINTER(C.c_float))
        self.sys = s


def _mk_args(render, n_points=None, point_offset=None, t=None):
    a = _Args()
    a.n_points = int(render.n_points if n_points is None else n_points)
    a.point_offset = int(render.point_offset if point_offset is None else point_offset)
    a.seed = int(render.seed)
    a.iterations = int(render.iterations)
    a.burn_in = int(render.burn_in)
    a.width = int(render.width)
    a.height = int(render.height)
    a.xmin, a.xmax, a.ymin, a.ymax = [float(np.float32(v)) for v in render.bounds]
    a.t = float(render.t if t is None else t)
    a.out_mode = _OUTS[render.out_mode]
    return a


def new_image(render):
    """Cleared oracle-side image: HIST uint32, RGBA float64[.,4], DEPTH uint64 (all ones)."""
    n = int(render.width) * int(render.height)
    if render.out_mode == "hist_u32":
        return np.zeros(n, dtype=np.uint32)
    if render.out_mode == "rgba_f32":
        return np.zeros((n, 4), dtype=np.float64)
    if render.out_mode == "depth_u64":
        return np.full(n, DEPTH_EMPTY, dtype=np.uint64)
    raise ValueError(render.out_mode)


def render(system, rnd, cloud=None, image=None, n_points=None, point_offset=None, t=None):
    """orc_render over [point_offset, point_offset+n_points). Returns (image, counters[2])."""
    pk = _Packed(system)
    a = _mk_args(rnd, n_points, point_offset, t)
    if image is None:
        image = new_image(rnd)
    counters = np.zeros(2, dtype=np.uint64)
    a.image = image.ctypes.data
    a.counters = counters.ctypes.data
    if cloud is not None:
        assert cloud.dtype == CLOUD_DTYPE and cloud.flags.c_contiguous
        a.cloud = cloud.ctypes.data
    rc = lib().orc_render(C.byref(pk.sys), C.byref(a))
    if rc != 0:
        raise ValueError("orc_render: invalid arguments")
    return image, counters


def render_parallel(system, rnd, cloud=None, n_points=None, point_offset=None, t=None, threads=None):
    """Same result as render(): disjoint point ranges on host threads (ctypes drops the GIL),
    partial images merged by sum (HIST, RGBA) or min (DEPTH).  Returns (image, counters, threads)."""
    n = int(rnd.n_points if n_points is None else n_points)
    off = int(rnd.point_offset if point_offset is None else point_offset)
    threads = threads or (os.cpu_count() or 1)
    threads = max(1, min(threads, max(1, n // 64)))
    if threads == 1:
        img, ctr = render(system, rnd, cloud, None, n, off, t)
        return img, ctr, 1
    edges = [off + (n * i) // threads for i in range(threads + 1)]

    def work(i):
        return render(system, rnd, cloud, None, edges[i + 1] - edges[i], edges[i], t)

    with ThreadPoolExecutor(threads) as ex:
        parts = list(ex.map(work, range(threads)))
    img, ctr = parts[0]
    for im2, c2 in parts[1:]:
        if rnd.out_mode == "depth_u64":
            np.minimum(img, im2, out=img)
        else:
            img += im2
        ctr += c2
    return img, ctr, threads


def trace(system, rnd, cloud=None, n_points=None, point_offset=None, t=None, want_picks=True):
    """Pick sequences [n,it] u8, final generator state [n,3], final chain output [n,3], alive [n]."""
    pk = _Packed(system)
    a = _mk_args(rnd, n_points, point_offset, t)
    n, it = int(a.n_points), int(a.iterations)
    picks = np.zeros((n, it), dtype=np.uint8) if want_picks else None
    fg = np.zeros((n, 3), dtype=np.float32)
    fq = np.zeros((n, 3), dtype=np.float32)
    al = np.zeros(n, dtype=np.uint8)
    if cloud is not None:
        a.cloud = cloud.ctypes.data
    rc = lib().orc_trace(C.byref(pk.sys), C.byref(a), picks.ctypes.data if want_picks else None,
                         fg.ctypes.data, fq.ctypes.data, al.ctypes.data)
    if rc != 0:
        raise ValueError("orc_trace: invalid arguments")
    return picks, fg, fq, al


def tonemap(image, out_mode, W, H, gamma, colour_scale):
    """image in the GPU path's format: HIST uint32, RGBA float32[.,4], DEPTH uint64."""
    want = {"hist_u32": np.uint32, "rgba_f32": np.float32, "depth_u64": np.uint64}[out_mode]
    img = np.ascontiguousarray(image, dtype=want)
    out = np.zeros(int(W) * int(H), dtype=np.uint32)
    rc = lib().orc_tonemap(img.ctypes.data, _OUTS[out_mode], int(W), int(H), float(gamma),
                           float(colour_scale), out.ctypes.data)
    if rc != 0:
        raise ValueError("orc_tonemap: invalid arguments")
    return out
