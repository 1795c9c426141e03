"""Seeded synthetic inputs for the CFS hot path -- the five BASELINE.json workloads.

This module serves BOTH the CUDA path and the CPU oracle and therefore holds none of
the method's arithmetic: no RNG of the method, no maps, no pixel rule.  It only
writes down *inputs*: function tables, transform chains, palettes, bounds, seeds and
the synthetic point cloud of config 3 (drawn with numpy's own generator; the same
host buffer is handed to both sides).  Descriptions are neutral (string type names);
each binding maps them to its own enums.

Workload recipes: BASELINE.json `configs[0..4]`, constants per SURVEY.md section 8(d)
(paper is silent on all coefficients: PAPER L19 names only "f1..f4" for the square).
"""
from __future__ import annotations

import math
from dataclasses import dataclass, field, replace
from typing import List, Optional, Sequence

import numpy as np

CLOUD_DTYPE = np.dtype([("x", "<f4"), ("y", "<f4"), ("z", "<f4"), ("rgba8", "<u4")])


@dataclass
class Func:
    type: str            # "affine" | "circle_half" (PAPER Eq. 1: params = [f_id, r2_flag])
    prob: float
    params: Sequence[float]


@dataclass
class Xform:
    type: str            # affine|swirl|sinusoidal|rotate_z|twist_z|bend|pinhole|stretch_cos|branch (separator)
    p0: Sequence[float] = ()
    p1: Sequence[float] = ()


@dataclass
class System:
    dim: int
    gen: str                                  # "ifs" | "cloud"
    funcs: List[Func] = field(default_factory=list)
    chain: List[Xform] = field(default_factory=list)
    color: str = "none"                       # none | map_index | point
    palette: Optional[np.ndarray] = None      # float32 [n_funcs, 4], integer-valued 0..255
    reuse: bool = False


@dataclass
class Render:
    n_points: int
    seed: int
    iterations: int
    burn_in: int
    width: int
    height: int
    bounds: Sequence[float]                   # xmin, xmax, ymin, ymax
    out_mode: str                             # hist_u32 | rgba_f32 | depth_u64
    t: float = 0.0
    point_offset: int = 0


@dataclass
class Workload:
    name: str
    system: System
    render: Render
    frames: List[float] = field(default_factory=lambda: [0.0])   # frame parameters t
    cloud_seed: Optional[int] = None

    def scaled(self, **kw) -> "Workload":
        """Same workload with some render fields replaced (smaller point counts for tests)."""
        return replace(self, render=replace(self.render, **kw))

    @property
    def point_iterations(self) -> int:
        return self.render.n_points * self.render.iterations * len(self.frames)

    @property
    def splats(self) -> int:
        return self.render.n_points * (self.render.iterations - self.render.burn_in) * len(self.frames)


# ----------------------------------------------------------------------------- function tables
def _f32(x: float) -> float:
    return float(np.float32(x))


def square_funcs(probs: Optional[Sequence[float]] = None) -> List[Func]:
    """Fig. 1 square: f_k(p) = 0.5 p + 0.5 c_k, c_k = (2(k&1)-1, 2(k>>1)-1)."""
    out = []
    for k in range(4):
        cx, cy = 2 * (k & 1) - 1, 2 * (k >> 1) - 1
        pr = 0.25 if probs is None else probs[k]
        out.append(Func("affine", _f32(pr), [0.5, 0.0, 0.0, 0.5, 0.5 * cx, 0.5 * cy]))
    return out


def sierpinski_vertices():
    h = math.sqrt(3.0) / 2.0
    return [(0.0, 1.0), (-h, -0.5), (h, -0.5)]


def circle_funcs(r2_reading: bool = False) -> List[Func]:
    """PAPER Eq. 1 (L47-60): the two maps sending the unit disc to its top (f_id 0) / bottom (f_id 1) half."""
    return [Func("circle_half", 0.5, [float(fid), 1.0 if r2_reading else 0.0]) for fid in (0, 1)]


def sierpinski_funcs(probs: Optional[Sequence[float]] = None) -> List[Func]:
    """3 maps of scale 0.5 towards the vertices of an equilateral triangle on the unit circle."""
    out = []
    for k, (vx, vy) in enumerate(sierpinski_vertices()):
        pr = (1.0 / 3.0) if probs is None else probs[k]
        out.append(Func("affine", _f32(pr), [0.5, 0.0, 0.0, 0.5, _f32(0.5 * vx), _f32(0.5 * vy)]))
    return out


def carpet_funcs() -> List[Func]:
    """Sierpinski carpet: 8 maps of scale 1/3 (2-D analogue of the Menger sponge; test use)."""
    out = []
    s = _f32(1.0 / 3.0)
    for iy in range(3):
        for ix in range(3):
            if ix == 1 and iy == 1:
                continue
            out.append(Func("affine", _f32(0.125),
                            [s, 0.0, 0.0, s, _f32(2.0 / 3.0 * (ix - 1)), _f32(2.0 / 3.0 * (iy - 1))]))
    return out


def menger_cells():
    """Kept cells (ix,iy,iz) in increasing ix+3iy+9iz, skipping those with >=2 indices equal to 1."""
    cells = []
    for iz in range(3):
        for iy in range(3):
            for ix in range(3):
                if (ix == 1) + (iy == 1) + (iz == 1) >= 2:
                    continue
                cells.append((ix, iy, iz))
    return cells


def menger_funcs() -> List[Func]:
    out = []
    s = _f32(1.0 / 3.0)
    for (ix, iy, iz) in menger_cells():
        b = [_f32(2.0 / 3.0 * (i - 1)) for i in (ix, iy, iz)]
        out.append(Func("affine", _f32(0.05), [s, 0, 0, 0, s, 0, 0, 0, s, b[0], b[1], b[2]]))
    return out


def palette_for(n: int) -> np.ndarray:
    """Integer-valued 0..255 RGBA palette, one entry per map (alpha 255)."""
    base = [(255, 0, 0), (0, 255, 0), (0, 0, 255), (255, 255, 0)]
    pal = np.zeros((n, 4), dtype=np.float32)
    for k in range(n):
        if k < 4 and n <= 4:
            r, g, b = base[k]
        else:
            r, g, b = 40 + (k * 67) % 216, 40 + (k * 131 + 50) % 216, 40 + (k * 29 + 120) % 216
        pal[k] = (r, g, b, 255)
    return pal


# ----------------------------------------------------------------------------- point cloud (config 3)
def gaussian_mixture_cloud(n_points: int, seed: int, components: int = 8, sigma: float = 0.1) -> np.ndarray:
    """Seeded isotropic Gaussian mixture: means uniform in [-1,1]^3, record p belongs to
    component p mod `components` (spatially unsorted stream), float32 xyz + rgba8."""
    rng = np.random.default_rng(seed)
    means = rng.uniform(-1.0, 1.0, size=(components, 3))
    pal = palette_for(components).astype(np.uint32)
    rgba = pal[:, 0] | (pal[:, 1] << 8) | (pal[:, 2] << 16) | (pal[:, 3] << 24)
    rec = np.empty(n_points, dtype=CLOUD_DTYPE)
    comp = np.arange(n_points, dtype=np.int64) % components
    chunk = 1 << 22
    for s in range(0, n_points, chunk):
        e = min(n_points, s + chunk)
        xyz = means[comp[s:e]] + sigma * rng.standard_normal(size=(e - s, 3))
        rec["x"][s:e] = xyz[:, 0].astype(np.float32)
        rec["y"][s:e] = xyz[:, 1].astype(np.float32)
        rec["z"][s:e] = xyz[:, 2].astype(np.float32)
    rec["rgba8"] = rgba[comp]
    return rec


# ----------------------------------------------------------------------------- the five configs
SEED_BASE = 0xC0FFEE00
PINHOLE = Xform("pinhole", [60.0, -4.0, 1e-3])


def config(i: int) -> Workload:
    """BASELINE.json configs[i] at full size."""
    if i == 0:
        return Workload(
            "cfg0_square_hist512",
            System(2, "ifs", square_funcs(), [], "none"),
            Render(1 << 16, SEED_BASE + 0, 1000, 20, 512, 512, (-1.0, 1.0, -1.0, 1.0), "hist_u32"))
    if i == 1:
        return Workload(
            "cfg1_square_swirl_rgba1024",
            System(2, "ifs", square_funcs(),
                   [Xform("swirl"), Xform("affine", [0.8, 0.0, 0.0, 0.8, 0.0, 0.0])],
                   "map_index", palette_for(4)),
            Render(1 << 20, SEED_BASE + 1, 1000, 20, 1024, 1024, (-1.25, 1.25, -1.25, 1.25), "rgba_f32"))
    if i == 2:
        frames = [float(np.float32(k / 15.0)) for k in range(16)]
        return Workload(
            "cfg2_sierpinski_rotate_sin_1080p",
            System(2, "ifs", sierpinski_funcs(),
                   [Xform("rotate_z", [0.0], [2.0 * math.pi]), Xform("sinusoidal")],
                   "map_index", palette_for(3)),
            Render(1 << 22, SEED_BASE + 2, 500, 20, 1920, 1080,
                   (-16.0 / 9.0, 16.0 / 9.0, -1.0, 1.0), "rgba_f32"),
            frames=frames)
    if i == 3:
        return Workload(
            "cfg3_cloud_twist_bend_pinhole_4k",
            System(3, "cloud", [], [Xform("twist_z", [3.0]), Xform("bend", [1.0]), PINHOLE], "point"),
            Render(1 << 24, SEED_BASE + 3, 1, 0, 3840, 2160, (-1.0, 1.0, -1.0, 1.0), "rgba_f32"),
            cloud_seed=SEED_BASE + 3)
    if i == 4:
        return Workload(
            "cfg4_menger_depth_4k",
            System(3, "ifs", menger_funcs(), [PINHOLE], "map_index", palette_for(20)),
            Render(1 << 26, SEED_BASE + 4, 1000, 20, 3840, 2160, (-1.0, 1.0, -1.0, 1.0), "depth_u64"))
    raise ValueError(f"no config {i}")


N_CONFIGS = 5


def fig4_like() -> Workload:
    """A scene with the STRUCTURE of the paper's Fig. 4 (planet, ring, stars and comet, all from ONE
    circle primitive; the paper prints none of its formulas, so the numbers here are this repo's): the Eq. 1 circle
    generator (r^2 reading: uniform disc) drives four branches per iteration -- a planet (uniform scale), a ring
    (the disc squashed and tilted), 64 stars (a tiny copy placed by the on-the-fly PRNG, L198) and a comet (a
    stretched, sheared copy) -- into the paper's 1920 x 1080 frame (L202).  One-to-many splatting:
    4 splats per point and iteration.  Used by bench.py to put numbers beside the paper's own (L200: compile time
    against frame time) and by the run-time specialisation tests."""
    c30, s30 = math.cos(math.radians(30.0)), math.sin(math.radians(30.0))
    planet = [Xform("affine", [0.42, 0.0, 0.0, 0.42, 0.0, 0.0])]
    ring = [Xform("affine", [0.95 * c30, -0.12 * s30, 0.95 * s30, 0.12 * c30, 0.0, 0.0])]
    stars = [Xform("affine", [0.006, 0.0, 0.0, 0.006, 0.0, 0.0]), Xform("scatter", [64, 1.7, 0.95, 0.0])]
    comet = [Xform("affine", [0.30, 0.06, -0.05, 0.05, 1.05, 0.55])]
    chain = planet + [Xform("branch")] + ring + [Xform("branch")] + stars + [Xform("branch")] + comet
    return Workload(
        "fig4_like_planet_ring_stars_comet_1080p",
        System(2, "ifs", circle_funcs(r2_reading=True), chain, "map_index", palette_for(2)),
        Render(1 << 20, SEED_BASE + 0x40, 200, 20, 1920, 1080, (-16.0 / 9.0, 16.0 / 9.0, -1.0, 1.0), "rgba_f32"))
