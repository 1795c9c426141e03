"""Pins of the CPU oracle, part 2: whole-path invariants, chain transforms, splat modes, tone map.

Invariants named by BASELINE.json north_star: uniform invariant density of the Fig. 1 square
(chi-square), zero hits in the removed regions of Sierpinski / carpet / Menger attractors, total
in-bounds hits = points x (iterations - burn-in); plus the composition semantics of PAPER L77
(Fig. 2 B vs C), colour = generating map, closed forms of every chain transform,
a brute-force depth buffer and closed-form tone-map values.
"""
import math

import numpy as np
import pytest

from paper_2606_02226_b200 import workloads as W


# ------------------------------------------------------------------ P5: uniform invariant density
def test_square_density_is_uniform_chi2(oracle):
    """One splat per point after 20 steps => i.i.d. uniform multinomial over 512^2 pixels."""
    w = W.config(0)
    n = 1 << 21
    rnd = w.scaled(n_points=n, iterations=21, burn_in=20).render
    img, ctr, _ = oracle.render_parallel(w.system, rnd)
    assert int(ctr[0]) == n
    exp = n / (512 * 512)
    chi2 = ((img.astype(np.float64) - exp) ** 2 / exp).sum()
    dof = 512 * 512 - 1
    assert abs(chi2 - dof) < 5 * math.sqrt(2 * dof)


# ------------------------------------------------------------------ P6: conservation
@pytest.mark.parametrize("cfg", [0, 1, 2, 4])
def test_conservation_all_in_bounds(oracle, cfg):
    w = W.config(cfg)
    n = 512
    rnd = w.scaled(n_points=n).render
    img, ctr = oracle.render(w.system, rnd, t=w.frames[len(w.frames) // 2])
    want = n * (rnd.iterations - rnd.burn_in)
    assert int(ctr[0]) == want and int(ctr[1]) == 0
    if rnd.out_mode == "hist_u32":
        assert int(img.sum()) == want
    elif rnd.out_mode == "rgba_f32":
        assert img[:, 3].sum() == want
    else:
        assert np.count_nonzero(img != oracle.DEPTH_EMPTY) > 0


def test_burn_in_and_iteration_count(oracle):
    """Splat happens iff it >= burn_in, it counted from 0; the initial point is never splatted."""
    w = W.config(0)
    for I, B in ((1, 0), (5, 0), (5, 4), (7, 3)):
        img, ctr = oracle.render(w.system, w.scaled(n_points=100, iterations=I, burn_in=B).render)
        assert int(img.sum()) == 100 * (I - B) == int(ctr[0])
    with pytest.raises(ValueError):
        oracle.render(w.system, w.scaled(n_points=1, iterations=5, burn_in=5).render)
    with pytest.raises(ValueError):
        oracle.render(w.system, w.scaled(n_points=1, iterations=0, burn_in=0).render)
    # n_points == 0 is a no-op
    img, ctr = oracle.render(w.system, w.scaled(n_points=0).render)
    assert int(img.sum()) == 0 and int(ctr.sum()) == 0


def test_point_ranges_compose(oracle):
    """RNG keyed by the global point id: [0,300) == [0,100) + [100,300), any order."""
    w = W.config(1).scaled(n_points=300, iterations=40)
    full, c_full = oracle.render(w.system, w.render)
    a, ca = oracle.render(w.system, w.render, n_points=200, point_offset=100)
    b, cb = oracle.render(w.system, w.render, n_points=100, point_offset=0)
    assert np.array_equal(full, a + b) and np.array_equal(c_full, ca + cb)
    par, c_par, _ = oracle.render_parallel(w.system, w.render, threads=3)
    assert np.array_equal(par, full) and np.array_equal(c_par, c_full)


# ------------------------------------------------------------------ P7: removed regions
def test_sierpinski_holes_empty(oracle):
    """Medial triangles of levels 1..3 (eroded by 1.5 pixels) receive no hit."""
    sys = W.System(2, "ifs", W.sierpinski_funcs(), [], "none")
    Wd = 768
    rnd = W.Render(1 << 13, 5, 220, 20, Wd, Wd, (-1, 1, -1, 1), "hist_u32")
    img, ctr, _ = oracle.render_parallel(sys, rnd)
    img = img.reshape(Wd, Wd)
    assert int(ctr[0]) + int(ctr[1]) == rnd.n_points * 200
    V = np.array(W.sierpinski_vertices())
    ys, xs = np.mgrid[0:Wd, 0:Wd]
    cx = (xs + 0.5) * 2 / Wd - 1
    cy = (ys + 0.5) * 2 / Wd - 1
    margin = 1.5 * 2 / Wd * math.sqrt(2)

    def inside(tri, m):
        """strictly inside triangle tri (3x2), at distance > m from every edge"""
        ok = np.ones_like(cx, dtype=bool)
        for i in range(3):
            a, b, c = tri[i], tri[(i + 1) % 3], tri[(i + 2) % 3]
            nrm = np.array([-(b - a)[1], (b - a)[0]])
            nrm = nrm / np.linalg.norm(nrm)
            if np.dot(c - a, nrm) < 0:
                nrm = -nrm
            ok &= ((cx - a[0]) * nrm[0] + (cy - a[1]) * nrm[1]) > m
        return ok

    tris = [V]
    holes = 0
    for _level in range(3):
        nxt = []
        for t in tris:
            mid = np.array([(t[0] + t[1]) / 2, (t[1] + t[2]) / 2, (t[2] + t[0]) / 2])
            hole = inside(mid, margin)
            holes += int(hole.sum())
            assert int(img[hole].sum()) == 0
            nxt += [np.array([t[0], mid[0], mid[2]]), np.array([mid[0], t[1], mid[1]]),
                    np.array([mid[2], mid[1], t[2]])]
        tris = nxt
    assert holes > 0.2 * Wd * Wd * 0.3          # the test really covers a sizeable area
    assert int(img[inside(V, -margin) == False].sum()) == 0      # nothing outside the triangle
    assert int(img.sum()) > 0


def test_carpet_holes_empty(oracle):
    """Sierpinski carpet (2-D analogue of Menger) on 729^2: a pixel whose base-3 (ix,iy) digits
    are both 1 at any of the first 4 levels is empty, after eroding holes by one pixel."""
    sys = W.System(2, "ifs", W.carpet_funcs(), [], "none")
    n = 729
    rnd = W.Render(1 << 13, 6, 220, 20, n, n, (-1, 1, -1, 1), "hist_u32")
    img, _, _ = oracle.render_parallel(sys, rnd)
    img = img.reshape(n, n)
    idx = np.arange(n)
    hole = np.zeros((n, n), dtype=bool)
    for level in range(4):
        size = n // 3 ** (level + 1)
        d = (idx // size) % 3 == 1
        off = idx % size
        core = d & (off >= 1) & (off <= size - 2)       # eroded by one pixel
        hole |= np.outer(core, core)
    assert hole.sum() > 0.15 * n * n
    assert int(img[hole].sum()) == 0
    assert np.count_nonzero(img[~hole]) > 0.9 * (~hole).sum() * 0.7


def test_menger_digit_test(oracle):
    """No state has >= 2 middle base-3 digits among (x,y,z) at any of the first 5 levels
    (cells eroded by 1e-5 because boundary points belong to the attractor)."""
    sys = W.System(3, "ifs", W.menger_funcs(), [], "none")
    bad = 0
    total = 0
    for I in (25, 26, 31, 40):
        rnd = W.Render(4096, 8, I, I - 1, 8, 8, (-1, 1, -1, 1), "hist_u32")
        _, fg, _, _ = oracle.trace(sys, rnd, want_picks=False)
        u = (fg.astype(np.float64) + 1.0) / 2.0
        assert u.min() >= -1e-6 and u.max() <= 1 + 1e-6
        for level in range(5):
            s = u * 3 ** (level + 1)
            frac = s - np.floor(s)
            digit = np.floor(s).astype(np.int64) % 3
            interior = (frac > 1e-4) & (frac < 1 - 1e-4)
            mid = (digit == 1) & interior
            bad += int((mid.sum(axis=1) >= 2).sum())
        total += len(fg)
    assert total == 4 * 4096 and bad == 0


# ------------------------------------------------------------------ P9: Fig. 2 (B) vs (C)
def test_copy_semantics_generator_independent_of_chain(oracle):
    base = W.config(0).scaled(n_points=256, iterations=50)
    with_chain = W.System(2, "ifs", W.square_funcs(), [W.Xform("swirl"), W.Xform("stretch_cos")], "none")
    p0, g0, q0, _ = oracle.trace(base.system, base.render)
    p1, g1, q1, _ = oracle.trace(with_chain, base.render)
    assert np.array_equal(p0, p1) and np.array_equal(g0, g1)     # Fig. 2(B): P untouched
    assert not np.array_equal(q0, q1)
    reuse = W.System(2, "ifs", W.square_funcs(), [W.Xform("affine", [0.5, 0, 0, 0.5, 0.25, 0])], "none",
                     reuse=True)
    p2, g2, q2, _ = oracle.trace(reuse, base.render)
    assert np.array_equal(p0, p2) and not np.array_equal(g0, g2)  # Fig. 2(C): P is P2
    assert np.array_equal(g2, q2)


# ------------------------------------------------------------------ P10: chain transforms
def _x(oracle, xf, q, dim=3, t=0.0, Wd=1, Hd=1):
    out, alive = oracle.apply_xform(xf, dim, np.array(q, dtype=np.float32), t, Wd, Hd)
    return out.astype(np.float64), alive


def test_swirl_closed_form(oracle):
    q, _ = _x(oracle, W.Xform("swirl"), [1.0, 0.0, 0.0])
    assert np.allclose(q[:2], [math.cos(1.0), math.sin(1.0)], atol=6e-8)
    q, _ = _x(oracle, W.Xform("swirl"), [0.0, 0.5, 0.0])          # r2 = .25: (-y sin, y cos)
    assert np.allclose(q[:2], [-0.5 * math.sin(0.25), 0.5 * math.cos(0.25)], atol=6e-8)
    rng = np.random.default_rng(0)
    for p in rng.uniform(-1, 1, size=(200, 3)):
        q, alive = _x(oracle, W.Xform("swirl"), p)
        pf = np.float32(p).astype(np.float64)
        assert alive and abs(np.hypot(*q[:2]) - np.hypot(*pf[:2])) < 2e-7 and q[2] == pf[2]
        ang = math.atan2(q[1], q[0]) - math.atan2(pf[1], pf[0]) - (pf[0] ** 2 + pf[1] ** 2)
        assert abs((ang + math.pi) % (2 * math.pi) - math.pi) < 1e-6


def test_swirl_preserves_area(oracle):
    """Unit Jacobian: the uniform square of cfg 0, swirled and scaled by 0.8, is uniform inside the
    disc r <= 0.8 (every circle of radius <= 1 lies inside the square and is rotated rigidly)."""
    w = W.config(1)
    n = 1 << 19
    Wd = 64
    rnd = w.scaled(n_points=n, iterations=21, burn_in=20, width=Wd, height=Wd).render
    img, ctr, _ = oracle.render_parallel(w.system, rnd)
    assert int(ctr[0]) == n
    cnt = img[:, 3].reshape(Wd, Wd)
    ys, xs = np.mgrid[0:Wd, 0:Wd]
    px = 2.5 / Wd
    far = np.hypot(np.maximum(np.abs(xs * px - 1.25), np.abs((xs + 1) * px - 1.25)),
                   np.maximum(np.abs(ys * px - 1.25), np.abs((ys + 1) * px - 1.25)))
    inside = far < 0.8
    exp = n * (px / 0.8) ** 2 / 4.0          # square of side 1.6 holds all n points uniformly
    k = int(inside.sum())
    assert k > 500
    chi2 = ((cnt[inside] - exp) ** 2 / exp).sum()
    assert abs(chi2 - k) < 5 * math.sqrt(2 * k)


def test_sinusoidal_twist_bend_stretch_closed_forms(oracle):
    q, _ = _x(oracle, W.Xform("sinusoidal"), [0.5, -1.25, 0.75])
    assert np.allclose(q, [math.sin(0.5), math.sin(-1.25), 0.75], atol=6e-8)
    q, _ = _x(oracle, W.Xform("twist_z", [3.0]), [1.0, 0.0, 0.5])  # angle 1.5
    assert np.allclose(q, [math.cos(1.5), math.sin(1.5), 0.5], atol=6e-8)
    q, _ = _x(oracle, W.Xform("twist_z", [3.0]), [0.25, -0.5, 0.0])  # z = 0: identity
    assert np.allclose(q, [0.25, -0.5, 0.0], atol=0)
    q, _ = _x(oracle, W.Xform("bend", [1.0]), [0.5, 0.0, 0.3])     # angle = x = 0.5
    assert np.allclose(q, [0.5 * math.cos(0.5), 0.5 * math.sin(0.5), 0.3], atol=6e-8)
    q, _ = _x(oracle, W.Xform("bend", [2.0]), [0.0, 0.7, -0.3])    # x = 0: identity
    assert np.allclose(q, [0.0, 0.7, -0.3], atol=0)
    # PAPER Eq. 2 (L62-67): x2 = 2x, y2 = y - cos(x)
    q, _ = _x(oracle, W.Xform("stretch_cos"), [0.5, 0.25, 0.0])
    assert np.allclose(q[:2], [1.0, 0.25 - math.cos(0.5)], atol=6e-8)
    q, _ = _x(oracle, W.Xform("stretch_cos"), [0.0, 0.0, 0.0])
    assert np.allclose(q[:2], [0.0, -1.0], atol=0)


def test_sinusoidal_range_on_image(oracle):
    """cfg 2: |sin| <= sin(1.0...) so no hit beyond |x'|,|y'| > sin 1 (attractor radius 1)."""
    w = W.config(2).scaled(n_points=2048, width=192, height=108)
    img, ctr = oracle.render(w.system, w.render, t=w.frames[5])
    assert int(ctr[1]) == 0
    cnt = img[:, 3].reshape(108, 192)
    s1 = math.sin(1.0)
    xs = (np.arange(192) + 0.5) / 192 * (32 / 9) - 16 / 9
    ys = (np.arange(108) + 0.5) / 108 * 2 - 1
    px = 32 / 9 / 192
    assert cnt[:, np.abs(xs) > s1 + px].sum() == 0 and cnt[np.abs(ys) > s1 + px, :].sum() == 0
    assert cnt.sum() == 2048 * 480


def test_rotate_resolves_to_affine(oracle):
    rot = W.Xform("rotate_z", [0.0], [2 * math.pi])
    ty, prm = oracle.resolve_xform(rot, 2, 0.0, 8, 8)
    assert ty == 0 and list(prm[:6]) == [1.0, -0.0, 0.0, 1.0, 0.0, 0.0]   # identity at t = 0
    ty, prm = oracle.resolve_xform(rot, 2, 0.25, 8, 8)                      # quarter turn
    assert np.allclose(prm[:6], [0, -1, 1, 0, 0, 0], atol=1e-7)
    q, _ = _x(oracle, rot, [1.0, 0.0, 0.0], dim=2, t=0.25)
    assert np.allclose(q[:2], [0.0, 1.0], atol=1e-7)
    q, _ = _x(oracle, rot, [0.3, -0.4, 0.9], dim=3, t=0.5)
    assert np.allclose(q, [-0.3, 0.4, 0.9], atol=1e-6)
    # parameter interpolation p0 + t p1 for AFFINE
    aff = W.Xform("affine", [1, 0, 0, 1, 0, 0], [1, 0, 0, -0.5, 2, 0])
    q, _ = _x(oracle, aff, [0.5, 0.5, 0.0], dim=2, t=0.5)
    assert np.allclose(q[:2], [1.5 * 0.5 + 1.0, 0.75 * 0.5], atol=1e-7)


def test_pinhole(oracle):
    ph = W.PINHOLE
    q, alive = _x(oracle, ph, [0.0, 0.0, 0.0], Wd=3840, Hd=2160)
    assert alive and list(q) == [0.0, 0.0, 4.0]
    assert oracle.pixel(q[0], q[1], (-1, 1, -1, 1), 3840, 2160) == 1080 * 3840 + 1920
    d = 4.0
    ytop = d * math.tan(math.radians(30.0))
    q, alive = _x(oracle, ph, [0.0, ytop, 0.0], Wd=3840, Hd=2160)
    assert alive and abs(q[1] - 1.0) < 2e-7                     # top edge of the frustum
    q, alive = _x(oracle, ph, [ytop * 3840 / 2160, 0.0, 0.0], Wd=3840, Hd=2160)
    assert alive and abs(q[0] - 1.0) < 2e-7                     # right edge: fx = f H / W
    _, alive = _x(oracle, ph, [0.0, 0.0, -4.0], Wd=16, Hd=9)
    assert not alive                                             # at the camera: d = 0 <= near
    _, alive = _x(oracle, ph, [0.0, 0.0, -5.0], Wd=16, Hd=9)
    assert not alive                                             # behind the camera
    ty, prm = oracle.resolve_xform(ph, 3, 0.0, 3840, 2160)
    assert ty == 6 and abs(prm[1] - 1.7320508) < 1e-7 and abs(prm[0] - 1.7320508 * 0.5625) < 1e-7
    assert prm[2] == -4.0 and abs(prm[3] - 1e-3) < 1e-9


# ------------------------------------------------------------------ P11: colour = generating map
def test_colour_is_map_of_this_iteration(oracle):
    sys = W.System(2, "ifs", W.square_funcs(), [], "map_index", W.palette_for(4))
    rnd = W.Render(4096, 21, 60, 20, 2, 2, (-1, 1, -1, 1), "rgba_f32")
    img, ctr = oracle.render(sys, rnd)
    pal = W.palette_for(4).astype(np.float64)
    for k in range(4):                      # quadrant k = pixel (k>>1, k&1) holds only colour k
        n = img[k, 3]
        assert n > 0 and np.array_equal(img[k, :3], pal[k, :3] * n)
    assert img[:, 3].sum() == 4096 * 40


# ------------------------------------------------------------------ P12: depth buffer
def test_depth_buffer_vs_bruteforce(oracle):
    w = W.config(4)
    n = 20000
    rnd = w.scaled(n_points=n, iterations=25, burn_in=24, width=96, height=54).render
    img, ctr = oracle.render(w.system, rnd)
    assert int(ctr[0]) == n
    picks, _, fq, alive = oracle.trace(w.system, rnd)
    assert alive.all() and fq[:, 2].min() >= 3.0 - 1e-5 and fq[:, 2].max() <= 5.0 + 1e-5
    pal = w.system.palette.astype(np.uint64)
    col = (pal[:, 0] | (pal[:, 1] << 8) | (pal[:, 2] << 16) | (pal[:, 3] << 24))[picks[:, -1]]
    key = (fq[:, 2].copy().view(np.uint32).astype(np.uint64) << np.uint64(32)) | col
    pix = np.array([oracle.pixel(x, y, rnd.bounds, 96, 54) for x, y in fq[:, :2]])
    want = np.full(96 * 54, oracle.DEPTH_EMPTY, dtype=np.uint64)
    order = np.lexsort((key, pix))          # brute force: sort by (pixel, key), first wins
    first = np.ones(n, dtype=bool)
    first[1:] = pix[order][1:] != pix[order][:-1]
    want[pix[order][first]] = key[order][first]
    assert np.array_equal(img, want)
    # order independence: sub-ranges merged in reverse
    parts = [oracle.render(w.system, rnd, n_points=5000, point_offset=o)[0] for o in (15000, 0, 10000, 5000)]
    assert np.array_equal(np.minimum.reduce(parts), img)
    # depth ordering really is float ordering: nearest (smallest d) wins
    d = (img[img != oracle.DEPTH_EMPTY] >> np.uint64(32)).astype(np.uint32).view(np.float32)
    assert d.min() >= 3.0 - 1e-5 and d.max() <= 5.0


# ------------------------------------------------------------------ P13: cloud
def test_cloud_conservation(oracle):
    w = W.config(3)
    n = 1 << 15
    cloud = W.gaussian_mixture_cloud(n, w.cloud_seed)
    rnd = w.scaled(n_points=n, width=384, height=216).render
    img, ctr = oracle.render(w.system, rnd, cloud=cloud)
    assert int(ctr[0]) + int(ctr[1]) == n and int(ctr[0]) > 0.5 * n
    assert img[:, 3].sum() == int(ctr[0])
    _, fg, fq, alive = oracle.trace(w.system, rnd, cloud=cloud, want_picks=False)
    assert np.array_equal(fg[:, 0], cloud["x"]) and np.array_equal(fg[:, 2], cloud["z"])
    inb = alive.astype(bool) & (np.abs(fq[:, 0]) <= 1) & (np.abs(fq[:, 1]) <= 1)
    assert int(inb.sum()) == int(ctr[0])
    for ch in range(3):
        want = ((cloud["rgba8"][inb] >> (8 * ch)) & 0xFF).astype(np.float64).sum()
        assert img[:, ch].sum() == want
    # twist and bend preserve x^2+y^2 and z: depth after pinhole is z + 4
    assert np.allclose(fq[alive.astype(bool), 2], cloud["z"][alive.astype(bool)] + 4.0, atol=1e-6)
    # sub-range addressing: record p is cloud[p]
    a, _ = oracle.render(w.system, rnd, cloud=cloud, n_points=n // 2, point_offset=n // 2)
    b, _ = oracle.render(w.system, rnd, cloud=cloud, n_points=n // 2, point_offset=0)
    assert np.array_equal(a + b, img)


# ------------------------------------------------------------------ P14: tone map
def test_tonemap_closed_forms(oracle):
    acc = np.zeros((16, 4), dtype=np.float32)
    acc[1] = (255 * 9, 0, 0, 9)              # n = n_max: L = 1 -> pure red, alpha 255
    acc[2] = (0, 255 * 2, 0, 2)              # L = log 3 / log 10
    acc[3] = (255 * 3, 255 * 3, 0, 3)
    out = oracle.tonemap(acc, "rgba_f32", 4, 4, 2.2, 1 / 255.0)
    assert out[0] == 0 and np.all(out[4:] == 0)
    assert out[1] == 0xFF0000FF
    L2 = math.log(3) / math.log(10)
    g2 = int(math.floor(255 * L2 ** (1 / 2.2) + 0.5))
    assert out[2] == (g2 << 8) | (int(math.floor(255 * L2 + 0.5)) << 24)
    L3 = math.log(4) / math.log(10)
    v3 = int(math.floor(255 * L3 ** (1 / 2.2) + 0.5))
    assert out[3] == v3 | (v3 << 8) | (int(math.floor(255 * L3 + 0.5)) << 24)
    # HIST: grey = L^(1/gamma), monotone in n
    hist = np.arange(16, dtype=np.uint32)
    out = oracle.tonemap(hist, "hist_u32", 4, 4, 1.0, 1.0)
    grey = out & 0xFF
    assert out[0] == 0 and grey[15] == 255 and np.all(np.diff(grey.astype(int)) >= 0)
    assert grey[3] == int(math.floor(255 * math.log(4) / math.log(16) + 0.5)) == 128
    assert np.all(((out >> 8) & 0xFF) == grey) and np.all(((out >> 16) & 0xFF) == grey)
    # DEPTH: resolve = colour, empty -> 0
    buf = np.full(4, oracle.DEPTH_EMPTY, dtype=np.uint64)
    buf[2] = (np.uint64(0x40800000) << np.uint64(32)) | np.uint64(0xFF112233)
    out = oracle.tonemap(buf, "depth_u64", 2, 2, 2.2, 1.0)
    assert list(out) == [0, 0, 0xFF112233, 0]


# ------------------------------------------------------------------ NEXT-2: one-to-many splatting
def _branches():
    a = [W.Xform("affine", [0.5, 0, 0, 0.5, -0.4, 0.3])]
    b = [W.Xform("swirl"), W.Xform("affine", [0.6, 0, 0, 0.6, 0.3, -0.2])]
    c = []                                                   # the generated point itself
    return [a, b, c]


def _join(branches):
    out = []
    for i, br in enumerate(branches):
        if i:
            out.append(W.Xform("branch"))
        out.extend(br)
    return out


@pytest.mark.parametrize("mode", ["hist_u32", "rgba_f32"])
def test_branches_equal_the_sum_of_single_chain_renders(oracle, mode):
    """"Many objects from a single primitive": every BRANCH of the chain gets its own
    copy of the generated point.  The generator never sees the chain (Fig. 2(B)), so the M-branch image is
    EXACTLY the sum of the M single-chain images -- which reduces this path to the pinned single-chain one.
    Splats per point = M (I - B)."""
    brs = _branches()
    rule, pal = ("none", None) if mode == "hist_u32" else ("map_index", W.palette_for(4))
    r = W.Render(3000, 5, 60, 10, 128, 128, (-1, 1, -1, 1), mode)
    multi, mc = oracle.render(W.System(2, "ifs", W.square_funcs(), _join(brs), rule, pal), r)
    total, n_in, n_drop = None, 0, 0
    for br in brs:
        img, c = oracle.render(W.System(2, "ifs", W.square_funcs(), br, rule, pal), r)
        total = img.copy() if total is None else total + img
        n_in += int(c[0]); n_drop += int(c[1])
    assert np.array_equal(multi, total)
    assert int(mc[0]) == n_in and int(mc[1]) == n_drop and n_in + n_drop == 3 * 3000 * 50
    # a trailing BRANCH opens one more (empty) branch: the generated point itself
    again, ac = oracle.render(W.System(2, "ifs", W.square_funcs(), _join(brs[:2]) + [W.Xform("branch")], rule, pal), r)
    assert np.array_equal(again, multi) and np.array_equal(ac, mc)


def test_branches_depth_is_the_min_of_single_chain_renders(oracle):
    pin = W.Xform("pinhole", [60.0, -4.0, 1e-3])
    brs = [[pin], [W.Xform("affine", [0.5, 0, 0, 0, 0.5, 0, 0, 0, 0.5, 0.3, 0.2, -1.0]), pin]]
    r = W.Render(2000, 9, 50, 10, 160, 90, (-1, 1, -1, 1), "depth_u64")
    pal = W.palette_for(20)
    multi, mc = oracle.render(W.System(3, "ifs", W.menger_funcs(), _join(brs), "map_index", pal), r)
    singles = [oracle.render(W.System(3, "ifs", W.menger_funcs(), br, "map_index", pal), r)[0] for br in brs]
    assert np.array_equal(multi, np.minimum(singles[0], singles[1])) and int(mc[0]) + int(mc[1]) == 2 * 2000 * 40
    with pytest.raises(ValueError):            # a branch that does not end in PINHOLE cannot feed a depth buffer
        oracle.render(W.System(3, "ifs", W.menger_funcs(), _join([[pin], []]), "map_index", pal), r)
    with pytest.raises(ValueError):            # reuse (Fig. 2(C)) has no meaning with several branches
        oracle.render(W.System(2, "ifs", W.square_funcs(), _join(_branches()), "none", None, reuse=True),
                      W.Render(10, 1, 20, 5, 32, 32, (-1, 1, -1, 1), "hist_u32"))


# ------------------------------------------------------------------ NEXT-2: PRNG-placed duplicates (DESIGN R14)
def _u24(w):
    return np.float32(np.float32(w >> 8) * np.float32(2.0 ** -23) - np.float32(1.0))


def test_scatter_places_copies_by_philox(oracle):
    """A SCATTER(D, rx, ry) step moves the copy onto duplicate d = floor(w D / 2^32), w = the AUX-domain word
    of (seed, p, it); the offset of duplicate d is a pure function of (seed, d) in the PLACE domain.  Checked
    per point against the pinned Philox (known-answer tests) with the keying written out here; the empty-chain
    generator state must not move (Fig. 2(B)); duplicates are drawn uniformly (chi-square)."""
    D, rx, ry = 5, 0.75, 0.5
    seed, n, I = 0xABCDEF12345, 4000, 24
    sys_s = W.System(2, "ifs", W.square_funcs(), [W.Xform("scatter", [D, rx, ry, 0.0])], "none")
    r = W.Render(n, seed, I, 4, 64, 64, (-2, 2, -2, 2), "hist_u32")
    _, g, q, alive = oracle.trace(sys_s, r)
    _, g0, _, _ = oracle.trace(W.System(2, "ifs", W.square_funcs(), [], "none"), r)
    assert np.array_equal(g, g0) and alive.all()
    key = [seed & 0xFFFFFFFF, seed >> 32]
    offs = []
    for d in range(D):
        v = oracle.philox4x32_10([d, 0, 0, 3], key)
        offs.append((np.float32(_u24(v[0]) * np.float32(rx)), np.float32(_u24(v[1]) * np.float32(ry))))
    assert len({(float(a), float(b)) for a, b in offs}) == D
    it = I - 1
    counts = np.zeros(D)
    for p in range(n):
        w = oracle.philox4x32_10([p, 0, it >> 2, 2], key)[it & 3]
        d = (w * D) >> 32
        counts[d] += 1
        assert q[p, 0] == np.float32(g[p, 0] + offs[d][0]) and q[p, 1] == np.float32(g[p, 1] + offs[d][1]) and q[p, 2] == g[p, 2]
    chi2 = ((counts - n / D) ** 2 / (n / D)).sum()
    assert chi2 < 30.0                                                   # 4 dof
    # D = 1: one copy; the offset is applied once per coordinate, z untouched in 2-D
    one = W.System(2, "ifs", W.square_funcs(), [W.Xform("scatter", [1, rx, ry, 0.0])], "none")
    _, g1, q1, _ = oracle.trace(one, r)
    assert np.all(q1[:, 0] == (g1[:, 0] + offs[0][0]).astype(np.float32)) and np.all(q1[:, 1] == (g1[:, 1] + offs[0][1]).astype(np.float32))
    with pytest.raises(ValueError):                                      # D must be a whole number in [1, 2^20]
        oracle.trace(W.System(2, "ifs", W.square_funcs(), [W.Xform("scatter", [2.5, rx, ry, 0.0])], "none"), r)
