"""Pins of the CPU oracle, part 1: RNG, pick, init, generator maps, pixel rule.

The paper prints no numeric output of the method (PAPER.md has no worked example), so the
oracle is pinned to what the mathematics fixes: published Philox known answers, exact integer
threshold tables, fixed points of the affine maps, the binary-expansion closed form of the
Fig. 1 square, brute-force composition over all map words of length <= 8.
None of these tests touches the CUDA path.
"""
import itertools
import math
import os

import numpy as np
import pytest

from paper_2606_02226_b200 import workloads as W

GOLD = os.path.join(os.path.dirname(__file__), "golden")


def _rows(name):
    with open(os.path.join(GOLD, name)) as fh:
        return [ln.strip() for ln in fh if ln.strip() and not ln.startswith("#")]


# ------------------------------------------------------------------ P1: Philox4x32-10
def test_philox_known_answers(oracle):
    for row in _rows("philox4x32_10_kat.txt"):
        v = [int(t, 16) for t in row.split()]
        assert oracle.philox4x32_10(v[0:4], v[4:6]) == v[6:10]


def test_pick_word_keying(oracle):
    """DESIGN R1: counter = (p lo, p hi, it>>2, domain 0), key = (seed lo, seed hi), word it&3."""
    seed, p = 0x0123456789ABCDEF, 0x00000002_00000007
    for it in (0, 1, 2, 3, 4, 7, 8, 999, 1000):
        blk = oracle.philox4x32_10([p & 0xFFFFFFFF, p >> 32, it >> 2, 0], [seed & 0xFFFFFFFF, seed >> 32])
        assert oracle.pick_word(seed, p, it) == blk[it & 3]
    # distinct points / seeds / blocks give distinct words (no accidental aliasing of fields)
    words = {oracle.pick_word(s, q, it) for s in (1, 2, 1 << 32) for q in (0, 1, 1 << 32) for it in (0, 4)}
    assert len(words) == 18


def test_init_point_is_24bit_uniform(oracle):
    """DESIGN R3: coord = (w >> 8) * 2^-23 - 1 from INIT-domain words 0,1,2."""
    seed = 77
    for p in (0, 1, 12345, (1 << 40) + 3):
        blk = oracle.philox4x32_10([p & 0xFFFFFFFF, p >> 32, 0, 1], [seed, 0])
        want = [(w >> 8) / 2.0 ** 23 - 1.0 for w in blk[:3]]          # exact in double
        g3 = oracle.init_point(seed, p, 3)
        g2 = oracle.init_point(seed, p, 2)
        assert [float(v) for v in g3] == want
        assert [float(v) for v in g2[:2]] == want[:2] and float(g2[2]) == 0.0
    pts = np.array([oracle.init_point(5, p, 3) for p in range(20000)], dtype=np.float64)
    assert pts.min() >= -1.0 and pts.max() < 1.0
    assert np.all(np.abs(pts.mean(axis=0)) < 5 * math.sqrt(1 / 3 / 20000))
    assert np.all(np.abs(pts.var(axis=0) - 1 / 3) < 0.02)


# ------------------------------------------------------------------ P2: thresholds and pick
def test_threshold_tables_exact(oracle):
    for row in _rows("pick_thresholds.txt"):
        n, vals = row.split(":")
        n = int(n)
        want = [int(v) for v in vals.split()] + [1 << 32]
        prob = [float(np.float32(1.0 / n))] * n
        assert oracle.thresholds(prob) == want


def test_pick_boundaries_bruteforce(oracle):
    for probs in ([0.25] * 4, [1 / 3] * 3, [0.05] * 20, [0.1, 0.2, 0.3, 0.4], [1.0], [0.0, 1.0, 0.0, 2.0]):
        probs = [float(np.float32(p)) for p in probs]
        T = oracle.thresholds(probs)
        n = len(probs)
        assert T[-1] == 1 << 32 and all(T[j] <= T[j + 1] for j in range(n - 1))
        us = {0, 0xFFFFFFFF}
        for tj in T[:-1]:
            us |= {max(0, tj - 1), min(tj, 0xFFFFFFFF), min(tj + 1, 0xFFFFFFFF)}
        for u in us:
            want = sum(1 for j in range(n - 1) if u >= T[j])          # the definition, by hand
            assert oracle.pick(u, T) == want
            assert 0 <= want < n
    # zero-probability maps are never chosen
    T = oracle.thresholds([0.0, 1.0, 0.0, 2.0])
    ks = {oracle.pick(u, T) for u in range(0, 1 << 32, 9999991)}
    assert ks == {1, 3}
    # n = 3 is not mulhi(u, 3): the switch is at 1431655765, not 1431655766
    T3 = oracle.thresholds([float(np.float32(1 / 3))] * 3)
    assert oracle.pick(1431655765, T3) == 1 and oracle.pick(1431655764, T3) == 0


def test_invalid_probabilities(oracle):
    for bad in ([-0.1, 1.0], [0.0, 0.0], [float("nan"), 1.0], [float("inf"), 1.0]):
        with pytest.raises(ValueError):
            oracle.thresholds(bad)


def test_pick_frequencies_chi2(oracle):
    probs = [0.1, 0.2, 0.3, 0.4]
    sys = W.System(2, "ifs", W.square_funcs(probs), [], "none")
    rnd = W.Render(4096, 99, 64, 0, 16, 16, (-1, 1, -1, 1), "hist_u32")
    picks, _, _, _ = oracle.trace(sys, rnd)
    cnt = np.bincount(picks.ravel(), minlength=4).astype(np.float64)
    pf = np.array([float(np.float32(p)) for p in probs])
    exp = pf / pf.sum() * picks.size
    chi2 = ((cnt - exp) ** 2 / exp).sum()
    assert chi2 < 21.1                      # 3 dof, p ~ 1e-4
    # and picks are exactly pick(pick_word)
    T = oracle.thresholds([f.prob for f in sys.funcs])
    for p in (0, 17, 4095):
        for it in (0, 1, 5, 63):
            assert picks[p, it] == oracle.pick(oracle.pick_word(99, p, it), T)


# ------------------------------------------------------------------ P3: fixed points
@pytest.mark.parametrize("name", ["square", "sierpinski", "menger", "carpet"])
def test_affine_fixed_points(oracle, name):
    """One-hot probabilities: the chaos game converges to the fixed point (I-A)^-1 b of that map."""
    if name == "square":
        funcs, dim = W.square_funcs(), 2
        fixed = [(2 * (k & 1) - 1, 2 * (k >> 1) - 1, 0) for k in range(4)]
    elif name == "sierpinski":
        funcs, dim = W.sierpinski_funcs(), 2
        fixed = [(x, y, 0) for x, y in W.sierpinski_vertices()]
    elif name == "carpet":
        funcs, dim = W.carpet_funcs(), 2
        fixed = [(ix - 1, iy - 1, 0) for iy in range(3) for ix in range(3) if not (ix == 1 and iy == 1)]
    else:
        funcs, dim = W.menger_funcs(), 3
        fixed = [(ix - 1, iy - 1, iz - 1) for ix, iy, iz in W.menger_cells()]
    assert len(funcs) == len(fixed)
    for k in range(len(funcs)):
        one_hot = [W.Func(f.type, 1.0 if j == k else 0.0, f.params) for j, f in enumerate(funcs)]
        sys = W.System(dim, "ifs", one_hot, [], "none")
        rnd = W.Render(8, 3, 60, 59, 8, 8, (-1, 1, -1, 1), "hist_u32")
        picks, fg, _, _ = oracle.trace(sys, rnd)
        assert np.all(picks == k)
        assert np.allclose(fg, np.array(fixed[k], dtype=np.float64), atol=3e-7, rtol=0)


def test_menger_table_structure():
    cells = W.menger_cells()
    assert len(cells) == 20 and cells[0] == (0, 0, 0) and cells[-1] == (2, 2, 2)
    assert all((c[0] == 1) + (c[1] == 1) + (c[2] == 1) < 2 for c in cells)
    ranks = [c[0] + 3 * c[1] + 9 * c[2] for c in cells]
    assert ranks == sorted(ranks)


# ------------------------------------------------------------------ P8: all words of length <= 8
@pytest.mark.parametrize("L", [1, 2, 3, 5, 8])
def test_words_bruteforce_square(oracle, L):
    """Apply every word w in {0..3}^L (L <= 5) or 4096 random words (L = 8) to a start point with
    the oracle's map, compare with the exact closed form in double:
    f_w(x) = 2^-L x + sum_j 2^-(L-j) c_{w_j}/..., all exact dyadic arithmetic."""
    funcs = W.square_funcs()
    x0 = np.array([0.3125, -0.65625, 0.0])
    if L <= 5:
        words = list(itertools.product(range(4), repeat=L))
    else:
        rng = np.random.default_rng(1)
        words = [tuple(rng.integers(0, 4, size=L)) for _ in range(4096)]
    for w in words:
        g = x0.astype(np.float32)
        exact = x0.copy()
        for k in w:
            g = oracle.apply_func(funcs[k], 2, g)
            c = np.array([2 * (k & 1) - 1, 2 * (k >> 1) - 1, 0.0])
            exact = 0.5 * exact + 0.5 * c
            exact[2] = 0.0
        assert np.array_equal(g.astype(np.float64), exact)    # dyadic: float32 is exact here


def test_words_support_and_measure_nonuniform(oracle):
    """After L steps a point lies in cell f_w([-1,1]^2), w = last L picks; on a 2^L x 2^L image
    that cell is one pixel and its mass is prod p_{w_i}.  One splat per point => i.i.d."""
    probs = [0.1, 0.2, 0.3, 0.4]
    L = 4
    sys = W.System(2, "ifs", W.square_funcs(probs), [], "none")
    n = 1 << 18
    rnd = W.Render(n, 4242, L + 5, L + 4, 1 << L, 1 << L, (-1, 1, -1, 1), "hist_u32")
    img, ctr, _ = oracle.render_parallel(sys, rnd)
    assert int(ctr[0]) == n and int(img.sum()) == n
    pf = np.array([float(np.float32(p)) for p in probs], dtype=np.float64)
    pf /= pf.sum()
    exp = np.zeros((1 << L, 1 << L))
    for w in itertools.product(range(4), repeat=L):           # w[0] = most recent pick
        px = sum((w[j] & 1) << (L - 1 - j) for j in range(L))
        py = sum((w[j] >> 1) << (L - 1 - j) for j in range(L))
        exp[py, px] = n * np.prod(pf[list(w)])
    chi2 = ((img.reshape(1 << L, 1 << L) - exp) ** 2 / exp).sum()
    dof = (1 << (2 * L)) - 1
    assert abs(chi2 - dof) < 5 * math.sqrt(2 * dof)


def test_words_sierpinski_cells(oracle):
    """Every post-burn-in state lies within 2^-8 of f_w(0), w = its last 8 picks (the attractor
    has radius 1 about the origin); f_w(0) computed independently in double."""
    sys = W.System(2, "ifs", W.sierpinski_funcs(), [], "none")
    rnd = W.Render(2048, 11, 40, 39, 8, 8, (-1, 1, -1, 1), "hist_u32")
    picks, fg, _, _ = oracle.trace(sys, rnd)
    V = np.array(W.sierpinski_vertices())
    z = np.zeros((2048, 2))
    for j in range(8):                       # oldest of the last 8 first
        k = picks[:, 40 - 8 + j]
        z = 0.5 * z + 0.5 * V[k]
    d = np.hypot(fg[:, 0] - z[:, 0], fg[:, 1] - z[:, 1])
    assert d.max() <= 2.0 ** -8 + 1e-6


# ------------------------------------------------------------------ P4: closed form for cfg 0
def test_cfg0_pixel_is_word_of_last_nine_picks(oracle):
    w = W.config(0)
    n, I = 1 << 14, 30
    rnd = w.scaled(n_points=n, iterations=I, burn_in=I - 1).render
    picks, fg, fq, alive = oracle.trace(w.system, rnd)
    px = np.zeros(n, dtype=np.int64)
    py = np.zeros(n, dtype=np.int64)
    for j in range(9):                       # j = 0: the most recent pick = most significant bit
        k = picks[:, I - 1 - j].astype(np.int64)
        px |= (k & 1) << (8 - j)
        py |= (k >> 1) << (8 - j)
    want = np.bincount(py * 512 + px, minlength=512 * 512)
    img, ctr = oracle.render(w.system, rnd)
    assert int(ctr[0]) == n and int(ctr[1]) == 0
    mism = np.abs(img.astype(np.int64) - want).sum() / 2
    assert mism / n < 1e-4                  # float ties at pixel edges only
    assert np.array_equal(fg, fq) and alive.all()     # empty chain: copy == state
    # and the pixel rule itself on the final states
    pix = np.array([oracle.pixel(x, y, rnd.bounds, 512, 512) for x, y in fg[:512, :2]])
    assert np.count_nonzero(pix != (py * 512 + px)[:512]) <= 1


# ------------------------------------------------------------------ pixel rule (DESIGN R8)
def test_pixel_rule_edges(oracle):
    b = (-1.0, 1.0, -1.0, 1.0)
    assert oracle.pixel(-1.0, -1.0, b, 512, 512) == 0                   # row 0 is ymin
    assert oracle.pixel(1.0, -1.0, b, 512, 512) == 511                  # closed upper bound, clamped
    assert oracle.pixel(-1.0, 1.0, b, 512, 512) == 511 * 512
    assert oracle.pixel(0.0, 0.0, b, 512, 512) == 256 * 512 + 256
    assert oracle.pixel(np.nextafter(np.float32(1.0), np.float32(2.0)), 0.0, b, 512, 512) == -1
    assert oracle.pixel(np.nextafter(np.float32(-1.0), np.float32(-2.0)), 0.0, b, 512, 512) == -1
    assert oracle.pixel(float("nan"), 0.0, b, 512, 512) == -1
    assert oracle.pixel(0.0, float("inf"), b, 512, 512) == -1
    # non-square image / bounds: x in [-16/9,16/9] on 1920 columns
    b2 = (-16 / 9, 16 / 9, -1.0, 1.0)
    assert oracle.pixel(0.0, 0.0, b2, 1920, 1080) == 540 * 1920 + 960
    assert oracle.pixel(-1.7, 0.999, b2, 1920, 1080) == 1079 * 1920 + int(math.floor((-1.7 + 16 / 9) * 540))


# ------------------------------------------------------------------ NEXT-1: PAPER Eq. 1, the circle IFS
def _golden_eq1():
    import os
    rows = []
    with open(os.path.join(os.path.dirname(__file__), "golden", "eq1_circle_half.txt")) as fh:
        for ln in fh:
            if ln.strip() and not ln.startswith("#"):
                rows.append([float(v) for v in ln.split()])
    return rows


def test_circle_half_golden_values(oracle):
    """Values worked by hand from the printed Eq. 1 (tests/golden/eq1_circle_half.txt)."""
    rows = _golden_eq1()
    assert len(rows) == 9
    for x, y, fid, flag, ex, ey in rows:
        g = oracle.apply_func(W.Func("circle_half", 0.5, [fid, flag]), 2, np.array([x, y, 0.0], dtype=np.float32))
        assert abs(float(g[0]) - ex) < 2e-7 and abs(float(g[1]) - ey) < 2e-7, (x, y, fid, flag, g)


@pytest.mark.parametrize("flag", [0.0, 1.0])
def test_circle_half_invariants(oracle, flag):
    """the maps send the disc "on to either the top or bottom half of itself": for r < 1 the
    sign of y2 is decided by f_id alone and r2 < 1.  The map swaps the polar coordinates: the output radius
    depends on the input ANGLE only, the output angle on the input RADIUS only."""
    rng = np.random.default_rng(7)
    for _ in range(300):
        r, th = rng.uniform(0.01, 0.99), rng.uniform(0.01, 2 * math.pi - 0.01)
        r_b, th_b = rng.uniform(0.01, 0.99), rng.uniform(0.01, 2 * math.pi - 0.01)
        for fid in (0.0, 1.0):
            f = W.Func("circle_half", 0.5, [fid, flag])
            def m(rr, tt):
                return oracle.apply_func(f, 2, np.array([rr * math.cos(tt), rr * math.sin(tt), 0.0], dtype=np.float32)).astype(np.float64)
            a, b, c = m(r, th), m(r_b, th), m(r, th_b)
            assert (a[1] >= 0) == (fid == 0.0) and np.hypot(a[0], a[1]) < 1.0
            assert abs(np.hypot(a[0], a[1]) - np.hypot(b[0], b[1])) < 1e-6          # same angle -> same radius
            assert abs(math.atan2(a[1], a[0]) - math.atan2(c[1], c[0])) < 1e-5      # same radius -> same angle


def test_circle_half_r2_reading_has_uniform_invariant_density(oracle):
    """In (s, u) = (r^2, theta / 2 pi) the r^2 reading is (s, u) -> (u, (s + f_id) / 2), which preserves
    the uniform measure of the unit square, i.e. the uniform AREA measure of the disc: the chaos game's
    histogram is flat over pixels wholly inside the disc (chi-square, one splat per point => i.i.d.)."""
    sys_c = W.System(2, "ifs", W.circle_funcs(r2_reading=True), [], "none")
    n, side = 400000, 32
    r = W.Render(n, 1, 40, 39, side, side, (-1, 1, -1, 1), "hist_u32")
    h, c = oracle.render(sys_c, r)
    assert int(c[0]) == n
    h = h.reshape(side, side).astype(np.float64)
    edges = np.linspace(-1, 1, side + 1)
    far = np.maximum(np.abs(edges[:-1]), np.abs(edges[1:]))
    inside = (far[:, None] ** 2 + far[None, :] ** 2) < 1.0                  # all four corners inside the disc
    exp = n * (2.0 / side) ** 2 / math.pi
    chi2 = ((h[inside] - exp) ** 2 / exp).sum()
    dof = int(inside.sum())
    assert dof > 600 and abs(chi2 - dof) < 6 * math.sqrt(2 * dof), (chi2, dof)
    # the as-printed reading (r, not r^2) is NOT uniform: same statistic, far outside the band
    h2, _ = oracle.render(W.System(2, "ifs", W.circle_funcs(False), [], "none"), r)
    h2 = h2.reshape(side, side).astype(np.float64)
    assert ((h2[inside] - exp) ** 2 / exp).sum() > dof + 50 * math.sqrt(2 * dof)
