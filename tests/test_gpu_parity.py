"""GPU parity: the CUDA path (through the C ABI) against the CPU oracle, element by element, on
the same seeded inputs.  Bars (BASELINE.json north_star / SURVEY 8(c) S10):
  (i)   map-index sequences bit-exact;
  (ii)  final float32 coordinates within 1e-4 absolute;
  (iii) affine-only images (cfg 0; cfg 4 incl. pinhole and depth) bit-exact per pixel;
  (iv)  otherwise normalised-density L1 <= 1e-3 on the count and on each colour channel;
  (v)   counters: in-bounds + dropped = points x (iterations - burn_in).
"""
import math

import numpy as np
import pytest

from paper_2606_02226_b200 import workloads as W
from tests._gpu_util import density_l1, gpu_render, gpu_trace

pytestmark = pytest.mark.gpu

COORD_TOL = 1e-4
L1_TOL = 1e-3


@pytest.fixture(scope="module")
def cfs():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    from paper_2606_02226_b200 import cfs as mod
    mod.lib()
    return mod


def _cloud_for(w, n):
    return W.gaussian_mixture_cloud(n, w.cloud_seed) if w.system.gen == "cloud" else None


# ------------------------------------------------------------------ (i), (ii): picks and coordinates
@pytest.mark.parametrize("cfg", [0, 1, 2, 3, 4])
def test_pick_sequences_and_coordinates(cfs, oracle, cfg):
    w = W.config(cfg)
    n = 1024 + 37                                   # several CTAs and a ragged tail
    cloud = _cloud_for(w, n)
    w = w.scaled(n_points=n)
    for t in (w.frames[0], w.frames[len(w.frames) // 2]) if len(w.frames) > 1 else (w.frames[0],):
        gp, gg, gq, ga = gpu_trace(cfs, w, t=t, cloud=cloud)
        op, og, oq, oa = oracle.trace(w.system, w.render, cloud=cloud, t=t)
        assert np.array_equal(gp, op)                               # (i) bit-exact
        assert np.array_equal(gg, og)                               # affine generators: bit-equal
        assert np.array_equal(ga, oa)
        live = oa.astype(bool)
        assert np.abs(gq[live].astype(np.float64) - oq[live]).max() <= COORD_TOL   # (ii)
        if cfg in (0, 4):
            assert np.array_equal(gq, oq)                           # affine + pinhole: bit-exact


def test_point_offset_beyond_32_bits(cfs, oracle):
    w = W.config(0).scaled(n_points=300, iterations=40)
    off = (1 << 33) + 12345
    gp, gg, _, _ = gpu_trace(cfs, w, point_offset=off)
    op, og, _, _ = oracle.trace(w.system, w.render, point_offset=off)
    assert np.array_equal(gp, op) and np.array_equal(gg, og)


# ------------------------------------------------------------------ (iii): bit-exact images
@pytest.mark.parametrize("variant", ["direct", "warp_agg", "cluster_hist", "auto"])
def test_cfg0_histogram_bit_exact(cfs, oracle, variant):
    w = W.config(0).scaled(n_points=4096 + 99)
    g, gc = gpu_render(cfs, w, variant=variant)
    o, oc, _ = oracle.render_parallel(w.system, w.render)
    assert np.array_equal(g, o)
    assert np.array_equal(gc, oc) and int(gc[0]) == w.render.n_points * 980 and int(gc[1]) == 0


@pytest.mark.parametrize("size", [(64, 64), (200, 120), (224, 224)])
@pytest.mark.parametrize("variant", ["shared_hist", "direct", "warp_agg", "cluster_hist", "auto"])
def test_small_histograms_all_variants(cfs, oracle, size, variant):
    """Per-CTA shared-memory privatised histogram (and the others) on images that fit shared memory;
    bounds narrower than the attractor so that some splats are dropped."""
    w = W.config(0).scaled(n_points=3000, iterations=200, width=size[0], height=size[1])
    w = w.scaled(bounds=(-0.75, 1.0, -1.0, 0.5))
    g, gc = gpu_render(cfs, w, variant=variant)
    o, oc, _ = oracle.render_parallel(w.system, w.render)
    assert np.array_equal(g, o) and np.array_equal(gc, oc)
    assert int(gc[1]) > 0 and int(gc[0]) + int(gc[1]) == 3000 * 180


def test_cfg0_full_size_bit_exact(cfs, oracle):
    w = W.config(0)
    g, gc = gpu_render(cfs, w)
    o, oc, _ = oracle.render_parallel(w.system, w.render)
    assert int(gc[0]) == 64225280 and int(g.sum(dtype=np.uint64)) == 64225280
    assert np.array_equal(g, o)


@pytest.mark.parametrize("n", [1, 31, 255, 256, 257, 5000])
def test_cfg4_depth_bit_exact(cfs, oracle, n):
    w = W.config(4).scaled(n_points=n, iterations=120, width=480, height=270)
    g, gc = gpu_render(cfs, w)
    o, oc = oracle.render(w.system, w.render)
    assert np.array_equal(g, o) and np.array_equal(gc, oc)
    assert int(gc[0]) == n * 100


def test_cfg4_full_image_subrange_bit_exact(cfs, oracle):
    """Full 3840x2160 buffer, bench launch shape, a point sub-range the oracle finishes in seconds;
    sub-ranges compose by min into the full-range result."""
    w = W.config(4).scaled(n_points=1 << 13)
    g, gc = gpu_render(cfs, w)
    o, oc, _ = oracle.render_parallel(w.system, w.render)
    assert np.array_equal(g, o) and np.array_equal(gc, oc)
    a, _ = gpu_render(cfs, w, n_points=5000, point_offset=0)
    b, _ = gpu_render(cfs, w, n_points=(1 << 13) - 5000, point_offset=5000)
    assert np.array_equal(np.minimum(a, b), g)


# ------------------------------------------------------------------ (iv): density L1
def _check_rgba(g, o, gc, oc):
    assert np.array_equal(gc, oc)                                    # (v)
    assert g[:, 3].astype(np.float64).sum() == o[:, 3].sum() == float(oc[0])
    for ch in range(4):
        assert density_l1(g[:, ch], o[:, ch]) <= L1_TOL


def test_cfg1_swirl_rgba(cfs, oracle):
    w = W.config(1).scaled(n_points=(1 << 14) + 5)
    g, gc = gpu_render(cfs, w)
    o, oc, _ = oracle.render_parallel(w.system, w.render)
    _check_rgba(g, o, gc, oc)
    assert int(gc[1]) == 0


@pytest.mark.parametrize("frame", [0, 7, 15])
def test_cfg2_animation_frames(cfs, oracle, frame):
    w = W.config(2).scaled(n_points=(1 << 14) + 3)
    t = w.frames[frame]
    g, gc = gpu_render(cfs, w, t=t)
    o, oc, _ = oracle.render_parallel(w.system, w.render, t=t)
    _check_rgba(g, o, gc, oc)


def test_cfg3_cloud(cfs, oracle):
    w = W.config(3)
    n = (1 << 18) + 11
    cloud = W.gaussian_mixture_cloud(n, w.cloud_seed)
    w = w.scaled(n_points=n)
    g, gc = gpu_render(cfs, w, cloud=cloud)
    o, oc, _ = oracle.render_parallel(w.system, w.render, cloud=cloud)
    assert int(gc[0]) + int(gc[1]) == n
    # a point within float rounding of the frustum edge may be dropped on one side only
    assert abs(int(gc[0]) - int(oc[0])) <= 4
    for ch in range(4):
        assert density_l1(g[:, ch], o[:, ch]) <= L1_TOL
    # sub-range of the whole cloud: record p is d_cloud[p]
    a, _ = gpu_render(cfs, w, cloud=cloud, n_points=n - 1000, point_offset=1000)
    b, _ = gpu_render(cfs, w, cloud=cloud, n_points=1000, point_offset=0)
    assert np.array_equal(a + b, g)                                  # integer-valued sums: exact


# ------------------------------------------------------------------ compiled chains, interpreter, fast sin/cos
@pytest.mark.parametrize("cfg", [1, 2, 3, 4])
def test_compiled_chain_equals_interpreter(cfs, oracle, cfg):
    """A kernel compiled for the chain's signature and the chain interpreter evaluate the same device
    functions: traces and images are bit-identical (integer-valued colour sums are order-free)."""
    w = W.config(cfg)
    n = (1 << 17) + 77 if cfg == 3 else (1 << 14) + 77      # >= 2 M splats (cfg 3: 2^17 records): edge flips stay far below the bar
    cloud = _cloud_for(w, n)
    w = w.scaled(n_points=n, iterations=min(w.render.iterations, 150), width=640, height=360)
    t = w.frames[len(w.frames) // 2]
    a = gpu_trace(cfs, w, t=t, cloud=cloud)
    b = gpu_trace(cfs, w, t=t, cloud=cloud, flags=["interpret_chain"])
    for x, y in zip(a, b):
        assert np.array_equal(x, y)
    ga, ca = gpu_render(cfs, w, t=t, cloud=cloud)
    gb, cb = gpu_render(cfs, w, t=t, cloud=cloud, flags=["interpret_chain"])
    assert np.array_equal(ga, gb) and np.array_equal(ca, cb)
    o, oc, _ = oracle.render_parallel(w.system, w.render, cloud=cloud, t=t)
    if cfg == 4:
        assert np.array_equal(ga, o) and np.array_equal(ca, oc)
    else:
        for ch in range(4):
            assert density_l1(ga[:, ch], o[:, ch]) <= L1_TOL, (cfg, ch, density_l1(ga[:, ch], o[:, ch]))


# ------------------------------------------------------------------ NEXT-4: run-time specialisation (NVRTC)
@pytest.mark.parametrize("fast", [False, True])
@pytest.mark.parametrize("cfg", [0, 1, 2, 3, 4])
def test_three_ways_to_run_a_chain_are_bit_identical(cfs, oracle, cfg, fast):
    """interpreter / ahead-of-time kernel / run-time-compiled kernel (CFS_FLAG_JIT): the same
    device functions three ways -- traces and images identical to the last bit, in the direct variant and
    through the tile bins (hybrid), with sincosf and with MUFU sin/cos."""
    w = W.config(cfg)
    n = (1 << 13) + 77
    cloud = _cloud_for(w, n)
    w = w.scaled(n_points=n, iterations=min(w.render.iterations, 150), width=640, height=360)
    t = w.frames[len(w.frames) // 2]
    base = ["fast_trig"] if fast else []
    ways = {"interpreter": base + ["interpret_chain"], "aot": base, "jit": base + ["jit"]}
    traces = {k: gpu_trace(cfs, w, t=t, cloud=cloud, flags=f) for k, f in ways.items()}
    images = {k: gpu_render(cfs, w, t=t, cloud=cloud, variant="direct", flags=f) for k, f in ways.items()}
    for k in ("aot", "jit"):
        for x, y in zip(traces[k], traces["interpreter"]):
            assert np.array_equal(x, y), k
        assert np.array_equal(images[k][0], images["interpreter"][0]) and np.array_equal(images[k][1], images["interpreter"][1]), k
    if cfg in (0, 1, 2):
        for k, f in ways.items():
            g, c = gpu_render(cfs, w, t=t, variant="binned", flags=f + ["bin_hybrid"])
            assert np.array_equal(g, images["interpreter"][0]) and np.array_equal(c, images["interpreter"][1]), k


@pytest.mark.parametrize("n", [5, 6, 7, 12, 20, 24])
def test_map_pick_forms_agree_with_the_oracle(cfs, oracle, n):
    """n equal maps: the run-time compiled kernel picks the map with one multiply (pick form 4; n = 6, 12, 24 have
    thresholds that are exact integers, n = 5, 7, 20 none), the linked kernels read the table -- both bit-identical
    to the oracle's threshold walk (DESIGN R2), picks traced and histograms rendered."""
    funcs = [W.Func("affine", float(np.float32(1.0 / n)),
                    [0.45, 0.0, 0.0, 0.45, 0.55 * math.cos(2 * math.pi * k / n), 0.55 * math.sin(2 * math.pi * k / n)]) for k in range(n)]
    w = W.Workload("pick", W.System(2, "ifs", funcs), W.Render(6007, 31 + n, 96, 8, 160, 120, (-1.1, 1.1, -1.1, 1.1), "hist_u32"))
    sysh = cfs.cfs_create(w.system)
    form = cfs.cfs_host_resolve(sysh, cfs.make_args(w.render))["pick_form"]
    sysh.close()
    assert form == 4, (n, form)
    o, oc, _ = oracle.render_parallel(w.system, w.render)
    tr_ref = gpu_trace(cfs, w, flags=["interpret_chain"])
    for flags in ([], ["jit"]):
        g, c = gpu_render(cfs, w, variant="direct", flags=flags)
        assert np.array_equal(g, o) and np.array_equal(c, oc), (n, flags)
        for x, y in zip(gpu_trace(cfs, w, flags=flags), tr_ref):
            assert np.array_equal(x, y), (n, flags)


def _random_system(rng, dim):
    """A random IFS of affine contractions with a random chain and random image bounds (sometimes generous enough for
    the host to prove "no splat is dropped", sometimes not)."""
    n = int(rng.integers(2, 8))
    probs = rng.uniform(0.5, 1.5, n) if rng.random() < 0.5 else np.ones(n)
    probs = probs / probs.sum()
    funcs = []
    for k in range(n):
        if dim == 2:
            sc, th = rng.uniform(0.2, 0.6), rng.uniform(0, 2 * math.pi)
            A = sc * np.array([[math.cos(th), -math.sin(th)], [math.sin(th), math.cos(th)]])
            if rng.random() < 0.3:
                A = np.diag(rng.uniform(0.2, 0.7, 2))
        else:
            A = np.diag(rng.uniform(0.2, 0.6, 3)) + rng.uniform(-0.1, 0.1, (3, 3))
        b = rng.uniform(-0.6, 0.6, dim)
        funcs.append(W.Func("affine", float(np.float32(probs[k])), [float(v) for v in A.ravel()] + [float(v) for v in b]))
    chain = []
    for _ in range(int(rng.integers(0, 4))):
        if dim == 2:
            kind = rng.choice(["affine", "swirl", "sinusoidal", "stretch_cos", "scatter"])
        else:
            kind = rng.choice(["affine", "twist_z", "bend", "scatter"])
        if kind == "affine":
            M = rng.uniform(-0.7, 0.7, (dim, dim)) + np.eye(dim) * rng.uniform(0.3, 0.9)
            chain.append(W.Xform("affine", [float(v) for v in M.ravel()] + [float(v) for v in rng.uniform(-0.3, 0.3, dim)]))
        elif kind in ("twist_z", "bend"):
            chain.append(W.Xform(kind, [float(rng.uniform(-3.0, 3.0))]))
        elif kind == "scatter":
            chain.append(W.Xform("scatter", [int(rng.integers(2, 40)), float(rng.uniform(0, 0.5)), float(rng.uniform(0, 0.5)),
                                             float(rng.uniform(0, 0.5)) if dim == 3 else 0.0]))
        else:
            chain.append(W.Xform(kind))
    if dim == 3:
        chain.append(W.Xform("pinhole", [float(rng.uniform(40, 85)), -float(rng.uniform(2.0, 9.0)), float(rng.choice([1e-3, 0.1, 1.0]))]))
    half = float(rng.choice([0.6, 1.2, 2.5, 6.0]))
    bounds = (-half, half, -half * 0.75, half * 0.75) if rng.random() < 0.7 else (-half, half * 0.5, -half * 0.3, half)
    out = "hist_u32" if dim == 2 else "depth_u64"
    color, pal = ("none", None) if dim == 2 else ("map_index", W.palette_for(n))
    return W.Workload("random", W.System(dim, "ifs", funcs, chain, color, pal),
                      W.Render(int(rng.integers(1500, 4000)), int(rng.integers(1, 1 << 30)), 64, 8, 200, 150, bounds, out))


def test_proved_options_are_sound_on_random_systems(cfs):
    """What the host proves about a render (bounded attractor pushed through the chain: "every depth is a normal float",
    "no splat is dropped") is compiled into the run-time specialised kernel as a DROPPED test.  On random systems the
    specialised kernel must give the interpreter's image and counters to the last bit, whether the proof succeeded or
    not -- an unsound proof shows as a splat that should have been dropped (or a clamp that should have bound)."""
    rng = np.random.default_rng(20261105)
    proved = {0: 0, 1: 0, 2: 0, 3: 0}
    for i in range(36):
        w = _random_system(rng, 2 if i % 2 == 0 else 3)
        sysh = cfs.cfs_create(w.system)
        proved[cfs.cfs_host_resolve(sysh, cfs.make_args(w.render))["proved"]] += 1
        sysh.close()
        ref, cref = gpu_render(cfs, w, variant="direct", flags=["interpret_chain"])
        g, c = gpu_render(cfs, w, variant="direct", flags=["jit"])
        assert np.array_equal(g, ref) and np.array_equal(c, cref), (i, w.system.chain, w.render.bounds)
        if w.system.dim == 2:
            g, c = gpu_render(cfs, w, variant="binned", flags=["jit", "bin_hybrid"])
            assert np.array_equal(g, ref) and np.array_equal(c, cref), (i, "bins", w.system.chain, w.render.bounds)
        else:
            g, c = gpu_render(cfs, w, variant="depth_hiz", flags=["jit"],
                              scratch_bytes=cfs.cfs_hiz_scratch_bytes(w.render.width, w.render.height))
            assert np.array_equal(g, ref) and np.array_equal(c, cref), (i, "hiz", w.system.chain, w.render.bounds)
    # both outcomes of the proof were exercised
    assert proved[2] + proved[3] >= 5 and proved[0] + proved[1] >= 5, proved


def test_jit_compiles_branch_scatter_reuse_and_the_eq1_generator(cfs, oracle):
    """The NEXT-1 / NEXT-2 systems have no ahead-of-time kernel; CFS_FLAG_JIT compiles their chain in (BRANCH
    structure, SCATTER draws, Fig. 2(C) reuse, the Eq. 1 generator) -- identical to the interpreter and, where
    the arithmetic is exact, to the oracle.  cfs_specialize reports the compile time, the second call is cached."""
    pin = W.Xform("pinhole", [60.0, -4.0, 1e-3])
    a = [W.Xform("affine", [0.5, 0, 0, 0.5, -0.4, 0.3])]
    b = [W.Xform("affine", [0.3, 0.1, -0.1, 0.3, 0.3, -0.5])]
    sw = [W.Xform("swirl"), W.Xform("affine", [0.6, 0, 0, 0.6, 0.3, -0.2])]
    stars = [W.Xform("affine", [0.03, 0, 0, 0.03, 0, 0]), W.Xform("scatter", [64, 0.95, 0.95, 0.0])]
    br = [W.Xform("branch")]
    systems = [
        ("branches_hist", W.System(2, "ifs", W.square_funcs(), a + br + b + br, "none"),
         W.Render(6005, 5, 80, 10, 200, 160, (-1, 1, -1, 0.9), "hist_u32"), True),
        ("branches_rgba", W.System(2, "ifs", W.square_funcs(), sw + br + a, "map_index", W.palette_for(4)),
         W.Render(20000, 6, 60, 10, 256, 256, (-1.2, 1.2, -1.2, 1.2), "rgba_f32"), False),
        ("sky", W.System(2, "ifs", W.square_funcs(), a + br + stars, "map_index", W.palette_for(4)),
         W.Render(8000, 77, 60, 10, 256, 256, (-1, 1, -1, 1), "rgba_f32"), True),
        ("scatter3d", W.System(3, "ifs", W.menger_funcs(), [W.Xform("affine", [0.2, 0, 0, 0, 0.2, 0, 0, 0, 0.2, 0, 0, 0]),
                                                             W.Xform("scatter", [9, 0.7, 0.7, 0.7]), pin], "map_index", W.palette_for(20)),
         W.Render(3000, 5, 50, 10, 320, 180, (-1, 1, -1, 1), "depth_u64"), True),
        ("depth_branches", W.System(3, "ifs", W.menger_funcs(), [pin] + br + [W.Xform("affine", [0.5, 0, 0, 0, 0.5, 0, 0, 0, 0.5, 0.3, 0.2, -1.0]), pin],
                                    "map_index", W.palette_for(20)),
         W.Render(3000, 9, 60, 10, 320, 180, (-1, 1, -1, 1), "depth_u64"), True),
        ("reuse_eq2", W.System(2, "ifs", W.square_funcs(), [W.Xform("stretch_cos"), W.Xform("affine", [0.4, 0, 0, 0.4, 0, 0.3])],
                               "map_index", W.palette_for(4), reuse=True),
         W.Render(4000, 12, 60, 10, 256, 256, (-1.5, 1.5, -1.5, 1.5), "rgba_f32"), False),
        ("eq1_B", W.System(2, "ifs", W.circle_funcs(False), [W.Xform("stretch_cos"), W.Xform("affine", [0.4, 0, 0, 0.4, 0, 0.3])],
                           "map_index", W.palette_for(2)),
         W.Render(5000, 21, 60, 10, 256, 256, (-1.5, 1.5, -1.5, 1.5), "rgba_f32"), False),
        ("eq1_C", W.System(2, "ifs", W.circle_funcs(True), [W.Xform("stretch_cos"), W.Xform("affine", [0.4, 0, 0, 0.4, 0, 0.3])],
                           "map_index", W.palette_for(2), reuse=True),
         W.Render(5000, 22, 60, 10, 256, 256, (-1.5, 1.5, -1.5, 1.5), "rgba_f32"), False),
    ]
    for name, system, render, exact_vs_oracle in systems:
        w = W.Workload(name, system, render)
        gi, ci = gpu_render(cfs, w, variant="direct", flags=["interpret_chain"])
        gj, cj = gpu_render(cfs, w, variant="direct", flags=["jit"])
        assert np.array_equal(gi, gj) and np.array_equal(ci, cj), name
        if render.out_mode != "depth_u64":
            gb, cb = gpu_render(cfs, w, variant="binned", flags=["jit", "bin_hybrid"])
            assert np.array_equal(gb, gi) and np.array_equal(cb, ci), name
        if exact_vs_oracle:
            o, oc = oracle.render(system, render)
            assert np.array_equal(gj.astype(o.dtype), o) and np.array_equal(cj, oc), name
    # compile time is reported once, then the kernel comes from the process cache
    w = W.Workload("timing", W.System(2, "ifs", W.square_funcs(), sw + br + a + br + stars, "map_index", W.palette_for(4)),
                   W.Render(1000, 3, 40, 10, 128, 128, (-1.2, 1.2, -1.2, 1.2), "rgba_f32"))
    sysh = cfs.cfs_create(w.system)
    n0, _ = cfs.cfs_jit_stats()
    ms_first = cfs.cfs_specialize(sysh, cfs.make_args(w.render))
    ms_again = cfs.cfs_specialize(sysh, cfs.make_args(w.render))
    n1, total = cfs.cfs_jit_stats()
    sysh.close()
    assert ms_first > 0.0 and ms_again == 0.0 and n1 >= n0 + 2 and total >= ms_first


@pytest.mark.parametrize("interp", [False, True])
@pytest.mark.parametrize("cfg", [1, 2, 3])
def test_fast_trig_within_tolerance(cfs, oracle, cfg, interp):
    """CFS_FLAG_FAST_TRIG (MUFU sin/cos): pick sequences unchanged, coordinates within 1e-4 of the
    oracle (BASELINE north_star), density L1 within 1e-3."""
    flags = ["fast_trig"] + (["interpret_chain"] if interp else [])
    w = W.config(cfg)
    n = (1 << 14) + 5 if cfg != 3 else (1 << 18) + 11
    cloud = _cloud_for(w, n)
    w = w.scaled(n_points=n)
    t = w.frames[len(w.frames) // 2]
    nt = 1024 + 37
    gp, gg, gq, ga = gpu_trace(cfs, w, t=t, cloud=cloud, n_points=nt, flags=flags)
    op, og, oq, oa = oracle.trace(w.system, w.scaled(n_points=nt).render, cloud=cloud, t=t)
    assert np.array_equal(gp, op) and np.array_equal(gg, og) and np.array_equal(ga, oa)
    live = oa.astype(bool)
    assert np.abs(gq[live].astype(np.float64) - oq[live]).max() <= COORD_TOL
    g, gc = gpu_render(cfs, w, t=t, cloud=cloud, flags=flags)
    o, oc, _ = oracle.render_parallel(w.system, w.render, cloud=cloud, t=t)
    assert int(gc[0]) + int(gc[1]) == int(oc[0]) + int(oc[1]) and abs(int(gc[0]) - int(oc[0])) <= 4
    for ch in range(4):
        assert density_l1(g[:, ch], o[:, ch]) <= L1_TOL


# ------------------------------------------------------------------ tile-binned variant
@pytest.mark.parametrize("hybrid", [False, True])
@pytest.mark.parametrize("n", [1, 1000, 1024, 5000 + 13])
def test_binned_histogram_bit_exact(cfs, oracle, n, hybrid):
    """CFS_VARIANT_BINNED on the cfg 0 image: records through the block pool, tiles accumulated in
    shared memory; identical per pixel to the oracle, counters included; ragged CTAs.  With
    CFS_FLAG_BIN_HYBRID every other splat goes straight to L2 instead: same histogram."""
    w = W.config(0).scaled(n_points=n, iterations=300)
    g, gc = gpu_render(cfs, w, variant="binned", flags=["bin_hybrid"] if hybrid else 0)
    o, oc, _ = oracle.render_parallel(w.system, w.render)
    assert np.array_equal(g, o) and np.array_equal(gc, oc)


def test_binned_chunks_and_small_scratch(cfs, oracle):
    """A scratch buffer far below the one-chunk size forces several (pass 1, pass 2) chunks; one that
    cannot hold a partial block per (CTA, tile) is refused with UNSUPPORTED."""
    w = W.config(0).scaled(n_points=400000, iterations=120)
    sysh = cfs.cfs_create(w.system)
    need = cfs.cfs_binned_scratch_bytes(sysh, cfs.make_args(w.render))
    sysh.close()
    assert need > (120 << 20)
    o, oc, _ = oracle.render_parallel(w.system, w.render)
    g, gc = gpu_render(cfs, w, variant="binned", scratch_bytes=need * 2 // 3)       # two chunks
    assert np.array_equal(g, o) and np.array_equal(gc, oc)
    g, gc = gpu_render(cfs, w, variant="binned", flags=["bin_hybrid"], scratch_bytes=need * 2 // 3)    # hybrid, in chunks
    assert np.array_equal(g, o) and np.array_equal(gc, oc)
    g, gc = gpu_render(cfs, w, variant="auto", scratch_bytes=need * 3 // 5)         # AUTO: hybrid, in chunks
    assert np.array_equal(g, o) and np.array_equal(gc, oc)
    with pytest.raises(cfs.CfsError) as ei:
        gpu_render(cfs, w, variant="binned", scratch_bytes=1 << 20)
    assert ei.value.status == cfs.CFS_ERR_UNSUPPORTED
    g, gc = gpu_render(cfs, w, variant="auto", scratch_bytes=1 << 20)      # AUTO falls back to direct
    assert np.array_equal(g, o)


@pytest.mark.parametrize("hybrid", [False, True])
@pytest.mark.parametrize("cfg", [1, 2])
def test_binned_rgba_equals_direct(cfs, oracle, cfg, hybrid):
    """Binned RGBA (counters per pixel and map, sum_k n_k * palette[k]) against the direct variant
    on the same device functions: integer-valued colour sums below 2^24 are exact, so the images
    are identical; and against the oracle within the density bar."""
    w = W.config(cfg).scaled(n_points=(1 << 14) + 5)
    t = w.frames[len(w.frames) // 2]
    gb, cb = gpu_render(cfs, w, t=t, variant="binned", flags=["bin_hybrid"] if hybrid else 0)
    gd, cd = gpu_render(cfs, w, t=t, variant="direct")
    assert np.array_equal(gb, gd) and np.array_equal(cb, cd)
    o, oc, _ = oracle.render_parallel(w.system, w.render, t=t)
    _check_rgba(gb, o, cb, oc)


@pytest.mark.parametrize("size,mode,jit", [((1000, 777), "rgba_f32", True), ((333, 555), "hist_u32", True), ((1921, 1079), "rgba_f32", False),
                                           ((64, 64), "hist_u32", False), ((4099, 61), "rgba_f32", True)])
def test_interleaved_tiles_on_awkward_image_sizes(cfs, oracle, size, mode, jit):
    """The tiles of the binned variant are interleaved (pixel p in tile p & mask as its pixel p >> shift): images
    whose pixel count is no multiple of the tile count, whose rows are no multiple of it, tiny and very wide ones --
    binned (pure, hybrid, run-time compiled or linked) must equal the direct variant bit for bit (integer colour
    sums), and the oracle on the histogram."""
    wd, ht = size
    w = W.config(1 if mode == "rgba_f32" else 0).scaled(n_points=(1 << 15) + 77, iterations=120, width=wd, height=ht)
    flags = ["jit"] if jit else []
    gd, cd = gpu_render(cfs, w, variant="direct")
    for extra in ([], ["bin_hybrid"]):
        gb, cb = gpu_render(cfs, w, variant="binned", flags=flags + extra)
        assert np.array_equal(gb, gd) and np.array_equal(cb, cd), (size, mode, extra)
    if mode == "hist_u32":           # the affine-only system of configs[0]: bit-exact against the oracle
        o, oc, _ = oracle.render_parallel(w.system, w.render)
        assert np.array_equal(gd, o) and np.array_equal(cd, oc)


@pytest.mark.parametrize("cfg", [1, 2])
def test_hist_output_of_a_coloured_system_through_the_bins(cfs, oracle, cfg):
    """HIST_U32 output from a system created with COLOR_MAP_INDEX (colour ignored, include/cfs.h): the tile
    bins must lay out ONE counter per pixel (round-1 ADVICE: they keyed on the colour rule and wrote 16-byte
    reductions into a 4-byte histogram).  Every variant that can serve a histogram gives the same image as
    the direct one, exactly; conservation exact; oracle within the density bar."""
    w = W.config(cfg).scaled(n_points=(1 << 15) + 9, out_mode="hist_u32")
    t = w.frames[len(w.frames) // 2]
    gd, cd = gpu_render(cfs, w, t=t, variant="direct")
    S = w.render.n_points * (w.render.iterations - w.render.burn_in)
    assert int(cd[0]) == S and int(gd.sum(dtype=np.uint64)) == S
    sysh = cfs.cfs_create(w.system)
    need = cfs.cfs_binned_scratch_bytes(sysh, cfs.make_args(w.render))
    sysh.close()
    assert need > 0
    for variant, flags in (("binned", 0), ("binned", ["bin_hybrid"]), ("auto", 0), ("binned", ["interpret_chain"]),
                           ("binned", ["bin_hybrid", "interpret_chain"]), ("warp_agg", 0)):
        g, c = gpu_render(cfs, w, t=t, variant=variant, flags=flags, scratch_bytes=need)
        assert np.array_equal(g, gd) and np.array_equal(c, cd), (variant, flags)
    o, oc, _ = oracle.render_parallel(w.system, w.render, t=t)
    assert np.array_equal(cd, oc) and density_l1(gd, o) <= L1_TOL


@pytest.mark.parametrize("jit", [False, True])
@pytest.mark.parametrize("cfg,n", [(1, 1 << 18), (2, 1 << 19)])
def test_bench_launch_configuration_against_the_oracle(cfs, oracle, cfg, n, jit):
    """The EXACT configuration bench.py times -- variant AUTO with scratch (-> hybrid: one splat in four straight to
    L2, the rest through the tile bins), CFS_FLAG_FAST_TRIG (MUFU sin/cos) and the kernels compiled at run time for the
    system (CFS_FLAG_JIT; also the linked ones) -- on a point sub-range large enough for AUTO's hybrid threshold, at
    full image size, DIRECTLY against the oracle: counters equal, normalised-density L1 <= 1e-3 on the count and on
    every colour channel."""
    import torch
    w = W.config(cfg).scaled(n_points=n)
    t = w.frames[len(w.frames) // 2]
    flags = ["fast_trig"] + (["jit"] if jit else [])
    sysh = cfs.cfs_create(w.system)
    need = cfs.cfs_binned_scratch_bytes(sysh, cfs.make_args(w.render))
    assert need > 0
    scratch = torch.empty(need, dtype=torch.uint8, device="cuda")
    img = cfs.new_image(w.render)
    ctr = torch.zeros(2, dtype=torch.int64, device="cuda")
    if jit:
        cfs.cfs_specialize(sysh, cfs.make_args(w.render, t=t, variant="auto", flags=flags))
    cfs.cfs_launch_count(reset=True)
    cfs.cfs_render(sysh, cfs.make_args(w.render, d_image=img, d_counters=ctr, t=t, variant="auto", flags=flags, d_scratch=scratch))
    torch.cuda.synchronize()
    assert cfs.cfs_launch_count() == 2, "AUTO did not take the hybrid stage (pass 1 + pass 2 in one chunk)"
    g, gc = img.cpu().numpy(), ctr.cpu().numpy().astype(np.uint64)
    sysh.close()
    o, oc, _ = oracle.render_parallel(w.system, w.render, t=t)
    assert np.array_equal(gc, oc) and int(gc[1]) == 0
    assert g[:, 3].astype(np.float64).sum() == o[:, 3].sum() == float(oc[0])
    for ch in range(4):
        assert density_l1(g[:, ch], o[:, ch]) <= L1_TOL, (cfg, ch, density_l1(g[:, ch], o[:, ch]))


def test_bench_launch_configuration_cfg3_cfg4_against_the_oracle(cfs, oracle):
    """configs[3] and configs[4] as bench.py launches them (AUTO with scratch, MUFU sin/cos, run-time compiled kernels):
    the streamed cloud on 2^20 records (L1 <= 1e-3 per channel), and the Menger depth render on 1.18 M points -- enough
    splats for AUTO to take the Hi-Z variant (plain slice, map build, Hi-Z phase) -- bit for bit against the oracle,
    full 4K images."""
    import torch
    flags = ["fast_trig", "jit"]
    w = W.config(3)
    n = 1 << 20
    cloud = W.gaussian_mixture_cloud(n, w.cloud_seed)
    w = w.scaled(n_points=n)
    g, gc = gpu_render(cfs, w, cloud=cloud, variant="auto", flags=flags)
    o, oc, _ = oracle.render_parallel(w.system, w.render, cloud=cloud)
    assert int(gc[0]) + int(gc[1]) == n and abs(int(gc[0]) - int(oc[0])) <= 4
    for ch in range(4):
        assert density_l1(g[:, ch], o[:, ch]) <= L1_TOL, (3, ch, density_l1(g[:, ch], o[:, ch]))
    w = W.config(4).scaled(n_points=(1 << 20) + (1 << 17) + 8)   # >= 2^30 splats: AUTO's threshold for the Hi-Z variant
    sysh = cfs.cfs_create(w.system)
    img = cfs.new_image(w.render)
    ctr = torch.zeros(2, dtype=torch.int64, device="cuda")
    scratch = torch.empty(cfs.cfs_hiz_scratch_bytes(w.render.width, w.render.height), dtype=torch.uint8, device="cuda")
    cfs.cfs_specialize(sysh, cfs.make_args(w.render, variant="auto", flags=flags))
    cfs.cfs_launch_count(reset=True)
    cfs.cfs_render(sysh, cfs.make_args(w.render, d_image=img, d_counters=ctr, variant="auto", flags=flags, d_scratch=scratch))
    torch.cuda.synchronize()
    assert cfs.cfs_launch_count() in (3, 5), "AUTO did not take the Hi-Z depth variant"      # plain slice, map build, Hi-Z phase (+ rebuild, phase)
    g, gc = cfs.image_to_numpy(img, "depth_u64"), ctr.cpu().numpy().astype(np.uint64)
    sysh.close()
    o, oc, _ = oracle.render_parallel(w.system, w.render)
    assert np.array_equal(g, o) and np.array_equal(gc, oc)


def test_binned_hot_tile_overflow_and_limits(cfs, oracle):
    """All splats in ONE pixel (one-hot probabilities: the point sits on the map's fixed point): the
    staging row of that tile overflows constantly and the surplus takes the direct path; nothing
    is lost.  16 maps use 4 colour bits; 17 maps and DEPTH output are refused."""
    funcs = W.square_funcs(probs=[0.0, 0.0, 1.0, 0.0])
    sys1 = W.System(2, "ifs", funcs, [], "map_index", W.palette_for(4))
    # 400 x 160 splats x 255 < 2^24: the float sum is exact whatever the order of the additions
    w = W.Workload("hot", sys1, W.Render(400, 5, 200, 40, 512, 512, (-1, 1, -1, 1), "rgba_f32"))
    o, oc = oracle.render(sys1, w.render)
    for flags in (0, ["bin_hybrid"]):
        g, gc = gpu_render(cfs, w, variant="binned", flags=flags)
        assert np.array_equal(g.astype(np.float64), o) and np.array_equal(gc, oc)
        assert np.count_nonzero(g[:, 3]) == 1 and g[:, 3].sum() == 400 * 160

    f16 = [W.Func("affine", float(np.float32(1 + (k % 3))), [0.5, 0, 0, 0.5, 0.5 * math.cos(k), 0.5 * math.sin(k)])
           for k in range(17)]
    s16 = W.System(2, "ifs", f16[:16], [], "map_index", W.palette_for(16))
    w16 = W.Workload("n16", s16, W.Render(4000, 6, 90, 10, 300, 200, (-1, 1, -1, 1), "rgba_f32"))
    g, gc = gpu_render(cfs, w16, variant="binned")
    o, oc = oracle.render(s16, w16.render)
    assert np.array_equal(g.astype(np.float64), o) and np.array_equal(gc, oc)
    s17 = W.System(2, "ifs", f16, [], "map_index", W.palette_for(17))
    w17 = W.Workload("n17", s17, w16.render)
    for bad in (w17, W.config(4).scaled(n_points=100, iterations=30)):
        with pytest.raises(cfs.CfsError) as ei:
            gpu_render(cfs, bad, variant="binned", scratch_bytes=64 << 20)
        assert ei.value.status == cfs.CFS_ERR_UNSUPPORTED


def test_depth_hiz_equals_direct_and_oracle(cfs, oracle):
    """CFS_VARIANT_DEPTH_HIZ: occluded splats stop at a shared-memory Hi-Z map built from a snapshot of
    the depth image.  The map is conservative (the image only decreases), so the image is identical per
    pixel to the direct variant and to the oracle; sized so that all three phases run (plain slice, first
    map, rebuilt map).  Without enough scratch the variant is refused."""
    w = W.config(4).scaled(n_points=300000 + 7, iterations=100, width=256, height=144)
    need = cfs.cfs_hiz_scratch_bytes(256, 144)
    assert 0 < need < (1 << 20)
    gh, ch = gpu_render(cfs, w, variant="depth_hiz", scratch_bytes=need)
    gd, cd = gpu_render(cfs, w, variant="direct")
    assert np.array_equal(gh, gd) and np.array_equal(ch, cd)
    o, oc, _ = oracle.render_parallel(w.system, w.render)
    assert np.array_equal(gh, o) and np.array_equal(ch, oc)
    with pytest.raises(cfs.CfsError) as ei:
        gpu_render(cfs, w, variant="depth_hiz", scratch_bytes=need // 2)
    assert ei.value.status == cfs.CFS_ERR_UNSUPPORTED
    with pytest.raises(cfs.CfsError) as ei:                          # not a depth render
        gpu_render(cfs, W.config(1).scaled(n_points=100), variant="depth_hiz", scratch_bytes=need)
    assert ei.value.status == cfs.CFS_ERR_UNSUPPORTED


# ------------------------------------------------------------------ general tables and edge cases
def test_general_pick_and_general_affine(cfs, oracle):
    """Non-uniform probabilities incl. zero-probability maps (table + compare pick), non-diagonal
    affine maps in 2-D and 3-D (general coefficient rows)."""
    rng = np.random.default_rng(3)
    funcs2 = []
    probs = [0.05, 0.0, 0.4, 0.25, 0.3, 0.0, 1e-4]
    for pr in probs:
        th = rng.uniform(0, 2 * math.pi)
        s = rng.uniform(0.2, 0.6)
        funcs2.append(W.Func("affine", float(np.float32(pr)),
                             [s * math.cos(th), -s * math.sin(th), s * math.sin(th), s * math.cos(th),
                              rng.uniform(-0.4, 0.4), rng.uniform(-0.4, 0.4)]))
    sys2 = W.System(2, "ifs", funcs2, [], "none")
    w2 = W.Workload("gen2", sys2, W.Render(2000, 9, 64, 4, 300, 200, (-1, 1, -1, 1), "hist_u32"))
    gp, gg, _, _ = gpu_trace(cfs, w2)
    op, og, _, _ = oracle.trace(sys2, w2.render)
    assert np.array_equal(gp, op) and np.array_equal(gg, og)
    assert set(np.unique(gp)) <= {0, 2, 3, 4, 6}
    g, gc = gpu_render(cfs, w2, variant="direct")
    o, oc = oracle.render(sys2, w2.render)
    assert np.array_equal(g, o) and np.array_equal(gc, oc)

    funcs3 = []
    for k in range(37):
        A = rng.uniform(-0.35, 0.35, size=(3, 3))
        b = rng.uniform(-0.5, 0.5, size=3)
        funcs3.append(W.Func("affine", float(np.float32(rng.uniform(0.0, 1.0))), list(A.ravel()) + list(b)))
    pal = W.palette_for(37)
    sys3 = W.System(3, "ifs", funcs3, [W.PINHOLE], "map_index", pal)
    w3 = W.Workload("gen3", sys3, W.Render(3000, 10, 50, 5, 160, 90, (-1, 1, -1, 1), "depth_u64"))
    gp, gg, gq, ga = gpu_trace(cfs, w3)
    op, og, oq, oa = oracle.trace(sys3, w3.render)
    assert np.array_equal(gp, op) and np.array_equal(gg, og) and np.array_equal(gq, oq) and np.array_equal(ga, oa)
    g, gc = gpu_render(cfs, w3)
    o, oc = oracle.render(sys3, w3.render)
    assert np.array_equal(g, o) and np.array_equal(gc, oc)


def test_n64_funcs_and_single_func(cfs, oracle):
    funcs = [W.Func("affine", float(np.float32(1 + (k % 5))), [0.5, 0, 0, 0.5, 0.5 * math.cos(k), 0.5 * math.sin(k)])
             for k in range(64)]
    sysm = W.System(2, "ifs", funcs, [], "map_index", W.palette_for(64))
    w = W.Workload("n64", sysm, W.Render(1500, 4, 80, 8, 128, 128, (-1, 1, -1, 1), "rgba_f32"))
    gp, _, _, _ = gpu_trace(cfs, w)
    op, _, _, _ = oracle.trace(sysm, w.render)
    assert np.array_equal(gp, op) and gp.max() == 63
    g, gc = gpu_render(cfs, w)
    o, oc = oracle.render(sysm, w.render)
    assert np.array_equal(g.astype(np.float64), o) and np.array_equal(gc, oc)     # integer sums: exact
    one = W.System(2, "ifs", funcs[:1], [], "none")
    w1 = W.Workload("n1", one, W.Render(100, 4, 30, 0, 64, 64, (-1, 1, -1, 1), "hist_u32"))
    g, _ = gpu_render(cfs, w1, variant="direct")
    o, _ = oracle.render(one, w1.render)
    assert np.array_equal(g, o)


def test_reuse_composition_and_eq2(cfs, oracle):
    """Fig. 2(C) reuse flag and the paper's Eq. 2 transform."""
    chain = [W.Xform("stretch_cos"), W.Xform("affine", [0.4, 0, 0, 0.4, 0, 0.3])]
    for reuse in (False, True):
        sysr = W.System(2, "ifs", W.square_funcs(), chain, "map_index", W.palette_for(4), reuse=reuse)
        w = W.Workload("reuse", sysr, W.Render(40000, 12, 60, 10, 256, 256, (-1.5, 1.5, -1.5, 1.5), "rgba_f32"))
        gp, gg, gq, ga = gpu_trace(cfs, w, n_points=2000)
        op, og, oq, oa = oracle.trace(sysr, w.render, n_points=2000)
        assert np.array_equal(gp, op) and np.array_equal(ga, oa)
        assert np.abs(gg.astype(np.float64) - og).max() <= COORD_TOL
        assert np.abs(gq.astype(np.float64) - oq).max() <= COORD_TOL
        g, gc = gpu_render(cfs, w)
        o, oc, _ = oracle.render_parallel(sysr, w.render)
        assert np.array_equal(gc, oc)
        for ch in range(4):
            assert density_l1(g[:, ch], o[:, ch]) <= L1_TOL, (reuse, ch, density_l1(g[:, ch], o[:, ch]))


@pytest.mark.parametrize("r2_reading", [False, True])
@pytest.mark.parametrize("composition", ["A", "B", "C"])
def test_eq1_circle_generator_fig2(cfs, oracle, r2_reading, composition):
    """NEXT-1, the paper's own worked example (Fig. 2): the non-affine circle IFS of Eq. 1
    alone (A), with Eq. 2 applied to a copy (B), and with the transformed point reused (C).  The maps are
    non-affine and only contractive on average, so float32 and the double-evaluating oracle agree within
    1e-4 on all but a sliver of points (those that passed within rounding of the angle cut or of r = 0);
    pick sequences are bit-exact, counters conserve, densities agree."""
    chain = [] if composition == "A" else [W.Xform("stretch_cos"), W.Xform("affine", [0.4, 0, 0, 0.4, 0, 0.3])]
    sysc = W.System(2, "ifs", W.circle_funcs(r2_reading), chain, "map_index", W.palette_for(2),
                    reuse=(composition == "C"))
    w = W.Workload("eq1", sysc, W.Render(20000, 21, 60, 10, 256, 256, (-1.5, 1.5, -1.5, 1.5), "rgba_f32"))
    gp, gg, gq, ga = gpu_trace(cfs, w)
    op, og, oq, oa = oracle.trace(sysc, w.render)
    assert np.array_equal(gp, op) and np.array_equal(ga, oa)
    far_g = np.abs(gg.astype(np.float64) - og).max(axis=1) > COORD_TOL
    far_q = np.abs(gq.astype(np.float64) - oq).max(axis=1) > COORD_TOL
    assert far_g.mean() <= 2e-3 and far_q.mean() <= 2e-3, (far_g.mean(), far_q.mean())
    if composition == "A":       # f_id decides the half of the disc, and the point stays inside it
        last = gp[:, -1]
        assert np.all((gg[:, 1] >= 0) == (last == 0)) and np.all(np.hypot(gg[:, 0], gg[:, 1]) < 1.0 + 1e-6)
    # density bar (iv) at 100 M splats on a 64 x 64 image: the trajectories that float32 and double take apart
    # (non-contractive maps: ~1 % of the splats, measured) are independent samples of the same invariant density,
    # and their sampling noise, ~ sqrt(fraction x pixels / splats), is what has to stay below the bar
    wd = W.Workload("eq1d", sysc, W.Render(2000000, 21, 60, 10, 64, 64, (-1.5, 1.5, -1.5, 1.5), "rgba_f32"))
    o, oc, _ = oracle.render_parallel(sysc, wd.render)
    for variant in ("direct", "binned"):
        g, gc = gpu_render(cfs, wd, variant=variant, flags=["bin_hybrid"] if variant == "binned" else 0)
        assert int(gc[0]) + int(gc[1]) == 2000000 * 50 and abs(int(gc[0]) - int(oc[0])) <= 2000
        for ch in range(4):
            if o[:, ch].sum() > 0:
                assert density_l1(g[:, ch], o[:, ch]) <= L1_TOL, (variant, ch, density_l1(g[:, ch], o[:, ch]))


def test_branches_one_to_many(cfs, oracle):
    """NEXT-2: a chain with BRANCH markers splats every generated point once per branch.
    HIST: identical per pixel to the oracle and to the sum of the single-chain GPU renders, in every
    variant; RGBA within the density bar; DEPTH = min of the single-chain renders, bit-exact."""
    a = [W.Xform("affine", [0.5, 0, 0, 0.5, -0.4, 0.3])]
    b = [W.Xform("affine", [0.3, 0.1, -0.1, 0.3, 0.3, -0.5])]
    c = []
    sw = [W.Xform("swirl"), W.Xform("affine", [0.6, 0, 0, 0.6, 0.3, -0.2])]
    def join(brs):
        out = []
        for i, br in enumerate(brs):
            out += ([W.Xform("branch")] if i else []) + br
        return out
    r = W.Render(6000 + 5, 5, 80, 10, 200, 160, (-1, 1, -1, 0.9), "hist_u32")
    multi = W.Workload("m", W.System(2, "ifs", W.square_funcs(), join([a, b, c]), "none"), r)
    o, oc = oracle.render(multi.system, r)
    assert int(oc[0]) + int(oc[1]) == 3 * 6005 * 70 and int(oc[1]) > 0
    total = None
    for br in (a, b, c):
        g1, _ = gpu_render(cfs, W.Workload("s", W.System(2, "ifs", W.square_funcs(), br, "none"), r), variant="direct")
        total = g1 if total is None else total + g1
    for variant, flags in (("direct", 0), ("auto", 0), ("shared_hist", 0), ("warp_agg", 0), ("binned", 0), ("binned", ["bin_hybrid"])):
        if variant == "shared_hist":
            continue                                    # 200 x 160 u32 does fit: exercised just below
        g, gc = gpu_render(cfs, multi, variant=variant, flags=flags)
        assert np.array_equal(g, o) and np.array_equal(gc, oc) and np.array_equal(g, total), variant
    g, gc = gpu_render(cfs, multi, variant="shared_hist")
    assert np.array_equal(g, o) and np.array_equal(gc, oc)
    # RGBA + a non-affine branch
    r2 = W.Render(20000, 6, 60, 10, 256, 256, (-1.2, 1.2, -1.2, 1.2), "rgba_f32")
    m2 = W.Workload("m2", W.System(2, "ifs", W.square_funcs(), join([sw, a]), "map_index", W.palette_for(4)), r2)
    o2, oc2 = oracle.render(m2.system, r2)
    for variant in ("direct", "binned"):
        g2, gc2 = gpu_render(cfs, m2, variant=variant)
        assert int(gc2[0]) + int(gc2[1]) == 2 * 20000 * 50 and abs(int(gc2[0]) - int(oc2[0])) <= 4
        for ch in range(4):
            assert density_l1(g2[:, ch], o2[:, ch]) <= L1_TOL
    # DEPTH: two objects from one Menger primitive
    pin = W.Xform("pinhole", [60.0, -4.0, 1e-3])
    small = [W.Xform("affine", [0.5, 0, 0, 0, 0.5, 0, 0, 0, 0.5, 0.3, 0.2, -1.0]), pin]
    r3 = W.Render(3000, 9, 60, 10, 320, 180, (-1, 1, -1, 1), "depth_u64")
    m3 = W.Workload("m3", W.System(3, "ifs", W.menger_funcs(), join([[pin], small]), "map_index", W.palette_for(20)), r3)
    o3, oc3 = oracle.render(m3.system, r3)
    g3, gc3 = gpu_render(cfs, m3)
    assert np.array_equal(g3, o3) and np.array_equal(gc3, oc3)
    # refused: reuse with branches, a depth branch without PINHOLE, cfs_trace
    with pytest.raises(cfs.CfsError) as ei:
        cfs.cfs_create(W.System(2, "ifs", W.square_funcs(), join([a, b]), "none", None, reuse=True))
    assert ei.value.status == cfs.CFS_ERR_INVALID_ARG
    with pytest.raises(cfs.CfsError) as ei:
        gpu_render(cfs, W.Workload("bad", W.System(3, "ifs", W.menger_funcs(), join([[pin], []]), "map_index", W.palette_for(20)), r3))
    assert ei.value.status == cfs.CFS_ERR_INVALID_ARG
    with pytest.raises(cfs.CfsError) as ei:
        gpu_trace(cfs, multi)
    assert ei.value.status == cfs.CFS_ERR_UNSUPPORTED


def test_scatter_duplicates(cfs, oracle):
    """NEXT-2 (DESIGN R14): PRNG-placed duplicates.  SCATTER is exact float32 arithmetic, so traced
    coordinates and the histogram are identical to the oracle's, in 2-D and 3-D, alone and as one branch of a
    one-to-many chain (an object plus a field of 64 small copies of it: the paper's "stars")."""
    sc = W.Xform("scatter", [7, 0.6, 0.4, 0.0])
    s2 = W.System(2, "ifs", W.square_funcs(), [W.Xform("affine", [0.25, 0, 0, 0.25, 0, 0]), sc], "none")
    w = W.Workload("sc", s2, W.Render(5000 + 3, 0x1234567890, 61, 9, 192, 128, (-1, 1, -1, 1), "hist_u32"))
    gp, gg, gq, ga = gpu_trace(cfs, w)
    op, og, oq, oa = oracle.trace(s2, w.render)
    assert np.array_equal(gp, op) and np.array_equal(gg, og) and np.array_equal(gq, oq) and np.array_equal(ga, oa)
    o, oc = oracle.render(s2, w.render)
    for variant in ("direct", "binned"):
        g, gc = gpu_render(cfs, w, variant=variant)
        assert np.array_equal(g, o) and np.array_equal(gc, oc)
    stars = [W.Xform("affine", [0.03, 0, 0, 0.03, 0, 0]), W.Xform("scatter", [64, 0.95, 0.95, 0.0])]
    planet = [W.Xform("affine", [0.4, 0, 0, 0.4, 0.1, -0.2])]
    s3 = W.System(2, "ifs", W.square_funcs(), planet + [W.Xform("branch")] + stars, "map_index", W.palette_for(4))
    w3 = W.Workload("sky", s3, W.Render(8000, 77, 60, 10, 256, 256, (-1, 1, -1, 1), "rgba_f32"))
    o3, oc3 = oracle.render(s3, w3.render)
    g3, gc3 = gpu_render(cfs, w3)
    assert np.array_equal(g3.astype(np.float64), o3) and np.array_equal(gc3, oc3)      # integer sums < 2^24: exact
    assert int(oc3[0]) + int(oc3[1]) == 2 * 8000 * 50
    # 3-D: the z offset is applied too, before the projection
    pin = W.Xform("pinhole", [60.0, -4.0, 1e-3])
    s4 = W.System(3, "ifs", W.menger_funcs(), [W.Xform("affine", [0.2, 0, 0, 0, 0.2, 0, 0, 0, 0.2, 0, 0, 0]),
                                                W.Xform("scatter", [9, 0.7, 0.7, 0.7]), pin], "map_index", W.palette_for(20))
    w4 = W.Workload("sc3", s4, W.Render(3000, 5, 50, 10, 320, 180, (-1, 1, -1, 1), "depth_u64"))
    o4, oc4 = oracle.render(s4, w4.render)
    g4, gc4 = gpu_render(cfs, w4)
    assert np.array_equal(g4, o4) and np.array_equal(gc4, oc4)
    with pytest.raises(cfs.CfsError) as ei:
        gpu_render(cfs, W.Workload("bad", W.System(2, "ifs", W.square_funcs(), [W.Xform("scatter", [0, 1, 1, 0])], "none"), w.render))
    assert ei.value.status == cfs.CFS_ERR_INVALID_ARG


def test_empty_and_accumulate(cfs, oracle):
    import torch
    w = W.config(0).scaled(n_points=0)
    g, gc = gpu_render(cfs, w)
    assert int(g.sum()) == 0 and int(gc.sum()) == 0
    # accumulation into a caller-owned image: two sub-ranges into one buffer
    w = W.config(0).scaled(n_points=700, iterations=50)
    img = cfs.new_image(w.render)
    gpu_render(cfs, w, n_points=300, point_offset=0, image=img, variant="direct")
    g, _ = gpu_render(cfs, w, n_points=400, point_offset=300, image=img, variant="direct")
    o, _ = oracle.render(w.system, w.render)
    assert np.array_equal(g, o)
    torch.cuda.synchronize()


def test_invalid_arguments(cfs):
    import torch
    w = W.config(0).scaled(n_points=10)
    sysh = cfs.cfs_create(w.system)
    img = cfs.new_image(w.render)

    def status(**kw):
        r = w.scaled(**kw).render
        try:
            cfs.cfs_render(sysh, cfs.make_args(r, d_image=img))
        except cfs.CfsError as e:
            return e.status
        return 0

    assert status(iterations=0) == cfs.CFS_ERR_INVALID_ARG
    assert status(burn_in=1000) == cfs.CFS_ERR_INVALID_ARG
    assert status(burn_in=-1) == cfs.CFS_ERR_INVALID_ARG
    assert status(bounds=(1.0, -1.0, -1.0, 1.0)) == cfs.CFS_ERR_INVALID_ARG
    assert status(bounds=(float("nan"), 1.0, -1.0, 1.0)) == cfs.CFS_ERR_INVALID_ARG
    assert status(width=0) == cfs.CFS_ERR_INVALID_ARG
    assert status(width=65536, height=65536) == cfs.CFS_ERR_INVALID_ARG
    assert status(out_mode="rgba_f32") == cfs.CFS_ERR_INVALID_ARG      # COLOR_NONE needs HIST
    assert status(out_mode="depth_u64") == cfs.CFS_ERR_INVALID_ARG
    with pytest.raises(cfs.CfsError) as ei:                            # shared variant on a 1 MiB image
        cfs.cfs_render(sysh, cfs.make_args(w.render, d_image=img, variant="shared_hist"))
    assert ei.value.status == cfs.CFS_ERR_UNSUPPORTED
    with pytest.raises(cfs.CfsError):
        cfs.cfs_render(sysh, cfs.make_args(w.render, d_image=None))
    assert status() == 0
    torch.cuda.synchronize()
    sysh.close()
    bad = W.System(2, "ifs", [W.Func("affine", -1.0, [0.5, 0, 0, 0.5, 0, 0])], [], "none")
    with pytest.raises(cfs.CfsError):
        cfs.cfs_create(bad)
    with pytest.raises(cfs.CfsError):
        cfs.cfs_create(W.System(2, "ifs", W.square_funcs(), [], "point"))
    with pytest.raises(cfs.CfsError):
        cfs.cfs_create(W.System(4, "ifs", W.square_funcs(), [], "none"))
    with pytest.raises(cfs.CfsError):
        cfs.cfs_create(W.System(3, "cloud", [], [], "map_index", W.palette_for(4)))


# ------------------------------------------------------------------ tone map and host entry point
@pytest.mark.parametrize("cfg", [0, 1, 2, 4])
def test_tonemap_matches_oracle(cfs, oracle, cfg):
    import torch
    w = W.config(cfg).scaled(n_points=1 << 13, iterations=200)
    sysh = cfs.cfs_create(w.system)
    img = cfs.new_image(w.render)
    cfs.cfs_render(sysh, cfs.make_args(w.render, d_image=img))
    n = w.render.width * w.render.height
    out = torch.zeros(n, dtype=torch.int32, device="cuda")
    scratch = torch.zeros(2, dtype=torch.int32, device="cuda")
    cfs.cfs_tonemap(img, w.render.out_mode, w.render.width, w.render.height, 2.2, 1 / 255.0, out, scratch)
    torch.cuda.synchronize()
    got = out.cpu().numpy().view(np.uint32)
    want = oracle.tonemap(cfs.image_to_numpy(img, w.render.out_mode), w.render.out_mode, w.render.width,
                          w.render.height, 2.2, 1 / 255.0)
    if cfg == 4:
        assert np.array_equal(got, want)
    else:
        for sh in (0, 8, 16, 24):
            d = np.abs(((got >> sh) & 0xFF).astype(np.int32) - ((want >> sh) & 0xFF).astype(np.int32))
            assert d.max() <= 1
        assert np.array_equal(got == 0, want == 0) and np.count_nonzero(got) > 1000
    sysh.close()


@pytest.mark.parametrize("cfg", [0, 1, 2])
def test_resolve_rgba8_single_pass_with_a_given_maximum(cfs, oracle, cfg):
    """NEXT-3 (the output layer is an RGBA8888 image): cfs_resolve_rgba8 with n_max GIVEN reads every
    accumulator once; with the image's true maximum it writes exactly what cfs_tonemap (maximum measured inside the
    same launch) writes, and it leaves this image's maximum in the scratch word for the next frame.  One kernel
    launch either way.  A different maximum changes the curve as the closed form says (alpha = log1p n / log1p n_max)."""
    import torch
    w = W.config(cfg).scaled(n_points=1 << 13, iterations=200)
    t = w.frames[len(w.frames) // 2]
    sysh = cfs.cfs_create(w.system)
    img = cfs.new_image(w.render)
    cfs.cfs_render(sysh, cfs.make_args(w.render, d_image=img, t=t))
    npx = w.render.width * w.render.height
    out_a = torch.zeros(npx, dtype=torch.int32, device="cuda")
    out_b = torch.zeros(npx, dtype=torch.int32, device="cuda")
    out_c = torch.zeros(npx, dtype=torch.int32, device="cuda")
    scr = torch.zeros(2, dtype=torch.int32, device="cuda")
    cfs.cfs_launch_count(reset=True)
    cfs.cfs_tonemap(img, w.render.out_mode, w.render.width, w.render.height, 2.2, 1 / 255.0, out_a, scr)
    torch.cuda.synchronize()
    assert cfs.cfs_launch_count() == 1
    host = cfs.image_to_numpy(img, w.render.out_mode)
    counts = host.astype(np.float32) if w.render.out_mode == "hist_u32" else host[:, 3]
    n_max = float(counts.max())
    assert scr.cpu().numpy().view(np.float32)[0] == np.float32(n_max)
    cfs.cfs_launch_count(reset=True)
    cfs.cfs_resolve_rgba8(img, w.render.out_mode, w.render.width, w.render.height, 2.2, 1 / 255.0, n_max, out_b, scr)
    torch.cuda.synchronize()
    assert cfs.cfs_launch_count() == 1 and torch.equal(out_a, out_b)
    assert scr.cpu().numpy().view(np.float32)[0] == np.float32(n_max)            # measured on the fly for the next frame
    want = oracle.tonemap(host, w.render.out_mode, w.render.width, w.render.height, 2.2, 1 / 255.0)
    got = out_b.cpu().numpy().view(np.uint32)
    for sh in (0, 8, 16, 24):
        assert np.abs(((got >> sh) & 0xFF).astype(np.int32) - ((want >> sh) & 0xFF).astype(np.int32)).max() <= 1
    # twice the maximum: alpha byte = floor(255 log1p(n) / log1p(2 n_max) + 0.5), +-1 code (float32 log1p against numpy's double)
    cfs.cfs_resolve_rgba8(img, w.render.out_mode, w.render.width, w.render.height, 2.2, 1 / 255.0, 2.0 * n_max, out_c, scr)
    torch.cuda.synchronize()
    alpha = (out_c.cpu().numpy().view(np.uint32) >> 24).astype(np.int32)
    hit = counts > 0
    exp = np.floor(255.0 * np.log1p(counts[hit].astype(np.float64)) / math.log1p(2.0 * n_max) + 0.5).astype(np.int32)
    assert np.abs(alpha[hit] - exp).max() <= 1 and np.all(alpha[~hit] == 0)
    sysh.close()


def test_resolve_with_the_previous_frames_maximum_and_the_rgba8_host_entry(cfs, oracle):
    """An animation (BASELINE configs[2]; PAPER L9, L206 in-betweens) resolved frame by frame: frame 0 measures its
    maximum inside the launch (n_max = 0), frame k > 0 is mapped with frame k-1's maximum taken from the scratch word
    on the device (n_max < 0: no host round trip) -- the same bytes as passing that maximum explicitly.  And the
    end-to-end host entry (cfs_render_rgba8_host: H2D, clear, render, resolve, D2H of the RGBA8888 image only) returns
    what the device calls produce."""
    import torch
    w = W.config(2).scaled(n_points=1 << 14, iterations=120)
    r = w.render
    npx = r.width * r.height
    sysh = cfs.cfs_create(w.system)
    img = cfs.new_image(r)
    out = torch.zeros(npx, dtype=torch.int32, device="cuda")
    ref = torch.zeros(npx, dtype=torch.int32, device="cuda")
    scr = torch.zeros(4, dtype=torch.int32, device="cuda")
    scr2 = torch.zeros(4, dtype=torch.int32, device="cuda")
    prev_max = None
    h_out = np.zeros(npx, dtype=np.uint32)
    h_ctr = np.zeros(2, dtype=np.uint64)
    h_max = np.zeros(1, dtype=np.float32)
    for k, t in enumerate(w.frames[:4]):
        img.zero_()
        cfs.cfs_render(sysh, cfs.make_args(r, d_image=img, t=t, variant="direct"))
        cfs.cfs_resolve_rgba8(img, r.out_mode, r.width, r.height, 2.2, 1 / 255.0, 0.0 if k == 0 else -1.0, out, scr)
        cfs.cfs_resolve_rgba8(img, r.out_mode, r.width, r.height, 2.2, 1 / 255.0, 0.0 if k == 0 else prev_max, ref, scr2)
        torch.cuda.synchronize()
        assert torch.equal(out, ref), k
        this_max = float(img[:, 3].max().item())
        assert scr.cpu().numpy().view(np.float32)[0] == np.float32(this_max) == scr2.cpu().numpy().view(np.float32)[0]
        # the host entry point, same frame, same maximum
        cfs.cfs_render_rgba8_host(sysh, cfs.make_args(r, t=t, variant="direct"), 2.2, 1 / 255.0, 0.0 if k == 0 else prev_max,
                                  h_out, None, h_ctr, h_max)
        assert np.array_equal(h_out, out.cpu().numpy().view(np.uint32)) and h_max[0] == np.float32(this_max)
        assert int(h_ctr[0]) + int(h_ctr[1]) == r.n_points * (r.iterations - r.burn_in)
        prev_max = this_max
    sysh.close()


def test_render_and_resolve_replay_from_a_cuda_graph(cfs, oracle):
    """cfs_render / cfs_resolve_rgba8 allocate nothing and never synchronise (include/cfs.h), so a frame -- clear, render
    through the tile bins (memset + pass 1 + pass 2), resolve (memset + cooperative kernel) -- is captured once into a
    CUDA graph and replayed; run-time compiled kernels are compiled before the capture (cfs_specialize).  Each replay
    reproduces the eagerly rendered frame bit for bit."""
    import torch
    w = W.config(1).scaled(n_points=(1 << 15) + 3, iterations=200)
    r = w.render
    flags = ["fast_trig", "jit"]
    sysh = cfs.cfs_create(w.system)
    need = cfs.cfs_binned_scratch_bytes(sysh, cfs.make_args(r, variant="binned", flags=flags + ["bin_hybrid"]))
    scratch = torch.empty(need, dtype=torch.uint8, device="cuda")
    img = cfs.new_image(r)
    out = torch.zeros(r.width * r.height, dtype=torch.int32, device="cuda")
    tone = torch.zeros(4, dtype=torch.int32, device="cuda")
    args = cfs.make_args(r, d_image=img, variant="binned", flags=flags + ["bin_hybrid"], d_scratch=scratch)
    cfs.cfs_specialize(sysh, args)

    def frame():
        img.zero_()
        cfs.cfs_render(sysh, args)
        cfs.cfs_resolve_rgba8(img, r.out_mode, r.width, r.height, 2.2, 1 / 255.0, 0.0, out, tone)

    frame()
    torch.cuda.synchronize()
    want_img, want_out = img.clone(), out.clone()
    side = torch.cuda.Stream()
    side.wait_stream(torch.cuda.current_stream())
    with torch.cuda.stream(side):
        frame()                                   # warm-up on the capture stream
    torch.cuda.current_stream().wait_stream(side)
    torch.cuda.synchronize()
    graph = torch.cuda.CUDAGraph()
    with torch.cuda.graph(graph):
        frame()
    for _ in range(3):
        img.fill_(7.0)
        out.zero_()
        graph.replay()
        torch.cuda.synchronize()
        assert torch.equal(img, want_img) and torch.equal(out, want_out)
    sysh.close()


@pytest.mark.parametrize("cfg", [0, 3, 4])
def test_render_host_entry_point(cfs, oracle, cfg):
    """cfs_render_host: HOST buffers in and out (the end-to-end call bench.py times)."""
    w = W.config(cfg)
    n = 5000
    cloud = _cloud_for(w, n + 100)
    if cfg == 3:
        n = 1 << 17                          # one splat per record: enough of them that an edge flip weighs 1.5e-5
        cloud = _cloud_for(w, n + 100)
    w = w.scaled(n_points=n, iterations=min(w.render.iterations, 60), burn_in=min(w.render.burn_in, 20),
                 width=320, height=180)
    npx = 320 * 180
    h_img = {"hist_u32": np.empty(npx, np.uint32), "rgba_f32": np.empty((npx, 4), np.float32),
             "depth_u64": np.empty(npx, np.uint64)}[w.render.out_mode]
    h_ctr = np.zeros(2, np.uint64)
    sysh = cfs.cfs_create(w.system)
    off = 100 if cloud is not None else 0
    cfs.cfs_render_host(sysh, cfs.make_args(w.render, point_offset=off), h_img, cloud, h_ctr)
    o, oc = oracle.render(w.system, w.render, cloud=cloud, point_offset=off)
    if cfg == 3:
        for ch in range(4):
            assert density_l1(h_img[:, ch], o[:, ch]) <= L1_TOL, (ch, density_l1(h_img[:, ch], o[:, ch]))
    else:
        assert np.array_equal(h_img, o)
    assert np.array_equal(h_ctr, oc) or cfg == 3
    sysh.close()


# ------------------------------------------------------------------ full-size properties (bench launch shape)
def test_cfg1_full_size_properties(cfs, oracle):
    """BASELINE configs[1] as bench.py launches it: conservation (exact, every pixel count < 2^24),
    colour sums = 255 x picks of each map, and sub-ranges compose; oracle parity on the first 2^15
    points rendered into the full-size image."""
    w = W.config(1)
    g, gc = gpu_render(cfs, w)
    P, S = w.render.n_points, w.render.n_points * 980
    assert int(gc[0]) == S and int(gc[1]) == 0
    assert g[:, 3].max() < 2 ** 24 and g[:, 3].astype(np.float64).sum() == S
    col = g[:, :3].astype(np.float64).sum(axis=0) / 255.0            # map 0: R, 1: G, 2: B, 3: R+G
    assert g[:, :3].max() < 2 ** 24 and np.all(col == np.round(col))
    assert abs(col[2] / S - 0.25) < 1e-3 and abs(col[1] / S - 0.5) < 1e-3 and abs(col[0] / S - 0.5) < 1e-3
    # the same render through the tile bins, in one chunk and in several; integer-valued sums below 2^24 are exact, so all three images are identical.
    # A scratch too small for the bins makes AUTO fall back to the direct path.
    sysh = cfs.cfs_create(w.system)
    need = cfs.cfs_binned_scratch_bytes(sysh, cfs.make_args(w.render))
    sysh.close()
    assert need > (3 << 29)                       # 2 bytes per binned splat (three in four under AUTO) + head-room + block lists
    # AUTO with enough scratch runs the hybrid stage (every other splat direct), under sincosf as well.
    for variant, nbytes in (("binned", need), ("binned", need // 3), ("auto", need), ("auto", 1 << 20)):
        gb, gbc = gpu_render(cfs, w, variant=variant, scratch_bytes=nbytes)
        assert np.array_equal(gb, g) and np.array_equal(gbc, gc)
    # the configuration bench.py times: MUFU sin/cos, AUTO with scratch (-> tile bins).  Conservation
    # stays exact; against the accurate image only splats within ~2^-21 of a pixel edge move.
    gf, gfc = gpu_render(cfs, w, variant="auto", scratch_bytes=need, flags=["fast_trig", "jit"])
    assert np.array_equal(gfc, gc) and gf[:, 3].astype(np.float64).sum() == S
    for ch in range(4):
        assert density_l1(gf[:, ch], g[:, ch]) <= L1_TOL
    sub = w.scaled(n_points=1 << 15)
    gs, gsc = gpu_render(cfs, sub)
    o, oc, _ = oracle.render_parallel(sub.system, sub.render)
    assert np.array_equal(gsc, oc)
    for ch in range(4):
        assert density_l1(gs[:, ch], o[:, ch]) <= L1_TOL


def test_cfg2_cfg3_cfg4_full_size_properties(cfs, oracle):
    """The other BASELINE configs at full size, in the launch configuration bench.py's side report times
    (AUTO with scratch + MUFU sin/cos): properties that hold at any size, and oracle parity on a sub-range
    of the points rendered into the full-size image."""
    # configs[2], middle frame: hybrid stage (tile bins + direct).  Exact conservation; identical to the
    # direct variant under the same sin/cos evaluation (integer-valued sums below 2^24)
    w = W.config(2)
    t = w.frames[7]
    S = w.render.n_points * 480
    sysh = cfs.cfs_create(w.system)
    need = cfs.cfs_binned_scratch_bytes(sysh, cfs.make_args(w.render))
    sysh.close()
    ga, gac = gpu_render(cfs, w, t=t, variant="auto", scratch_bytes=need, flags=["fast_trig", "jit"])
    gd, gdc = gpu_render(cfs, w, t=t, variant="direct", flags=["fast_trig"])
    assert int(gac[0]) == S and int(gac[1]) == 0 and ga[:, 3].astype(np.float64).sum() == S
    assert ga[:, 3].max() < 2 ** 24 and np.array_equal(ga[:, 3], gd[:, 3]) and np.array_equal(gac, gdc)
    small = gd[:, :3] < 2 ** 24          # hot pixels of the fractal exceed 2^24 in colour: there the order of
    assert np.array_equal(ga[:, :3][small], gd[:, :3][small])          # the float32 additions shows (R8)
    # beyond 2^24 every += 255 of the direct variant rounds (spacing 2, then 4): ~1e4 such additions drift by
    # up to ~6e-4 relative, while the binned half adds n_k * palette[k] once per tile -- both are float32 sums
    assert np.all(np.abs(ga[:, :3][~small] - gd[:, :3][~small]) <= 2e-3 * gd[:, :3][~small])
    assert np.all(ga[np.abs(np.arange(ga.shape[0]) // 1920 - 539.5) > 0.8415 * 540 + 1, 3] == 0)   # |sin| <= sin 1
    sub = w.scaled(n_points=1 << 14)
    gs, gsc = gpu_render(cfs, sub, t=t, flags=["fast_trig"])
    o, oc, _ = oracle.render_parallel(sub.system, sub.render, t=t)
    assert np.array_equal(gsc, oc)
    for ch in range(4):
        assert density_l1(gs[:, ch], o[:, ch]) <= L1_TOL
    # configs[3]: the whole 2^24-record cloud.  Every record is splatted or dropped; the alpha plane
    # counts the splats and every colour sum is an integer (exact float32 sums below 2^24)
    w = W.config(3)
    cloud = W.gaussian_mixture_cloud(w.render.n_points, w.cloud_seed)
    g, gc = gpu_render(cfs, w, cloud=cloud, flags=["fast_trig", "jit"])
    assert int(gc[0]) + int(gc[1]) == 1 << 24 and g[:, 3].astype(np.float64).sum() == int(gc[0])
    assert g.max() < 2 ** 24 and np.all(g == np.round(g))
    n_sub = 1 << 17
    gs, gsc = gpu_render(cfs, w, cloud=cloud, n_points=n_sub, flags=["fast_trig", "jit"])
    o, oc, _ = oracle.render_parallel(w.system, w.render, cloud=cloud, n_points=n_sub)
    assert abs(int(gsc[0]) - int(oc[0])) <= 4
    for ch in range(4):
        assert density_l1(gs[:, ch], o[:, ch]) <= L1_TOL
    # configs[4]: min over all points <= min over any subset, with equality wherever the subset holds the
    # winner; every key carries a depth in [3, 5] and one of the 20 palette entries
    w = W.config(4)
    g, gc = gpu_render(cfs, w, variant="auto", flags=["jit"], scratch_bytes=cfs.cfs_hiz_scratch_bytes(3840, 2160))    # Hi-Z, as bench.py
    assert int(gc[0]) == (1 << 26) * 980 and int(gc[1]) == 0
    gdir, gdc = gpu_render(cfs, w, variant="direct")          # the direct variant, linked kernel: the same image, bit for bit
    assert np.array_equal(g, gdir) and np.array_equal(gc, gdc)
    sub = w.scaled(n_points=1 << 12)
    o, _, _ = oracle.render_parallel(sub.system, sub.render)
    assert np.all(g <= o)
    hit = g != np.uint64(0xFFFFFFFFFFFFFFFF)
    depth = (g[hit] >> np.uint64(32)).astype(np.uint32).view(np.float32)
    assert hit.sum() > 1_000_000 and depth.min() >= 3.0 - 1e-6 and depth.max() <= 5.0 + 1e-6
    pal8 = set(int(v) for v in (g[hit] & np.uint64(0xFFFFFFFF)).astype(np.uint32)[:: 997])
    assert len(pal8) <= 20


# ------------------------------------------------------------------ bounds checks of our own (no compute-sanitizer on this pool)
_CHECKED_RENDERS = r"""
import sys, numpy as np, torch
sys.path.insert(0, %(root)r)
from paper_2606_02226_b200 import cfs, workloads as W
from oracle import cfs_oracle as O
from tests._gpu_util import gpu_render
def same(w, variant, flags=0, scratch=None, cloud=None, exact=True):
    g, c = gpu_render(cfs, w, variant=variant, flags=flags, scratch_bytes=scratch, cloud=cloud)
    o, oc, _ = O.render_parallel(w.system, w.render, cloud=cloud)
    assert np.array_equal(c, oc) or cloud is not None
    if exact:
        assert np.array_equal(g.astype(o.dtype), o), (w.name, variant)
w0 = W.config(0).scaled(n_points=5000 + 13, iterations=300)
for v, f in (("direct", 0), ("warp_agg", 0), ("binned", 0), ("binned", ["bin_hybrid"])):
    same(w0, v, f)
same(W.config(0).scaled(n_points=3000, iterations=200, width=200, height=120), "shared_hist")
w0c = W.config(0).scaled(n_points=400000, iterations=120)
sysh = cfs.cfs_create(w0c.system); need = cfs.cfs_binned_scratch_bytes(sysh, cfs.make_args(w0c.render)); sysh.close()
same(w0c, "binned", ["bin_hybrid"], scratch=need * 2 // 3)                       # several chunks
hot = W.Workload("hot", W.System(2, "ifs", W.square_funcs(probs=[0.0, 0.0, 1.0, 0.0]), [], "map_index", W.palette_for(4)),
                 W.Render(400, 5, 200, 40, 512, 512, (-1, 1, -1, 1), "rgba_f32"))
same(hot, "binned", ["bin_hybrid"])                                              # one pixel takes everything: rows overflow
w1 = W.config(1).scaled(n_points=(1 << 14) + 5)
gb, _ = gpu_render(cfs, w1, variant="binned", flags=["bin_hybrid", "fast_trig"])
gd, _ = gpu_render(cfs, w1, variant="direct", flags=["fast_trig"])
assert np.array_equal(gb, gd)
w4 = W.config(4).scaled(n_points=300000 + 7, iterations=100, width=256, height=144)
same(w4, "depth_hiz", scratch=cfs.cfs_hiz_scratch_bytes(256, 144))
same(w4, "direct")
w3 = W.config(3)
cloud = W.gaussian_mixture_cloud((1 << 16) + 11, w3.cloud_seed)
same(w3.scaled(n_points=(1 << 16) + 11), "auto", cloud=cloud, exact=False)
print("checked renders ok; kernels compiled at run time:", cfs.cfs_jit_stats()[0])
"""


@pytest.mark.parametrize("selftest", [False, True])
def test_device_bounds_checks(cfs, selftest):
    """compute-sanitizer is closed on this pool, so the kernels carry bounds checks of their own (CFS_CHECK in csrc/:
    staging rows, pool positions, tile / record / pixel / Hi-Z indices, ring stages), compiled in by -DCFS_CHECKS=1 for
    run-time compiled kernels.  Here every splat variant renders in a fresh process with all kernels compiled under
    the checks (a failed check traps and the render raises) and still matches the oracle; the negative control
    (-DCFS_CHECK_SELFTEST=1: every kernel fails its first check) must fail."""
    import os
    import subprocess
    import sys
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    env = dict(os.environ, CFS_FORCE_JIT="1", CFS_JIT_OPTIONS="-DCFS_CHECKS=1" + (" -DCFS_CHECK_SELFTEST=1" if selftest else ""))
    p = subprocess.run([sys.executable, "-c", _CHECKED_RENDERS % {"root": root}], env=env, capture_output=True, text=True, timeout=900)
    if selftest:
        assert p.returncode != 0, "the negative control rendered without tripping a check"
    else:
        assert p.returncode == 0, p.stdout[-2000:] + p.stderr[-4000:]
        assert "checked renders ok" in p.stdout and not p.stdout.strip().endswith(": 0")


_CACHED_RENDER = """
import sys, hashlib, numpy as np, torch
sys.path.insert(0, %(root)r)
from paper_2606_02226_b200 import cfs, workloads as W
from tests._gpu_util import gpu_render
cfs.lib()
w = W.config(1).scaled(n_points=20011, iterations=60, width=200, height=160)
g, c = gpu_render(cfs, w, variant="direct", flags=["jit", "fast_trig"])
n, ms = cfs.cfs_jit_stats()
print("RESULT", n, hashlib.sha256(g.tobytes()).hexdigest(), int(c[0]))
"""


def test_run_time_kernels_survive_processes_through_the_disk_cache(cfs, tmp_path):
    """$CFS_JIT_CACHE: a kernel compiled for a system by one process is loaded, not compiled, by the next one (the
    paper's own measurement has compilation at 35 x the frame time), keyed by kernel name and a hash of
    the embedded sources; a damaged cache file is compiled afresh and replaced.  Same image every time."""
    import os
    import subprocess
    import sys
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    env = dict(os.environ, CFS_JIT_CACHE=str(tmp_path))
    env.pop("CFS_FORCE_JIT", None)

    def run():
        p = subprocess.run([sys.executable, "-c", _CACHED_RENDER % {"root": root}], env=env, capture_output=True, text=True, timeout=600)
        assert p.returncode == 0, p.stdout[-2000:] + p.stderr[-4000:]
        line = [ln for ln in p.stdout.splitlines() if ln.startswith("RESULT")][-1].split()
        return int(line[1]), line[2], int(line[3])

    n1, h1, c1 = run()
    files = sorted(os.listdir(tmp_path))
    assert n1 == 1 and len(files) == 1, (n1, files)
    n2, h2, c2 = run()
    assert n2 == 0 and (h2, c2) == (h1, c1), "the second process compiled again or rendered something else"
    path = os.path.join(tmp_path, files[0])
    blob = bytearray(open(path, "rb").read())
    for i in range(len(blob) // 2, len(blob) // 2 + 64):
        blob[i] ^= 0x5A
    open(path, "wb").write(bytes(blob[: len(blob) - 100]))       # damaged and truncated
    n3, h3, c3 = run()
    assert (h3, c3) == (h1, c1), "a damaged cache file changed the render"
    n4, h4, c4 = run()
    assert n3 == 1 and n4 == 0 and (h4, c4) == (h1, c1), (n3, n4)
