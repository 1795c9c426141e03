"""CPU-side checks of the C ABI (no compute): the library loads, exports every function
include/cfs.h declares, validates arguments on the host, refuses to work without a device (there is
no CPU fallback), and plans the tiles of the binned variant with exact integer arithmetic."""
import ctypes as C
import os
import re

import numpy as np
import pytest

from paper_2606_02226_b200 import build as cuda_build
from paper_2606_02226_b200 import workloads as W

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def cfs():
    cuda_build.build()                       # nvcc cross-compiles without a GPU
    from paper_2606_02226_b200 import cfs as mod
    mod.lib()
    return mod


def _declared_functions():
    text = open(os.path.join(ROOT, "include", "cfs.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(cfs_[a-z0-9_]+)\s*\(", text)))


def test_library_exports_every_declared_function(cfs):
    names = _declared_functions()
    assert {"cfs_create", "cfs_render", "cfs_tonemap", "cfs_destroy", "cfs_render_host", "cfs_trace",
            "cfs_microbench", "cfs_binned_scratch_bytes", "cfs_binned_plan", "cfs_last_error"} <= set(names)
    lib = C.CDLL(cfs.LIB_PATH)
    for n in names:
        assert hasattr(lib, n), f"{n} is declared in include/cfs.h but not exported"
    assert set(cfs.EXPORTS) == set(names)                 # the Python binding carries the same names
    assert "sm_100a" in cfs.cfs_version()


def test_create_validates_on_the_host(cfs):
    sysh = cfs.cfs_create(W.config(1).system)             # host only: no device work
    sysh.close()
    for bad in (W.System(4, "ifs", W.square_funcs(), [], "none"),
                W.System(2, "ifs", [W.Func("affine", -1.0, [0.5, 0, 0, 0.5, 0, 0])], [], "none"),
                W.System(2, "ifs", [W.Func("affine", 0.0, [0.5, 0, 0, 0.5, 0, 0])], [], "none"),
                W.System(2, "ifs", W.square_funcs(), [], "point"),
                W.System(2, "ifs", W.square_funcs(), [W.Xform("affine")] * 9, "none"),
                W.System(2, "ifs", W.square_funcs(), [], "map_index", None)):
        with pytest.raises(cfs.CfsError) as ei:
            cfs.cfs_create(bad)
        assert ei.value.status == cfs.CFS_ERR_INVALID_ARG and cfs.cfs_last_error()


def test_no_cpu_fallback(cfs):
    """Without a CUDA device every working call fails loudly with CFS_ERR_CUDA."""
    import torch
    if torch.cuda.is_available():
        pytest.skip("a CUDA device is present")
    w = W.config(0).scaled(n_points=16)
    sysh = cfs.cfs_create(w.system)
    img = np.zeros(512 * 512, np.uint32)
    with pytest.raises(cfs.CfsError) as ei:
        cfs.cfs_render(sysh, cfs.make_args(w.render, d_image=img), stream=0)
    assert ei.value.status == cfs.CFS_ERR_CUDA and "no CPU fallback" in str(ei.value)
    with pytest.raises(cfs.CfsError) as ei:
        cfs.cfs_render_host(sysh, cfs.make_args(w.render), img, None, None, stream=0)
    assert ei.value.status == cfs.CFS_ERR_CUDA
    assert cfs.cfs_binned_scratch_bytes(sysh, cfs.make_args(w.render)) == 0
    sysh.close()


SIZES = [(512, 512), (1024, 1024), (1920, 1080), (3840, 2160), (64, 64), (200, 120), (1, 1), (4097, 3), (7, 9001),
         (16384, 16384), (12288, 1), (333, 777)]


@pytest.mark.parametrize("mode,n_funcs", [("hist_u32", 1), ("rgba_f32", 3), ("rgba_f32", 4), ("rgba_f32", 16)])
@pytest.mark.parametrize("size", SIZES)
def test_binned_plan_tile_arithmetic_is_exact(cfs, size, mode, n_funcs):
    """Interleaved tiles: pixel p belongs to tile p & mask and is its pixel p >> shift.  The map must be a
    bijection between the pixels of the image and (tile, pixel in tile) pairs below the planned sizes, and
    the plan must respect the shared-memory budgets of both passes."""
    wd, ht = size
    n_pix = wd * ht
    try:
        pl = cfs.cfs_binned_plan(wd, ht, mode, n_funcs)
    except cfs.CfsError as e:
        assert e.status == cfs.CFS_ERR_UNSUPPORTED          # too many tiles for 320-record staging rows
        nk = 1 if mode == "hist_u32" else n_funcs
        assert -(-n_pix // (49152 // nk)) > 200
        return
    tp, nt, sh, mask = pl["tile_pixels"], pl["n_tiles"], pl["tile_shift"], pl["tile_mask"]
    assert nt == 1 << sh and mask == nt - 1 and 64 <= nt <= 1024
    assert tp == -(-n_pix // nt)                                                        # ceil(n_pix / n_tiles)
    assert tp * pl["nk"] * 4 <= 192 << 10                                              # pass 2 counters
    assert pl["nk"] == (1 if mode == "hist_u32" else n_funcs)
    assert pl["cap"] >= 320 and pl["cap"] % 64 == 0
    assert nt * pl["cap"] * 2 + (nt + 4) * 4 <= 232448                                  # pass 1 staging rows (u16)
    assert tp * pl["nk"] <= 1 << 16                                                     # a record fits 16 bits
    assert pl["check_every"] % 4 == 0 and 4 <= pl["check_every"] <= 128 and pl["split"] >= 1     # whole Philox blocks
    p = np.unique(np.concatenate([np.arange(0, min(n_pix, 4 * nt), dtype=np.uint64),
                                  np.random.default_rng(1).integers(0, n_pix, 4096, dtype=np.uint64),
                                  np.array([0, n_pix - 1, max(n_pix - nt, 0), max(n_pix - nt - 1, 0)], dtype=np.uint64)]))
    p = p[p < n_pix]
    tile, inner = p & np.uint64(mask), p >> np.uint64(sh)
    assert tile.max() < nt and inner.max() < tp
    assert np.array_equal((inner << np.uint64(sh)) | tile, p)                           # the inverse pass 2 uses
    assert len(np.unique(tile * np.uint64(tp) + inner)) == len(p)                       # no two pixels share a counter


def test_hiz_scratch_bytes_is_host_arithmetic(cfs):
    """The Hi-Z map of CFS_VARIANT_DEPTH_HIZ: smallest 8/16/32-pixel block whose u16 map fits 96 KiB."""
    for wd, ht, side in ((256, 144, 8), (1920, 1080, 8), (3840, 2160, 16), (7680, 4320, 32)):
        n = -(-wd // side) * -(-ht // side)
        assert (n + 7) // 8 * 8 * 2 <= 96 << 10
        if side > 8:
            assert -(-wd // (side // 2)) * -(-ht // (side // 2)) * 2 > 96 << 10
        assert cfs.cfs_hiz_scratch_bytes(wd, ht) == (n + 7) // 8 * 8 * 2 + 256
    assert cfs.cfs_hiz_scratch_bytes(16384, 16384) == 0 and cfs.cfs_hiz_scratch_bytes(0, 10) == 0


def test_eq1_generator_validation(cfs):
    f = W.circle_funcs()
    with pytest.raises(cfs.CfsError) as ei:                      # mixed affine + circle
        cfs.cfs_create(W.System(2, "ifs", [f[0], W.square_funcs()[0]], [], "none"))
    assert ei.value.status == cfs.CFS_ERR_UNSUPPORTED
    with pytest.raises(cfs.CfsError) as ei:                      # 3-D
        cfs.cfs_create(W.System(3, "ifs", f, [], "none"))
    assert ei.value.status == cfs.CFS_ERR_INVALID_ARG
    with pytest.raises(cfs.CfsError) as ei:                      # f_id outside {0, 1}
        cfs.cfs_create(W.System(2, "ifs", [W.Func("circle_half", 1.0, [2.0, 0.0])], [], "none"))
    assert ei.value.status == cfs.CFS_ERR_INVALID_ARG


def test_branch_marker_validation(cfs):
    """CFS_T_BRANCH (one-to-many splatting) is checked on the host: not with reuse, known type ids only."""
    a = [W.Xform("affine", [0.5, 0, 0, 0.5, 0, 0])]
    ok = cfs.cfs_create(W.System(2, "ifs", W.square_funcs(), a + [W.Xform("branch")] + a, "none"))
    ok.close()
    with pytest.raises(cfs.CfsError) as ei:
        cfs.cfs_create(W.System(2, "ifs", W.square_funcs(), a + [W.Xform("branch")] + a, "none", None, reuse=True))
    assert ei.value.status == cfs.CFS_ERR_INVALID_ARG


def test_run_time_specialiser_compiles_without_a_device(cfs):
    """NEXT-4: the kernel templates compile under NVRTC for sm_100a from the sources embedded in
    the library -- the five BASELINE systems, and chains no ahead-of-time kernel exists for (BRANCH, SCATTER,
    reuse, the Eq. 1 generator).  Compile-only: no device needed."""
    for cfg in range(W.N_CONFIGS):
        w = W.config(cfg)
        sysh = cfs.cfs_create(w.system)
        nbytes, ms = cfs.cfs_jit_check(sysh, cfs.make_args(w.render, flags=["fast_trig"]))
        assert nbytes > 10000 and ms > 0.0
        sysh.close()
    br = [W.Xform("branch")]
    chain = [W.Xform("swirl"), W.Xform("affine", [0.6, 0, 0, 0.6, 0.3, -0.2])] + br + \
            [W.Xform("affine", [0.03, 0, 0, 0.03, 0, 0]), W.Xform("scatter", [64, 0.95, 0.95, 0.0])]
    r = W.Render(1000, 3, 40, 10, 128, 128, (-1.2, 1.2, -1.2, 1.2), "rgba_f32")
    for system in (W.System(2, "ifs", W.square_funcs(), chain, "map_index", W.palette_for(4)),
                   W.System(2, "ifs", W.circle_funcs(True), [W.Xform("stretch_cos")], "map_index", W.palette_for(2), reuse=True)):
        sysh = cfs.cfs_create(system)
        for kind in (-1, 6):                       # direct sink and the tile-bin pass 1
            nbytes, _ = cfs.cfs_jit_check(sysh, cfs.make_args(r), kind)
            assert nbytes > 10000
        sysh.close()
