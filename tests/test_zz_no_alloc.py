"""cfs_render_depth_noalloc (include/cfs.h): the Hi-Z depth render whose scratch is a static device array inside the
library, for callers that cannot call cudaMalloc.  Collected LAST on purpose (the suite runs with pytest -x).

Checked against the existing paths on the same seeded inputs: depth images are integer work (u64 keys, atomicMin),
so the bar is bit-exact, image and counters -- the tolerance the other DEPTH tests use.  Two calls in a row on
different images: the second call finds the first call's Hi-Z map in the shared array and must not be affected by it.
"""
import numpy as np
import pytest

from paper_2606_02226_b200 import workloads as W
from tests._gpu_util import gpu_render

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def cfs():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    from paper_2606_02226_b200 import cfs as mod
    mod.lib()
    return mod


def _noalloc_render(cfs, w, flags=0):
    import torch
    sysh = cfs.cfs_create(w.system)
    img = cfs.new_image(w.render)
    ctr = torch.zeros(2, dtype=torch.int64, device="cuda")
    # variant and d_scratch are ignored by the entry point: pass the defaults, no scratch
    args = cfs.make_args(w.render, d_image=img, d_counters=ctr, flags=flags)
    before = torch.cuda.memory_allocated()
    cfs.cfs_launch_count(reset=True)
    cfs.cfs_render_depth_noalloc(sysh, args)
    launches = cfs.cfs_launch_count()
    torch.cuda.synchronize()
    assert torch.cuda.memory_allocated() == before
    out = cfs.image_to_numpy(img, w.render.out_mode)
    c = ctr.cpu().numpy().astype(np.uint64)
    sysh.close()
    return out, c, launches


def _workloads():
    base = W.config(4)
    # a: sized so that all three phases of the Hi-Z render run (plain slice, first map, rebuilt map: 5 launches);
    # b: the plain slice and one map (3 launches)
    a = base.scaled(n_points=700_077, iterations=200, width=640, height=360)
    b = base.scaled(n_points=(1 << 16) + 5, iterations=120, width=333, height=190, seed=base.render.seed + 9)
    return a, b


def test_noalloc_depth_render_equals_the_existing_paths_twice_in_a_row(cfs):
    import os
    if os.environ.get("CFS_FORCE_JIT", "") not in ("", "0"):
        pytest.skip("$CFS_FORCE_JIT compiles every kernel at run time; the no-allocation entry point refuses that by contract")
    a, b = _workloads()
    want = {}
    for name, w in (("a", a), ("b", b)):
        hiz = gpu_render(cfs, w, variant="depth_hiz", scratch_bytes=cfs.cfs_hiz_scratch_bytes(w.render.width, w.render.height))
        direct = gpu_render(cfs, w, variant="direct")
        assert np.array_equal(hiz[0], direct[0]) and np.array_equal(hiz[1], direct[1]), name
        want[name] = hiz
    # two calls in a row, then the first again: every call finds another image's map in the shared array
    for name, w in (("a", a), ("b", b), ("a", a)):
        got, c, launches = _noalloc_render(cfs, w)
        assert np.array_equal(got, want[name][0]), name
        assert np.array_equal(c, want[name][1]), name
        assert launches == {"a": 5, "b": 3}[name], (name, launches)      # the map in the static array really was used
    # the interpreter flag is honoured too (linked kernels either way)
    got, c, _ = _noalloc_render(cfs, b, flags=["interpret_chain"])
    assert np.array_equal(got, want["b"][0]) and np.array_equal(c, want["b"][1])


def test_noalloc_rejects_what_it_cannot_serve(cfs):
    import torch
    a, _ = _workloads()
    sysh = cfs.cfs_create(a.system)
    img = torch.zeros(16, dtype=torch.int64, device="cuda")
    # beyond the built-in scratch: more than 49152 blocks of 32 x 32 pixels (the image is never touched)
    big = a.scaled(width=8192, height=8192).render
    assert cfs.cfs_hiz_scratch_bytes(8192, 8192) == 0
    with pytest.raises(cfs.CfsError) as e:
        cfs.cfs_render_depth_noalloc(sysh, cfs.make_args(big, d_image=img))
    assert e.value.status == cfs.CFS_ERR_INVALID_ARG and "built-in scratch holds" in str(e.value)
    # the largest image the map serves fits the stated maximum
    assert 0 < cfs.cfs_hiz_scratch_bytes(7000, 7000) <= cfs.NOALLOC_SCRATCH_BYTES
    assert 0 < cfs.cfs_hiz_scratch_bytes(3840, 2160) <= cfs.NOALLOC_SCRATCH_BYTES
    # run-time compilation allocates: refused
    with pytest.raises(cfs.CfsError) as e:
        cfs.cfs_render_depth_noalloc(sysh, cfs.make_args(a.render, d_image=cfs.new_image(a.render), flags=["jit"]))
    assert e.value.status == cfs.CFS_ERR_INVALID_ARG
    sysh.close()
    # not a DEPTH render of an IFS: unsupported
    w1 = W.config(1).scaled(n_points=1000, iterations=30, width=64, height=64)
    s1 = cfs.cfs_create(w1.system)
    with pytest.raises(cfs.CfsError) as e:
        cfs.cfs_render_depth_noalloc(s1, cfs.make_args(w1.render, d_image=cfs.new_image(w1.render)))
    assert e.value.status == cfs.CFS_ERR_UNSUPPORTED
    s1.close()
