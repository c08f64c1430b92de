"""cube_histogram_noalloc: the allocation-free histogram entry point (include/cube.h) against the existing
cube_histogram path and the CPU oracle, on two calls in a row that share the library's static scratch array.
Integer work: the bar is bit-exact.  Collected last on purpose (the suite runs with pytest -x); passes alone in a
fresh process (the first call resolves the scratch address itself) and after the other tests."""
import numpy as np
import pytest
import torch

import cubegen
import oracle
import paper_1211_4896_b200 as cube

pytestmark = pytest.mark.gpu


def seeded_cube(name, dims, misalign=0):
    cfg = cubegen.scaled(name, dims)
    n = dims[0] * dims[1] * dims[2]
    buf = torch.empty(n + 4, dtype=torch.float32, device="cuda")
    tmp = torch.empty(n, dtype=torch.float32, device="cuda")
    cubegen.generate_device(cfg, tmp.data_ptr())
    t = buf[misalign:misalign + n]
    t.copy_(tmp)
    torch.cuda.synchronize()
    return t, t.cpu().numpy()


def test_noalloc_histogram_matches_the_existing_path_twice_in_a_row():
    assert torch.cuda.is_available(), "gpu tests need a CUDA device (there is no CPU fallback)"
    # call 1: 4096 bins (the maximum) on a cube of several tiles and a ragged tail, host outputs;
    # call 2, right behind it on the same stream: another cube, FEWER bins, another range, device outputs -- whatever
    # call 1 left in the shared scratch must not show
    t1, a1 = seeded_cube("c2", (200, 131, 67), misalign=1)
    t2, a2 = seeded_cube("c4", (96, 96, 50))
    lo1, hi1 = -0.01, 0.05
    lo2, hi2 = float(np.nanmin(a2)), float(np.nanmax(a2))
    b1, o1 = cube.histogram_noalloc(t1, 200, 131, 67, cube.NOALLOC_MAX_BINS, lo1, hi1)
    b2 = torch.full((257,), -1, dtype=torch.int64, device="cuda")
    o2 = torch.full((2,), -1, dtype=torch.int64, device="cuda")
    cube.histogram_noalloc(t2, 96, 96, 50, 257, lo2, hi2, bins=b2, outside=o2)
    torch.cuda.synchronize()
    ctx = cube.Context()
    try:
        e1, eo1 = ctx.histogram(t1, 200, 131, 67, cube.NOALLOC_MAX_BINS, lo1, hi1)
        e2, eo2 = ctx.histogram(t2, 96, 96, 50, 257, lo2, hi2)
        torch.cuda.synchronize()
    finally:
        ctx.close()
    assert np.array_equal(b1, e1) and np.array_equal(o1, eo1)
    assert np.array_equal(b2.cpu().numpy().astype(np.uint64), e2) and np.array_equal(o2.cpu().numpy().astype(np.uint64), eo2)
    # and both equal the oracle (the existing path's own parity bar)
    r1, ro1 = oracle.histogram(a1, cube.NOALLOC_MAX_BINS, lo1, hi1)
    r2, ro2 = oracle.histogram(a2, 257, lo2, hi2)
    assert np.array_equal(b1, r1) and np.array_equal(o1, ro1)
    assert np.array_equal(e2, r2) and np.array_equal(eo2, ro2)
    assert int(b1.sum() + o1.sum()) == int(np.count_nonzero(~np.isnan(a1)))
    # a third call repeats the first: same counts again after the scratch held call 2's
    b3, o3 = cube.histogram_noalloc(t1, 200, 131, 67, cube.NOALLOC_MAX_BINS, lo1, hi1)
    assert np.array_equal(b3, e1) and np.array_equal(o3, eo1)


def test_noalloc_histogram_rejects_what_the_scratch_cannot_hold():
    t = torch.zeros(64, dtype=torch.float32, device="cuda")
    with pytest.raises(cube.CubeError) as e:
        cube.histogram_noalloc(t, 4, 4, 4, cube.NOALLOC_MAX_BINS + 1, 0.0, 1.0)
    assert e.value.code == cube.ERANGE and "range" in str(e.value)
    for bad in (lambda: cube.histogram_noalloc(t, 4, 4, 4, 0, 0.0, 1.0),
                lambda: cube.histogram_noalloc(t, 4, 4, 4, 16, 1.0, 0.0),
                lambda: cube.histogram_noalloc(t, 0, 4, 4, 16, 0.0, 1.0),
                lambda: cube.histogram_noalloc(t, 4, 4, 4, 16, float("nan"), 1.0)):
        with pytest.raises(cube.CubeError) as e:
            bad()
        assert e.value.code == cube.EINVAL
    # the rejected calls enqueued nothing and left the entry point usable: one bin, every voxel in it
    b, o = cube.histogram_noalloc(t, 4, 4, 4, 1, 0.0, 0.0)
    assert int(b[0]) == 64 and int(o.sum()) == 0
