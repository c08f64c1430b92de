"""GPU parity for the NEXT rows of SURVEY.md sec. 8(f): cube_mad, cube_clipped_moments, cube_sigma_clip (NEXT-1)
and cube_minimap (NEXT-2), through the C ABI, against the CPU oracle on the same seeded inputs.
Bar: bit-exact count / min / max / median / MAD / iteration count / window; mean, std <= 1e-9 relative.
"""
import math

import numpy as np
import pytest
import torch

import cubegen
import oracle
import paper_1211_4896_b200 as cube

pytestmark = pytest.mark.gpu
REL = 1e-9


@pytest.fixture(scope="module")
def ctx():
    assert torch.cuda.is_available(), "gpu tests need a CUDA device (there is no CPU fallback)"
    c = cube.Context()
    yield c
    c.close()


def dev(a, misalign=0):
    a = np.ascontiguousarray(a, dtype=np.float32).reshape(-1)
    buf = torch.empty(a.size + 4 + misalign, dtype=torch.float32, device="cuda")
    view = buf[misalign:misalign + a.size]
    view.copy_(torch.from_numpy(a))
    return view


def same_float(a, b):
    a, b = np.float32(a), np.float32(b)
    if math.isnan(float(a)) or math.isnan(float(b)):
        return math.isnan(float(a)) and math.isnan(float(b))
    return a.view(np.uint32) == b.view(np.uint32)


def check_moments(got, ref, scale=None):
    assert got["count"] == ref["count"] and got["nan_count"] == ref["nan_count"], (got, ref)
    assert same_float(got["min"], ref["min"]) and same_float(got["max"], ref["max"]), (got, ref)
    if ref["count"] == 0:
        assert math.isnan(got["mean"]) and math.isnan(got["std"])
        return
    mext = max(abs(float(ref["min"])), abs(float(ref["max"])))
    assert abs(got["mean"] - ref["mean"]) <= REL * max(abs(ref["mean"]), 1e-6 * mext), (got, ref)
    if math.isnan(ref["std"]):
        assert math.isnan(got["std"])
    else:
        assert abs(got["std"] - ref["std"]) <= REL * max(ref["std"], 1e-6 * mext), (got, ref)


def scaled_cube(name, dims, **kw):
    cfg = cubegen.scaled(name, dims, **kw)
    nx, ny, nz = cfg["dims"]
    t = torch.empty(nx * ny * nz, dtype=torch.float32, device="cuda")
    cubegen.generate_device(cfg, t.data_ptr())
    torch.cuda.synchronize()
    return t, t.cpu().numpy(), cfg["dims"]


# --------------------------------------------------------------------------------------- MAD
@pytest.mark.parametrize("n,misalign", [(1, 0), (2, 1), (33, 3), (4097, 0), (300001, 2)])
def test_mad_random_sizes(ctx, n, misalign):
    r = np.random.default_rng(n)
    a = (r.standard_normal(n) * 0.002 + 0.0005).astype(np.float32)
    if n > 100:
        a[r.integers(0, n, n // 50)] = np.nan
        a[r.integers(0, n, n // 100)] *= 300
    med, mad = ctx.mad(dev(a, misalign), n, 1, 1)
    rmed, rmad = oracle.mad(a)
    assert same_float(med, rmed) and same_float(mad, rmad)


def test_mad_ties_zero_and_empty(ctx):
    a = np.array([1.0] * 60 + [9.0] * 40 + [np.nan] * 7, dtype=np.float32)
    assert ctx.mad(dev(a), a.size, 1, 1) == oracle.mad(a)
    a = np.round(np.random.default_rng(5).standard_normal(100000) * 3).astype(np.float32)     # heavy ties
    got, ref = ctx.mad(dev(a), a.size, 1, 1), oracle.mad(a)
    assert same_float(got[0], ref[0]) and same_float(got[1], ref[1])
    e = np.full(1000, np.nan, dtype=np.float32)
    med, mad = ctx.mad(dev(e), e.size, 1, 1)
    assert math.isnan(med) and math.isnan(mad)
    c = np.full(5000, -0.0, dtype=np.float32)
    med, mad = ctx.mad(dev(c), c.size, 1, 1)
    assert same_float(med, -0.0) and same_float(mad, 0.0)       # |(-0) - (-0)| = +0


@pytest.mark.parametrize("name,dims", [("c1", (96, 80, 64)), ("c2", (128, 128, 96)), ("c3", (64, 64, 300)),
                                       ("c4", (256, 128, 40))])
def test_mad_scaled_configs(ctx, name, dims):
    t, a, (nx, ny, nz) = scaled_cube(name, dims)
    med, mad = ctx.mad(t, nx, ny, nz)
    rmed, rmad = oracle.mad(a)
    assert same_float(med, rmed) and same_float(mad, rmad)
    # after a cube_stats on the same data the first digit pass of the median is reused
    ctx.stats(t, nx, ny, nz, 0)
    med2, mad2 = ctx.mad(t, nx, ny, nz, flags=cube.REUSE_COARSE)
    assert same_float(med2, rmed) and same_float(mad2, rmad)
    # device outputs on a side stream
    s = torch.cuda.Stream()
    o = torch.zeros(2, dtype=torch.float32, device="cuda")
    with torch.cuda.stream(s):
        ctx.mad(t, nx, ny, nz, median_out=o[0:1], mad_out=o[1:2], stream=s.cuda_stream)
    s.synchronize()
    assert same_float(o[0].item(), rmed) and same_float(o[1].item(), rmad)


def test_mad_small_candidate_buffer_takes_the_third_pass():
    c = cube.Context(scratch_bytes_hint=4096)
    a = np.round(np.random.default_rng(9).standard_normal(400000) * 2).astype(np.float32)
    got, ref = c.mad(dev(a), a.size, 1, 1), oracle.mad(a)
    assert same_float(got[0], ref[0]) and same_float(got[1], ref[1])
    c.close()


# --------------------------------------------------------------------------------------- clipped moments
@pytest.mark.parametrize("n,misalign", [(1, 0), (7, 1), (1025, 2), (300001, 3)])
def test_clipped_moments_random(ctx, n, misalign):
    r = np.random.default_rng(1000 + n)
    a = r.standard_normal(n).astype(np.float32)
    if n > 10:
        a[r.integers(0, n, n // 20 + 1)] = np.nan
    t = dev(a, misalign)
    for lo, hi in [(-0.5, 1.25), (-100.0, 100.0), (0.0, 0.0), (2.0, -2.0), (float(np.nanmin(a)), float(np.nanmax(a)))]:
        for flags, sample in [(0, False), (cube.SAMPLE_STD, True)]:
            check_moments(ctx.clipped_moments(t, n, 1, 1, lo, hi, flags=flags), oracle.clipped_moments(a, lo, hi, sample))


def test_clipped_moments_edges_are_closed_and_ramp_closed_form(ctx):
    N = 1 << 20
    a = np.arange(N, dtype=np.float32)
    t = dev(a)
    m = ctx.clipped_moments(t, N, 1, 1, 1000.0, 4999.0)
    assert m["count"] == 4000 and m["min"] == 1000.0 and m["max"] == 4999.0 and m["nan_count"] == N - 4000
    assert m["mean"] == 2999.5
    assert m["std"] == pytest.approx(math.sqrt((4000 ** 2 - 1) / 12.0), rel=1e-12)
    with pytest.raises(cube.CubeError):
        ctx.clipped_moments(t, N, 1, 1, float("nan"), 1.0)
    inf = np.array([-np.inf, -1.0, 0.0, 2.0, np.inf, np.nan], dtype=np.float32)
    m = ctx.clipped_moments(dev(inf), inf.size, 1, 1, -1.0, 2.0)
    check_moments(m, oracle.clipped_moments(inf, -1.0, 2.0))
    assert m["count"] == 3


# --------------------------------------------------------------------------------------- sigma clipping
def check_clip(ctx, t, a, dims, kappa, max_iter, flags=0):
    nx, ny, nz = dims
    got, it, win = ctx.sigma_clip(t, nx, ny, nz, kappa, max_iter, flags=flags)
    ref, rit, rwin = oracle.sigma_clip(a, kappa, max_iter, sample_std=bool(flags & cube.SAMPLE_STD))
    assert it == rit, (it, rit)
    assert same_float(win[0], rwin[0]) and same_float(win[1], rwin[1]), (win, rwin)
    check_moments(got, ref)
    return got, it


@pytest.mark.parametrize("name,dims,kappa", [("c1", (96, 80, 64), 3.0), ("c2", (128, 128, 96), 3.0),
                                             ("c2", (128, 128, 96), 2.0), ("c3", (64, 64, 300), 2.5),
                                             ("c4", (256, 128, 40), 3.0)])
def test_sigma_clip_scaled_configs(ctx, name, dims, kappa):
    t, a, dims = scaled_cube(name, dims)
    got, it = check_clip(ctx, t, a, dims, kappa, 25)
    assert it >= 1
    check_clip(ctx, t, a, dims, kappa, 3, flags=cube.SAMPLE_STD)
    check_clip(ctx, t, a, dims, kappa, 0)


def test_sigma_clip_degenerate_and_async(ctx):
    c = np.full(10000, 2.5, dtype=np.float32)
    got, it = check_clip(ctx, dev(c), c, (c.size, 1, 1), 3.0, 10)
    assert it == 1 and got["std"] == 0.0
    e = np.full(999, np.nan, dtype=np.float32)
    got, it = check_clip(ctx, dev(e), e, (e.size, 1, 1), 3.0, 10)
    assert it == 0 and got["count"] == 0
    one = np.array([7.0], dtype=np.float32)
    check_clip(ctx, dev(one), one, (1, 1, 1), 3.0, 5, flags=cube.SAMPLE_STD)     # sample std of one voxel: NaN -> stop
    a = np.random.default_rng(3).standard_normal(200000).astype(np.float32)
    a[:2000] = 50.0
    t = dev(a)
    got, it = check_clip(ctx, t, a, (a.size, 1, 1), 3.0, 30)
    assert 0.95 < got["std"] < 1.0 and it >= 2
    with pytest.raises(cube.CubeError):
        ctx.sigma_clip(t, a.size, 1, 1, -1.0, 3)
    # device outputs, side stream, no host synchronisation inside
    s = torch.cuda.Stream()
    om = torch.zeros(40, dtype=torch.uint8, device="cuda")
    oi = torch.zeros(1, dtype=torch.int32, device="cuda")
    ow = torch.zeros(2, dtype=torch.float32, device="cuda")
    with torch.cuda.stream(s):
        ctx.sigma_clip(t, a.size, 1, 1, 3.0, 30, out=om, iters=oi, window=ow, stream=s.cuda_stream)
    s.synchronize()
    m = cube.MomentsT.from_buffer_copy(om.cpu().numpy().tobytes()).as_dict()
    assert m["count"] == got["count"] and m["mean"] == got["mean"] and oi.item() == it


# --------------------------------------------------------------------------------------- mini-map
def run_minimap(ctx, t, dims, part, flags=0):
    nx, ny, nz = dims
    mx, my, mz = ctx.minimap_dims(nx, ny, nz, *part)
    cells = torch.zeros(mx * my * mz * 40, dtype=torch.uint8, device="cuda")
    ctx.minimap(t, nx, ny, nz, part[0], part[1], part[2], cells, flags=flags)
    torch.cuda.synchronize()
    return np.frombuffer(cells.cpu().numpy().tobytes(), dtype=cube.MINIMAP_DTYPE).reshape(mz, my, mx)


def check_minimap(got, ref):
    assert got.shape == ref.shape
    assert (got["count"] == ref["count"]).all() and (got["nan_count"] == ref["nan_count"]).all()
    assert (got["min"].view(np.uint32)[ref["count"] > 0] == ref["min"].view(np.uint32)[ref["count"] > 0]).all()
    assert (got["max"].view(np.uint32)[ref["count"] > 0] == ref["max"].view(np.uint32)[ref["count"] > 0]).all()
    empty = ref["count"] == 0
    assert np.isnan(got["mean"][empty]).all() and np.isnan(got["std"][empty]).all() and np.isnan(got["min"][empty]).all()
    ok = ~empty
    mext = np.maximum(np.abs(ref["min"][ok]), np.abs(ref["max"][ok])).astype(np.float64)
    assert (np.abs(got["mean"][ok] - ref["mean"][ok]) <= REL * np.maximum(np.abs(ref["mean"][ok]), 1e-6 * mext)).all()
    rs = ref["std"][ok]
    fin = ~np.isnan(rs)
    assert np.isnan(got["std"][ok][~fin]).all()
    assert (np.abs(got["std"][ok][fin] - rs[fin]) <= REL * np.maximum(rs[fin], 1e-6 * mext[fin])).all()


@pytest.mark.parametrize("dims,part", [((64, 48, 40), (30, 30, 30)), ((96, 80, 64), (16, 16, 16)),
                                       ((100, 33, 17), (7, 5, 3)), ((37, 29, 11), (37, 29, 11)),
                                       ((1200, 9, 5), (600, 4, 2)), ((1300, 6, 4), (1300, 3, 2)),
                                       ((130, 70, 50), (1, 1, 1)), ((50, 40, 30), (64, 64, 64)),
                                       ((513, 20, 19), (30, 30, 30)), ((960, 20, 19), (30, 30, 30)),
                                       ((1024, 35, 9), (30, 7, 9)), ((484, 12, 10), (480, 5, 5))])
@pytest.mark.parametrize("variant", [0, 1, 2, 3])   # automatic / 128-bit register kernel / scalar kernel / TMA ring
def test_minimap_shapes(ctx, dims, part, variant):
    nx, ny, nz = dims
    r = np.random.default_rng(nx * 31 + ny)
    a = (r.standard_normal(nx * ny * nz) * 0.002 + 0.001).astype(np.float32)
    a[r.integers(0, a.size, a.size // 30)] = np.nan
    cubev = a.reshape(nz, ny, nx)
    cubev[0:min(part[2], nz), 0:min(part[1], ny), 0:min(part[0], nx)] = np.nan          # one fully blanked cell
    t = dev(a, misalign=nx % 4)
    ctx.set_knob(cube.KNOB_MINIMAP, variant)
    try:
        check_minimap(run_minimap(ctx, t, dims, part), oracle.minimap(a, dims, part))
        check_minimap(run_minimap(ctx, t, dims, part, flags=cube.SAMPLE_STD),
                      oracle.minimap(a, dims, part, sample_std=True))
    finally:
        ctx.set_knob(cube.KNOB_MINIMAP, 0)


def test_minimap_variants_agree_on_nan_free_and_nan_heavy_rows(ctx):
    # hot path (no NaN), safe path (scattered NaN) and whole blanked planes in one cube; the three kernels must
    # give the same integers and the oracle's values
    nx, ny, nz = 480, 64, 45
    r = np.random.default_rng(77)
    a = (r.standard_normal(nx * ny * nz) * 0.002).astype(np.float32).reshape(nz, ny, nx)
    a[10:20][r.random((10, ny, nx)) < 0.01] = np.nan
    a[30:33] = np.nan
    a = a.reshape(-1)
    t = dev(a)
    ref = oracle.minimap(a, (nx, ny, nz), (30, 30, 30))
    for variant in (0, 1, 2, 3):
        ctx.set_knob(cube.KNOB_MINIMAP, variant)
        try:
            check_minimap(run_minimap(ctx, t, (nx, ny, nz), (30, 30, 30)), ref)
        finally:
            ctx.set_knob(cube.KNOB_MINIMAP, 0)


def test_minimap_merge_pivot_far_from_the_cell_mean(ctx):
    # first column of a cell: blanked except one voxel of 1e6; the other columns 1e-3 noise -- the per-cell merge
    # starts from a pivot hundreds of standard deviations away and has to refine it (every kernel variant)
    nx, ny, nz = 64, 32, 32
    r = np.random.default_rng(5)
    a = (r.standard_normal(nx * ny * nz) * 1e-3).astype(np.float32).reshape(nz, ny, nx)
    a[:, :, 0] = np.nan
    a[3, 4, 0] = 1e6
    a[:, :, 32] = np.nan
    a[7, 1, 32] = -1e6
    a = a.reshape(-1)
    t = dev(a)
    ref = oracle.minimap(a, (nx, ny, nz), (32, 32, 32))
    for variant in (0, 1, 2, 3):
        ctx.set_knob(cube.KNOB_MINIMAP, variant)
        try:
            check_minimap(run_minimap(ctx, t, (nx, ny, nz), (32, 32, 32)), ref)
        finally:
            ctx.set_knob(cube.KNOB_MINIMAP, 0)


def test_minimap_scaled_config_and_global_consistency(ctx):
    t, a, dims = scaled_cube("c2", (160, 128, 96))
    nx, ny, nz = dims
    got = run_minimap(ctx, t, dims, (30, 30, 30))
    check_minimap(got, oracle.minimap(a, dims, (30, 30, 30)))
    g = ctx.moments(t, nx, ny, nz)
    assert int(got["count"].sum()) == g["count"] and int(got["nan_count"].sum()) == g["nan_count"]
    ok = got["count"] > 0
    assert np.float32(got["min"][ok].min()) == g["min"] and np.float32(got["max"][ok].max()) == g["max"]
    # count-weighted mean of the cell means is the global mean
    wm = float((got["mean"][ok] * got["count"][ok]).sum() / got["count"].sum())
    assert abs(wm - g["mean"]) <= 1e-9 * abs(g["mean"])


def test_minimap_invalid_arguments(ctx):
    t = dev(np.zeros(64, dtype=np.float32))
    cells = torch.zeros(40 * 8, dtype=torch.uint8, device="cuda")
    with pytest.raises(cube.CubeError):
        ctx.minimap(t, 4, 4, 4, 0, 2, 2, cells)
    with pytest.raises(cube.CubeError):
        ctx.minimap(t, 4, 4, 4, 2, 2, 2, np.zeros(40 * 8, dtype=np.uint8))      # pageable host memory
    with pytest.raises(cube.CubeError):
        ctx.minimap_dims(4, 4, 4, 2, -1, 2)


# --------------------------------------------------------------------------------------- Torben (Alg. 1) on the GPU
def check_torben(ctx, t, a, dims, cap):
    nx, ny, nz = dims
    val, it, conv = ctx.median_torben(t, nx, ny, nz, cap)
    rval, rit, rconv = oracle.torben_capped(a, cap)
    if rit < 0:                                           # no non-NaN voxel
        assert math.isnan(float(val)) and it == 0 and not conv
        return val, it, conv
    assert it == rit and conv == rconv, (cap, it, rit, conv, rconv)
    # Alg. 1 compares numerically: +0.0 and -0.0 are one value (cube.h), everything else is bit-exact
    assert (math.isnan(float(val)) and math.isnan(float(rval))) or float(val) == float(rval), (cap, val, rval)
    return val, it, conv


@pytest.mark.parametrize("name,dims", [("c1", (96, 80, 64)), ("c2", (128, 128, 96)), ("c3", (64, 64, 300)),
                                       ("c4", (256, 128, 40))])
def test_torben_scaled_configs(ctx, name, dims):
    t, a, dims = scaled_cube(name, dims)
    val, it, conv = check_torben(ctx, t, a, dims, 200)
    assert conv and same_float(val, oracle.median(a)) or float(val) == float(oracle.median(a))   # the exact lower median
    assert 1 <= it <= 200
    for cap in (0, 1, 2, 5, 10, 20, it - 1, it, it + 1):
        if cap >= 0:
            check_torben(ctx, t, a, dims, cap)
    # the radix select reads the cube twice, Alg. 1 `it` times: same value
    assert float(ctx.median(t, *dims)) == float(val)


def test_torben_edge_cases_and_async(ctx):
    for a in (np.full(1000, np.nan, np.float32), np.array([3.5], np.float32), np.full(4097, -2.0, np.float32),
              np.array([1, 2, 3, 4], np.float32), np.array([0.0, -0.0, 0.0, -0.0, 1.0], np.float32),
              np.array([-np.inf, 1.0, 2.0, np.inf, np.nan], np.float32),
              np.round(np.random.default_rng(4).standard_normal(100001) * 2).astype(np.float32)):
        for cap in (0, 1, 3, 300):
            check_torben(ctx, dev(a, 1), a, (a.size, 1, 1), cap)
    with pytest.raises(cube.CubeError):
        ctx.median_torben(dev(np.zeros(8, np.float32)), 8, 1, 1, -1)
    a = (np.random.default_rng(6).standard_normal(300000) * 0.002).astype(np.float32)
    t = dev(a)
    s = torch.cuda.Stream()
    o = torch.zeros(1, dtype=torch.float32, device="cuda")
    oi = torch.zeros(2, dtype=torch.int32, device="cuda")
    with torch.cuda.stream(s):
        ctx.median_torben(t, a.size, 1, 1, 100, out=o, iters=oi[0:1], converged=oi[1:2], stream=s.cuda_stream)
    s.synchronize()
    rval, rit, rconv = oracle.torben_capped(a, 100)
    assert float(o.item()) == float(rval) and oi[0].item() == rit and bool(oi[1].item()) == rconv


# --------------------------------------------------------------------------------------- mini-map: per-cell median
def run_minimap_median(ctx, t, dims, part):
    """every kernel variant (CUBE_KNOB_MAPMEDIAN: two reads / keys staged in shared memory) must give the same bits"""
    nx, ny, nz = dims
    mx, my, mz = ctx.minimap_dims(nx, ny, nz, *part)
    outs = []
    try:
        for variant in (0, 1, 2):
            ctx.set_knob(cube.KNOB_MAPMEDIAN, variant)
            med = torch.full((mx * my * mz,), 123.0, dtype=torch.float32, device="cuda")
            ctx.minimap_median(t, nx, ny, nz, part[0], part[1], part[2], med)
            torch.cuda.synchronize()
            outs.append(med.cpu().numpy().reshape(mz, my, mx))
    finally:
        ctx.set_knob(cube.KNOB_MAPMEDIAN, 0)
    assert same_bits_map(outs[0], outs[1]) and same_bits_map(outs[0], outs[2])
    return outs[0]


def same_bits_map(got, ref):
    g, r = np.ascontiguousarray(got).view(np.uint32), np.ascontiguousarray(ref).view(np.uint32)
    return bool(((g == r) | (np.isnan(got) & np.isnan(ref))).all())


@pytest.mark.parametrize("dims,part", [((64, 48, 40), (30, 30, 30)), ((96, 80, 64), (16, 16, 16)),
                                       ((100, 33, 17), (7, 5, 3)), ((37, 29, 11), (37, 29, 11)),
                                       ((1200, 9, 5), (600, 4, 2)), ((130, 70, 50), (1, 1, 1)),
                                       ((50, 40, 30), (64, 64, 64)), ((513, 20, 19), (30, 30, 30)),
                                       ((70, 66, 65), (64, 64, 32)),     # 131072 voxels per cell: re-read per digit
                                       ((40, 40, 40), (38, 38, 38)),     # 54872 voxels: the largest staged cells
                                       ((33, 32, 31), (11, 10, 9)), ((9, 9, 9), (10, 10, 1024)),
                                       ((300, 40, 30), (150, 40, 30))])  # 180000 voxels per cell
def test_minimap_median_shapes(ctx, dims, part):
    nx, ny, nz = dims
    r = np.random.default_rng(nx * 131 + part[0])
    a = (r.standard_normal(nx * ny * nz) * 0.002 + 0.001).astype(np.float32)
    a[r.integers(0, a.size, a.size // 40)] = np.nan
    a[r.integers(0, a.size, a.size // 50)] = np.round(a[r.integers(0, a.size, a.size // 50)], 3)    # ties
    a[r.integers(0, a.size, 20)] = np.float32([np.inf, -np.inf, 0.0, -0.0] * 5)
    a[:min(a.size, part[0])] = np.nan                                       # a NULL run at the start of cell 0
    got = run_minimap_median(ctx, dev(a, 1), dims, part)
    assert same_bits_map(got, oracle.minimap_median(a, dims, part))


def test_minimap_median_degenerate_cells(ctx):
    dims, part = (64, 40, 36), (32, 20, 12)
    a = np.full(64 * 40 * 36, np.nan, dtype=np.float32)                      # every cell empty
    assert np.isnan(run_minimap_median(ctx, dev(a), dims, part)).all()
    vol = a.reshape(36, 40, 64)
    vol[:12, :20, :32] = 2.5                                                 # a constant cell
    vol[12:24, 20:, 32:] = -0.0
    vol[12, 20, 32] = 0.0                                                    # -0.0 < +0.0: the lower median stays -0.0
    vol[30, 5, 40] = 7.0                                                     # a cell with a single voxel
    got = run_minimap_median(ctx, dev(vol.reshape(-1)), dims, part)
    assert same_bits_map(got, oracle.minimap_median(vol.reshape(-1), dims, part))
    # buckets larger than the candidate buffer of the two-read kernel (4096 keys): a cell of two values, the median
    # among 20000 copies of the upper one; a cell whose first digit ties but whose second differs; 0 / 1 data
    r = np.random.default_rng(8)
    two = np.where(r.random(64 * 40 * 36) < 0.45, np.float32(1.0), np.float32(1.0000001)).astype(np.float32)
    got = run_minimap_median(ctx, dev(two), dims, (64, 40, 36))
    assert same_bits_map(got, oracle.minimap_median(two, dims, (64, 40, 36)))
    near = (1.0 + r.random(64 * 40 * 36) * 1e-3).astype(np.float32)           # 8000 distinct keys in one first-digit bin
    near[r.integers(0, near.size, 500)] = np.nan
    for p3 in ((64, 40, 36), (32, 20, 12)):
        assert same_bits_map(run_minimap_median(ctx, dev(near), dims, p3), oracle.minimap_median(near, dims, p3))
    flags = (r.random(64 * 40 * 36) < 0.5).astype(np.float32)
    assert same_bits_map(run_minimap_median(ctx, dev(flags), dims, (32, 20, 12)), oracle.minimap_median(flags, dims, (32, 20, 12)))
    # infinities and NaN patterns that share their top 11 bits with them (payload below 2^21), the median an infinity
    odd = r.standard_normal(64 * 40 * 36).astype(np.float32)
    bits = odd.view(np.uint32)
    where = r.random(odd.size)
    bits[where < 0.55] = 0x7F800000                                          # +Inf: the median of most cells
    bits[(where >= 0.55) & (where < 0.70)] = 0x7F800001 + r.integers(0, 1 << 20)   # signalling NaNs, same raw bucket
    bits[(where >= 0.70) & (where < 0.75)] = 0xFF800123                      # their negative twins, beside -Inf
    bits[(where >= 0.75) & (where < 0.77)] = 0xFF800000
    vol3 = odd.reshape(36, 40, 64)
    vol3[:12, :20, :32] = np.where(r.random((12, 20, 32)) < 0.6, np.float32(-np.inf), np.float32(np.nan))   # median -Inf
    assert np.isnan(odd).sum() > 1000
    for p3 in ((32, 20, 12), (64, 40, 36), (8, 8, 8)):
        got = run_minimap_median(ctx, dev(odd), dims, p3)
        assert same_bits_map(got, oracle.minimap_median(odd, dims, p3))
        if p3 == (32, 20, 12):
            assert np.isposinf(got).sum() >= 4 and np.isneginf(got[0, 0, 0])
    for name, d3 in (("c3", (64, 64, 90)), ("c4", (96, 64, 30))):
        t, b, _ = scaled_cube(name, d3)
        for p3 in ((30, 30, 30), (8, 8, 8)):
            assert same_bits_map(run_minimap_median(ctx, t, d3, p3), oracle.minimap_median(b, d3, p3))
