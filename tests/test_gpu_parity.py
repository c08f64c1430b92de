"""GPU parity: the CUDA path (libcube through its C ABI) against the CPU oracle, element by element on
the same seeded inputs.  Bar (BASELINE.json north_star): bit-exact count / nan_count / min / max /
histogram / k-th / median; |rel. error| <= 1e-9 for mean and std (floor of DESIGN.md R16 on
degenerate cubes).  Every test needs a CUDA device and FAILS without one (no CPU fallback)."""
import math

import numpy as np
import pytest
import torch

import cubegen
import oracle
import paper_1211_4896_b200 as cube

pytestmark = pytest.mark.gpu

REL = 1e-9


@pytest.fixture(scope="module", params=["l2_resident_single_launch", "general_path"])
def ctx(request):
    """Every test of this file runs twice: as a user gets it (cubes of at most 96 MiB: cube_stats with the median and
    cube_median are ONE cooperative launch), and with CUBE_KNOB_SMALL = 1 (the general multi-launch path that larger
    cubes take), so that both see every edge case here."""
    assert torch.cuda.is_available(), "gpu tests need a CUDA device (there is no CPU fallback)"
    torch.cuda.init()
    c = cube.Context()
    c.set_knob(cube.KNOB_SMALL, 1 if request.param == "general_path" else 0)
    yield c
    c.close()


def dev(a, misalign=0):
    """numpy float32 -> device tensor; `misalign` floats of offset from a 16-byte boundary."""
    a = np.ascontiguousarray(a, dtype=np.float32).reshape(-1)
    buf = torch.empty(a.size + 4 + misalign, dtype=torch.float32, device="cuda")
    view = buf[misalign:misalign + a.size]
    view.copy_(torch.from_numpy(a))
    assert view.data_ptr() % 16 == (4 * misalign) % 16
    return view


def bits(x):
    return int(np.float32(x).view(np.uint32))


def same_float(a, b):
    a, b = np.float32(a), np.float32(b)
    if math.isnan(float(a)) or math.isnan(float(b)):
        return math.isnan(float(a)) and math.isnan(float(b))
    return bits(a) == bits(b)


def check_minimap_cells(got, ref):
    """Mini-map cells against the oracle: count / nan_count / min / max exact, mean and std <= REL with the floor of
    DESIGN.md R16 (no cell is left out of the std check; empty cells must be NaN)."""
    assert got.shape == ref.shape
    assert (got["count"] == ref["count"]).all() and (got["nan_count"] == ref["nan_count"]).all()
    ok = ref["count"] > 0
    for f in ("min", "max"):
        g, r = np.ascontiguousarray(got[f]), np.ascontiguousarray(ref[f])
        assert (g.view(np.uint32)[ok] == r.view(np.uint32)[ok]).all() and np.isnan(g[~ok]).all()
    assert np.isnan(got["mean"][~ok]).all() and np.isnan(got["std"][~ok]).all()
    mext = np.maximum(np.abs(ref["min"][ok]), np.abs(ref["max"][ok])).astype(np.float64)
    assert (np.abs(got["mean"][ok] - ref["mean"][ok]) <= REL * np.maximum(np.abs(ref["mean"][ok]), 1e-6 * mext)).all()
    assert (np.abs(got["std"][ok] - ref["std"][ok]) <= REL * np.maximum(ref["std"][ok], 1e-6 * mext)).all()


def check_moments(got, ref, a):
    assert got["count"] == ref["count"] and got["nan_count"] == ref["nan_count"]
    assert same_float(got["min"], ref["min"]) and same_float(got["max"], ref["max"])
    if ref["count"] == 0:
        assert math.isnan(got["mean"]) and math.isnan(got["std"])
        return
    if math.isnan(ref["std"]):
        assert math.isnan(got["std"])
    if math.isnan(ref["mean"]):                      # reading R8: an infinite voxel makes mean and std NaN
        assert math.isnan(got["mean"]) and math.isnan(got["std"])
        return
    fin = a[np.isfinite(a)] if a is not None else None
    # R16: relative 1e-9, with a floor that only matters on degenerate cubes (std == 0, mean ~ 0)
    mabs = float(np.mean(np.abs(fin.astype(np.float64)))) if fin is not None and fin.size else 0.0
    mext = max(abs(float(ref["min"])), abs(float(ref["max"])))
    assert abs(got["mean"] - ref["mean"]) <= REL * max(abs(ref["mean"]), 1e-6 * mabs), (got, ref)
    if not math.isnan(ref["std"]):
        assert abs(got["std"] - ref["std"]) <= REL * max(ref["std"], 1e-6 * mext), (got, ref)


def full_check(ctx, a, hists=(), ks=(), misalign=0):
    a = np.ascontiguousarray(a, dtype=np.float32).reshape(-1)
    t = dev(a, misalign)
    n = a.size
    ref = oracle.moments(a)
    check_moments(ctx.moments(t, n, 1, 1), ref, a)
    check_moments(ctx.moments(t, n, 1, 1, flags=cube.SAMPLE_STD), oracle.moments(a, sample_std=True), a)
    for nbins, lo, hi in hists:
        try:
            rb, ro = oracle.histogram(a, nbins, lo, hi)
        except ValueError:                      # e.g. scale overflows float32 on a subnormal range (R19)
            with pytest.raises(cube.CubeError):
                ctx.histogram(t, n, 1, 1, nbins, lo, hi)
            continue
        b, o = ctx.histogram(t, n, 1, 1, nbins, lo, hi)
        assert (b == rb).all() and (o == ro).all(), (nbins, lo, hi)
        assert int(b.sum() + o.sum()) == ref["count"]
    cnt = ref["count"]
    med = ctx.median(t, n, 1, 1)
    assert same_float(med, oracle.median(a))
    check_stats(ctx, t, a, ref, hists)
    for k in ks:
        if k < cnt:
            assert same_float(ctx.kth(t, n, 1, 1, k), oracle.kth(a, k)), k
        else:
            assert math.isnan(float(ctx.kth(t, n, 1, 1, k)))
    return ref


def check_stats(ctx, t, a, ref, hists, dims=None):
    """cube_stats (everything in two reads) against the oracle: fixed ranges, [min,max], no histogram."""
    nx, ny, nz = dims if dims else (a.size, 1, 1)
    omed = oracle.median(a)
    m, b, o, med = ctx.stats(t, nx, ny, nz)                                   # moments + median only
    check_moments(m, ref, a)
    assert b is None and same_float(med, omed)
    for nbins, lo, hi in hists:
        try:
            rb, ro = oracle.histogram(a, nbins, lo, hi)
        except ValueError:
            with pytest.raises(cube.CubeError):
                ctx.stats(t, nx, ny, nz, nbins, lo, hi)
            continue
        m, b, o, med = ctx.stats(t, nx, ny, nz, nbins, lo, hi)
        check_moments(m, ref, a)
        assert (b == rb).all() and (o == ro).all(), (nbins, lo, hi)
        assert same_float(med, omed)
        m, b, o, med = ctx.stats(t, nx, ny, nz, nbins, lo, hi, want_median=False)
        assert med is None and (b == rb).all() and (o == ro).all()
    for nbins in (64, 4096, 16385):                                           # histogram over [min,max]
        m, b, o, med = ctx.stats(t, nx, ny, nz, nbins, flags=cube.SAMPLE_STD)
        check_moments(m, oracle.moments(a, sample_std=True), a)
        assert same_float(med, omed)
        usable = ref["count"] > 0 and np.isfinite(ref["min"]) and np.isfinite(ref["max"])
        if usable:
            try:
                rb, ro = oracle.histogram(a, nbins, float(ref["min"]), float(ref["max"]))
            except ValueError:
                usable = False
        if usable:
            assert (b == rb).all() and (o == ro).all() and int(b.sum()) == ref["count"], nbins
        else:
            assert not b.any() and (o == np.uint64(2 ** 64 - 1)).all()


def std_ks(n):
    return sorted(set(k for k in (0, 1, n // 100, (n - 1) // 2, n // 2, 99 * n // 100, n - 2, n - 1, n, n + 5)
                      if k >= 0))


# ------------------------------------------------------------------------------------------------ small
@pytest.mark.parametrize("n", [1, 2, 3, 4, 5, 7, 31, 257, 1023, 4099, 8192 * 4 + 3, 37 * 41 * 43, 300001])
@pytest.mark.parametrize("misalign", [0, 1, 3])
def test_small_noise_with_nans(ctx, n, misalign):
    r = np.random.default_rng(n * 7 + misalign)
    a = (r.standard_normal(n) * 0.002).astype(np.float32)
    if n > 4:
        a[r.integers(0, n, max(1, n // 50))] = np.nan
    cnt = int((~np.isnan(a)).sum())
    full_check(ctx, a, hists=[(256, -0.005, 0.005), (4096, -0.02, 0.5), (1, -1.0, 1.0), (7, 0.0, 0.001)],
               ks=std_ks(cnt), misalign=misalign)


def test_degenerate_cubes(ctx):
    qn = np.float32("nan")
    neg_nan = np.frombuffer(np.uint32(0xFFC00000).tobytes(), dtype=np.float32)[0]
    cases = [
        np.full(100000, 0.1, np.float32),                                  # constant: std == 0 exactly
        np.full(70001, -1234.567, np.float32),
        np.full(5000, qn, np.float32),                                     # all blanked
        np.array([qn, 2.5, neg_nan], np.float32),                          # single value
        np.array([0.0, -0.0, 0.0, -0.0, -0.0], np.float32),                # signed zeros (R7)
        np.array([1e-40, -1e-40, 0.0, -0.0, 1e-45, 3e-39], np.float32),    # subnormals (R9)
        np.array([np.inf, -np.inf, 1.0, qn, 2.0], np.float32),             # infinities (R8)
        np.concatenate([np.full(40000, 0.1, np.float32), np.full(30000, qn, np.float32),
                        np.full(40000, 0.1, np.float32)]),                 # constant with a blanked slab
        np.tile(np.array([0.0, -0.0], np.float32), 60000),                 # -0.0 < +0.0 inside one thread's batch
        np.tile(np.array([-0.0, 0.0, 0.0], np.float32), 40001),
        np.concatenate([np.full(50000, 0.0, np.float32), np.full(50000, -0.0, np.float32)]),
        np.arange(1 << 20, dtype=np.float32),                              # ramp: closed forms
        np.arange(1 << 20, dtype=np.float32)[::-1].copy() - np.float32(2 ** 19),
    ]
    for a in cases:
        cnt = int((~np.isnan(a)).sum())
        fin = a[np.isfinite(a)]
        hists = [(16, -1.0, 1.0), (1024, 0.0, float(1 << 20))]
        if fin.size:
            hists.append((64, float(fin.min()), float(fin.max())))         # hi == lo on constant cubes (R13)
        got = None
        if np.isinf(a).any():
            t = dev(a)
            got, ref = ctx.moments(t, a.size, 1, 1), oracle.moments(a)
            assert got["count"] == ref["count"] and same_float(got["min"], ref["min"]) and same_float(got["max"], ref["max"])
            assert np.isnan(got["mean"]) and np.isnan(got["std"]) and np.isnan(ref["mean"]) and np.isnan(ref["std"])   # R8
            assert same_float(ctx.median(t, a.size, 1, 1), oracle.median(a))
            for k in range(cnt):
                assert same_float(ctx.kth(t, a.size, 1, 1, k), oracle.kth(a, k))
            m, b, o, med = ctx.stats(t, a.size, 1, 1, 128)                    # [min,max] = [-inf,inf]: unusable
            assert same_float(med, oracle.median(a)) and not b.any() and (o == np.uint64(2 ** 64 - 1)).all()
            continue
        ref = full_check(ctx, a, hists=hists, ks=std_ks(cnt))
        if cnt and float(fin.min()) == float(fin.max()):
            t = dev(a)
            m = ctx.moments(t, a.size, 1, 1)
            assert m["std"] == 0.0 and m["mean"] == float(fin[0])           # exactly


def test_moments_merge_pivot_far_from_the_mean(ctx):
    # The last CTA merges the per-CTA partials as sums about the mean of the first non-empty partial.  Here that
    # partial is one voxel of 1e6 (the rest of CTA 0's first tile is blanked) in front of 2^24 voxels of 1e-3 noise:
    # the pivot is ~4000 standard deviations from the mean, q - s^2/n would lose 7 digits, and the merge has to
    # refine its pivot to stay within 1e-9 (moments numerics).
    n = 1 << 24
    r = np.random.default_rng(2024)
    a = (r.standard_normal(n) * 1e-3).astype(np.float32)
    a[:8192] = np.nan
    a[5] = 1e6
    t = dev(a)
    ref = oracle.moments(a)
    assert abs(1e6 - ref["mean"]) > 1000 * ref["std"]
    for per in (0, 1, 4):
        ctx.set_launch(per)
        check_moments(ctx.moments(t, n, 1, 1), ref, a)
        m = ctx.stats(t, n, 1, 1, 64, None, None)[0]
        check_moments(m, ref, a)
    ctx.set_launch(0)


def test_kth_multi_matches_single_selections(ctx):
    # cube_kth_multi: several ranks after ONE first-digit pass -- config 3's request (median, n/100, 99n/100) and
    # edge ranks, ties, a rank beyond the count (NaN), device output, reuse of the kept histogram
    cfg = cubegen.scaled("c3", (64, 64, 300))
    a = cubegen.generate_numpy(cfg).reshape(-1)
    t = dev(a)
    n = a.size
    cnt = int(np.count_nonzero(a == a))
    ks = [(cnt - 1) // 2, cnt // 100, 99 * cnt // 100, 0, cnt - 1, cnt, cnt + 5]
    got = ctx.kth_multi(t, n, 1, 1, ks)
    for k, g in zip(ks, got):
        if k >= cnt:
            assert math.isnan(float(g))
        else:
            assert same_float(g, oracle.kth(a, k)), (k, g)
    assert same_float(got[0], oracle.median(a))
    # the first-digit histogram stays in the context: more ranks of the same cube without the first pass
    more = ctx.kth_multi(t, n, 1, 1, [cnt // 2, cnt // 3], flags=cube.REUSE_COARSE)
    assert same_float(more[0], oracle.kth(a, cnt // 2)) and same_float(more[1], oracle.kth(a, cnt // 3))
    out = torch.zeros(3, dtype=torch.float32, device="cuda")
    ctx.kth_multi(t, n, 1, 1, ks[:3], out=out, stream=torch.cuda.current_stream().cuda_stream)
    torch.cuda.synchronize()
    assert (out.cpu().numpy().view(np.uint32) == got[:3].view(np.uint32)).all()
    # heavy ties and signed zeros
    b = np.array([0.0, -0.0, 1.0, 1.0, 1.0, -2.5, np.nan, 7.0] * 500, dtype=np.float32)
    tb = dev(b)
    nb = int(np.count_nonzero(b == b))
    kb = list(range(0, nb, 377)) + [nb - 1]
    gb = ctx.kth_multi(tb, b.size, 1, 1, kb)
    for k, g in zip(kb, gb):
        assert same_float(g, oracle.kth(b, k)), (k, g)
    with pytest.raises(cube.CubeError):
        ctx.kth_multi(t, n, 1, 1, [])


def test_kth_multi_two_reads_edges_and_fallback(ctx):
    # cube_kth_multi gathers the first-digit buckets of up to four ranks in ONE read (cube_select_multi.cuh):
    # +-Inf share their first-digit bucket with NaNs, duplicated ranks, ranks of one bucket, a misaligned
    # ragged cube, only invalid ranks -- and the per-rank selections that take over on the device when the
    # buckets do not fit the candidate buffer (a context with a 4 KiB buffer, and a constant cube)
    rng = np.random.default_rng(77)
    a = rng.standard_normal(200003).astype(np.float32)
    a[::97] = np.nan
    a[5::1013] = np.inf
    a[7::2027] = -np.inf
    a[11::31] = 0.25          # a heavy tie
    cnt = int(np.count_nonzero(a == a))
    ks = [0, 3, cnt // 2, cnt // 2, cnt // 2 + 1, cnt - 1, cnt - 2, cnt // 7, 5 * cnt // 7, cnt + 1]
    ref = [oracle.kth(a, k) if k < cnt else np.float32(np.nan) for k in ks]
    small = cube.Context(scratch_bytes_hint=4096)
    try:
        for mis in (0, 1, 3):
            t = dev(a, misalign=mis)
            for c in (ctx, small):
                got = c.kth_multi(t, a.size, 1, 1, ks)
                for k, g, r in zip(ks, got, ref):
                    assert same_float(g, r), (mis, c is small, k, g, r)
        t = dev(a)
        for c in (ctx, small):
            bad = c.kth_multi(t, a.size, 1, 1, [cnt, cnt + 9, 1 << 60])
            assert all(math.isnan(float(g)) for g in bad)
            one = c.kth_multi(t, a.size, 1, 1, [cnt // 3])
            assert same_float(one[0], oracle.kth(a, cnt // 3))
        # every voxel is a candidate: overflow of the small buffer on a constant cube, exact fit questions aside
        cst = np.full(70001, -3.5, dtype=np.float32)
        tc = dev(cst)
        for c in (ctx, small):
            g = c.kth_multi(tc, cst.size, 1, 1, [0, 35000, 70000, 70001, 12])
            assert [bits(x) for x in g[:3]] == [bits(-3.5)] * 3 and math.isnan(float(g[3])) and bits(g[4]) == bits(-3.5)
        # all NaN
        tn = dev(np.full(5000, np.nan, dtype=np.float32))
        assert all(math.isnan(float(x)) for x in ctx.kth_multi(tn, 5000, 1, 1, [0, 1, 2]))
        # the digit bins are left clean: a plain selection afterwards is still right
        assert same_float(ctx.kth(t, a.size, 1, 1, cnt // 5), oracle.kth(a, cnt // 5))
        assert same_float(small.median(t, a.size, 1, 1), oracle.median(a))
    finally:
        small.close()


def test_ramp_closed_forms_direct(ctx):
    # independent of the oracle: north_star's closed forms
    N = 1 << 24
    t = torch.arange(N, dtype=torch.float32, device="cuda")
    m = ctx.moments(t, 256, 256, 256)
    assert m["count"] == N and m["min"] == 0.0 and m["max"] == np.float32(N - 1)
    assert abs(m["mean"] - (N - 1) / 2.0) <= REL * (N - 1) / 2.0
    assert abs(m["std"] - math.sqrt((N * N - 1) / 12.0)) <= REL * math.sqrt((N * N - 1) / 12.0)
    b, o = ctx.histogram(t, 256, 256, 256, 65536, 0.0, float(N))
    assert (b == N // 65536).all() and o.tolist() == [0, 0]
    b, o = ctx.histogram(t, 256, 256, 256, 4096, 0.0, float(N))
    assert (b == N // 4096).all()
    for k in (0, 12345, (N - 1) // 2, N - 1):
        assert ctx.kth(t, 256, 256, 256, k) == np.float32(k)
    assert ctx.median(t, 256, 256, 256) == np.float32((N - 1) // 2)


def test_heavy_ties_and_hot_bins(ctx):
    r = np.random.default_rng(4)
    n = 1 << 21
    a = cubegen.generate_numpy(cubegen.scaled("c4", (256, 256, 32))).reshape(-1)
    ref = full_check(ctx, a, hists=[(256, 0.0, float(a.max())), (65536, 0.0, float(a.max())), (4096, 0.0, 1.0)],
                     ks=std_ks(n))
    assert ref["min"] == 0.0
    b = r.integers(0, 3, n).astype(np.float32)                             # three values only
    full_check(ctx, b, hists=[(3, 0.0, 2.0), (65536, 0.0, 2.0)], ks=std_ks(n))


@pytest.mark.parametrize("nbins", [1, 2, 255, 1024, 4096, 16384, 16385, 40000, 65536])
def test_histogram_bin_counts_all_sizes(ctx, nbins):
    r = np.random.default_rng(nbins)
    a = np.concatenate([(r.standard_normal(200000) * 0.3).astype(np.float32),
                        r.uniform(-2, 2, 100001).astype(np.float32)])
    a[::97] = np.nan
    t = dev(a)
    for lo, hi in ((-1.0, 1.0), (float(np.nanmin(a)), float(np.nanmax(a))), (0.25, 0.25000003)):
        b, o = ctx.histogram(t, a.size, 1, 1, nbins, lo, hi)
        rb, ro = oracle.histogram(a, nbins, lo, hi)
        assert (b == rb).all() and (o == ro).all()


def test_invalid_arguments(ctx):
    t = dev(np.zeros(16, np.float32))
    for bad in ((0, 0.0, 1.0), (65537, 0.0, 1.0), (4, 1.0, 0.0), (4, float("nan"), 1.0), (4, 0.0, float("inf")),
                (4, -3e38, 3e38)):
        with pytest.raises(cube.CubeError) as e:
            ctx.histogram(t, 16, 1, 1, *bad)
        assert e.value.code == cube.EINVAL
    for dims in ((0, 1, 1), (-4, 1, 1), (1 << 20, 1 << 20, 1 << 20)):
        with pytest.raises(cube.CubeError):
            ctx.moments(t, *dims)
    with pytest.raises(cube.CubeError):
        ctx.median(None, 16, 1, 1)


def test_tiling_invariance(ctx):
    # any tiling of the cube over CTAs gives identical integers (order-free merges)
    a = cubegen.generate_numpy(cubegen.scaled("c3", (128, 128, 64))).reshape(-1)
    t = dev(a, 2)
    base = None
    try:
        for per_sm in (1, 2, 3, 5, 8):
            ctx.set_launch(per_sm)
            m = ctx.moments(t, a.size, 1, 1)
            b, o = ctx.histogram(t, a.size, 1, 1, 1000, -0.01, 0.02)
            med = ctx.median(t, a.size, 1, 1)
            cur = (m["count"], m["nan_count"], bits(m["min"]), bits(m["max"]), b.tobytes(), o.tobytes(), bits(med))
            if base is None:
                base, m0 = cur, m
            assert cur == base
            assert abs(m["mean"] - m0["mean"]) <= 1e-13 * abs(m0["mean"]) + 1e-300
            assert abs(m["std"] - m0["std"]) <= 1e-13 * m0["std"]
    finally:
        ctx.set_launch(0)
    m1 = ctx.moments(t, a.size, 1, 1)
    m2 = ctx.moments(t, a.size, 1, 1)
    assert m1 == m2 or (m1["mean"] == m2["mean"] and m1["std"] == m2["std"])   # run-to-run deterministic


def test_device_and_pinned_outputs_on_a_stream(ctx):
    a = cubegen.generate_numpy(cubegen.scaled("c1", (64, 64, 64), nsrc=3)).reshape(-1)
    t = dev(a)
    s = torch.cuda.Stream()
    out_m = torch.zeros(40, dtype=torch.uint8, device="cuda")
    out_b = torch.zeros(1024, dtype=torch.int64, device="cuda")
    out_o = torch.zeros(2, dtype=torch.int64, device="cuda")
    out_med = torch.zeros(1, dtype=torch.float32).pin_memory()
    with torch.cuda.stream(s):
        ctx.moments(t, 64, 64, 64, out=out_m, stream=s.cuda_stream)
        ctx.histogram(t, 64, 64, 64, 1024, -5.0, 5.0, bins=out_b, outside=out_o, stream=s.cuda_stream)
        ctx.median(t, 64, 64, 64, out=out_med, stream=s.cuda_stream)
    s.synchronize()
    m = cube.MomentsT.from_buffer_copy(out_m.cpu().numpy().tobytes()).as_dict()
    check_moments(m, oracle.moments(a), a)
    rb, ro = oracle.histogram(a, 1024, -5.0, 5.0)
    assert (out_b.cpu().numpy().astype(np.uint64) == rb).all() and (out_o.cpu().numpy().astype(np.uint64) == ro).all()
    assert same_float(out_med.numpy()[0], oracle.median(a))


def test_coarse_histogram_reuse(ctx):
    a = cubegen.generate_numpy(cubegen.scaled("c2", (64, 64, 256), nsrc=4)).reshape(-1)
    t = dev(a)
    m = ctx.moments(t, a.size, 1, 1, flags=cube.COARSE_HIST)
    check_moments(m, oracle.moments(a), a)
    assert same_float(ctx.median(t, a.size, 1, 1, flags=cube.REUSE_COARSE), oracle.median(a))
    m = ctx.moments(t, a.size, 1, 1, flags=cube.COARSE_HIST)
    k = m["count"] // 100
    assert same_float(ctx.kth(t, a.size, 1, 1, k, flags=cube.REUSE_COARSE), oracle.kth(a, k))


# ------------------------------------------------------------------------------------------------ configs
def _config_case(ctx, cfg, hists, extra_ks=()):
    nx, ny, nz = cfg["dims"]
    n = nx * ny * nz
    t = torch.empty(n, dtype=torch.float32, device="cuda")
    cubegen.generate_device(cfg, t.data_ptr())
    torch.cuda.synchronize()
    a = t.cpu().numpy()
    ref = oracle.moments(a)
    check_moments(ctx.moments(t, nx, ny, nz), ref, a)
    for nbins, lo, hi in hists:
        if lo is None:
            lo, hi = float(ref["min"]), float(ref["max"])
        b, o = ctx.histogram(t, nx, ny, nz, nbins, lo, hi)
        rb, ro = oracle.histogram(a, nbins, lo, hi)
        assert (b == rb).all() and (o == ro).all()
    med = ctx.median(t, nx, ny, nz)
    assert same_float(med, oracle.median(a))
    for nbins, lo, hi in hists:                                               # the fused two-read path
        m, b, o, smed = ctx.stats(t, nx, ny, nz, nbins, lo, hi)
        check_moments(m, ref, a)
        rb, ro = oracle.histogram(a, nbins, *((float(ref["min"]), float(ref["max"])) if lo is None else (lo, hi)))
        assert (b == rb).all() and (o == ro).all() and same_float(smed, med)
    less, equal = oracle.rank_counts(a, med)
    kmed = (ref["count"] - 1) // 2
    assert equal >= 1 and less <= kmed < less + equal
    for k in extra_ks:
        k = int(k(ref["count"]))
        assert same_float(ctx.kth(t, nx, ny, nz, k), oracle.kth(a, k))
    return a, ref


def test_config1_full(ctx):
    # BASELINE.json configs[0]: 256^3, seed 1; 1024 bins over [min,max]; exact lower median
    a, ref = _config_case(ctx, cubegen.CONFIGS["c1"], [(1024, None, None)])
    assert ref["nan_count"] == 0 and (ref["count"] - 1) // 2 == 8388607


def test_config2_scaled(ctx):
    _config_case(ctx, cubegen.scaled("c2", (256, 256, 1024)), [(4096, -0.02, 0.5)])


def test_config3_scaled(ctx):
    _config_case(ctx, cubegen.scaled("c3", (256, 256, 512)), [(65536, None, None)],
                 extra_ks=(lambda n: n // 100, lambda n: 99 * n // 100))


def test_config4_scaled(ctx):
    a, ref = _config_case(ctx, cubegen.scaled("c4", (512, 512, 64)), [(256, None, None), (65536, None, None)])
    assert ref["min"] == 0.0


def test_config5_scaled_out_of_core(ctx):
    # 8 bricks of 64^3 out of a 128^3 cube, streamed in brick order, vs the whole cube in-core and the oracle
    cfg = cubegen.scaled("c5", (128, 128, 128), nsrc=40)
    bricks = []
    for oz in (0, 64):
        for oy in (0, 64):
            for ox in (0, 64):
                t = torch.empty(64 ** 3, dtype=torch.float32, device="cuda")
                cubegen.generate_device(cfg, t.data_ptr(), origin=(ox, oy, oz), brick=(64, 64, 64))
                bricks.append(t)
    torch.cuda.synchronize()
    whole = torch.cat(bricks)
    a = whole.cpu().numpy()
    ctx.ooc_begin(4096, -0.02, 0.5, want_median=True)
    more = True
    sweeps = 0
    while more:
        for t in bricks:
            ctx.ooc_brick(t, t.numel())
        more = ctx.ooc_next_sweep()
        sweeps += 1
    assert sweeps == 2                      # the median's bucket fitted the candidate buffer: no third sweep
    m, b, o, med = ctx.ooc_result(4096)
    check_moments(m, oracle.moments(a), a)
    rb, ro = oracle.histogram(a, 4096, -0.02, 0.5)
    assert (b == rb).all() and (o == ro).all()
    assert same_float(med, oracle.median(a))
    # identical integers to the in-core path on the same voxels
    mi = ctx.moments(whole, a.size, 1, 1)
    assert (mi["count"], bits(mi["min"]), bits(mi["max"])) == (m["count"], bits(m["min"]), bits(m["max"]))
    assert abs(mi["mean"] - m["mean"]) <= REL * abs(m["mean"]) and abs(mi["std"] - m["std"]) <= REL * m["std"]
    assert same_float(ctx.median(whole, a.size, 1, 1), med)
    ms = ctx.ooc_result(4096, flags=cube.SAMPLE_STD)[0]
    check_moments(ms, oracle.moments(a, sample_std=True), a)


def test_candidate_buffer_overflow_falls_back_to_a_third_pass():
    # a 4 KiB candidate buffer cannot hold the median's bucket: pass 2 must stream the cube again (in-core)
    # and the brick-streamed path must ask for a third sweep -- same exact results either way
    small = cube.Context(scratch_bytes_hint=4096)
    try:
        cases = [cubegen.generate_numpy(cubegen.scaled("c2", (64, 64, 128), nsrc=3)).reshape(-1),
                 cubegen.generate_numpy(cubegen.scaled("c2", (128, 128, 128), nsrc=3)).reshape(-1),
                 np.full(300000, 0.25, np.float32),                       # every key in one bucket
                 cubegen.generate_numpy(cubegen.scaled("c4", (128, 128, 16))).reshape(-1)]
        for a in cases:
            t = dev(a, 1)
            assert same_float(small.median(t, a.size, 1, 1), oracle.median(a))
            cnt = int((~np.isnan(a)).sum())
            for k in (0, cnt // 3, cnt - 1):
                assert same_float(small.kth(t, a.size, 1, 1, k), oracle.kth(a, k))
            small.ooc_begin(0, 0.0, 0.0, want_median=True)
            sweeps, more = 0, True
            half = (a.size // 2) & ~3
            while more:
                small.ooc_brick(t[:half], half)
                small.ooc_brick(t[half:], a.size - half)
                more = small.ooc_next_sweep()
                sweeps += 1
            # the bucket = voxels sharing the top 13 bits of the median's order-preserving key; 3 sweeps iff it
            # does not fit the 1024-key buffer
            u = a[~np.isnan(a)].view(np.uint32)
            key = np.where(u >> 31 == 1, ~u, u | np.uint32(0x80000000))
            mu = np.array([oracle.median(a)], np.float32).view(np.uint32)
            mkey = np.where(mu >> 31 == 1, ~mu, mu | np.uint32(0x80000000))[0]
            bucket = int((key >> 19 == mkey >> 19).sum())
            assert sweeps == (3 if bucket > 1024 else 2), (sweeps, bucket)
            assert same_float(small.ooc_result(0)[3], oracle.median(a))
    finally:
        small.close()


def test_packed_histogram_counter_wraps(ctx):
    # > 65535 voxels in even bins, odd bins and adjacent (even, odd) pairs of the 16-bit packed layout
    r = np.random.default_rng(11)
    n = 1 << 21
    nb = 65536
    centres = np.array([0, 1, 2, 100, 101, 32767, 32768, 65534, 65535], dtype=np.int64)
    b = centres[r.integers(0, len(centres), n)]
    b[r.integers(0, n, n // 16)] = r.integers(0, nb, n // 16)               # plus a uniform floor
    a = ((b.astype(np.float64) + 0.5) / nb).astype(np.float32)             # lo=0, hi=1: exact bin centres
    t = dev(a)
    for nbins in (nb, nb - 1, 40001, 16385):
        got, go = ctx.histogram(t, n, 1, 1, nbins, 0.0, 1.0)
        rb, ro = oracle.histogram(a, nbins, 0.0, 1.0)
        assert (got == rb).all() and (go == ro).all()
    assert rb.max() > 3 * 65536


@pytest.mark.parametrize("nbins", [16, 256, 4096, 65536])
def test_histogram_underflow_below_lo(ctx, nbins):
    # (x - lo) * scale underflows to -0.0 for subnormal x just below lo = 0 when scale < 1: such voxels are
    # outside[0], not bin 0 (the fast functors place voxels by floor(v) without a range test)
    r = np.random.default_rng(nbins)
    n = 70001
    a = r.uniform(0.0, 1000.0, n).astype(np.float32)
    tiny = np.array([-1e-45, -3e-45, -1e-40, 1e-45, -0.0, 0.0], dtype=np.float32)
    a[r.integers(0, n, 600)] = tiny[r.integers(0, tiny.size, 600)]
    a[::501] = np.nan
    for misalign in (0, 1):
        t = dev(a, misalign)
        for lo, hi in ((0.0, 1000.0), (0.0, 1e6), (-1e-42, 4000.0)):
            b, o = ctx.histogram(t, n, 1, 1, nbins, lo, hi)
            rb, ro = oracle.histogram(a, nbins, lo, hi)
            assert (b == rb).all() and (o == ro).all(), (nbins, lo, hi, o, ro, b[:2], rb[:2])
            if nbins <= 16384:
                m, b2, o2, med = ctx.stats(t, n, 1, 1, nbins, lo, hi)
                assert (b2 == rb).all() and (o2 == ro).all()


@pytest.mark.parametrize("seed", range(10))
def test_moments_nan_patterns_switch_hot_and_safe_paths(ctx, seed):
    # the moments kernels run a NaN-blind hot path and a per-voxel safe path and switch per warp and tile (8192
    # voxels per CTA tile, 1024 per warp): NULL runs of every length and alignment, single NULL voxels at tile
    # edges, all-NULL stretches followed by data (late pivots), +-0 and constant stretches
    r = np.random.default_rng(5000 + seed)
    n = int(r.integers(200000, 1200000))
    a = (r.standard_normal(n) * 0.002 + 0.0007).astype(np.float32)
    for _ in range(int(r.integers(1, 40))):
        start = int(r.integers(0, n))
        length = int(r.choice([1, 2, 3, 4, 31, 32, 33, 1023, 1024, 1025, 8191, 8192, 8193, 50000]))
        if r.random() < 0.5:
            start = (start // 1024) * 1024 + int(r.choice([0, -1, 1, 4]))          # hug the warp-tile edges
        a[max(start, 0):start + length] = np.nan
    if seed % 3 == 0:
        a[:int(r.integers(1, n // 2))] = np.nan                                    # every thread starts without a pivot
    if seed % 4 == 1:
        a[r.integers(0, n, n // 200)] = np.nan                                     # scattered: warps stay on the safe path
    if seed % 5 == 2:
        a[n // 3:n // 3 + 70000] = np.float32(0.125)                               # constant stretch
    t = dev(a, seed % 4)
    ref = oracle.moments(a)
    check_moments(ctx.moments(t, n, 1, 1), ref, a)
    check_moments(ctx.moments(t, n, 1, 1, flags=cube.COARSE_HIST), ref, a)
    m, b, o, med = ctx.stats(t, n, 1, 1, 4096, -0.02, 0.5)
    check_moments(m, ref, a)
    rb, ro = oracle.histogram(a, 4096, -0.02, 0.5)
    assert (b == rb).all() and (o == ro).all() and same_float(med, oracle.median(a))
    k = ref["count"] // 3
    assert same_float(ctx.kth(t, n, 1, 1, k, flags=cube.REUSE_COARSE), oracle.kth(a, k))   # digit bins after the NaN repairs
    lo, hi = np.float32(ref["mean"] - ref["std"]), np.float32(ref["mean"] + 2 * ref["std"])
    got, want = ctx.clipped_moments(t, n, 1, 1, float(lo), float(hi)), oracle.clipped_moments(a, lo, hi)
    assert got["count"] == want["count"] and abs(got["mean"] - want["mean"]) <= REL * abs(want["mean"])
    # mini-map rows over the same voxels (hot / safe groups of 8 lines)
    nx, ny = 256, 64
    nz = n // (nx * ny)
    if nz >= 2:
        sub = a[:nx * ny * nz]
        mx, my, mz = ctx.minimap_dims(nx, ny, nz, 30, 30, 30)
        cells = torch.zeros(mx * my * mz * 40, dtype=torch.uint8, device="cuda")
        ts = dev(sub, 0)
        ctx.minimap(ts, nx, ny, nz, 30, 30, 30, cells)
        torch.cuda.synchronize()
        gotm = np.frombuffer(cells.cpu().numpy().tobytes(), dtype=cube.MINIMAP_DTYPE).reshape(mz, my, mx)
        refm = oracle.minimap(sub, (nx, ny, nz), (30, 30, 30))
        check_minimap_cells(gotm, refm)


@pytest.mark.parametrize("seed", range(16))
def test_selection_randomised_values_and_ranks(ctx, seed):
    # differential test of the radix select (three fused pass kernels, candidate compaction, bucket location in the
    # last CTA) on mixtures with heavy ties, both zeros, subnormals, +-Inf, NaN of both signs, at random ranks
    r = np.random.default_rng(7000 + seed)
    n = int(r.integers(1, 400000))
    kind = seed % 4
    if kind == 0:
        a = (r.standard_normal(n) * 10.0 ** r.uniform(-30, 30)).astype(np.float32)
    elif kind == 1:
        a = r.integers(-3, 4, n).astype(np.float32)                              # seven values
    elif kind == 2:
        a = np.exp(np.round(r.standard_normal(n) * 2, 1)).astype(np.float32) * np.float32(r.choice([1.0, -1.0]))
    else:
        a = (r.standard_normal(n) * 1e-41).astype(np.float32)                    # subnormals
    specials = np.array([0.0, -0.0, np.inf, -np.inf, np.nan, 1e-45, -1e-45, 3.4e38, -3.4e38], dtype=np.float32)
    idx = r.integers(0, n, n // 8 + 1)
    a[idx] = specials[r.integers(0, specials.size, idx.size)]
    a[r.integers(0, n, 3)] = np.frombuffer(np.uint32(0xFFC00001).tobytes(), dtype=np.float32)[0]
    t = dev(a, seed % 4)
    cnt = int((~np.isnan(a)).sum())
    assert same_float(ctx.median(t, n, 1, 1), oracle.median(a))
    ks = {0, max(cnt - 1, 0), cnt // 2, cnt // 100, int(r.integers(0, max(cnt, 1)))}
    for k in sorted(ks):
        if k < cnt:
            assert same_float(ctx.kth(t, n, 1, 1, k), oracle.kth(a, k)), (seed, k, cnt)
    assert math.isnan(float(ctx.kth(t, n, 1, 1, cnt)))                          # k >= count -> NaN
    m = ctx.moments(t, n, 1, 1, flags=cube.COARSE_HIST)
    assert m["count"] == cnt
    if cnt:
        k = int(r.integers(0, cnt))
        assert same_float(ctx.kth(t, n, 1, 1, k, flags=cube.REUSE_COARSE), oracle.kth(a, k))
    s_m, _, _, s_med = ctx.stats(t, n, 1, 1, 0)
    assert same_float(s_med, oracle.median(a)) and s_m["count"] == cnt


@pytest.mark.parametrize("seed", range(24))
def test_histogram_randomised_ranges_and_specials(ctx, seed):
    # differential test of every histogram path (general / fast / window / packed functors, cube_histogram and the
    # fused cube_stats pass B) on random ranges of every magnitude with the awkward values planted: the range ends
    # and their float neighbours, +-0, subnormals, +-Inf, NaN of both signs, values far outside
    r = np.random.default_rng(9000 + seed)
    nbins = int(r.choice([1, 2, 7, 8, 9, 255, 1000, 4096, 16384, 16385, 32768, 32769, 50000, 65536]))
    mag = 10.0 ** r.uniform(-42, 30) if seed % 3 else 10.0 ** r.uniform(-3, 3)
    lo = np.float32(r.uniform(-1, 1) * mag)
    width = np.float32(abs(r.standard_normal()) * mag * 10.0 ** r.uniform(-6, 2))
    hi = np.float32(lo + width) if seed % 7 else lo                      # hi == lo now and then (R13)
    if not np.isfinite(hi) or hi < lo:
        hi = lo
    n = int(r.integers(1000, 200000))
    centre, spread = (float(lo) + float(hi)) / 2, max(float(hi) - float(lo), abs(float(lo)) * 1e-6 + 1e-45)
    a = (centre + r.standard_normal(n) * spread * 10.0 ** r.uniform(-1.5, 0.5)).astype(np.float32)
    specials = np.array([lo, hi, np.nextafter(lo, np.float32(-np.inf)), np.nextafter(lo, np.float32(np.inf)),
                         np.nextafter(hi, np.float32(-np.inf)), np.nextafter(hi, np.float32(np.inf)),
                         0.0, -0.0, 1e-45, -1e-45, 1e-39, -1e-39, np.inf, -np.inf, np.nan, 3e38, -3e38],
                        dtype=np.float32)
    idx = r.integers(0, n, n // 10)
    a[idx] = specials[r.integers(0, specials.size, idx.size)]
    a[r.integers(0, n, 5)] = np.frombuffer(np.uint32(0xFFC00001).tobytes(), dtype=np.float32)[0]   # negative NaN
    t = dev(a, seed % 4)
    try:
        rb, ro = oracle.histogram(a, nbins, lo, hi)
    except ValueError:
        with pytest.raises(cube.CubeError):
            ctx.histogram(t, n, 1, 1, nbins, float(lo), float(hi))
        return
    b, o = ctx.histogram(t, n, 1, 1, nbins, float(lo), float(hi))
    assert (o == ro).all() and (b == rb).all(), (nbins, lo, hi, o, ro, np.nonzero(b != rb)[0][:5])
    m, b2, o2, med = ctx.stats(t, n, 1, 1, nbins, float(lo), float(hi))
    assert (o2 == ro).all() and (b2 == rb).all(), (nbins, lo, hi, o2, ro)
    fin = a[~np.isnan(a)]
    assert same_float(med, oracle.median(a)) and m["count"] == fin.size
    assert int(b.sum() + o.sum()) == fin.size


@pytest.mark.parametrize("knob", [0, 1, 2])
def test_big_histogram_variants(ctx, knob):
    # > 16384 bins: 0 = automatic (32-bit window of 32768 bins + global REDs, or 16-bit packed when the sampled
    # voxels do not fit a window), 1 = cluster DSM, 2 = always packed.  Same integers from all of them.
    r = np.random.default_rng(77)
    n = 700001
    noise_low = (r.standard_normal(n) * 0.002).astype(np.float32)
    noise_low[r.integers(0, n, n // 200)] = r.uniform(0.0, 0.9, n // 200).astype(np.float32)   # sparse sources
    noise_high = (0.8 + r.standard_normal(n) * 0.004).astype(np.float32)                       # window with w0 > 0
    noise_high[r.integers(0, n, n // 100)] = r.uniform(-0.1, 0.2, n // 100).astype(np.float32)
    uniform = r.uniform(-1.0, 1.0, n).astype(np.float32)                                        # no window fits
    mid = (r.standard_normal(n) * 0.05 + 0.47).astype(np.float32)                               # straddles bin 32768
    ctx.set_knob(cube.KNOB_BIGHIST, knob)
    try:
        for a in (noise_low, noise_high, uniform, mid):
            a = a.copy()
            a[::131] = np.nan
            t = dev(a, 1)
            lo, hi = float(np.nanmin(a)), float(np.nanmax(a))
            for nbins, (l, h) in ((65536, (lo, hi)), (65536, (-0.05, 0.95)), (40000, (lo, hi)), (16385, (0.0, 1.0)),
                                  (32768, (lo, hi)), (32769, (lo, hi))):
                b, o = ctx.histogram(t, a.size, 1, 1, nbins, l, h)
                rb, ro = oracle.histogram(a, nbins, l, h)
                assert (b == rb).all() and (o == ro).all(), (knob, nbins, l, h)
            m, b, o, med = ctx.stats(t, a.size, 1, 1, 65536)                # [min,max] resolved on the device
            rb, ro = oracle.histogram(a, 65536, lo, hi)
            assert (b == rb).all() and (o == ro).all() and same_float(med, oracle.median(a))
    finally:
        ctx.set_knob(cube.KNOB_BIGHIST, 0)


@pytest.mark.parametrize("resident", [False, True])
def test_stats_host_matches_oracle(ctx, resident):
    a = cubegen.generate_numpy(cubegen.scaled("c2", (96, 96, 200), nsrc=5)).reshape(-1)
    h = torch.from_numpy(a).pin_memory()
    ctx.host_workspace(resident_bytes=(a.nbytes + 4096) if resident else 0, chunk_bytes=1 << 20)
    m, b, o, med = ctx.stats_host(h, 96, 96, 200, 4096, -0.02, 0.5)
    check_moments(m, oracle.moments(a), a)
    rb, ro = oracle.histogram(a, 4096, -0.02, 0.5)
    assert (b == rb).all() and (o == ro).all()
    assert same_float(med, oracle.median(a))
    # histogram over [min, max] found by the first sweep (CUBE_RANGE_MINMAX), small and big bin counts, with and
    # without the median (without it the second sweep exists for the histogram alone)
    ref = oracle.moments(a)
    for nb in (1024, 65536):
        rb, ro = oracle.histogram(a, nb, float(ref["min"]), float(ref["max"]))
        for want_median in (True, False):
            m, b, o, med = ctx.stats_host(h, 96, 96, 200, nb, 0.0, 0.0, flags=cube.RANGE_MINMAX, want_median=want_median)
            check_moments(m, ref, a)
            assert (b == rb).all() and (o == ro).all() and int(b.sum()) == ref["count"]
            assert (not want_median) or same_float(med, oracle.median(a))
    ctx.host_workspace(0, 1 << 20)


@pytest.mark.parametrize("mode", ["gpu_fill", "cpu_fill", "resident_half", "ragged_last_brick"])
def test_stats_stream_brick_callback(ctx, mode):
    # config 5 scaled: 128^3 produced brick by brick (8 x 64^3) by a callback into pinned staging buffers;
    # same integers as the oracle on the concatenated bricks, exact median in two sweeps
    import ctypes
    cfg = cubegen.scaled("c5", (128, 128, 128), nsrc=40)
    brick = (64, 64, 64)
    bvox = 64 ** 3
    origins = cubegen.brick_grid(cfg, brick)
    scratch = torch.empty(bvox, dtype=torch.float32, device="cuda")
    host_bricks = []
    for org in origins:
        cubegen.generate_device(cfg, scratch.data_ptr(), origin=org, brick=brick)
        torch.cuda.synchronize()
        host_bricks.append(scratch.cpu().numpy().copy())
    a = np.concatenate(host_bricks)
    total = a.size
    nbricks = len(origins)
    if mode == "ragged_last_brick":                 # bricks of 100000 voxels over the same bytes, last one short
        bvox = 100000
        nbricks = (total + bvox - 1) // bvox
    calls = []

    def fill(b, sweep, h_dst, nvox, fs):
        calls.append((b, sweep, nvox))
        if mode == "gpu_fill":
            cubegen.generate_to_host(cfg, h_dst, scratch.data_ptr(), origin=origins[b], brick=brick, stream=fs)
        else:
            src = a[b * bvox: b * bvox + nvox]
            assert src.size == nvox
            ctypes.memmove(h_dst, src.ctypes.data, nvox * 4)
        return 0

    ctx.stream_workspace(bvox * 4, host_slots=3, resident_bytes=(4 * bvox * 4 if mode == "resident_half" else 0))
    m, b, o, med, info = ctx.stats_stream(nbricks, bvox, total, fill, 4096, -0.02, 0.5)
    check_moments(m, oracle.moments(a), a)
    rb, ro = oracle.histogram(a, 4096, -0.02, 0.5)
    assert (b == rb).all() and (o == ro).all()
    assert same_float(med, oracle.median(a))
    assert info["sweeps"] == 2
    moved = nbricks * 2 - (4 if mode == "resident_half" else 0)
    assert len(calls) == moved and info["h2d_bytes"] == (2 * total - (4 * bvox if mode == "resident_half" else 0)) * 4
    assert [c[0] for c in calls if c[1] == 0] == list(range(nbricks))
    # a failing callback aborts with CUBE_ECALLBACK and the context stays usable
    with pytest.raises(cube.CubeError) as e:
        ctx.stats_stream(nbricks, bvox, total, lambda *args: 7, 4096, -0.02, 0.5)
    assert e.value.code == cube.ECALLBACK
    with pytest.raises(ZeroDivisionError):
        ctx.stats_stream(nbricks, bvox, total, lambda *args: 1 // 0, 4096, -0.02, 0.5)
    m2, b2, o2, med2, _ = ctx.stats_stream(nbricks, bvox, total, fill, 4096, -0.02, 0.5, want_median=False)
    assert (b2 == rb).all() and m2["count"] == m["count"]
    ctx.host_workspace(0, 1 << 20)


def test_infinite_voxels_give_nan_mean_and_std_whatever_the_grid(ctx):
    # reading R8: count / min / max / selections stay exact, mean and std are NaN -- for one sign of infinity or both,
    # wherever the infinite voxels sit (first voxel of a thread, a whole tile, scattered), for every grid size, in
    # cube_moments, cube_stats, cube_clipped_moments (window holding an infinity) and the mini-map cells that hold one
    r = np.random.default_rng(77)
    base = (r.standard_normal(300001) * 0.002 + 0.001).astype(np.float32)
    variants = []
    a = base.copy(); a[0] = np.inf; variants.append(a)
    a = base.copy(); a[::4099] = np.inf; variants.append(a)
    a = base.copy(); a[5::1013] = np.inf; a[7::2027] = -np.inf; a[11::997] = np.nan; variants.append(a)
    a = base.copy(); a[:70000] = -np.inf; variants.append(a)                     # whole tiles of one infinity
    a = np.full(50000, np.inf, np.float32); variants.append(a)                   # nothing finite at all
    for a in variants:
        t = dev(a)
        ref = oracle.moments(a)
        assert np.isnan(ref["mean"]) and np.isnan(ref["std"])
        for per_sm in (0, 1, 3, 8):
            ctx.set_launch(per_sm)
            for got in (ctx.moments(t, a.size, 1, 1), ctx.stats(t, a.size, 1, 1, 0)[0]):
                assert got["count"] == ref["count"] and got["nan_count"] == ref["nan_count"]
                assert same_float(got["min"], ref["min"]) and same_float(got["max"], ref["max"])
                assert np.isnan(got["mean"]) and np.isnan(got["std"])
        ctx.set_launch(0)
        assert same_float(ctx.median(t, a.size, 1, 1), oracle.median(a))
        got, want = ctx.clipped_moments(t, a.size, 1, 1, 0.0, float("inf")), oracle.clipped_moments(a, 0.0, np.inf)
        assert got["count"] == want["count"] and same_float(got["max"], want["max"])
        assert np.isnan(got["mean"]) == np.isnan(want["mean"]) and np.isnan(got["std"]) == np.isnan(want["std"])
        got, want = ctx.clipped_moments(t, a.size, 1, 1, -1.0, 1.0), oracle.clipped_moments(a, -1.0, 1.0)   # infinities clipped away
        assert got["count"] == want["count"]
        if want["count"]:
            assert abs(got["mean"] - want["mean"]) <= REL * abs(want["mean"]) and abs(got["std"] - want["std"]) <= REL * want["std"]
    a = base[:256 * 64 * 18].copy()
    a[12345] = np.inf                 # two cells hold an infinity, the others none
    a[200000] = -np.inf
    a[11::997] = np.nan
    t = dev(a)
    mx, my, mz = ctx.minimap_dims(256, 64, 18, 30, 30, 30)
    for variant in (0, 1, 2, 3):
        ctx.set_knob(cube.KNOB_MINIMAP, variant)
        cells = torch.zeros(mx * my * mz * 40, dtype=torch.uint8, device="cuda")
        ctx.minimap(t, 256, 64, 18, 30, 30, 30, cells)
        torch.cuda.synchronize()
        gotm = np.frombuffer(cells.cpu().numpy().tobytes(), dtype=cube.MINIMAP_DTYPE).reshape(mz, my, mx)
        refm = oracle.minimap(a, (256, 64, 18), (30, 30, 30))
        assert (gotm["count"] == refm["count"]).all()
        assert (np.isnan(gotm["mean"]) == np.isnan(refm["mean"])).all() and (np.isnan(gotm["std"]) == np.isnan(refm["std"])).all()
        assert np.isnan(refm["mean"]).any() and not np.isnan(refm["mean"]).all()
        fin = ~np.isnan(refm["mean"])
        assert (np.abs(gotm["mean"][fin] - refm["mean"][fin]) <= REL * np.abs(refm["mean"][fin])).all()
    ctx.set_knob(cube.KNOB_MINIMAP, 0)


@pytest.mark.parametrize("frac_one_value", [1.0, 0.85])
def test_big_fused_pass_b_ragged_tile_with_a_dense_bucket(frac_one_value):
    # cube_stats with more than 16384 bins and the median (hist_win_select_kernel): a ragged last tile whose voxels
    # nearly all fall into the median's first-digit bucket.  n / 4 mod 8192 = 8166 float4, so the ragged tile gives a
    # warp up to 1024 keys between two fill checks -- more than its stage slice holds; single voxels therefore go
    # straight to the candidate buffer.  Constant cube, and a cube that is 85 % one value.
    n = 150 ** 3
    assert 5120 < (n // 4) % 8192 < 8192
    r = np.random.default_rng(3)
    a = np.full(n, 0.375, np.float32)
    if frac_one_value < 1.0:
        idx = r.random(n) > frac_one_value
        a[idx] = (0.375 + r.standard_normal(int(idx.sum())) * 0.01).astype(np.float32)
    t = dev(a)
    c = cube.Context(scratch_bytes_hint=64 << 20)
    try:
        for nb, lo, hi in ((65536, 0.0, 1.0), (40000, 0.3, 0.5)):
            m, b, o, med = c.stats(t, 150, 150, 150, nb, lo, hi)
            ref = oracle.moments(a)
            rb, ro = oracle.histogram(a, nb, lo, hi)
            check_moments(m, ref, a)
            assert (b == rb).all() and (o == ro).all() and same_float(med, oracle.median(a))
    finally:
        c.close()


@pytest.mark.parametrize("scratch", [0, 4096])
def test_single_launch_path_for_l2_resident_cubes(scratch):
    # cube_stats on a cube of at most 96 MiB with <= 4096 bins and the median is ONE cooperative launch
    # (csrc/cube_small.cuh): against the oracle, against the general three-launch path (CUBE_KNOB_SMALL = 1: identical
    # integers, mean / std within the tolerance), for several grid sizes; scratch = 4096 bytes makes the median's bucket
    # overflow the candidate buffer, so the last digit is counted over the cube by all CTAs (a fourth grid barrier)
    r = np.random.default_rng(41)
    noise = (r.standard_normal(700001) * 0.002 + 0.0003).astype(np.float32)
    noise[r.integers(0, noise.size, 9000)] = np.nan
    noise[r.integers(0, noise.size, 500)] *= 200
    ties = np.round(r.standard_normal(400003) * 2).astype(np.float32)
    cases = [noise, ties, np.full(150001, 0.25, np.float32), np.full(5000, np.nan, np.float32),
             np.array([3.5], np.float32), np.array([np.inf, -np.inf, 1.0, np.nan, 2.0], np.float32),
             np.tile(np.array([0.0, -0.0], np.float32), 70000)]
    c = cube.Context(scratch_bytes_hint=scratch)
    try:
        for a in cases:
            t = dev(a, 1)
            ref, omed = oracle.moments(a), oracle.median(a)
            for nb, lo, hi in ((4096, -0.02, 0.5), (64, None, None), (1, -1.0, 1.0), (7, 0.0, 0.001)):
                want = None
                if lo is not None:
                    want = oracle.histogram(a, nb, lo, hi)
                elif ref["count"] and np.isfinite(ref["min"]) and np.isfinite(ref["max"]):
                    want = oracle.histogram(a, nb, float(ref["min"]), float(ref["max"]))
                c.set_knob(cube.KNOB_SMALL, 1)
                l0 = c.launch_count
                gm, gb, go, gmed = c.stats(t, a.size, 1, 1, nb, lo, hi)
                assert c.launch_count - l0 >= 3
                c.set_knob(cube.KNOB_SMALL, 0)
                for per_sm in (0, 1, 3):
                    c.set_launch(per_sm)
                    l0 = c.launch_count
                    m, b, o, med = c.stats(t, a.size, 1, 1, nb, lo, hi, flags=0)
                    assert c.launch_count - l0 == 1                        # one launch
                    check_moments(m, ref, a)
                    assert same_float(med, omed) and same_float(med, gmed)
                    assert (b == gb).all() and (o == go).all()
                    if want is not None:
                        assert (b == want[0]).all() and (o == want[1]).all()
                    else:
                        assert not b.any() and (o == np.uint64(2 ** 64 - 1)).all()
                c.set_launch(0)
                # device-resident outputs are written by the kernel itself (no copy is enqueued)
                d_m = torch.zeros(40, dtype=torch.uint8, device="cuda")
                d_b = torch.full((nb,), -1, dtype=torch.int64, device="cuda")
                d_o = torch.full((2,), -1, dtype=torch.int64, device="cuda")
                d_f = torch.zeros(1, dtype=torch.float32, device="cuda")
                c.stats(t, a.size, 1, 1, nb, lo, hi, out=d_m, bins=d_b, outside=d_o, median=d_f)
                torch.cuda.synchronize()
                assert (d_b.cpu().numpy().astype(np.uint64) == gb).all() and (d_o.cpu().numpy().astype(np.uint64) == go).all()
                assert same_float(d_f.cpu()[0].item(), gmed)
                dm = cube.MomentsT.from_buffer_copy(d_m.cpu().numpy().tobytes()).as_dict()
                assert dm["count"] == ref["count"] and same_float(dm["min"], ref["min"]) and same_float(dm["max"], ref["max"])
                # the first-digit histogram is left in the context as by the general path
                k = ref["count"] // 3
                if ref["count"]:
                    assert same_float(c.kth(t, a.size, 1, 1, k, flags=cube.REUSE_COARSE), oracle.kth(a, k))
                ms = c.stats(t, a.size, 1, 1, nb, lo, hi, flags=cube.SAMPLE_STD)[0]
                check_moments(ms, oracle.moments(a, sample_std=True), a)
            # cube_median alone takes the same single launch, without the histogram; the three-launch path under the knob
            c.set_knob(cube.KNOB_SMALL, 1)
            l0 = c.launch_count
            gmed = c.median(t, a.size, 1, 1)
            assert c.launch_count - l0 >= 3 and same_float(gmed, omed)
            c.set_knob(cube.KNOB_SMALL, 0)
            for per_sm in (0, 1, 3):
                c.set_launch(per_sm)
                l0 = c.launch_count
                assert same_float(c.median(t, a.size, 1, 1), omed)
                assert c.launch_count - l0 == 1
                d_f = torch.full((1,), 7.0, dtype=torch.float32, device="cuda")
                c.median(t, a.size, 1, 1, out=d_f)
                torch.cuda.synchronize()
                assert same_float(d_f.cpu()[0].item(), omed)
            c.set_launch(0)
            # cube_kth takes the same launch with the rank it is given: first, last, a middle one, one beyond the count
            for kk in sorted({0, ref["count"] // 7, max(ref["count"] - 1, 0), ref["count"], ref["count"] + 5}):
                want = oracle.kth(a, kk) if kk < ref["count"] else np.float32(np.nan)
                l0 = c.launch_count
                assert same_float(c.kth(t, a.size, 1, 1, kk), want)
                assert c.launch_count - l0 == 1
            # and the state it leaves serves a later selection on the same cube
            if ref["count"]:
                assert same_float(c.kth(t, a.size, 1, 1, ref["count"] // 5, flags=cube.REUSE_COARSE), oracle.kth(a, ref["count"] // 5))
    finally:
        c.close()
