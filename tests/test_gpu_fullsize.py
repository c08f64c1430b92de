"""GPU parity at BASELINE.json's FULL sizes, all five configs, in the launch configuration bench.py times (same
context sizing, cube_stats with device-resident outputs on torch's current stream, default grid).

config 1 / config 2 (64 MiB / 4 GiB): the oracle computes everything on the identical bytes in one piece
(moments, histogram, nth_element median and k-th); config 2 also carries the NEXT rows at bench size (MAD, sigma
clipping, 30^3 mini-map, Alg. 1).
configs 3, 4 (64 / 32 GiB) and 5 (256 GiB, out of core): the single-threaded oracle runs CHUNK BY CHUNK on the same
bytes, several chunks at a time in a thread pool (SURVEY.md sec. 8(c) "oracle at scale"; each oracle call stays
single-threaded and sees a contiguous run of the cube's voxels):
  * count / nan_count / bins / outside : exact sums of the per-chunk oracle results; min / max their extrema;
  * mean / std : the exact regrouping of the per-chunk (count, mean, std) in rational arithmetic -- the definition of
    the population variance regrouped by chunk, nothing else;
  * median / k-th : the rank certificate  #{x<m} <= k < #{x<m} + #{x==m},  #{x==m} >= 1  summed over the chunks, which
    is necessary and sufficient and independent of both selection algorithms (oracle.rank_counts).
The histogram range of configs 3 and 4 is [min, max]: the chunks are binned over the extrema the GPU reported, and
those are then required to equal the oracle's extrema bit for bit, so the range is the oracle's own.

CUBE_SKIP_FULLSIZE=1 skips the three big configs (quick local iterations only; the default run includes them).
"""
import gc
import math
import os
import threading
from concurrent.futures import ThreadPoolExecutor
from fractions import Fraction

import numpy as np
import pytest
import torch

import cubegen
import oracle
import paper_1211_4896_b200 as cube

pytestmark = pytest.mark.gpu

REL = 1e-9
SKIP_BIG = os.environ.get("CUBE_SKIP_FULLSIZE", "0") == "1"
big = pytest.mark.skipif(SKIP_BIG, reason="CUBE_SKIP_FULLSIZE=1")
CHUNK = 1 << 27                      # voxels per oracle call on the in-HBM cubes (512 MiB)


def bits(x):
    return int(np.float32(x).view(np.uint32))


def bench_like_context(n):
    # bench.py: candidate buffer = 1/16 of the cube, at least 256 MiB
    return cube.Context(scratch_bytes_hint=max(256 << 20, n * 4 // 16))


def device_results(ctx, t, dims, nb, lo, hi):
    """One cube_stats call exactly as bench.py's step issues it (device outputs, current stream)."""
    nx, ny, nz = dims
    out_m = torch.zeros(40, dtype=torch.uint8, device="cuda")
    out_b = torch.zeros(nb, dtype=torch.int64, device="cuda")
    out_o = torch.zeros(2, dtype=torch.int64, device="cuda")
    out_f = torch.zeros(1, dtype=torch.float32, device="cuda")
    stream = torch.cuda.current_stream().cuda_stream
    ctx.stats(t, nx, ny, nz, nb, lo, hi, out=out_m, bins=out_b, outside=out_o, median=out_f, stream=stream)
    torch.cuda.synchronize()
    m = cube.MomentsT.from_buffer_copy(out_m.cpu().numpy().tobytes()).as_dict()
    return m, out_b.cpu().numpy().astype(np.uint64), out_o.cpu().numpy().astype(np.uint64), np.float32(out_f.cpu()[0])


def check_moments(got, ref):
    assert got["count"] == ref["count"] and got["nan_count"] == ref["nan_count"]
    assert bits(got["min"]) == bits(ref["min"]) and bits(got["max"]) == bits(ref["max"])
    assert abs(got["mean"] - ref["mean"]) <= REL * abs(ref["mean"]), (got, ref)
    assert abs(got["std"] - ref["std"]) <= REL * ref["std"], (got, ref)


def certify(a, value, k):
    less, equal = oracle.rank_counts(a, value)
    assert equal >= 1 and less <= k < less + equal, (float(value), k, less, equal)


def generate(name):
    cfg = cubegen.CONFIGS[name]
    nx, ny, nz = cfg["dims"]
    gc.collect()
    torch.cuda.empty_cache()
    t = torch.empty(nx * ny * nz, dtype=torch.float32, device="cuda")
    cubegen.generate_device(cfg, t.data_ptr())
    torch.cuda.synchronize()
    return cfg, t


def workers():
    return max(1, min(14, (os.cpu_count() or 2) - 2))


# ------------------------------------------------------------------------------------------------ oracle by chunks
def oracle_by_chunks(chunks, fn):
    """chunks: iterator of device tensors (contiguous runs of the cube, in order); fn(host float32 array) -> result.
    Every chunk goes device -> pinned host buffer -> one single-threaded oracle call in a pool thread; at most
    workers() + 2 chunks are on the host at any time.  -> list of results in chunk order."""
    nw = workers()
    free, cond, ring = [], threading.Condition(), {}

    def run(a, key):
        try:
            return fn(a)
        finally:
            with cond:
                free.append(key)
                cond.notify()

    futs = []
    with ThreadPoolExecutor(nw) as pool:
        for ch in chunks:
            n = ch.numel()
            with cond:
                key = next((k for k in free if ring[k].numel() >= n), None)
                while key is None and len(ring) >= nw + 2:
                    cond.wait()
                    key = next((k for k in free if ring[k].numel() >= n), None)
                if key is None:
                    key = len(ring)
                    ring[key] = torch.empty(n, dtype=torch.float32, pin_memory=True)
                else:
                    free.remove(key)
            h = ring[key][:n]
            h.copy_(ch, non_blocking=True)
            torch.cuda.synchronize()
            futs.append(pool.submit(run, h.numpy(), key))
        return [f.result() for f in futs]


def merge_chunk_moments(parts):
    """Whole-cube (count, mean, population std) from the oracle's per-chunk records, in exact rational arithmetic
    (a double is a dyadic rational): mean = sum n_i mean_i / n, M2 = sum M2_i + sum n_i (mean_i - mean)^2 with
    M2_i = n_i std_i^2 (the definition of the population variance regrouped by chunk, nothing else)."""
    n = sum(p["count"] for p in parts)
    mean = sum(Fraction(p["mean"]) * p["count"] for p in parts if p["count"]) / n
    m2 = sum(Fraction(p["std"]) ** 2 * p["count"] + (Fraction(p["mean"]) - mean) ** 2 * p["count"]
             for p in parts if p["count"])
    return n, float(mean), math.sqrt(float(m2 / n))


def total_order_key(v):
    return (float(v), not math.copysign(1.0, float(v)) < 0)


def merged_reference(parts):
    """parts: per-chunk oracle.moments records -> the whole cube's record."""
    count, mean, std = merge_chunk_moments(parts)
    live = [r for r in parts if r["count"]]
    return dict(count=count, nan_count=sum(r["nan_count"] for r in parts), mean=mean, std=std,
                min=min((r["min"] for r in live), key=total_order_key),
                max=max((r["max"] for r in live), key=total_order_key))


# ------------------------------------------------------------------------------------------------ configs 1, 2
def test_config1_full_size():
    # BASELINE.json configs[0]: 256^3, seed 1, 1024 bins over [min,max] (the single-launch path of cube_stats)
    cfg, t = generate("c1")
    dims = cfg["dims"]
    a = t.cpu().numpy()
    ctx = bench_like_context(t.numel())
    try:
        ref = oracle.moments(a)
        assert ref["nan_count"] == 0 and ref["count"] == 256 ** 3
        m, b, o, med = device_results(ctx, t, dims, 1024, None, None)
        check_moments(m, ref)
        rb, ro = oracle.histogram(a, 1024, float(ref["min"]), float(ref["max"]))
        assert (b == rb).all() and (o == ro).all() and int(b.sum()) == ref["count"]
        assert bits(med) == bits(oracle.median(a)) and (ref["count"] - 1) // 2 == 8388607
        check_moments(ctx.moments(t, *dims), ref)
        assert bits(ctx.median(t, *dims)) == bits(med)
    finally:
        ctx.close()


def test_config2_full_size():
    # BASELINE.json configs[1]: 1024^3, seed 2, 4096 bins over [-0.02, 0.5]
    cfg, t = generate("c2")
    dims = cfg["dims"]
    n = t.numel()
    a = t.cpu().numpy()
    ctx = bench_like_context(n)
    try:
        # the oracle's NEXT rows at this size take a minute each: run them beside the main checks
        pool = ThreadPoolExecutor(5)
        f_mad = pool.submit(oracle.mad, a)
        f_clip = pool.submit(oracle.sigma_clip, a, 3.0, 5)
        f_map = pool.submit(oracle.minimap, a, dims, (30, 30, 30))
        f_torben = pool.submit(oracle.torben_capped, a, 20)
        f_mapmed = pool.submit(oracle.minimap_median, a, dims, (30, 30, 30))
        ref = oracle.moments(a)
        assert ref["nan_count"] > 0 and ref["nan_count"] % (dims[0] * dims[1]) == 0      # whole blanked planes
        rb, ro = oracle.histogram(a, 4096, -0.02, 0.5)
        assert int(ro[1]) > 0                                                            # sources above hi
        omed = oracle.median(a)
        m, b, o, med = device_results(ctx, t, dims, 4096, -0.02, 0.5)                    # the fused two-read step
        check_moments(m, ref)
        assert (b == rb).all() and (o == ro).all() and bits(med) == bits(omed)
        # the three entry points on their own
        check_moments(ctx.moments(t, *dims), ref)
        b2, o2 = ctx.histogram(t, *dims, 4096, -0.02, 0.5)
        assert (b2 == rb).all() and (o2 == ro).all()
        assert bits(ctx.median(t, *dims)) == bits(omed)
        k = ref["count"] // 100
        assert bits(ctx.kth(t, *dims, k)) == bits(oracle.kth(a, k))
        certify(a, med, (ref["count"] - 1) // 2)
        # the three ranks bench.py asks cube_kth_multi for (two reads of the cube), and a second group of ranks
        ks = [(ref["count"] - 1) // 2, k, 99 * ref["count"] // 100, 0, ref["count"] - 1, ref["count"]]
        got = ctx.kth_multi(t, *dims, ks)
        assert bits(got[0]) == bits(omed) and bits(got[1]) == bits(oracle.kth(a, k))
        for kk, g in zip(ks[2:5], got[2:5]):
            certify(a, g, kk)
        assert np.isnan(got[5])
        # NEXT rows at bench size: MAD, sigma clipping, mini-map, Alg. 1 stopped at 20 passes
        gmed, gmad = ctx.mad(t, *dims)
        rmed, rmad = f_mad.result()
        assert bits(gmed) == bits(rmed) == bits(omed) and bits(gmad) == bits(rmad)
        cm, cit, cwin = ctx.sigma_clip(t, *dims, 3.0, 5)
        rm, rit, rwin = f_clip.result()
        assert cit == rit and bits(cwin[0]) == bits(rwin[0]) and bits(cwin[1]) == bits(rwin[1])
        check_moments(cm, rm)
        tv, tit, tconv = ctx.median_torben(t, *dims, 20)
        rv, rit2, rconv = f_torben.result()
        assert (float(tv) == float(rv)) and tit == rit2 and tconv == rconv
        mx, my, mz = ctx.minimap_dims(*dims, 30, 30, 30)
        cells = torch.zeros(mx * my * mz * 40, dtype=torch.uint8, device="cuda")
        ctx.minimap(t, *dims, 30, 30, 30, cells)
        torch.cuda.synchronize()
        gmap = np.frombuffer(cells.cpu().numpy().tobytes(), dtype=cube.MINIMAP_DTYPE).reshape(mz, my, mx)
        check_minimap(gmap, f_map.result())
        gmed = torch.zeros(mx * my * mz, dtype=torch.float32, device="cuda")
        ctx.minimap_median(t, *dims, 30, 30, 30, gmed)
        torch.cuda.synchronize()
        gm, rmm = gmed.cpu().numpy().reshape(mz, my, mx), f_mapmed.result()
        assert ((gm.view(np.uint32) == rmm.view(np.uint32)) | (np.isnan(gm) & np.isnan(rmm))).all()
        # NEXT-4 through the full cube: a small image (64 x 48 rays of ~1775 samples) and two profiles, bit for bit
        view = cubegen.view_orbit(dims, 30.0, 20.0, 64, 48, step=1.0)
        img = torch.zeros(64 * 48, dtype=torch.float32, device="cuda")
        ctx.render_mip(t, *dims, view, img)
        tab = np.linspace(0.0, 1.0, 64, dtype=np.float32)[:, None] * np.array([1.0, 0.5, 0.25, 0.05], dtype=np.float32)
        rgba = torch.zeros(64 * 48 * 4, dtype=torch.float32, device="cuda")
        ctx.render_tf(t, *dims, view, tab, 0.004, 0.1, rgba, opacity_cut=0.98)
        prof = torch.zeros(view["nsteps"], dtype=torch.float32, device="cuda")
        ctx.spectrum(t, *dims, view, 31, 25, prof)
        torch.cuda.synchronize()
        for got_a, ref_a in ((img.cpu().numpy().reshape(48, 64), oracle.render_mip(a, dims, view)),
                             (rgba.cpu().numpy().reshape(48, 64, 4), oracle.render_tf(a, dims, view, tab, 0.004, 0.1, 0.98)),
                             (prof.cpu().numpy(), oracle.spectrum(a, dims, view, 31, 25))):
            assert ((got_a.view(np.uint32) == ref_a.view(np.uint32)) | (np.isnan(got_a) & np.isnan(ref_a))).all()
        # the sigma-clipping transfer function on the oracle's 30^3 mini-map (uploaded, so both sides read the same
        # records): 3-sigma threshold, bit for bit
        ref_cells = f_map.result()
        cells_o = torch.frombuffer(bytearray(np.ascontiguousarray(ref_cells, dtype=cube.MINIMAP_DTYPE).tobytes()),
                                   dtype=torch.uint8).cuda()
        sig = torch.zeros(64 * 48 * 4, dtype=torch.float32, device="cuda")
        ctx.render_sigma(t, *dims, view, cells_o, 30, 30, 30, tab, 3.0, 12.0, sig, opacity_cut=0.98)
        torch.cuda.synchronize()
        got_s = sig.cpu().numpy().reshape(48, 64, 4)
        assert (got_s.view(np.uint32) == oracle.render_sigma(a, dims, view, ref_cells, (30, 30, 30), tab, 3.0, 12.0, 0.98)
                .view(np.uint32)).all()
        assert (got_s[..., 3] > 0).any()
        pool.shutdown()
    finally:
        ctx.close()


def check_minimap(got, ref):
    """Every cell: count / nan_count / min / max exact (NaN == NaN), mean and std within REL (with the floor of
    DESIGN.md R16 for cells whose mean or std is ~0)."""
    assert got.shape == ref.shape
    assert (got["count"] == ref["count"]).all() and (got["nan_count"] == ref["nan_count"]).all()
    for f in ("min", "max"):
        g, r = np.ascontiguousarray(got[f]), np.ascontiguousarray(ref[f])
        assert ((g.view(np.uint32) == r.view(np.uint32)) | (np.isnan(g) & np.isnan(r))).all()
    live = ref["count"] > 0
    mext = np.maximum(np.abs(ref["min"][live].astype(np.float64)), np.abs(ref["max"][live].astype(np.float64)))
    assert (np.abs(got["mean"][live] - ref["mean"][live]) <= REL * np.maximum(np.abs(ref["mean"][live]), 1e-6 * mext)).all()
    assert (np.abs(got["std"][live] - ref["std"][live]) <= REL * np.maximum(ref["std"][live], 1e-6 * mext)).all()
    assert np.isnan(got["mean"][~live]).all() and np.isnan(got["std"][~live]).all()


# ------------------------------------------------------------------------------------------------ configs 3, 4
def _big_config(name, hists, ks):
    cfg, t = generate(name)
    dims = cfg["dims"]
    n = t.numel()
    ctx = bench_like_context(n)
    try:
        gpu = [device_results(ctx, t, dims, nb, None, None) for nb in hists]            # histogram over [min,max]
        m0, _, _, med0 = gpu[0]
        count = m0["count"]
        kmed = (count - 1) // 2
        kk = [int(kf(count)) for kf in ks]
        assert bits(ctx.median(t, *dims)) == bits(med0)
        singles = [ctx.kth(t, *dims, k) for k in kk]
        # the same ranks and the median through cube_kth_multi (two reads): bit-identical to the single selections
        multi = ctx.kth_multi(t, *dims, [kmed] + kk)
        assert [bits(g) for g in multi] == [bits(med0)] + [bits(v) for v in singles]
        claimed = [np.float32(med0)] + [np.float32(v) for v in singles]
        lo, hi = float(m0["min"]), float(m0["max"])

        def one(a):
            return (oracle.moments(a), [oracle.histogram(a, nb, lo, hi) for nb in hists],
                    [oracle.rank_counts(a, v) for v in claimed])

        parts = oracle_by_chunks((t[o:o + CHUNK] for o in range(0, n, CHUNK)), one)
        ref = merged_reference([p[0] for p in parts])
        assert bits(ref["min"]) == bits(m0["min"]) and bits(ref["max"]) == bits(m0["max"])   # the range was the oracle's
        for i, nb in enumerate(hists):
            m, b, o, med = gpu[i]
            check_moments(m, ref)
            rb = sum(p[1][i][0].astype(np.uint64) for p in parts)
            ro = sum(p[1][i][1].astype(np.uint64) for p in parts)
            assert (b == rb).all() and (o == ro).all() and int(b.sum()) == ref["count"]
            assert bits(med) == bits(med0)
        for j, k in enumerate([kmed] + kk):                                               # rank certificates
            less = sum(p[2][j][0] for p in parts)
            equal = sum(p[2][j][1] for p in parts)
            assert equal >= 1 and less <= k < less + equal, (float(claimed[j]), k, less, equal)
        return ref
    finally:
        ctx.close()
        del t
        gc.collect()
        torch.cuda.empty_cache()


@big
def test_config3_full_size():
    ref = _big_config("c3", [65536], [lambda c: c // 100, lambda c: 99 * c // 100])
    assert 0.004 < ref["nan_count"] / (ref["count"] + ref["nan_count"]) < 0.006


@big
def test_config4_full_size():
    # rank 0 is one of the 30 % of voxels that are exactly +0.0: its first-digit bucket cannot fit the candidate
    # buffer, so cube_kth_multi's group falls back, on the device, to the per-rank selections -- at full size
    ref = _big_config("c4", [256, 65536], [lambda c: 0])
    assert bits(ref["min"]) == 0 and (ref["count"] - 1) // 2 == 2 ** 32 - 1


# ------------------------------------------------------------------------------------------------ config 5
@big
def test_config5_full_size():
    """BASELINE.json configs[4] at full size, through the call bench.py times for c5 (cube_stats_stream, 512 bricks
    of 512^3 produced by a callback, 128 GiB kept in HBM after sweep 1).  The oracle cannot hold 256 GiB, so it runs
    brick by brick on the SAME bytes (each brick regenerated by the same device generator)."""
    cfg = cubegen.CONFIGS["c5"]
    nx, ny, nz = cfg["dims"]
    n = nx * ny * nz
    brick = (512, 512, 512)
    bvox = 512 ** 3
    origins = cubegen.brick_grid(cfg, brick)
    assert len(origins) == 512 and n == 512 * bvox
    nb, lo, hi = 4096, -0.02, 0.5
    gc.collect()
    torch.cuda.empty_cache()          # the 64 / 32 GiB cubes of the tests before this one: libcube allocates with cudaMalloc
    scr = torch.empty(bvox, dtype=torch.float32, device="cuda")
    ctx = cube.Context(scratch_bytes_hint=1 << 30)
    try:
        ctx.stream_workspace(bvox * 4, host_slots=4, resident_bytes=256 * bvox * 4)

        def fill(b, sweep, h_dst, nvox, fs):
            cubegen.generate_to_host(cfg, h_dst, scr.data_ptr(), origin=origins[b], brick=brick, stream=fs)
            return 0

        m, bins, outside, med, info = ctx.stats_stream(len(origins), bvox, n, fill, nb, lo, hi)
        assert info["sweeps"] == 2
    finally:
        ctx.close()
    medv = np.float32(med)

    def oracle_brick(a):
        hb, ho = oracle.histogram(a, nb, lo, hi)
        return oracle.moments(a), hb.astype(np.uint64), ho.astype(np.uint64), oracle.rank_counts(a, medv)

    scr2 = [torch.empty(bvox, dtype=torch.float32, device="cuda") for _ in range(2)]

    def bricks():
        for i, org in enumerate(origins):
            cubegen.generate_device(cfg, scr2[i & 1].data_ptr(), origin=org, brick=brick)
            yield scr2[i & 1]

    parts = oracle_by_chunks(bricks(), oracle_brick)
    ref = merged_reference([p[0] for p in parts])
    assert ref["nan_count"] == n - ref["count"]
    check_moments(m, ref)
    rb = sum(p[1] for p in parts)
    ro = sum(p[2] for p in parts)
    assert (bins == rb).all() and (outside == ro).all()
    assert int(rb.sum()) + int(ro.sum()) == ref["count"] and int(ro[1]) > 0
    less = sum(p[3][0] for p in parts)
    equal = sum(p[3][1] for p in parts)
    k = (ref["count"] - 1) // 2
    assert equal >= 1 and less <= k < less + equal, (float(medv), k, less, equal)
