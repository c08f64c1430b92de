"""The calls of the hot path can be recorded into a CUDA graph and replayed (every decision between
the passes is taken on the device, no call synchronises or allocates once the context exists): cube_stats -- the single
cooperative launch of an L2-resident cube and the general three-launch path --, cube_median and cube_histogram_noalloc
are captured on a stream with device-resident outputs, the input buffer is then overwritten with other cubes and the
graph replayed: every replay must give the oracle's results for the data it found."""
import numpy as np
import pytest
import torch

import oracle
import paper_1211_4896_b200 as cube

pytestmark = pytest.mark.gpu


def moments_of(buf):
    return cube.MomentsT.from_buffer_copy(buf.cpu().numpy().tobytes()).as_dict()


@pytest.mark.parametrize("general_path", [False, True])
def test_cube_stats_replays_from_a_cuda_graph(general_path):
    assert torch.cuda.is_available(), "gpu tests need a CUDA device (there is no CPU fallback)"
    n, nb, lo, hi = 300007, 512, -0.01, 0.02
    r = np.random.default_rng(5)
    cubes = [(r.standard_normal(n) * s + m).astype(np.float32) for s, m in ((0.002, 0.0003), (0.01, -0.004), (0.0005, 0.015))]
    cubes[1][r.integers(0, n, 3000)] = np.nan
    cubes[2][::7] = 0.0
    ctx = cube.Context()
    try:
        ctx.set_knob(cube.KNOB_SMALL, 1 if general_path else 0)
        t = torch.from_numpy(cubes[0]).cuda()
        d_m = torch.zeros(40, dtype=torch.uint8, device="cuda")
        d_b = torch.zeros(nb, dtype=torch.int64, device="cuda")
        d_o = torch.zeros(2, dtype=torch.int64, device="cuda")
        d_f = torch.zeros(1, dtype=torch.float32, device="cuda")
        d_f2 = torch.zeros(1, dtype=torch.float32, device="cuda")
        d_nb = torch.zeros(nb, dtype=torch.int64, device="cuda")
        d_no = torch.zeros(2, dtype=torch.int64, device="cuda")
        side = torch.cuda.Stream()
        # one eager call first (occupancy queries are cached, the allocation-free entry point resolves its scratch)
        ctx.stats(t, n, 1, 1, nb, lo, hi, out=d_m, bins=d_b, outside=d_o, median=d_f, stream=side.cuda_stream)
        ctx.median(t, n, 1, 1, out=d_f2, stream=side.cuda_stream)
        cube.histogram_noalloc(t, n, 1, 1, nb, lo, hi, bins=d_nb, outside=d_no, stream=side.cuda_stream)
        side.synchronize()
        g = torch.cuda.CUDAGraph()
        with torch.cuda.graph(g, stream=side):
            s = torch.cuda.current_stream().cuda_stream
            ctx.stats(t, n, 1, 1, nb, lo, hi, out=d_m, bins=d_b, outside=d_o, median=d_f, stream=s)
            ctx.median(t, n, 1, 1, out=d_f2, stream=s)
            cube.histogram_noalloc(t, n, 1, 1, nb, lo, hi, bins=d_nb, outside=d_no, stream=s)
        for a in (cubes[1], cubes[2], cubes[0], cubes[2]):
            t.copy_(torch.from_numpy(a))
            for buf in (d_m, d_b, d_o, d_f, d_f2, d_nb, d_no):
                buf.zero_()
            torch.cuda.synchronize()
            g.replay()
            torch.cuda.synchronize()
            ref, (rb, ro), rmed = oracle.moments(a), oracle.histogram(a, nb, lo, hi), oracle.median(a)
            m = moments_of(d_m)
            assert m["count"] == ref["count"] and m["nan_count"] == ref["nan_count"]
            assert np.float32(m["min"]).tobytes() == np.float32(ref["min"]).tobytes()
            assert abs(m["mean"] - ref["mean"]) <= 1e-9 * max(abs(ref["mean"]), 1e-6 * float(np.nanmax(np.abs(a))))
            assert abs(m["std"] - ref["std"]) <= 1e-9 * ref["std"]
            assert (d_b.cpu().numpy().astype(np.uint64) == rb).all() and (d_o.cpu().numpy().astype(np.uint64) == ro).all()
            assert (d_nb.cpu().numpy().astype(np.uint64) == rb).all() and (d_no.cpu().numpy().astype(np.uint64) == ro).all()
            assert np.float32(d_f.item()).tobytes() == np.float32(rmed).tobytes()
            assert np.float32(d_f2.item()).tobytes() == np.float32(rmed).tobytes()
    finally:
        ctx.close()


def test_single_operations_replay_from_a_cuda_graph():
    # cube_moments, cube_histogram with 65536 bins (the window / packed kernels and their device-side plan), cube_kth and
    # cube_kth_multi: captured once, replayed on other data
    n, nb = 262144 + 77, 65536
    r = np.random.default_rng(6)
    cubes = [(r.standard_normal(n) * s + m).astype(np.float32) for s, m in ((0.002, 0.0003), (0.3, 2.0), (0.0005, -0.015))]
    cubes[2][r.integers(0, n, 2000)] = np.nan
    lo, hi = -0.02, 3.0
    ks = [n // 100, n // 2, n - n // 50]
    ctx = cube.Context()
    try:
        t = torch.from_numpy(cubes[0]).cuda()
        d_m = torch.zeros(40, dtype=torch.uint8, device="cuda")
        d_b = torch.zeros(nb, dtype=torch.int64, device="cuda")
        d_o = torch.zeros(2, dtype=torch.int64, device="cuda")
        d_k = torch.zeros(1, dtype=torch.float32, device="cuda")
        d_ks = torch.zeros(len(ks), dtype=torch.float32, device="cuda")
        side = torch.cuda.Stream()

        def calls(s):
            ctx.moments(t, n, 1, 1, out=d_m, stream=s)
            ctx.histogram(t, n, 1, 1, nb, lo, hi, bins=d_b, outside=d_o, stream=s)
            ctx.kth(t, n, 1, 1, ks[0], out=d_k, stream=s)
            ctx.kth_multi(t, n, 1, 1, ks, out=d_ks, stream=s)

        calls(side.cuda_stream)
        side.synchronize()
        g = torch.cuda.CUDAGraph()
        with torch.cuda.graph(g, stream=side):
            calls(torch.cuda.current_stream().cuda_stream)
        for a in (cubes[1], cubes[2], cubes[0]):
            t.copy_(torch.from_numpy(a))
            for buf in (d_m, d_b, d_o, d_k, d_ks):
                buf.zero_()
            torch.cuda.synchronize()
            g.replay()
            torch.cuda.synchronize()
            ref, (rb, ro) = oracle.moments(a), oracle.histogram(a, nb, lo, hi)
            m = moments_of(d_m)
            assert m["count"] == ref["count"] and np.float32(m["max"]).tobytes() == np.float32(ref["max"]).tobytes()
            assert abs(m["std"] - ref["std"]) <= 1e-9 * ref["std"]
            assert (d_b.cpu().numpy().astype(np.uint64) == rb).all() and (d_o.cpu().numpy().astype(np.uint64) == ro).all()
            cnt = ref["count"]
            want = [oracle.kth(a, k) if k < cnt else np.float32(np.nan) for k in ks]
            got = d_ks.cpu().numpy()
            assert all(np.float32(x).tobytes() == np.float32(y).tobytes() or (np.isnan(x) and np.isnan(y)) for x, y in zip(got, want))
            assert np.float32(d_k.item()).tobytes() == np.float32(want[0]).tobytes()
    finally:
        ctx.close()
