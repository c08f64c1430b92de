"""GPU parity for the z-slab sharded path: one cube split into slabs, one libcube
context per slab, the per-rank buffers combined exactly as shard.run() combines them -- here in ONE process, the
"ranks" taken in lock step on one stream (nothing waits on anything: every rank's kernels simply follow the previous
rank's), because the box has a single GPU.  Results: bit-exact against the oracle on the WHOLE cube, identical on
every rank.  Also shard.run() itself with NCCL (world size 1) to exercise the aliasing of libcube's device buffers
by torch.distributed.
"""
import math
import os
import socket

import numpy as np
import pytest
import torch

import cubegen
import oracle
import paper_1211_4896_b200 as cube
from paper_1211_4896_b200 import shard

pytestmark = pytest.mark.gpu
REL = 1e-9


def same_float(a, b):
    a, b = np.float32(a), np.float32(b)
    if math.isnan(float(a)) or math.isnan(float(b)):
        return math.isnan(float(a)) and math.isnan(float(b))
    return a.view(np.uint32) == b.view(np.uint32)


class SeveralBricks(shard.ShardedStats):
    """A rank that presents its slab as three bricks per stage (cube.h allows any split into contiguous runs)."""

    def local_pass(self):
        step = (self.nvox + 2) // 3
        for o in range(0, self.nvox, step):
            self.ctx.ooc_brick(self.slab[o:o + step], min(step, self.nvox - o), self.stream)


def lockstep(slabs, nbins, lo, hi, want_median=True, flags=0, scratch=0, cls=shard.ShardedStats, ctxs=None):
    """Drive len(slabs) ranks through shard.ShardedStats in one process; the combine step is what the collectives do."""
    world = len(slabs)
    own = ctxs is None
    if own:
        ctxs = [cube.Context(scratch_bytes_hint=scratch) for _ in slabs]
    sts = [cls(c, s, s.numel(), nbins, lo, hi, want_median, flags) for c, s in zip(ctxs, slabs)]
    rounds = 0
    while sts[0].more:
        for st in sts:
            st.local_pass()
        payloads = [st.payload() for st in sts]
        if payloads[0][0] is not None:                                   # all-gather of the records, rank order
            gathered = torch.cat([p[0] for p in payloads]).clone()
            for st in sts:
                st.merge_records(gathered, world)
        for i in range(len(payloads[0][1])):                             # all-reduce SUM
            total = torch.stack([p[1][i] for p in payloads]).sum(dim=0)
            for p in payloads:
                p[1][i].copy_(total)
        for st in sts:
            st.advance()
        rounds += 1
    res = [st.result() for st in sts]
    if own:
        for c in ctxs:
            c.close()
    return res, rounds


def check_against_oracle(res, a, nbins, lo, hi, flags=0):
    ref = oracle.moments(a, sample_std=bool(flags & cube.SAMPLE_STD))
    rb, ro = oracle.histogram(a, nbins, lo, hi) if nbins else (None, None)
    rmed = oracle.median(a)
    m0 = res[0][0]
    for m, b, o, med in res:
        assert m["count"] == ref["count"] and m["nan_count"] == ref["nan_count"]
        assert same_float(m["min"], ref["min"]) and same_float(m["max"], ref["max"])
        assert abs(m["mean"] - ref["mean"]) <= REL * abs(ref["mean"]) and abs(m["std"] - ref["std"]) <= REL * ref["std"]
        assert m["mean"] == m0["mean"] and m["std"] == m0["std"]         # same bits on every rank
        if nbins:
            assert (b == rb).all() and (o == ro).all()
        assert same_float(med, rmed)


@pytest.mark.parametrize("name,dims,world,nbins,lo,hi", [
    ("c2", (96, 80, 64), 2, 4096, -0.02, 0.5), ("c2", (64, 64, 37), 3, 4096, -0.02, 0.5),
    ("c3", (64, 64, 128), 4, 65536, -0.02, 1.0), ("c4", (128, 128, 24), 2, 256, 0.0, 3000.0),
    ("c1", (48, 48, 8), 8, 1024, -5.0, 300.0)])
def test_sharded_matches_oracle_on_the_whole_cube(name, dims, world, nbins, lo, hi):
    cfg = cubegen.scaled(name, dims)
    nx, ny, nz = dims
    t = torch.empty(nx * ny * nz, dtype=torch.float32, device="cuda")
    cubegen.generate_device(cfg, t.data_ptr())
    torch.cuda.synchronize()
    a = t.cpu().numpy()
    slabs = []
    for r in range(world):
        z0, z1 = shard.slab_bounds(nz, world, r)
        slabs.append(t[z0 * nx * ny:z1 * nx * ny])
    res, rounds = lockstep(slabs, nbins, lo, hi)
    assert rounds == 3                                                   # three collective rounds for an exact median
    check_against_oracle(res, a, nbins, lo, hi)
    res, rounds = lockstep(slabs, nbins, lo, hi, want_median=False, flags=cube.SAMPLE_STD)
    assert rounds == 1
    ref = oracle.moments(a, sample_std=True)
    assert all(abs(m["std"] - ref["std"]) <= REL * ref["std"] for m, _, _, _ in res)


def test_sharded_edge_cases():
    r = np.random.default_rng(8)
    a = (r.standard_normal(50000) * 0.01).astype(np.float32)
    a[:20000] = np.nan                                                   # rank 0 sees only NULL voxels
    t = torch.from_numpy(a).cuda()
    slabs = [t[:20000], t[20000:20001], t[20001:]]                       # an all-NaN rank and a one-voxel rank
    res, _ = lockstep(slabs, 100, -0.05, 0.05)
    check_against_oracle(res, a, 100, -0.05, 0.05)
    # heavy ties + a candidate buffer too small for the bucket on every rank: stage 2 re-reads the slabs
    b = np.round(r.standard_normal(300000) * 2).astype(np.float32)
    tb = torch.from_numpy(b).cuda()
    res, _ = lockstep([tb[:100000], tb[100000:]], 16, -8.0, 8.0, scratch=4096)
    check_against_oracle(res, b, 16, -8.0, 8.0)


def test_run_with_nccl_world1():
    import torch.distributed as dist
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    port = s.getsockname()[1]
    s.close()
    dist.init_process_group("nccl", init_method="tcp://127.0.0.1:%d" % port, world_size=1, rank=0,
                            device_id=torch.device("cuda", 0))
    try:
        cfg = cubegen.scaled("c2", (64, 64, 48))
        t = torch.empty(64 * 64 * 48, dtype=torch.float32, device="cuda")
        cubegen.generate_device(cfg, t.data_ptr())
        torch.cuda.synchronize()
        ctx = cube.Context()
        res = shard.run(ctx, t, t.numel(), 4096, -0.02, 0.5)
        check_against_oracle([res], t.cpu().numpy(), 4096, -0.02, 0.5)
        ctx.close()
    finally:
        dist.destroy_process_group()


def test_sharded_empty_slab_and_reused_contexts():
    # world > nz: the last rank has NO voxel and presents no brick -- it all-gathers the empty record that
    # cube_ooc_begin leaves, also when its context still holds the record of an earlier run
    cfg = cubegen.scaled("c2", (64, 48, 3))
    t = torch.empty(64 * 48 * 3, dtype=torch.float32, device="cuda")
    cubegen.generate_device(cfg, t.data_ptr())
    torch.cuda.synchronize()
    a = t.cpu().numpy()
    slabs = []
    for r in range(4):
        z0, z1 = shard.slab_bounds(3, 4, r)
        slabs.append(t[z0 * 64 * 48:z1 * 64 * 48])
    assert slabs[3].numel() == 0
    ctxs = [cube.Context() for _ in slabs]
    try:
        junk = torch.full((5000,), 1e6, dtype=torch.float32, device="cuda")
        for c in ctxs:                                   # leave a stale running record in every context
            c.ooc_begin(16, 0.0, 1.0, True)
            c.ooc_brick(junk, junk.numel())
        for _ in range(2):
            res, rounds = lockstep(slabs, 4096, -0.02, 0.5, ctxs=ctxs)
            assert rounds == 3
            check_against_oracle(res, a, 4096, -0.02, 0.5)
        res, _ = lockstep(slabs, 4096, -0.02, 0.5, want_median=False, ctxs=ctxs)
        ref = oracle.moments(a)
        rb, ro = oracle.histogram(a, 4096, -0.02, 0.5)
        for m, b, o, _ in res:
            assert m["count"] == ref["count"] and (b == rb).all() and (o == ro).all()
    finally:
        for c in ctxs:
            c.close()


@pytest.mark.parametrize("scratch", [0, 4096])
@pytest.mark.parametrize("nbins,lo,hi", [(64, -8.0, 8.0), (40000, -8.0, 8.0)])
def test_sharded_slab_presented_as_several_bricks(scratch, nbins, lo, hi):
    # three bricks per rank and stage: the candidates of a rank are counted ONCE (in cube_shard_advance), whether they
    # fitted the buffer (scratch 0 = default size) or not (4096 bytes: stage 2 re-reads the bricks, each once);
    # both pass-B kernels (<= 16384 bins, and the window / packed ones above)
    r = np.random.default_rng(21)
    b = np.round(r.standard_normal(400003) * 2).astype(np.float32)       # heavy ties: big buckets
    b[r.integers(0, b.size, 4000)] = np.nan
    tb = torch.from_numpy(b).cuda()
    cuts = [0, 150001, 150002, 400003]
    slabs = [tb[cuts[i]:cuts[i + 1]] for i in range(3)]
    res, rounds = lockstep(slabs, nbins, lo, hi, scratch=scratch, cls=SeveralBricks)
    assert rounds == 3
    check_against_oracle(res, b, nbins, lo, hi)
    c2 = (r.standard_normal(300000) * 0.002 + 0.0004).astype(np.float32)  # continuous data: small bucket
    tc = torch.from_numpy(c2).cuda()
    res, _ = lockstep([tc[:100000], tc[100000:]], 4096, -0.02, 0.5, scratch=scratch, cls=SeveralBricks)
    check_against_oracle(res, c2, 4096, -0.02, 0.5)


@pytest.mark.parametrize("name,dims,world,nbins", [("c3", (64, 64, 96), 3, 65536), ("c4", (128, 64, 24), 2, 256),
                                                   ("c1", (48, 48, 30), 4, 1024)])
def test_sharded_histogram_over_the_merged_min_max(name, dims, world, nbins):
    # lo=None: the range is [min, max] of the WHOLE cube, known on every rank after the records are merged and
    # resolved on the device; the histogram is accumulated in stage 1 (configs 1, 3, 4 bin over [min, max])
    cfg = cubegen.scaled(name, dims)
    nx, ny, nz = dims
    t = torch.empty(nx * ny * nz, dtype=torch.float32, device="cuda")
    cubegen.generate_device(cfg, t.data_ptr())
    torch.cuda.synchronize()
    a = t.cpu().numpy()
    slabs = []
    for r in range(world):
        z0, z1 = shard.slab_bounds(nz, world, r)
        slabs.append(t[z0 * nx * ny:z1 * nx * ny])
    ref = oracle.moments(a)
    lo, hi = float(ref["min"]), float(ref["max"])
    res, rounds = lockstep(slabs, nbins, None, None)
    assert rounds == 3
    check_against_oracle(res, a, nbins, lo, hi)
    res, rounds = lockstep(slabs, nbins, None, None, want_median=False)
    assert rounds == 2
    rb, ro = oracle.histogram(a, nbins, lo, hi)
    for m, b, o, _ in res:
        assert m["count"] == ref["count"] and (b == rb).all() and (o == ro).all() and int(b.sum()) == ref["count"]
