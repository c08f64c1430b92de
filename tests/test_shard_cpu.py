"""Host-side logic of the z-slab sharded path (paper_1211_4896_b200/shard.py) on CPU:
slab partition, and the driver's sequence of local passes / collectives / advances in two real gloo processes.

No CUDA here, so the libcube context is replaced by a STUB that keeps the same buffers (record, bins, outside,
digits) in numpy memory and fills them with numpy arithmetic (test scaffolding, not the product: it exists only so
that shard.run() can be driven end to end without a GPU; the real kernels are checked against the oracle in
tests/test_gpu_shard.py).  What is checked is the plumbing: every rank ends with the whole cube's count, histogram
and exact lower median although it has only seen its own slab.
"""
import json
import os
import socket
import subprocess
import sys

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)


def test_slab_bounds_partition_without_overlap():
    from paper_1211_4896_b200.shard import slab_bounds
    for nz in (1, 2, 7, 8, 1024, 1031):
        for world in (1, 2, 3, 8):
            b = [slab_bounds(nz, world, r) for r in range(world)]
            assert b[0][0] == 0 and b[-1][1] == nz
            assert all(b[i][1] == b[i + 1][0] for i in range(world - 1))          # contiguous, no overlap
            sizes = [z1 - z0 for z0, z1 in b]
            assert max(sizes) - min(sizes) <= 1 and min(sizes) >= 0


WORKER = r"""
import json, os, sys
sys.path.insert(0, %(root)r)
import numpy as np
import torch
import torch.distributed as dist
from paper_1211_4896_b200 import shard

BITS = (13, 10, 9)


def keys_of(a):
    u = a.view(np.uint32)
    return np.where(u >> 31 == 1, ~u, u | np.uint32(0x80000000)).astype(np.uint32)


class StubContext:
    # same call surface as paper_1211_4896_b200.Context for the sharded path, numpy inside
    def __init__(self):
        self.record = np.zeros(5, dtype=np.float64)        # n, sum, sumsq, min, max  (40 bytes, opaque to the driver)
        self.bins = np.zeros(65536, dtype=np.int64)
        self.outside = np.zeros(2, dtype=np.int64)
        self.digits = np.zeros(8192, dtype=np.int64)
        self.calls = []

    def shard_buffers(self):
        return dict(record=self.record, bins=self.bins, outside=self.outside, digits=self.digits)

    def ooc_begin(self, nbins, lo, hi, want_median, stream):
        self.nbins, self.lo, self.hi, self.stage = nbins, np.float32(lo), np.float32(hi), 0
        self.prefix, self.k, self.total = 0, None, None
        self.record[:] = [0, 0, 0, np.inf, -np.inf]          # the empty record: a rank without voxels gathers this
        self.cand = np.zeros(0, dtype=np.uint32)
        self.calls.append("begin")

    def ooc_brick(self, slab, nvox, stream):
        a = slab[~np.isnan(slab)]
        key = keys_of(a)
        if self.stage == 0:
            self.record[:] = [a.size, a.astype(np.float64).sum(), (a.astype(np.float64) ** 2).sum(),
                              a.min() if a.size else np.inf, a.max() if a.size else -np.inf]
            self.digits += np.bincount(key >> 19, minlength=8192)
        elif self.stage == 1:                                # the histogram shares the second read of the slab
            inr = a[(a >= self.lo) & (a <= self.hi)]
            scale = np.float32(self.nbins) / np.float32(self.hi - self.lo)
            b = np.minimum(np.floor((inr - self.lo) * scale).astype(np.int64), self.nbins - 1)
            self.bins[:self.nbins] += np.bincount(b, minlength=self.nbins)
            self.outside += [int((a < self.lo).sum()), int((a > self.hi).sum())]
            sel = key[(key >> 19) == self.prefix]
            self.cand = sel
            self.digits[:1024] += np.bincount((sel >> 9) & 1023, minlength=1024)
        self.calls.append("pass%%d" %% self.stage)           # stage 2: the candidates were counted by advance()

    def shard_merge_records(self, gathered, world, flags, stream):
        g = gathered.numpy().view(np.float64).reshape(world, 5)
        self.merged = [g[:, 0].sum(), g[:, 1].sum(), g[:, 2].sum(), g[:, 3].min(), g[:, 4].max()]
        self.calls.append("merge%%d" %% world)

    def shard_advance(self, stream):
        nb = 1 << BITS[self.stage]
        c = self.digits[:nb]
        if self.stage == 0:
            self.total = int(c.sum())
            self.k = (self.total - 1) // 2
        cum = np.cumsum(c)
        b = int(np.searchsorted(cum, self.k, side="right"))
        self.k -= int(cum[b - 1]) if b else 0
        self.prefix = (self.prefix << BITS[self.stage]) | b
        self.digits[:] = 0
        self.stage += 1
        if self.stage == 2:                                  # this rank's own candidates, once (as cube_shard_advance)
            sel = self.cand[(self.cand >> 9) == self.prefix]
            self.digits[:512] += np.bincount(sel & 511, minlength=512)
        self.calls.append("advance")
        return self.stage < 3

    def ooc_result(self, nbins, flags, want_median, stream):
        key = np.uint32(self.prefix)
        bits = key ^ np.uint32(0x80000000) if key & np.uint32(0x80000000) else ~key
        return self.merged, self.bins[:nbins].copy(), self.outside.copy(), np.array([bits], dtype=np.uint32).view(np.float32)[0]


def alias(buf, nbytes, dtype, device):                       # numpy memory instead of a device address
    return torch.from_numpy(buf.view(np.uint8)[:nbytes]).view(dtype)


shard.alias = alias
dist.init_process_group("gloo")
rank, world = dist.get_rank(), dist.get_world_size()
nx, ny, nz = 16, 12, int(os.environ.get("SHARD_TEST_NZ", "37"))
rng = np.random.default_rng(5)
cube = (rng.standard_normal(nx * ny * nz) * 0.002 + 0.0005).astype(np.float32)
cube[rng.integers(0, cube.size, 200)] = np.nan
cube[rng.integers(0, cube.size, 50)] = 0.4
z0, z1 = shard.slab_bounds(nz, world, rank)
slab = cube[z0 * nx * ny:z1 * nx * ny]
ctx = StubContext()
"""

WORKER_MAIN = r"""
merged, bins, outside, med = shard.run(ctx, slab, slab.size, 64, -0.01, 0.01, device=torch.device("cpu"), stream=0)
ok = cube[~np.isnan(cube)]
ref_med = np.sort(ok)[(ok.size - 1) // 2]
out = {"rank": rank, "count": merged[0], "ref_count": int(ok.size), "med_bits": int(np.float32(med).view(np.uint32)),
       "ref_bits": int(np.float32(ref_med).view(np.uint32)), "bins_sum": int(bins.sum()), "outside": outside.tolist(),
       "min": merged[3], "max": merged[4], "ref_min": float(ok.min()), "ref_max": float(ok.max()),
       "calls": ctx.calls, "slab": [z0, z1]}
res = [None] * world
dist.all_gather_object(res, out)
if rank == 0:
    print("RESULT " + json.dumps(res))
dist.destroy_process_group()
"""


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


# (4, 3): world size 4 over 3 z-planes -- the last rank's slab is EMPTY (it presents no brick and all-gathers the
# empty record left by cube_ooc_begin)
@pytest.mark.parametrize("nproc,nz", [(2, 37), (3, 37), (4, 3)])
def test_sharded_driver_sequence_gloo(tmp_path, nproc, nz):
    w = tmp_path / "worker.py"
    w.write_text(WORKER % {"root": ROOT} + WORKER_MAIN)
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", str(nproc),
           "--master-addr", "127.0.0.1", "--master-port", str(_free_port()), str(w)]
    env = dict(os.environ, MASTER_ADDR="127.0.0.1", OMP_NUM_THREADS="1", SHARD_TEST_NZ=str(nz))
    r = subprocess.run(cmd, cwd=ROOT, env=env, capture_output=True, text=True, timeout=300)
    assert r.returncode == 0, r.stderr[-3000:]
    line = [l for l in r.stdout.splitlines() if l.startswith("RESULT ")]
    assert line, r.stdout[-2000:]
    res = json.loads(line[0][len("RESULT "):])
    assert len(res) == nproc
    for o in res:
        assert o["count"] == o["ref_count"]                                  # whole-cube count on every rank
        assert o["med_bits"] == o["ref_bits"]                                # exact lower median of the WHOLE cube
        assert o["bins_sum"] + sum(o["outside"]) == o["ref_count"]
        assert o["min"] == o["ref_min"] and o["max"] == o["ref_max"]
        empty = o["slab"][0] == o["slab"][1]
        assert o["calls"] == (["begin", "merge%d" % nproc, "advance", "advance", "advance"] if empty else
                              ["begin", "pass0", "merge%d" % nproc, "advance", "pass1", "advance", "pass2", "advance"])
    assert [o["slab"][0] for o in res] == sorted(o["slab"][0] for o in res)
    assert res[0]["slab"][0] == 0 and res[-1]["slab"][1] == nz
    assert (nz >= nproc) or any(o["slab"][0] == o["slab"][1] for o in res)
