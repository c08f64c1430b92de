"""Host-side logic of the N>1 bench path, on CPU with the gloo backend and world_size 2.

The statistics path does not shard across GPUs in this build ("replicas only"): under
torchrun every rank runs the whole hot path on its own cube and bench.py only combines the timings --
max over ranks of the device time, sum of the voxels processed.  These tests drive exactly that plumbing
(bench.aggregate_over_ranks, the per-rank seeds, the reference arm's rank-0-only rule) in two real processes.
No CUDA, no libcube compute call.
"""
import json
import os
import socket
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

WORKER = r"""
import json, os, sys
sys.path.insert(0, %(root)r)
import torch
import torch.distributed as dist
import bench
dist.init_process_group("gloo")
rank, world = dist.get_rank(), dist.get_world_size()
local_ms = 10.0 + 5.0 * rank              # rank 1 is the slow one
units = 1000 * (rank + 1)
t, u = bench.aggregate_over_ranks(dist, local_ms, units)
seed = bench.replica_seed(2, rank)
out = {"rank": rank, "world": world, "ms": t, "units": u, "seed": seed}
gathered = [None] * world
dist.all_gather_object(gathered, out)
if rank == 0:
    print("RESULT " + json.dumps(gathered))
dist.destroy_process_group()
"""


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def _torchrun(nproc, script_args, timeout=240):
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", str(nproc),
           "--master-addr", "127.0.0.1", "--master-port", str(_free_port())] + script_args
    env = dict(os.environ, MASTER_ADDR="127.0.0.1", OMP_NUM_THREADS="1")
    return subprocess.run(cmd, cwd=ROOT, env=env, capture_output=True, text=True, timeout=timeout)


def test_aggregate_over_ranks_gloo_world2(tmp_path):
    w = tmp_path / "worker.py"
    w.write_text(WORKER % {"root": ROOT})
    r = _torchrun(2, [str(w)])
    assert r.returncode == 0, r.stderr[-2000:]
    line = [l for l in r.stdout.splitlines() if l.startswith("RESULT ")]
    assert len(line) == 1
    res = json.loads(line[0][7:])
    assert [x["rank"] for x in res] == [0, 1] and all(x["world"] == 2 for x in res)
    # every rank sees max-over-ranks time and the whole-job unit count
    assert all(x["ms"] == 15.0 for x in res)
    assert all(x["units"] == 3000.0 for x in res)
    # independent replicas: rank 0 keeps the config's seed, the others get distinct ones
    assert res[0]["seed"] == 2 and res[1]["seed"] != 2


def test_aggregate_single_process_is_identity():
    sys.path.insert(0, ROOT)
    import bench
    assert bench.aggregate_over_ranks(None, 12.5, 77) == (12.5, 77.0)
    assert bench.replica_seed(5, 0) == 5
    assert len({bench.replica_seed(5, r) for r in range(8)}) == 8


def test_reference_arm_runs_on_rank0_only():
    # under torchrun the oracle arm prints ONE line (rank 0) and the other rank exits 0 without work
    r = _torchrun(2, ["bench.py", "--impl", "reference", "--gpus", "2", "--steps", "1", "--warmup", "0",
                      "--config", "c1", "--ref-voxels", "65536"], timeout=600)
    assert r.returncode == 0, r.stderr[-2000:]
    lines = [l for l in r.stdout.splitlines() if l.startswith("{")]
    assert len(lines) == 1
    j = json.loads(lines[0])
    assert j["impl"] == "reference" and j["n_gpus"] == 2 and j["unit"] == "voxels/s" and j["value"] > 0
    assert j["cpu_baseline"]["kind"] == "oracle" and j["e2e"]["h2d_bytes_per_step"] == 0


@pytest.mark.parametrize("flag", ["--help"])
def test_bench_cli_parses(flag):
    r = subprocess.run([sys.executable, "bench.py", flag], cwd=ROOT, capture_output=True, text=True, timeout=120)
    assert r.returncode == 0 and "--gpus" in r.stdout
