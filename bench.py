#!/usr/bin/env python
"""bench.py -- headline benchmark of libcube (BASELINE.json metric: voxels/s and % of HBM peak for
moments, histogram and exact median of a float32 cube).

A "step" is one pass of the whole hot path over the workload: cube_moments,
cube_histogram(nbins, lo, hi) and cube_median on the cube resident in HBM.  The workload at N=1 is
BASELINE.json configs[1] (c2: 1024^3 float32, 4 GiB, seed 2), generated on the device by cubegen.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config c2] [--impl reference]

Prints ONE JSON line (rank 0).  With --gpus N>1 (launched under torchrun) every rank runs an independent
replica of the workload on its own GPU (the path has no data-path collective: "replicas only",
DESIGN.md sec. 8); value = total voxels / max-over-ranks device time.

--impl reference times the CPU oracle (oracle/, as it stands) on a bounded sample of the same workload.
"""
import argparse
import json
import os
import subprocess
import sys
import tempfile
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

import cubegen  # noqa: E402

HIST = {"c1": (1024, None, None), "c2": (4096, -0.02, 0.5), "c3": (65536, None, None),
        "c4": (65536, None, None), "c5": (4096, -0.02, 0.5)}
METRIC = "voxels/s & % HBM peak for moments, histogram, exact median (float32 cube)"
# algorithmic bytes per voxel of each kernel kind, per launch (DESIGN.md sec. 4 / SURVEY.md sec. 8(d))
ALGO_BYTES_PER_VOXEL = 4.0


def measured_peak():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        try:
            return float(json.load(open(p))["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs, copy read+write)"
        except Exception:
            pass
    return 6650.0, "fallback (B200_PROFILING.md 6.65 TB/s)"


def workload_desc(name, cfg):
    nx, ny, nz = cfg["dims"]
    nb, lo, hi = HIST[name]
    rng = "[min,max]" if lo is None else "[%g,%g]" % (lo, hi)
    return "%s: %dx%dx%d float32 cube (%.2f GiB), seed %d; moments + %d-bin histogram over %s + exact lower median" % (
        name, nx, ny, nz, nx * ny * nz * 4 / 2 ** 30, cfg["seed"], nb, rng)


# ------------------------------------------------------------------------------------------------ clocks
class ClockSampler:
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.f = tempfile.NamedTemporaryFile("w+", suffix=".csv", delete=False)
        try:
            self.p = subprocess.Popen(["nvidia-smi", "-i", str(index), "--query-gpu=" + self.Q,
                                       "--format=csv,noheader,nounits", "-lms", "20"],
                                      stdout=self.f, stderr=subprocess.DEVNULL)
        except OSError:
            self.p = None

    def stop(self):
        out = {"sm_mhz": None, "sm_max_mhz": None, "reasons": []}
        if self.p is None:
            return out
        self.p.terminate()
        try:
            self.p.wait(timeout=5)
        except Exception:
            self.p.kill()
        self.f.flush()
        self.f.seek(0)
        sm, mx, reasons = [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for line in self.f:
            t = [v.strip() for v in line.split(",")]
            if len(t) < 7:
                continue
            try:
                sm.append(float(t[0]))
                mx.append(float(t[1]))
            except ValueError:
                continue
            for nme, v in zip(names, t[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(nme)
        os.unlink(self.f.name)
        if sm:
            out = {"sm_mhz": float(np.median(sm)), "sm_max_mhz": float(max(mx)), "reasons": sorted(reasons),
                   "samples": len(sm)}
        return out


# ------------------------------------------------------------------------------------------------ oracle legs
def replica_seed(seed, rank):
    """Seed of rank `rank`'s independent replica of the workload (rank 0 keeps the config's own seed)."""
    return seed + 1000 * rank if rank else seed


_SAMPLE_CACHE = {}


def sample_planes(cfg, sample_voxels):
    nx, ny, nz = cfg["dims"]
    return max(1, min(nz, sample_voxels // (nx * ny)))


def oracle_sample(name, cfg, sample_voxels=1 << 24, a=None):
    """Time the CPU oracle (as it stands, single thread) on a bounded sample of the workload: the first
    `planes` z-planes of the cube -- `a` when the caller already holds those voxels (bench copies them from the
    device cube it times), else generated here (CUDA generator when a device is present, numpy otherwise).
    Returns (voxels/s, description, seconds)."""
    import oracle
    nx, ny, nz = cfg["dims"]
    planes = sample_planes(cfg, sample_voxels)
    if a is None:
        key = (name, cfg["seed"], planes)
        if key not in _SAMPLE_CACHE:
            _SAMPLE_CACHE.clear()
            _SAMPLE_CACHE[key] = generate_sample(cfg, planes)
        a = _SAMPLE_CACHE[key]
    nb, lo, hi = HIST[name]
    t0 = time.perf_counter()
    m = oracle.moments(a)
    if lo is None:
        lo, hi = float(m["min"]), float(m["max"])
    oracle.histogram(a, nb, lo, hi)
    oracle.median(a)
    dt = time.perf_counter() - t0
    desc = "first %d z-planes of %s (%d voxels): oracle moments + %d-bin histogram + median, 1 thread" % (
        planes, name, a.size, nb)
    return a.size / dt, desc, dt


def generate_sample(cfg, planes):
    """First `planes` z-planes of the workload as a host float32 array (inputs only: cubegen)."""
    nx, ny, nz = cfg["dims"]
    try:
        import torch
        if torch.cuda.is_available():
            t = torch.empty(nx * ny * planes, dtype=torch.float32, device="cuda")
            cubegen.generate_device(cfg, t.data_ptr(), origin=(0, 0, 0), brick=(nx, ny, planes))
            torch.cuda.synchronize()
            return t.cpu().numpy()
    except ImportError:
        pass
    planes = min(planes, max(1, (1 << 25) // (nx * ny)))     # numpy generator: keep it to ~32 Mi voxels
    return cubegen.generate_numpy(cfg, origin=(0, 0, 0), brick=(nx, ny, planes)).reshape(-1)


def reference_sample_voxels(args):
    """Per-step sample of the oracle arm: ~120 s of single-thread oracle work (~40 Mvoxel/s for the three
    operations) over the whole --steps/--warmup run, between 2^20 and 2^29 voxels per step."""
    if args.ref_voxels:
        return args.ref_voxels
    per = int(5e9 / max(1, args.steps + (1 if args.warmup > 0 else 0)))
    return max(1 << 20, min(1 << 29, per))


def run_reference(args):
    """--impl reference: the oracle on the host cores, same metric/config, bounded sample per step."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return 0
    name = args.config
    cfg = cubegen.CONFIGS[name]
    sv = reference_sample_voxels(args)
    oracle_sample(name, cfg, sv) if args.warmup > 0 else None     # one warm-up (page-in, build)
    vals, secs, desc = [], [], ""
    for _ in range(max(1, args.steps)):
        v, desc, dt = oracle_sample(name, cfg, sv)
        vals.append(v)
        secs.append(dt)
    value = float(np.mean(vals))
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": "voxels/s", "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": float(np.mean(secs)) * 1e3,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f32",
            "data": "synthetic", "config": {"workload": workload_desc(name, cfg)},
            "cpu_baseline": {"value": value, "unit": "voxels/s", "cores": 1, "kind": "oracle", "sample": desc},
            "e2e": {"value": value, "unit": "voxels/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line))
    return 0


# ------------------------------------------------------------------------------------------------ rank plumbing
def aggregate_over_ranks(dist, local_ms, local_units, device=None):
    """max over ranks of the device time, sum of the units processed (works with nccl and gloo)."""
    import torch
    t = torch.tensor([local_ms], dtype=torch.float64, device=device)
    u = torch.tensor([float(local_units)], dtype=torch.float64, device=device)
    if dist is not None and dist.is_initialized() and dist.get_world_size() > 1:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        dist.all_reduce(u, op=dist.ReduceOp.SUM)
    return float(t.item()), float(u.item())


def run_out_of_core(args):
    """--config c5: 4096^3 (256 GiB) produced per 512^3 brick into pinned host staging buffers (generated on the
    device from the seed, copied D2H on the fill stream) and streamed H2D through cube_stats_stream.  One step =
    the whole job: moments + 4096-bin histogram + exact lower median over all 512 bricks."""
    import torch
    import paper_1211_4896_b200 as cube

    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: libcube has no CPU fallback")
    if int(os.environ.get("WORLD_SIZE", "1")) > 1:
        raise SystemExit("--config c5 is a single-GPU job")
    torch.cuda.set_device(0)
    name = "c5"
    cfg = cubegen.CONFIGS[name]
    nx, ny, nz = cfg["dims"]
    n = nx * ny * nz
    brick = (512, 512, 512)
    bvox = brick[0] * brick[1] * brick[2]
    origins = cubegen.brick_grid(cfg, brick)
    nb, lo, hi = HIST[name]
    scratch = torch.empty(bvox, dtype=torch.float32, device="cuda")
    scr = [scratch, torch.empty(bvox, dtype=torch.float32, device="cuda")]
    for org in origins:                        # per-brick source lists, cached outside the timed region
        cubegen.sources_in_brick(cfg, org, brick)
    ctx = cube.Context(scratch_bytes_hint=1 << 30)
    nres = int(args.resident_gib * 2 ** 30) // (bvox * 4)
    ctx.stream_workspace(bvox * 4, host_slots=4, resident_bytes=nres * bvox * 4)

    # measured pinned H2D peak of this box: 512 MiB copies, two in flight
    hp = torch.empty(bvox, dtype=torch.float32, pin_memory=True)
    s1, s2 = torch.cuda.Stream(), torch.cuda.Stream()
    d2 = torch.empty(bvox, dtype=torch.float32, device="cuda")
    torch.cuda.synchronize()
    t0 = time.perf_counter()
    reps = 16
    for i in range(reps):
        with torch.cuda.stream(s1 if i & 1 else s2):
            (scratch if i & 1 else d2).copy_(hp, non_blocking=True)
    torch.cuda.synchronize()
    h2d_peak = reps * bvox * 4 / (time.perf_counter() - t0) / 1e9
    del hp, d2

    # producer: brick generated on the device (gen stream, two scratch buffers) and copied D2H on the driver's
    # fill stream, so that generating brick i+1 overlaps the D2H of brick i and the H2D of brick i-1
    gen = torch.cuda.Stream()
    ev_gen = [torch.cuda.Event(), torch.cuda.Event()]
    ev_d2h = [torch.cuda.Event(), torch.cuda.Event()]
    produced = [0]

    def fill(b, sweep, h_dst, nvox, fs):
        k = produced[0] & 1
        produced[0] += 1
        fst = torch.cuda.ExternalStream(fs)
        gen.wait_event(ev_d2h[k])
        cubegen.generate_device(cfg, scr[k].data_ptr(), origin=origins[b], brick=brick, stream=gen.cuda_stream)
        ev_gen[k].record(gen)
        fst.wait_event(ev_gen[k])
        cubegen.to_host(h_dst, scr[k].data_ptr(), nvox, fs)
        ev_d2h[k].record(fst)

    results = []
    secs = []
    sampler = None
    for it in range(args.warmup + args.steps):
        if it == args.warmup:
            sampler = ClockSampler(0)
        l0 = ctx.launch_count
        torch.cuda.synchronize()
        t0 = time.perf_counter()
        m, b, o, med, info = ctx.stats_stream(len(origins), bvox, n, fill, nb, lo, hi)
        dt = time.perf_counter() - t0
        if it >= args.warmup:
            secs.append(dt)
            results.append((m, med, info, ctx.launch_count - l0))
    clocks = sampler.stop() if sampler else None
    dt = float(np.mean(secs))
    m, med, info, launches = results[-1]
    h2d_gbs = info["h2d_bytes"] / dt / 1e9
    cpu = None
    if not args.no_cpu_baseline:
        v, desc, cdt = oracle_sample(name, cfg, min(args.cpu_voxels, 1 << 28))
        cpu = {"value": v, "unit": "voxels/s", "cores": 1, "kind": "oracle", "sample": desc, "seconds": cdt}
    line = {"metric": METRIC, "value": n / dt, "unit": "voxels/s", "n_gpus": 1, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": dt * 1e3, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f32", "data": "synthetic",
            "config": {"workload": workload_desc(name, cfg) + "; out of core: 512 bricks of 512^3, %d kept in HBM after "
                                   "sweep 1, the rest produced and streamed again in sweep 2" % min(nres, len(origins)),
                       "l2": "bricks (512 MiB) are larger than the 126 MB L2",
                       "timer": "host perf_counter around the synchronous cube_stats_stream call"},
            "e2e": {"value": n / dt, "unit": "voxels/s", "h2d_bytes_per_step": info["h2d_bytes"],
                    "d2h_bytes_per_step": 40 + nb * 8 + 16 + 4, "note": "the job IS end to end: every brick crosses the "
                    "host link inside the timed region"},
            "gpu_launches": launches, "clocks": clocks,
            "roofline": {"bound": "h2d", "kernel": "cudaMemcpyAsync H2D of the bricks (the kernels have ~100x slack)",
                         "achieved": h2d_gbs, "peak": h2d_peak, "unit": "GB/s", "frac": h2d_gbs / h2d_peak,
                         "traffic": None, "peak_source": "pinned H2D copy, 512 MiB x 16, two streams, measured in this run",
                         "sweeps": info["sweeps"]},
            "cpu_baseline": cpu,
            "result_check": {"median": float(med), "count": m["count"], "mean": m["mean"], "std": m["std"],
                             "min": float(m["min"]), "max": float(m["max"])}}
    print(json.dumps(line))
    return 0


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=None, help="timed steps (default 200; 1 for c5)")
    ap.add_argument("--warmup", type=int, default=None, help="untimed warm-up steps (default 3; 1 for c5)")
    ap.add_argument("--config", default="c2", choices=sorted(cubegen.CONFIGS))
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--ref-voxels", type=int, default=0,
                    help="voxels of the bounded oracle sample per step of --impl reference (0 = sized from --steps)")
    ap.add_argument("--cpu-voxels", type=int, default=1 << 29,
                    help="voxels of the cpu_baseline sample (first z-planes of the timed device cube)")
    ap.add_argument("--resident-gib", type=float, default=128.0, help="c5: GiB of bricks kept in HBM after sweep 1")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-next", action="store_true", help="skip the timings of the NEXT rows (MAD, clipping, mini-map)")
    args = ap.parse_args()
    if args.steps is None:
        args.steps = 1 if args.config == "c5" else 200
    if args.warmup is None:
        args.warmup = 1 if args.config == "c5" else 3
    if args.impl == "reference":
        return run_reference(args)
    if args.config == "c5":
        return run_out_of_core(args)
    args.warmup = max(args.warmup, 3)

    import torch
    import torch.distributed as dist
    import paper_1211_4896_b200 as cube

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: libcube has no CPU fallback")
    torch.cuda.set_device(local_rank)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local_rank))
    dev = torch.device("cuda", local_rank)

    name = args.config
    cfg = dict(cubegen.CONFIGS[name])
    cfg["seed"] = replica_seed(cfg["seed"], rank)                        # independent replica per rank
    nx, ny, nz = cfg["dims"]
    n = nx * ny * nz
    nb, lo, hi = HIST[name]
    cube_t = torch.empty(n, dtype=torch.float32, device=dev)
    cubegen.generate_device(cfg, cube_t.data_ptr())
    torch.cuda.synchronize()

    # candidate buffer of the select: 1/16 of the cube (config 4's median bucket holds 2.2 % of it), >= 256 MiB
    ctx = cube.Context(scratch_bytes_hint=max(256 << 20, n * 4 // 16))
    stream = torch.cuda.current_stream().cuda_stream
    out_m = torch.zeros(40, dtype=torch.uint8, device=dev)
    out_b = torch.zeros(nb, dtype=torch.int64, device=dev)
    out_o = torch.zeros(2, dtype=torch.int64, device=dev)
    out_f = torch.zeros(1, dtype=torch.float32, device=dev)
    s_lo, s_hi = lo, hi                    # None -> cube_stats bins over [min,max] found on the device
    if lo is None:
        m0 = ctx.moments(cube_t, nx, ny, nz)
        lo, hi = float(m0["min"]), float(m0["max"])

    def step():
        # the whole hot path in one call: moments + histogram + exact lower median, two reads of the cube
        ctx.stats(cube_t, nx, ny, nz, nb, s_lo, s_hi, out=out_m, bins=out_b, outside=out_o, median=out_f, stream=stream)

    def op_moments():
        ctx.moments(cube_t, nx, ny, nz, out=out_m, stream=stream)

    def op_histogram():
        ctx.histogram(cube_t, nx, ny, nz, nb, lo, hi, bins=out_b, outside=out_o, stream=stream)

    def op_histogram_256():                 # config 4 also asks for a 256-bin histogram (hot-bin contention)
        ctx.histogram(cube_t, nx, ny, nz, 256, lo, hi, bins=out_b, outside=out_o, stream=stream)

    def op_median():
        ctx.median(cube_t, nx, ny, nz, out=out_f, stream=stream)

    # NEXT rows: MAD, clipped moments, sigma clipping, 30^3 statistical mini-map
    out_w = torch.zeros(2, dtype=torch.float32, device=dev)
    out_i = torch.zeros(1, dtype=torch.int32, device=dev)
    out_w2 = torch.zeros(1, dtype=torch.int32, device=dev)
    part = (30, 30, 30)
    mmx, mmy, mmz = ctx.minimap_dims(nx, ny, nz, *part)
    out_cells = torch.zeros(mmx * mmy * mmz * 40, dtype=torch.uint8, device=dev)

    def op_mad():
        ctx.mad(cube_t, nx, ny, nz, median_out=out_f, mad_out=out_w[0:1], stream=stream)

    def op_clipped():
        ctx.clipped_moments(cube_t, nx, ny, nz, lo, hi, out=out_m, stream=stream)

    def op_sigma_clip():
        ctx.sigma_clip(cube_t, nx, ny, nz, 3.0, 5, out=out_m, iters=out_i, window=out_w, stream=stream)

    def op_torben():                         # the paper's own median method (Alg. 1), ~30 passes over the cube
        ctx.median_torben(cube_t, nx, ny, nz, 64, out=out_f, iters=out_i, converged=out_w2, stream=stream)

    def op_minimap():
        ctx.minimap(cube_t, nx, ny, nz, part[0], part[1], part[2], out_cells, stream=stream)

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    def timed(fn, reps):
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        torch.cuda.synchronize()
        a.record()
        for _ in range(reps):
            fn()
        b.record()
        torch.cuda.synchronize()
        return a.elapsed_time(b) / reps

    for _ in range(args.warmup):
        step()
    barrier()
    sampler = ClockSampler(local_rank) if rank == 0 else None
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    l0 = ctx.launch_count
    e0.record()
    for _ in range(args.steps):
        step()
    e1.record()
    barrier()
    launches = ctx.launch_count - l0
    local_ms = e0.elapsed_time(e1)
    total_ms, total_units = aggregate_over_ranks(dist if world > 1 else None, local_ms, n * args.steps, dev)

    # the three operations of the metric through their own entry points (each its own timed region)
    peak, peak_src = measured_peak()
    ops = {}
    op_list = [("moments", op_moments, 4.0), ("histogram", op_histogram, 4.0), ("median", op_median, 8.0)]
    if name == "c4":
        op_list.append(("histogram_256", op_histogram_256, 4.0))
    if name in ("c2", "c3"):
        # BASELINE.json configs[2]: "median and k-th at k=N/100 and k=99N/100" -- three ranks of one cube in TWO
        # reads (cube_kth_multi: first digit of every voxel, then one gather of the three buckets; the other two
        # digits are counted on the gathered candidates) instead of three selections of two reads each
        cnt3 = int(ctx.moments(cube_t, nx, ny, nz)["count"])
        ks3 = [(cnt3 - 1) // 2, cnt3 // 100, 99 * cnt3 // 100]
        out_k3 = torch.zeros(3, dtype=torch.float32, device=dev)
        op_list.append(("median_p1_p99_multi", lambda: ctx.kth_multi(cube_t, nx, ny, nz, ks3, out=out_k3, stream=stream), 8.0))
    for nm, fn, bpv in op_list:
        for _ in range(3):
            fn()
        ms = timed(fn, args.steps)
        ops[nm] = {"ms": ms, "voxels_per_s": n / (ms * 1e-3), "algorithmic_bytes_per_voxel": bpv,
                   "algorithmic_gbs": bpv * n / (ms * 1e-3) / 1e9, "frac_of_peak": bpv * n / (ms * 1e-3) / 1e9 / peak}
    if not args.no_next:
        reps_n = max(3, args.steps // 4)
        op_sigma_clip()
        torch.cuda.synchronize()
        clip_passes = int(out_i.item()) + 1          # the plain pass + the clipped passes actually made
        op_torben()
        torch.cuda.synchronize()
        torben_passes = int(out_i.item()) + 1        # the moments pass (Min, Max, n) + the passes of Alg. 1
        op_sigma_clip()
        torch.cuda.synchronize()
        for nm, fn, bpv in [("paper_alg1_torben_median", op_torben, 4.0 * torben_passes),
                            ("next_mad", op_mad, 16.0), ("next_clipped_moments", op_clipped, 4.0),
                            ("next_sigma_clip_3sigma_max5", op_sigma_clip, 4.0 * clip_passes),
                            ("next_minimap_30x30x30", op_minimap, 4.0)]:
            for _ in range(2):
                fn()
            ms = timed(fn, reps_n)
            ops[nm] = {"ms": ms, "voxels_per_s": n / (ms * 1e-3), "algorithmic_bytes_per_voxel": bpv,
                       "algorithmic_gbs": bpv * n / (ms * 1e-3) / 1e9, "frac_of_peak": bpv * n / (ms * 1e-3) / 1e9 / peak}
    ops["stats_fused"] = {"ms": total_ms / args.steps, "voxels_per_s": total_units / (total_ms * 1e-3) / world,
                          "algorithmic_bytes_per_voxel": 8.0,
                          "algorithmic_gbs": 8.0 * n / (local_ms / args.steps * 1e-3) / 1e9,
                          "frac_of_peak": 8.0 * n / (local_ms / args.steps * 1e-3) / 1e9 / peak}
    # a cube that fits the 126 MB L2 (config 1) is also timed COLD: 512 MiB written between the repetitions, each
    # repetition bracketed by its own event pair ("c1: flush L2 between reps; report cold and warm")
    ops_cold = None
    if n * 4 <= (256 << 20):
        flush = torch.empty(512 << 20, dtype=torch.uint8, device=dev)
        ops_cold = {}
        for nm, fn, bpv in op_list + [("stats_fused", step, 8.0)]:
            ts = []
            for _ in range(23):
                flush.fill_(1)
                a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                a.record()
                fn()
                b.record()
                torch.cuda.synchronize()
                ts.append(a.elapsed_time(b))
            ms = float(np.median(ts[3:]))
            ops_cold[nm] = {"ms": ms, "voxels_per_s": n / (ms * 1e-3), "algorithmic_bytes_per_voxel": bpv,
                            "algorithmic_gbs": bpv * n / (ms * 1e-3) / 1e9,
                            "frac_of_peak": bpv * n / (ms * 1e-3) / 1e9 / peak}
        del flush
    for _ in range(3):
        ctx.probe_read(cube_t, n, stream=stream)
    probe_ms = timed(lambda: ctx.probe_read(cube_t, n, stream=stream), args.steps)
    read_peak = 4.0 * n / (probe_ms * 1e-3) / 1e9

    # per-kernel durations, live, with CUDA events on the launching stream (cube_profile_*)
    ctx.profile_reset()
    ctx.profile(True)
    for _ in range(args.steps):
        step()
    torch.cuda.synchronize()
    prof = ctx.profile_read()
    ctx.profile(False)
    clocks = sampler.stop() if sampler else None
    streams_cube = {"moments", "moments_coarse", "histogram", "select_pass0", "select_pass1", "hist_select"}
    tot_k = sum(ms for ms, _ in prof.values()) or 1.0
    # a launch that returns at once (an enqueued fallback whose turn did not come: DESIGN.md sec. 4) has read nothing:
    # it gets no bandwidth figure (anything "faster" than twice the read probe cannot have streamed the cube)
    kernels = {k: {"launches": c, "avg_ms": ms / c, "share": ms / tot_k,
                   "achieved_gbs": (ALGO_BYTES_PER_VOXEL * n / (ms / c * 1e-3) / 1e9)
                   if k in streams_cube and ms / c > 0.5 * probe_ms else None}
               for k, (ms, c) in prof.items() if c}
    dom = max(kernels, key=lambda k: kernels[k]["share"])
    achieved = kernels[dom]["achieved_gbs"]
    roofline = {"bound": "hbm", "kernel": dom, "achieved": achieved, "peak": peak, "unit": "GB/s",
                "frac": achieved / peak if achieved else None, "traffic": None, "peak_source": peak_src,
                "algorithmic_bytes_per_launch": ALGO_BYTES_PER_VOXEL * n,
                "read_probe_gbs": read_peak, "frac_of_read_probe": achieved / read_peak if achieved else None,
                "per_kernel": kernels}
    tr = os.path.join(ROOT, "profiles", "traffic.json")
    if os.path.exists(tr):
        try:
            roofline["traffic"] = json.load(open(tr)).get(name, {}).get(dom)
        except Exception:
            pass

    # median / moments sanity (device results of the last step), reported for the record
    med = float(out_f.cpu()[0])
    mom = cube.MomentsT.from_buffer_copy(out_m.cpu().numpy().tobytes()).as_dict()

    # end to end: host cube in pinned memory -> cube_stats_host (H2D inside the timed region)
    e2e = None
    if not args.no_e2e:
        host = torch.empty(n, dtype=torch.float32, pin_memory=True)
        host.copy_(cube_t)
        torch.cuda.synchronize()
        ctx.host_workspace(resident_bytes=n * 4, chunk_bytes=128 << 20)
        e_steps = max(2, min(args.steps, 5))
        ctx.stats_host(host, nx, ny, nz, nb, lo, hi)                    # warm-up
        barrier()
        t0 = time.perf_counter()
        for _ in range(e_steps):
            m_e, b_e, o_e, med_e = ctx.stats_host(host, nx, ny, nz, nb, lo, hi)
        torch.cuda.synchronize()
        e_ms = (time.perf_counter() - t0) * 1e3
        e_ms_max, e_units = aggregate_over_ranks(dist if world > 1 else None, e_ms, n * e_steps, dev)
        assert np.float32(med_e).tobytes() == np.float32(med).tobytes()
        e2e = {"value": e_units / (e_ms_max * 1e-3), "unit": "voxels/s", "h2d_bytes_per_step": n * 4,
               "d2h_bytes_per_step": 40 + nb * 8 + 16 + 4, "ms_per_step": e_ms_max / e_steps,
               "h2d_gbs": n * 4 / (e_ms_max / e_steps * 1e-3) / 1e9,
               "timer": "host perf_counter around the synchronous cube_stats_host call (pinned host cube, "
                        "128 MiB chunks, cube kept resident after sweep 1)"}
        ctx.host_workspace(0, 1 << 20)
        del host

    cpu = None
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        planes = sample_planes(cfg, args.cpu_voxels)
        a_host = cube_t[:nx * ny * planes].cpu().numpy()          # the very bytes the GPU path was timed on
        v, desc, dt = oracle_sample(name, cfg, args.cpu_voxels, a=a_host)
        cpu = {"value": v, "unit": "voxels/s", "cores": 1, "kind": "oracle", "sample": desc, "seconds": dt}

    if rank == 0:
        value = total_units / (total_ms * 1e-3)
        line = {"metric": METRIC, "value": value, "unit": "voxels/s", "n_gpus": world, "steps": args.steps,
                "warmup": args.warmup, "ms_per_step": total_ms / args.steps, "higher_is_better": True,
                "scaling": "weak", "vs_baseline": None, "dtype": "f32", "data": "synthetic",
                "config": {"workload": workload_desc(name, cubegen.CONFIGS[name]),
                           "l2": "input (%.2f GiB) is larger than the 126 MB L2" % (n * 4 / 2 ** 30)
                           if n * 4 > (256 << 20) else "input fits L2: warm-L2 numbers",
                           "parallelism": "replicas only (one independent cube per GPU)" if world > 1 else "1 GPU",
                           "step": "one cube_stats call = moments + histogram + exact lower median in two reads of "
                                   "the cube (pass A moments+digit, pass B histogram+digit+compaction, pass C on "
                                   "the candidates); the per-entry-point timings are under 'ops'"},
                "e2e": e2e, "gpu_launches": launches, "clocks": clocks, "roofline": roofline,
                "cpu_baseline": cpu,
                "result_check": {"median": med, "count": mom["count"], "mean": mom["mean"], "std": mom["std"]},
                "ops": ops}
        if ops_cold is not None:
            line["ops_cold_l2"] = ops_cold
            line["config"]["l2"] = ("input fits L2: 'value' and 'ops' are warm-L2 numbers (back-to-back calls); "
                                    "'ops_cold_l2' flushes L2 (512 MiB written) before every repetition")
        print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()
    return 0


if __name__ == "__main__":
    sys.exit(main())
