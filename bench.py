#!/usr/bin/env python
"""bench.py -- headline benchmark of libcube (BASELINE.json metric: voxels/s and % of HBM peak for
moments, histogram and exact median of a float32 cube).

A "step" is one pass of the whole hot path over the workload: ONE cube_stats call = moments +
histogram + exact lower median, two reads of the cube resident in HBM.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config cX] [--sub c1,c2,c4,c5|none] [--impl reference]
                    [--replicas]

N = 1 (default): the headline workload is the largest in-HBM configuration of BASELINE.json, c3 (2048 x 2048 x 4096,
64 GiB); the other configurations are measured in the same run and reported under "configs" (c1 warm and cold L2, c2
with the NEXT rows, c4, and the out-of-core c5 against the host-link roofline).  --config cX makes cX the headline and
drops the sub-records (unless --sub names some).
N > 1 (under torchrun): ONE cube sharded over the ranks as contiguous z-slabs (paper_1211_4896_b200/shard.py, NCCL:
all-gather of the moments records, all-reduce of histogram and digit counts), value = voxels of the one cube / max
over ranks of the device time, "scaling": "strong".  --replicas runs the old mode instead: every rank the whole hot
path on its own independent cube, "scaling": "weak".

Prints ONE JSON line (rank 0).  --impl reference times the CPU oracle (oracle/, as it stands, one thread) on a bounded
sample of the same workload.
"""
import argparse
import json
import math
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
HEADLINE = "c3"
METRIC = "voxels/s & % HBM peak for moments, histogram, exact median (float32 cube)"
# algorithmic bytes per voxel of each kernel kind, per launch (DESIGN.md sec. 4 / SURVEY.md sec. 8(d))
ALGO_BYTES_PER_VOXEL = 4.0
STREAMS_CUBE = {"moments", "moments_coarse", "histogram", "select_pass0", "select_pass1", "hist_select", "stats_small"}


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


def config_dict(name, world, mode):
    """The `config` object of the JSON line -- the same for our arm and the reference arm."""
    cfg = cubegen.CONFIGS[name]
    n = int(np.prod(cfg["dims"], dtype=np.int64))
    if name == "c5":
        l2 = "bricks (512 MiB) are larger than the 126 MB L2"
    elif n * 4 > (256 << 20):
        l2 = "input (%.2f GiB) is larger than the 126 MB L2" % (n * 4 / 2 ** 30)
    else:
        l2 = "input fits L2: warm-L2 numbers; 'ops_cold_l2' flushes L2 (512 MiB written) before every repetition"
    if world == 1:
        par = "1 GPU"
    elif mode == "sharded":
        par = "one cube sharded over %d GPUs as z-slabs (NCCL all-gather / all-reduce of O(bins) counters)" % world
    else:
        par = "replicas only (one independent cube per GPU)"
    return {"workload": workload_desc(name, cfg), "l2": l2, "parallelism": par,
            "step": "one cube_stats call = moments + histogram + exact lower median in two reads of the cube"}


def box_facts():
    model = ""
    try:
        for line in open("/proc/cpuinfo"):
            if line.startswith("model name"):
                model = line.split(":", 1)[1].strip()
                break
    except OSError:
        pass
    return {"nproc": os.cpu_count(), "cpu_model": model}


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
        sm, mx, pw, reasons = [], [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for line in self.f:
            t = [v.strip() for v in line.split(",")]
            if len(t) < 7:
                continue
            try:
                sm.append(float(t[0]))
                mx.append(float(t[1]))
                pw.append(float(t[2]))
            except ValueError:
                continue
            for nme, v in zip(names, t[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(nme)
        os.unlink(self.f.name)
        if sm:
            out = {"sm_mhz": float(np.median(sm)), "sm_max_mhz": float(max(mx)), "reasons": sorted(reasons),
                   "samples": len(sm), "power_w_median": float(np.median(pw)) if pw else None}
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
    what = "the whole cube" if a.size == nx * ny * nz else "first %d z-planes" % planes
    desc = "%s of %s (%d voxels): oracle moments + %d-bin histogram + median, 1 thread" % (what, name, a.size, nb)
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
    name = args.config or HEADLINE
    cfg = cubegen.CONFIGS[name]
    sv = reference_sample_voxels(args)
    oracle_sample(name, cfg, sv) if args.warmup > 0 else None     # one warm-up (page-in, build)
    vals, secs, desc = [], [], ""
    for _ in range(max(1, args.steps)):
        v, desc, dt = oracle_sample(name, cfg, sv)
        vals.append(v)
        secs.append(dt)
    value = float(np.mean(vals))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    mode = "replicas" if (args.replicas or world == 1) else "sharded"
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": "voxels/s", "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": float(np.mean(secs)) * 1e3,
            "higher_is_better": True, "scaling": "strong" if mode == "sharded" else "weak", "vs_baseline": None,
            "dtype": "f32", "data": "synthetic", "config": config_dict(name, world, mode),
            "cpu_baseline": dict({"value": value, "unit": "voxels/s", "cores": 1, "kind": "oracle", "sample": desc},
                                 **box_facts()),
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


def op_record(ms, n, bpv, peak):
    return {"ms": ms, "voxels_per_s": n / (ms * 1e-3), "algorithmic_bytes_per_voxel": bpv,
            "algorithmic_gbs": bpv * n / (ms * 1e-3) / 1e9, "frac_of_peak": bpv * n / (ms * 1e-3) / 1e9 / peak}


def traffic_of(name, kernel):
    """ncu dram__bytes_read.sum + dram__bytes_write.sum per launch, from the committed capture summary."""
    tr = os.path.join(ROOT, "profiles", "traffic.json")
    try:
        j = json.load(open(tr))
        return j.get(name, {}).get(kernel), j.get("_source", {}).get(name)
    except Exception:
        return None, None


# ------------------------------------------------------------------------------------------------ out of core (c5)
def measure_out_of_core(args, jobs, warm):
    """c5: 4096^3 (256 GiB) produced per 512^3 brick into pinned host staging buffers (generated on the device from
    the seed, copied D2H on the fill stream) and streamed H2D through cube_stats_stream.  One step = the whole job:
    moments + 4096-bin histogram + exact lower median over all 512 bricks.  -> record dict."""
    import torch
    import paper_1211_4896_b200 as cube

    torch.cuda.set_device(0)
    name = "c5"
    cfg = cubegen.CONFIGS[name]
    nx, ny, nz = cfg["dims"]
    n = nx * ny * nz
    brick = (512, 512, 512)
    bvox = brick[0] * brick[1] * brick[2]
    origins = cubegen.brick_grid(cfg, brick)
    nb, lo, hi = HIST[name]
    scr = [torch.empty(bvox, dtype=torch.float32, device="cuda"), torch.empty(bvox, dtype=torch.float32, device="cuda")]
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
            (scr[0] if i & 1 else d2).copy_(hp, non_blocking=True)
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

    results, secs = [], []
    sampler = None
    for it in range(warm + jobs):
        if it == warm:
            sampler = ClockSampler(0)
        l0 = ctx.launch_count
        torch.cuda.synchronize()
        t0 = time.perf_counter()
        m, b, o, med, info = ctx.stats_stream(len(origins), bvox, n, fill, nb, lo, hi)
        dt = time.perf_counter() - t0
        if it >= warm:
            secs.append(dt)
            results.append((m, med, info, ctx.launch_count - l0))
    clocks = sampler.stop() if sampler else None
    dt = float(np.mean(secs))
    m, med, info, launches = results[-1]
    h2d_gbs = info["h2d_bytes"] / dt / 1e9
    ctx.close()
    del scr
    torch.cuda.empty_cache()
    return {"workload": workload_desc(name, cfg) + "; out of core: 512 bricks of 512^3, %d kept in HBM after sweep 1, "
                        "the rest produced and streamed again in sweep 2" % min(nres, len(origins)),
            "ms_per_step": dt * 1e3, "voxels_per_s": n / dt, "jobs": jobs, "warmup_jobs": warm,
            "timer": "host perf_counter around the synchronous cube_stats_stream call (the job IS end to end: every "
                     "brick crosses the host link inside the timed region)",
            "e2e": {"value": n / dt, "unit": "voxels/s", "h2d_bytes_per_step": info["h2d_bytes"],
                    "d2h_bytes_per_step": 40 + nb * 8 + 16 + 4},
            "gpu_launches": launches, "clocks": clocks,
            "roofline": {"bound": "h2d", "kernel": "cudaMemcpyAsync H2D of the bricks (the kernels have ~100x slack)",
                         "achieved": h2d_gbs, "peak": h2d_peak, "unit": "GB/s", "frac": h2d_gbs / h2d_peak,
                         "traffic": None, "peak_source": "pinned H2D copy, 512 MiB x 16, two streams, measured in this run",
                         "sweeps": info["sweeps"]},
            "result_check": {"median": float(med), "count": m["count"], "mean": m["mean"], "std": m["std"],
                             "min": float(m["min"]), "max": float(m["max"])}}


# ------------------------------------------------------------------------------------------------ in-HBM configs
def measure_in_hbm(name, args, dev, rank, world, dist, steps, warmup, sustain_s, headline):
    """One in-HBM configuration on this rank's GPU: the fused step (sustained), the three entry points on their own,
    live per-kernel durations, the read probe; for the headline also cube_kth_multi, e2e and the oracle sample; for c2
    the NEXT rows; for c1 the cold-L2 repetitions.  -> (record, extras for the headline line)."""
    import torch
    import paper_1211_4896_b200 as cube

    cfg = dict(cubegen.CONFIGS[name])
    if world > 1:
        cfg["seed"] = replica_seed(cfg["seed"], rank)                    # independent replica per rank
    nx, ny, nz = cfg["dims"]
    n = nx * ny * nz
    nb, lo, hi = HIST[name]
    cube_t = torch.empty(n, dtype=torch.float32, device=dev)
    cubegen.generate_device(cfg, cube_t.data_ptr())
    torch.cuda.synchronize()
    peak, peak_src = measured_peak()

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

    def reps_for(fn, seconds, lo_reps=5, hi_reps=5000):
        est = timed(fn, 3)
        return int(min(hi_reps, max(lo_reps, math.ceil(seconds * 1e3 / max(est, 1e-3)))))

    # ---- the fused step.  The timed region is EXACTLY `steps` steps; before it, `warmup` steps and then as many more
    # as it takes to have run for `sustain_s` seconds, so that the clocks are those of a sustained run (power cap)
    for _ in range(warmup):
        step()
    torch.cuda.synchronize()
    # clocks / throttle reasons are sampled from here on: the same steps, run back to back, through the timed region
    sampler = ClockSampler(dev.index or 0) if (rank == 0 and headline) else None
    pre_steps, t_pre = 0, time.perf_counter()
    while time.perf_counter() - t_pre < sustain_s:
        for _ in range(max(1, steps // 4)):
            step()
        torch.cuda.synchronize()
        pre_steps += max(1, steps // 4)
    pre_s = time.perf_counter() - t_pre
    barrier()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    l0 = ctx.launch_count
    e0.record()
    for _ in range(steps):
        step()
    e1.record()
    barrier()
    launches = ctx.launch_count - l0
    local_ms = e0.elapsed_time(e1)
    total_ms, total_units = aggregate_over_ranks(dist if world > 1 else None, local_ms, n * steps, dev)

    # per-kernel durations of the same step, live, with CUDA events on the launching stream (cube_profile_*)
    ctx.profile_reset()
    ctx.profile(True)
    for _ in range(steps):
        step()
    torch.cuda.synchronize()
    prof = ctx.profile_read()
    ctx.profile(False)
    clocks = sampler.stop() if sampler else None

    # ---- the three operations of the metric through their own entry points (each its own timed region)
    ops = {}
    op_list = [("moments", op_moments, 4.0), ("histogram", op_histogram, 4.0), ("median", op_median, 8.0)]
    if name == "c4":
        op_list.append(("histogram_256", op_histogram_256, 4.0))
    if name in ("c2", "c3"):
        # BASELINE.json configs[2]: "median and k-th at k=N/100 and k=99N/100" -- three ranks of one cube in TWO
        # reads (cube_kth_multi) instead of three selections of two reads each
        cnt3 = int(ctx.moments(cube_t, nx, ny, nz)["count"])
        ks3 = [(cnt3 - 1) // 2, cnt3 // 100, 99 * cnt3 // 100]
        out_k3 = torch.zeros(3, dtype=torch.float32, device=dev)
        op_list.append(("median_p1_p99_multi", lambda: ctx.kth_multi(cube_t, nx, ny, nz, ks3, out=out_k3, stream=stream), 8.0))
    op_s = 0.4 if headline else 0.25
    for nm, fn, bpv in op_list:
        ops[nm] = op_record(timed(fn, reps_for(fn, op_s)), n, bpv, peak)
    if name == "c4" and not args.no_next:
        # MAD on the adversarial config: 30 % of the voxels share one deviation, so the second selection's first-digit
        # bucket is dense (PASS 1 counts in its hot loop, PASS 2 reads the cube a third time: 20 B per voxel moved)
        out_w4 = torch.zeros(2, dtype=torch.float32, device=dev)
        fn_mad = lambda: ctx.mad(cube_t, nx, ny, nz, median_out=out_w4[0:1], mad_out=out_w4[1:2], stream=stream)   # noqa: E731
        ops["next_mad"] = op_record(timed(fn_mad, reps_for(fn_mad, 0.25)), n, 16.0, peak)
    if name == "c2" and not args.no_next:
        ops.update(next_rows(ctx, cube_t, (nx, ny, nz), lo, hi, out_m, out_f, dev, stream, timed, reps_for, peak))
    ops["stats_fused"] = {"ms": total_ms / steps, "voxels_per_s": total_units / (total_ms * 1e-3) / world,
                          "algorithmic_bytes_per_voxel": 8.0,
                          "algorithmic_gbs": 8.0 * n / (local_ms / steps * 1e-3) / 1e9,
                          "frac_of_peak": 8.0 * n / (local_ms / steps * 1e-3) / 1e9 / peak}
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
            ops_cold[nm] = op_record(float(np.median(ts[3:])), n, bpv, peak)
        del flush
    probe = lambda: ctx.probe_read(cube_t, n, stream=stream)   # noqa: E731
    probe_ms = timed(probe, reps_for(probe, 0.2))
    read_peak = 4.0 * n / (probe_ms * 1e-3) / 1e9

    tot_k = sum(ms for ms, _ in prof.values()) or 1.0
    # a launch that returns at once (an enqueued fallback whose turn did not come: DESIGN.md sec. 4) has read nothing:
    # it gets no bandwidth figure (anything "faster" than twice the read probe cannot have streamed the cube)
    # algorithmic bytes per launch: 4 B per voxel for a kernel that reads the cube once, 8 for the one cooperative
    # launch that reads it twice (stats_small)
    reads = lambda k: 2.0 if k == "stats_small" else 1.0   # noqa: E731
    kernels = {k: {"launches": c, "avg_ms": ms / c, "share": ms / tot_k,
                   "achieved_gbs": (reads(k) * ALGO_BYTES_PER_VOXEL * n / (ms / c * 1e-3) / 1e9)
                   if k in STREAMS_CUBE and ms / c > 0.5 * probe_ms else None}
               for k, (ms, c) in prof.items() if c}
    dom = max(kernels, key=lambda k: kernels[k]["share"])
    achieved = kernels[dom]["achieved_gbs"]
    traffic, traffic_src = traffic_of(name, dom)
    roofline = {"bound": "hbm", "kernel": dom, "achieved": achieved, "peak": peak, "unit": "GB/s",
                "frac": achieved / peak if achieved else None, "traffic": traffic,
                "traffic_source": traffic_src, "peak_source": peak_src,
                "algorithmic_bytes_per_launch": reads(dom) * ALGO_BYTES_PER_VOXEL * n,
                "read_probe_gbs": read_peak, "frac_of_read_probe": achieved / read_peak if achieved else None,
                "per_kernel": kernels}

    med = float(out_f.cpu()[0])
    mom = cube.MomentsT.from_buffer_copy(out_m.cpu().numpy().tobytes()).as_dict()
    value = total_units / (total_ms * 1e-3)
    rec = {"workload": workload_desc(name, cubegen.CONFIGS[name]), "ms_per_step": total_ms / steps,
           "voxels_per_s": value, "algorithmic_gbs": 8.0 * n / (local_ms / steps * 1e-3) / 1e9,
           "frac_of_peak": 8.0 * n / (local_ms / steps * 1e-3) / 1e9 / peak, "steps": steps,
           "timing": {"warmup_steps": warmup, "sustain_steps_before_timing": pre_steps, "sustain_seconds": pre_s,
                      "timed_region_s": total_ms * 1e-3, "profiled_kernel_sum_ms_per_step": tot_k / steps},
           "gpu_launches": launches, "roofline": roofline, "ops": ops,
           "result_check": {"median": med, "count": mom["count"], "mean": mom["mean"], "std": mom["std"]}}
    if ops_cold is not None:
        rec["ops_cold_l2"] = ops_cold

    extras = {"clocks": clocks, "total_ms": total_ms, "value": value}
    # ---- end to end: host cube in pinned memory -> cube_stats_host (H2D inside the timed region)
    if (headline and not args.no_e2e) or (name in ("c1", "c2") and not args.no_e2e and world == 1):
        host = torch.empty(n, dtype=torch.float32, pin_memory=True)
        host.copy_(cube_t)
        torch.cuda.synchronize()
        ctx.host_workspace(resident_bytes=n * 4, chunk_bytes=128 << 20)
        e_steps = 2 if n * 4 > (8 << 30) else 5
        eflags = cube.RANGE_MINMAX if s_lo is None else 0
        ctx.stats_host(host, nx, ny, nz, nb, s_lo or 0.0, s_hi or 0.0, flags=eflags)        # warm-up
        barrier()
        t0 = time.perf_counter()
        for _ in range(e_steps):
            m_e, b_e, o_e, med_e = ctx.stats_host(host, nx, ny, nz, nb, s_lo or 0.0, s_hi or 0.0, flags=eflags)
        torch.cuda.synchronize()
        e_ms = (time.perf_counter() - t0) * 1e3
        e_ms_max, e_units = aggregate_over_ranks(dist if world > 1 else None, e_ms, n * e_steps, dev)
        assert np.float32(med_e).tobytes() == np.float32(med).tobytes()
        rec["e2e"] = {"value": e_units / (e_ms_max * 1e-3), "unit": "voxels/s", "h2d_bytes_per_step": n * 4,
                      "d2h_bytes_per_step": 40 + nb * 8 + 16 + 4, "ms_per_step": e_ms_max / e_steps, "steps": e_steps,
                      "h2d_gbs": n * 4 / (e_ms_max / e_steps * 1e-3) / 1e9,
                      "timer": "host perf_counter around the synchronous cube_stats_host call (pinned host cube, "
                               "128 MiB chunks, cube kept resident after sweep 1)"}
        ctx.host_workspace(0, 1 << 20)
        del host
    # ---- the oracle on the host cores: a bounded sample for the headline, the WHOLE cube for c1 and c2
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        if headline or name in ("c1", "c2"):
            full = name in ("c1", "c2")
            planes = nz if full else sample_planes(cfg, args.cpu_voxels)
            a_host = cube_t[:nx * ny * planes].cpu().numpy()          # the very bytes the GPU path was timed on
            v, desc, dt = oracle_sample(name, cfg, nx * ny * planes, a=a_host)
            rec["cpu_baseline"] = dict({"value": v, "unit": "voxels/s", "cores": 1, "kind": "oracle", "sample": desc,
                                        "seconds": dt}, **box_facts())
            del a_host
    ctx.close()
    del cube_t
    torch.cuda.empty_cache()
    return rec, extras


def next_rows(ctx, cube_t, dims, lo, hi, out_m, out_f, dev, stream, timed, reps_for, peak):
    """Timings of the NEXT rows on the cube at hand: MAD, clipped moments, sigma clipping, 30^3
    statistical mini-map (with the per-cell median), Alg. 1 of the paper, and the ray-casting kernels."""
    import torch
    nx, ny, nz = dims
    n = nx * ny * nz
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

    op_sigma_clip()
    torch.cuda.synchronize()
    clip_passes = int(out_i.item()) + 1          # the plain pass + the clipped passes actually made
    op_torben()
    torch.cuda.synchronize()
    torben_passes = int(out_i.item()) + 1        # the moments pass (Min, Max, n) + the passes of Alg. 1
    ops = {}
    for nm, fn, bpv in [("paper_alg1_torben_median", op_torben, 4.0 * torben_passes),
                        ("next_mad", op_mad, 16.0), ("next_clipped_moments", op_clipped, 4.0),
                        ("next_sigma_clip_3sigma_max5", op_sigma_clip, 4.0 * clip_passes),
                        ("next_minimap_30x30x30", op_minimap, 4.0)]:
        ms = timed(fn, reps_for(fn, 0.25))
        ops[nm] = {"ms": ms, "voxels_per_s": n / (ms * 1e-3), "algorithmic_bytes_per_voxel": bpv,
                   "algorithmic_gbs": bpv * n / (ms * 1e-3) / 1e9, "frac_of_peak": bpv * n / (ms * 1e-3) / 1e9 / peak}
    if hasattr(ctx, "minimap_median"):
        out_med = torch.zeros(mmx * mmy * mmz, dtype=torch.float32, device=dev)
        fn = lambda: ctx.minimap_median(cube_t, nx, ny, nz, part[0], part[1], part[2], out_med, stream=stream)   # noqa: E731
        ms = timed(fn, reps_for(fn, 0.25))
        ops["next_minimap_median_30x30x30"] = op_record(ms, n, 4.0, peak)
    # NEXT-4: ray casting into headless buffers, 1024 x 1024 pixels, the camera of PAPER.md:400 turned by 30 / 20 degrees
    w = h = 1024
    view = cubegen.view_orbit(dims, 30.0, 20.0, w, h, step=1.0)
    img = torch.zeros(w * h, dtype=torch.float32, device=dev)
    rgba = torch.zeros(w * h * 4, dtype=torch.float32, device=dev)
    table = np.zeros((256, 4), dtype=np.float32)
    table[:, 0] = np.linspace(0, 1, 256)
    table[:, 2] = np.linspace(1, 0, 256)
    table[:, 3] = np.linspace(0, 0.2, 256) ** 2
    tab_d = torch.from_numpy(table).to(dev)
    axis_view = cubegen.view_axis(dims, 2)
    for nm, fn, vw in [("next4_mip_1024x1024_yaw30_pitch20", lambda: ctx.render_mip(cube_t, nx, ny, nz, view, img, stream=stream), view),
                       ("next4_mip_along_z", lambda: ctx.render_mip(cube_t, nx, ny, nz, axis_view, img[:nx * ny], stream=stream), axis_view),
                       ("next4_transfer_function_256_levels", lambda: ctx.render_tf(cube_t, nx, ny, nz, view, tab_d, 0.004, 0.1, rgba, opacity_cut=0.98, stream=stream), view),
                       # the sigma-clipping transfer function on the 30^3 mini-map computed above (3 sigma)
                       ("paper_sigma_clipping_tf_3sigma_256_levels", lambda: ctx.render_sigma(cube_t, nx, ny, nz, view, out_cells, part[0], part[1], part[2], tab_d, 3.0, 12.0, rgba, opacity_cut=0.98, stream=stream), view)]:
        ms = timed(fn, reps_for(fn, 0.25, lo_reps=3))
        rays = vw["width"] * vw["height"]
        ops[nm] = {"ms": ms, "frames_per_s": 1e3 / ms, "rays": rays, "samples_per_ray": vw["nsteps"],
                   "voxels_per_s": n / (ms * 1e-3), "algorithmic_bytes_per_voxel": 4.0,
                   "algorithmic_gbs": 4.0 * n / (ms * 1e-3) / 1e9, "frac_of_peak": 4.0 * n / (ms * 1e-3) / 1e9 / peak}
    # the paper's measurement: the cube turned through 360 degrees ("2 degrees steps"; here every 10th
    # of those views), pitch 0 and pitch 20, MIP: mean, best and worst frame
    for pitch in (0.0, 20.0):
        for kind in ("mip", "transfer_function", "sigma_clipping_tf"):
            per_view = []
            for yaw in range(0, 360, 20):
                vw = cubegen.view_orbit(dims, float(yaw), pitch, w, h, step=1.0)
                if kind == "mip":
                    fn = lambda: ctx.render_mip(cube_t, nx, ny, nz, vw, img, stream=stream)   # noqa: E731
                elif kind == "transfer_function":
                    fn = lambda: ctx.render_tf(cube_t, nx, ny, nz, vw, tab_d, 0.004, 0.1, rgba, opacity_cut=0.98, stream=stream)   # noqa: E731
                else:
                    fn = lambda: ctx.render_sigma(cube_t, nx, ny, nz, vw, out_cells, part[0], part[1], part[2], tab_d, 3.0, 12.0, rgba, opacity_cut=0.98, stream=stream)   # noqa: E731
                per_view.append(timed(fn, 2))
            ms = sum(per_view) / len(per_view)
            ops["next4_%s_orbit_18_views_pitch%d" % (kind, int(pitch))] = {
                "ms": ms, "frames_per_s": 1e3 / ms, "ms_best_view": min(per_view), "ms_worst_view": max(per_view),
                "rays": w * h, "voxels_per_s": n / (ms * 1e-3), "algorithmic_bytes_per_voxel": 4.0,
                "algorithmic_gbs": 4.0 * n / (ms * 1e-3) / 1e9, "frac_of_peak": 4.0 * n / (ms * 1e-3) / 1e9 / peak}
    return ops


# ------------------------------------------------------------------------------------------------ sharded (N > 1)
def run_sharded(args, name):
    """One cube sharded over the ranks as contiguous z-slabs.  Every rank generates its
    own slab of the SAME cube (cubegen is keyed by global voxel index), reads it twice per step, and only O(bins)
    counters cross NVLink.  value = voxels of the one cube / max-over-ranks device time ("scaling": "strong")."""
    import torch
    import torch.distributed as dist
    import paper_1211_4896_b200 as cube
    from paper_1211_4896_b200 import shard

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)
    if not dist.is_initialized():
        if "MASTER_ADDR" not in os.environ:
            os.environ["MASTER_ADDR"] = "127.0.0.1"
            os.environ.setdefault("MASTER_PORT", "29511")
        dist.init_process_group("nccl", rank=rank, world_size=world, device_id=dev)
    cfg = cubegen.CONFIGS[name]
    nx, ny, nz = cfg["dims"]
    n = nx * ny * nz
    nb, lo, hi = HIST[name]
    z0, z1 = shard.slab_bounds(nz, world, rank)
    nvox = (z1 - z0) * nx * ny
    slab = torch.empty(max(nvox, 1), dtype=torch.float32, device=dev)
    if nvox:
        cubegen.generate_device(cfg, slab.data_ptr(), origin=(0, 0, z0), brick=(nx, ny, z1 - z0))
    torch.cuda.synchronize()
    ctx = cube.Context(scratch_bytes_hint=max(256 << 20, nvox * 4 // 16))
    res = [None]

    def step():
        res[0] = shard.run(ctx, slab, nvox, nb, lo, hi)

    for _ in range(max(args.warmup, 3)):
        step()
    sampler = ClockSampler(local_rank) if rank == 0 else None
    t_pre = time.perf_counter()
    while time.perf_counter() - t_pre < 1.0:
        step()
    dist.barrier()
    torch.cuda.synchronize()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    l0 = ctx.launch_count
    e0.record()
    for _ in range(args.steps):
        step()
    e1.record()
    dist.barrier()
    torch.cuda.synchronize()
    launches = ctx.launch_count - l0
    total_ms, _ = aggregate_over_ranks(dist, e0.elapsed_time(e1), 0, dev)
    clocks = sampler.stop() if sampler else None
    peak, peak_src = measured_peak()
    m, b, o, med = res[0]
    if rank == 0:
        ms = total_ms / args.steps
        value = n / (ms * 1e-3)
        per_gpu_gbs = 8.0 * (n / world) / (ms * 1e-3) / 1e9
        line = {"metric": METRIC, "value": value, "unit": "voxels/s", "n_gpus": world, "steps": args.steps,
                "warmup": args.warmup, "ms_per_step": ms, "higher_is_better": True, "scaling": "strong",
                "vs_baseline": None, "dtype": "f32", "data": "synthetic", "config": config_dict(name, world, "sharded"),
                "e2e": None, "gpu_launches": launches, "clocks": clocks,
                "roofline": {"bound": "hbm", "kernel": "the two reads of a rank's slab (fused pass A, fused pass B)",
                             "achieved": per_gpu_gbs, "peak": peak, "unit": "GB/s", "frac": per_gpu_gbs / peak,
                             "traffic": None, "peak_source": peak_src,
                             "note": "per GPU: 8 B x voxels of one slab / step time (collectives included)"},
                "cpu_baseline": None,
                "result_check": {"median": float(med), "count": m["count"], "mean": m["mean"], "std": m["std"]},
                "collectives_per_step": "1 all-gather (40 B per rank) + all-reduce of %d bins + 3 all-reduces of 8192 digit counts" % nb}
        print(json.dumps(line))
    ctx.close()
    if world > 1 or dist.is_initialized():
        dist.destroy_process_group()
    return 0


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=None, help="timed steps (default: 40 for c3, 100 otherwise)")
    ap.add_argument("--warmup", type=int, default=None, help="untimed warm-up steps (default 3)")
    ap.add_argument("--config", default=None, choices=sorted(cubegen.CONFIGS),
                    help="headline workload (default c3, with the other configs as sub-records at N=1)")
    ap.add_argument("--sub", default=None, help="comma list of configs measured as sub-records ('none': none; "
                                                "default c1,c2,c4,c5 when --config is not given, else none)")
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--replicas", action="store_true", help="N > 1: independent replicas instead of one sharded cube")
    ap.add_argument("--sharded", action="store_true", help="force the sharded path (also at N = 1)")
    ap.add_argument("--ref-voxels", type=int, default=0,
                    help="voxels of the bounded oracle sample per step of --impl reference (0 = sized from --steps)")
    ap.add_argument("--cpu-voxels", type=int, default=1 << 29,
                    help="voxels of the cpu_baseline sample (first z-planes of the timed device cube)")
    ap.add_argument("--resident-gib", type=float, default=128.0, help="c5: GiB of bricks kept in HBM after sweep 1")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-next", action="store_true", help="skip the timings of the NEXT rows (MAD, clipping, mini-map, ray casting)")
    args = ap.parse_args()
    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    name = args.config or HEADLINE
    if args.steps is None:
        args.steps = 1 if name == "c5" else 40 if name == "c3" else 100
    if args.warmup is None:
        args.warmup = 1 if name == "c5" else 3
    if args.impl == "reference":
        return run_reference(args)

    import torch
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: libcube has no CPU fallback")
    if name == "c5":
        if world > 1:
            raise SystemExit("--config c5 is a single-GPU job")
        rec = measure_out_of_core(args, max(1, args.steps), args.warmup)
        cpu = None
        if not args.no_cpu_baseline:
            v, desc, cdt = oracle_sample(name, cubegen.CONFIGS[name], min(args.cpu_voxels, 1 << 28))
            cpu = dict({"value": v, "unit": "voxels/s", "cores": 1, "kind": "oracle", "sample": desc, "seconds": cdt},
                       **box_facts())
        line = {"metric": METRIC, "value": rec["voxels_per_s"], "unit": "voxels/s", "n_gpus": 1, "steps": args.steps,
                "warmup": args.warmup, "ms_per_step": rec["ms_per_step"], "higher_is_better": True, "scaling": "weak",
                "vs_baseline": None, "dtype": "f32", "data": "synthetic", "config": config_dict(name, 1, "replicas"),
                "e2e": rec["e2e"], "gpu_launches": rec["gpu_launches"], "clocks": rec["clocks"],
                "roofline": rec["roofline"], "cpu_baseline": cpu, "result_check": rec["result_check"]}
        print(json.dumps(line))
        return 0
    if args.sharded or (world > 1 and not args.replicas):
        return run_sharded(args, name)

    import torch.distributed as dist
    args.warmup = max(args.warmup, 3)
    torch.cuda.set_device(local_rank)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local_rank))
    dev = torch.device("cuda", local_rank)
    rec, extras = measure_in_hbm(name, args, dev, rank, world, dist, args.steps, args.warmup, 1.0, True)
    subs = {}
    sub_names = [] if (args.config or world > 1) else ["c1", "c2", "c4", "c5"]
    if args.sub is not None:
        sub_names = [] if args.sub == "none" else [s for s in args.sub.split(",") if s and s != name]
    for sn in sub_names:
        if sn == "c5":
            subs[sn] = measure_out_of_core(args, 1, 0)
        else:
            n_sub = int(np.prod(cubegen.CONFIGS[sn]["dims"], dtype=np.int64))
            k = 200 if n_sub * 4 < (1 << 30) else 100 if n_sub * 4 < (8 << 30) else 30
            subs[sn], _ = measure_in_hbm(sn, args, dev, rank, world, dist, k, 3, 0.5, False)

    if rank == 0:
        line = {"metric": METRIC, "value": extras["value"], "unit": "voxels/s", "n_gpus": world, "steps": args.steps,
                "warmup": args.warmup, "ms_per_step": rec["ms_per_step"], "higher_is_better": True,
                "scaling": "weak", "vs_baseline": None, "dtype": "f32", "data": "synthetic",
                "config": config_dict(name, world, "replicas"),
                "e2e": rec.get("e2e"), "gpu_launches": rec["gpu_launches"], "clocks": extras["clocks"],
                "roofline": rec["roofline"], "cpu_baseline": rec.get("cpu_baseline"),
                "result_check": rec["result_check"], "timing": rec["timing"], "ops": rec["ops"]}
        if "ops_cold_l2" in rec:
            line["ops_cold_l2"] = rec["ops_cold_l2"]
        if subs:
            line["configs"] = subs
        print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()
    return 0


if __name__ == "__main__":
    sys.exit(main())
