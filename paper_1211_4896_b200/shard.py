"""Z-slab sharding of ONE cube over several GPUs: one process and one ``Context`` per
GPU, the collectives through ``torch.distributed`` (NCCL over NVLink on a GPU node).

This is the paper's client/server decomposition: every merge on the statistics path is associative
and commutative, so each rank reduces its own slab with the single-GPU kernels and only O(bins)
counters cross the links -- an all-gather of one 40-byte moments record per rank, one all-reduce of the histogram and
three all-reduces of 64 KiB of digit counts, against the paper's ~31 rounds of five scalars for Torben's median
(PAPER.md:294-296); every rank reads its slab twice (8 B per voxel), as cube_stats reads the cube.  All payloads are latency-bound; every step is enqueued on one stream and nothing synchronises
the host.

Plumbing only: every arithmetic step (accumulation, record merge, bucket location) runs in libcube's kernels; this
module owns no formula.  ``ShardedStats`` is written as explicit phases (local pass -> combine -> advance) so that the
same code drives real ranks (``run``) and the single-process lock-step emulation used by the tests.
"""
import torch

from . import SHARD_DIGITS, SHARD_RECORD_BYTES, MAX_BINS, RANGE_MINMAX


def slab_bounds(nz, world, rank):
    """Contiguous z-planes [z0, z1) of ``rank``: the first ``nz % world`` ranks take one plane more.  No overlap
    (the paper's overlapping boundaries exist only for rendering and must not be counted twice)."""
    base, extra = divmod(int(nz), int(world))
    z0 = rank * base + min(rank, extra)
    return z0, z0 + base + (1 if rank < extra else 0)


class _DeviceView:
    """Wraps a raw device address as a CUDA array (``__cuda_array_interface__``) so that torch can alias it."""

    def __init__(self, ptr, nbytes):
        self.__cuda_array_interface__ = {"shape": (nbytes,), "typestr": "|u1", "data": (ptr, False), "version": 2}


def alias(ptr, nbytes, dtype, device):
    """torch tensor aliasing ``nbytes`` of device memory at ``ptr`` (no copy)."""
    return torch.as_tensor(_DeviceView(ptr, nbytes), device=device).view(dtype)


class ShardedStats:
    """One rank's side of a sharded moments + histogram + exact-median run.

    With the median the slab is read twice, like the cube in ``cube_stats`` (8 B per voxel): ``stage`` 0 = moments +
    first select digit (libcube's fused pass A), 1 = histogram + second digit + candidate compaction (fused pass B),
    2 = last digit on this rank's own candidates (counted once inside ``advance()``; the slab is read a third time
    only if they did not fit the candidate buffer -- decided on the device).  Without the median: one stage, moments
    and histogram.  Per stage: ``local_pass()`` -> combine ``payload()`` across ranks -> ``advance()``.
    """

    def __init__(self, ctx, slab, nvox, nbins, lo, hi, want_median=True, flags=0, stream=None, device=None):
        self.ctx, self.slab, self.nvox = ctx, slab, int(nvox)
        self.nbins, self.flags, self.want_median = int(nbins), flags, bool(want_median)
        self.device = device if device is not None else torch.device("cuda", torch.cuda.current_device())
        self.stream = stream if stream is not None else torch.cuda.current_stream(self.device).cuda_stream
        b = ctx.shard_buffers()
        self.record = alias(b["record"], SHARD_RECORD_BYTES, torch.uint8, self.device)
        self.bins = alias(b["bins"], MAX_BINS * 8, torch.int64, self.device)[:max(self.nbins, 0)]
        self.outside = alias(b["outside"], 16, torch.int64, self.device)
        self.digits = alias(b["digits"], SHARD_DIGITS * 8, torch.int64, self.device)
        self.stage, self.more = 0, True
        # lo=None: histogram over [min, max] of the WHOLE cube (the merged records), resolved on the device
        self.minmax = bool(self.nbins) and lo is None
        if self.minmax:
            ctx.ooc_begin(self.nbins, 0.0, 0.0, self.want_median, self.stream, flags=RANGE_MINMAX)
        else:
            ctx.ooc_begin(self.nbins, lo if self.nbins else 0.0, hi if self.nbins else 0.0, self.want_median, self.stream)

    def local_pass(self):
        if self.nvox:
            self.ctx.ooc_brick(self.slab, self.nvox, self.stream)

    def payload(self):
        """-> (record to all-gather or None, [tensors to all-reduce SUM])."""
        hist = [self.bins, self.outside] if self.nbins else []
        two_stage_hist = self.want_median or self.minmax          # the histogram is accumulated in stage 1 then
        digits = [self.digits] if self.want_median else []
        if self.stage == 0:
            return self.record, (digits if two_stage_hist else hist)
        return None, (hist if self.stage == 1 and two_stage_hist else []) + digits

    def merge_records(self, gathered, world):
        self.ctx.shard_merge_records(gathered, world, self.flags, self.stream)

    def advance(self):
        self.more = self.ctx.shard_advance(self.stream)
        self.stage += 1
        return self.more

    def result(self):
        """-> (moments dict, bins, outside, median) on the host (synchronises)."""
        return self.ctx.ooc_result(self.nbins, self.flags, self.want_median, self.stream)


def run(ctx, slab, nvox, nbins, lo, hi, want_median=True, flags=0, group=None, stream=None, device=None):
    """SPMD driver: call on every rank with its own slab (``nvox`` may be 0).  Uses torch's current stream; with the
    NCCL backend the collectives are enqueued on it, with gloo (CPU tensors are not supported here) it is an error.
    -> (moments dict, bins, outside, median), identical on every rank."""
    import torch.distributed as dist

    use_dist = dist.is_initialized()
    world = dist.get_world_size(group) if use_dist else 1
    st = ShardedStats(ctx, slab, nvox, nbins, lo, hi, want_median, flags, stream=stream, device=device)
    while st.more:
        st.local_pass()
        record, sums = st.payload()
        if record is not None:
            if use_dist:
                gathered = torch.empty(world * SHARD_RECORD_BYTES, dtype=torch.uint8, device=st.device)
                dist.all_gather_into_tensor(gathered, record, group=group)
            else:
                gathered = record
            st.merge_records(gathered, world)
        if use_dist:
            for t in sums:
                dist.all_reduce(t, op=dist.ReduceOp.SUM, group=group)
        st.advance()
    return st.result()
