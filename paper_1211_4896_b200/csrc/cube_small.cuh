// cube_small.cuh -- cube_stats for cubes that fit the L2 cache (config 1 of BASELINE.json: 256^3, 64 MiB) in ONE
// cooperative launch instead of three dependent ones.
//
// A 64 MiB cube streams in ~10 us; the three launches of the general path (pass A, pass B, pass C) then cost more in
// launch gaps and serial tails -- the last CTA of pass A alone merging 592 partials and scanning 8192 digit bins while
// 147 SMs idle -- than in reading (73 us against a 2 x 13 us floor, profiles/r1_v11_c2.md sec. 3).  Here all CTAs are
// resident (cooperative launch), the passes are separated by grid barriers, and what used to be a last-CTA tail is
// done by EVERY CTA for itself: each CTA merges the per-CTA partials and locates the first-digit bucket redundantly
// (the inputs are a few KiB in L2), so nobody waits for one CTA's chain of dependent L2 round trips and no
// selection state crosses a launch boundary.  The kernels' arithmetic is that of the general path -- the same functors
// (MomentsF, HistFastF / HistF, SelectF), the same merge, the same bucket location -- so the results are bit for bit
// the same integers; mean / std differ in the last bits only through the grid size (tolerance R20).
//
//   phase A  moments + first digit (pass A); the histogram bins are zeroed on the way  | grid barrier
//            every CTA: locate the median's first-digit bucket (from 256 chunk totals)
//   phase B  histogram + second digit + candidate compaction (pass B), from L2        | grid barrier
//            candidates fit (the usual case): CTA 0 counts the last digit on them and finishes; the other CTAs exit
//            else: every CTA locates the second-digit bucket, counts the last digit over the cube | grid barrier, CTA 0 finishes
#pragma once
#include "cube_fused.cuh"

namespace cube {

struct SmallArgs {
    const float* d; uint64_t n;
    int nbins; float lo, hi, scale; int minmax; unsigned flags;
    Partial* partials; Partial* acc; unsigned long long* nvox_acc; MomentsOut* mom_out; MomentsOut* out_user;
    unsigned long long* coarse;      // kDigitBins first-digit counts of THIS call: all zero on entry, left all zero
    unsigned long long* coarse_keep; // where they are kept for CUBE_REUSE_COARSE: copied there (and `coarse` zeroed for
                                     // the next call) by the CTAs that have nothing else left to do
    unsigned long long* chunk_tot;   // kDigitBins / 32 totals of 32 consecutive first digits, in KEY order; zero on
                                     // entry, left zeroed
    unsigned long long* gdigits;     // kDigitBins: [0, 1024) second digit, [4096, 4608) last digit; left zeroed
    unsigned long long* gout;        // [outside (2)][bins (nbins)]
    SelectState* sel; uint32_t* cand; unsigned long long cand_cap; float* result_out;
    unsigned long long k; int use_median;   // the rank asked for: the lower median of the non-NaN voxels, or k
    unsigned long long* bins_user;   // the caller's bins / outside when the device can reach them (no copy is enqueued then)
    unsigned long long* outside_user;
    unsigned int* bar;               // [0] the barrier counter (only grows), [1] its value when this launch starts: read
                                     // by every CTA at its start, advanced by CTA 0 at the very end -- no state of the
                                     // call lives on the host, so a CUDA graph holding the launch can be replayed
    unsigned int* ext;               // [0] = smallest key seen (0xFFFFFFFF between calls), [1] = largest (0), [2] = ticket (0)
    unsigned long long* tstamp;      // debug (-DCUBE_SMALL_TIMING): %globaltimer of CTA 0 at the phase boundaries
};

constexpr int kSmallMaxBins = 4096;
constexpr int kSmallDigit2Off = 4096;
constexpr int small_smem(int nbins) {
    const int b = (nbins + 2 + kBins1 + 1 + (kThreads / 32) * ((int)kStageCap + 1)) * 4;
    const int a = (kDigitBins + 1) * 4;
    return a > b ? a : b;
}

// Grid barrier for a cooperative launch (all CTAs resident).  The counter only grows: arrival number base + k * grid
// ends barrier k, so nothing has to be reset while CTAs may still be spinning.
__device__ __forceinline__ void small_grid_sync(unsigned int* bar, unsigned int target) {
    __syncthreads();
    if (threadIdx.x == 0) {
        __threadfence();
        atomicAdd(bar, 1u);
        unsigned int v;
        do {
            asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(v) : "l"(bar) : "memory");
        } while ((int)(v - target) < 0);
    }
    __syncthreads();
}
// The two halves of small_grid_sync, for work that can be done between arriving and being released.
__device__ __forceinline__ void small_grid_wait(unsigned int* bar, unsigned int target) {
    if (threadIdx.x == 0) {
        unsigned int v;
        do {
            asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(v) : "l"(bar) : "memory");
        } while ((int)(v - target) < 0);      // the acquire load orders what follows (bar.sync carries it to the CTA)
    }
    __syncthreads();
}
// Arrive without waiting (a CTA that is done): every launch makes the same number of arrivals, which is what the
// host advances the barrier base by.
__device__ __forceinline__ void small_grid_arrive(unsigned int* bar) {
    __syncthreads();
    if (threadIdx.x == 0) { __threadfence(); atomicAdd(bar, 1u); }
}
constexpr unsigned kSmallBarriers = 3;

// First-digit bucket of the median from the chunk totals (256 sums of 32 consecutive digits, key order) and the one
// chunk that holds the rank: two dependent L2 round trips of ONE warp instead of a scan of all 8192 bins.  Called by
// warp 0 of every CTA; fills the CTA's own SelectState.
__device__ __forceinline__ void small_locate0(SelectState* st, const unsigned long long* __restrict__ coarse,
                                              const unsigned long long* __restrict__ chunk_tot, unsigned long long cand_cap,
                                              unsigned long long k_asked, int use_median) {
    constexpr int NCH = kDigitBins / 32, PER = NCH / 32;
    const int lane = threadIdx.x & 31;
    unsigned long long c[PER], mine = 0;
#pragma unroll
    for (int j = 0; j < PER; ++j) { c[j] = __ldcg(&chunk_tot[lane * PER + j]); mine += c[j]; }
    unsigned long long incl = mine;
#pragma unroll
    for (int off = 1; off < 32; off <<= 1) {
        const unsigned long long u = __shfl_up_sync(0xffffffffu, incl, off);
        if (lane >= off) incl += u;
    }
    const unsigned long long total = __shfl_sync(0xffffffffu, incl, 31);
    const unsigned long long k = use_median ? (total ? (total - 1) / 2 : 0) : k_asked;
    const bool invalid = k >= total;                  // also: no non-NaN voxel
    unsigned long long excl = incl - mine;
    int ch = -1;
    unsigned long long kin = 0;
#pragma unroll
    for (int j = 0; j < PER; ++j) {
        if (c[j] && excl <= k && k < excl + c[j]) { ch = lane * PER + j; kin = k - excl; }   // exactly one lane (total > 0)
        excl += c[j];
    }
    const unsigned ball = __ballot_sync(0xffffffffu, ch >= 0);
    if (lane == 0) {
        st->count = total; st->invalid = invalid ? 1u : 0u; st->use_median = use_median ? 1u : 0u; st->cand_n = 0; st->cand_cap = cand_cap;
        st->cand_done = 0u; st->k = k; st->prefix = 0u; st->result = __int_as_float(0x7fc00000); st->bucket_n = 0ull;
    }
    if (!ball) return;
    const int src = __ffs(ball) - 1;
    ch = __shfl_sync(0xffffffffu, ch, src);
    kin = __shfl_sync(0xffffffffu, kin, src);
    const uint32_t digit = (uint32_t)ch * 32u + (uint32_t)lane;
    const unsigned long long x = __ldcg(&coarse[raw_of_digit(digit)]);
    unsigned long long inc2 = x;
#pragma unroll
    for (int off = 1; off < 32; off <<= 1) {
        const unsigned long long u = __shfl_up_sync(0xffffffffu, inc2, off);
        if (lane >= off) inc2 += u;
    }
    const unsigned long long ex2 = inc2 - x;
    __syncwarp();
    if (x && ex2 <= kin && kin < inc2) { st->prefix = digit; st->k = kin - ex2; st->bucket_n = x; }   // exactly one lane
}

#ifdef CUBE_SMALL_TIMING
#define SMALL_T(i) do { if (a.tstamp && blockIdx.x == 0 && threadIdx.x == 0) { unsigned long long t_; asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t_)); a.tstamp[i] = t_; } } while (0)
// per-CTA stamps (slot i < 8 of CTA b at tstamp[16 + 8 b + i])
#define SMALL_TC(i) do { if (a.tstamp && threadIdx.x == 0) { unsigned long long t_; asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t_)); a.tstamp[16 + 8 * blockIdx.x + (i)] = t_; } } while (0)
#else
#define SMALL_T(i) do { } while (0)
#define SMALL_TC(i) do { } while (0)
#endif

__global__ void __launch_bounds__(kThreads, 3)
stats_small_kernel(SmallArgs a) {
    extern __shared__ __align__(16) uint32_t dyn_bins[];
    __shared__ Partial scratch[kThreads / 32];
    __shared__ SelectState s_sel;
    __shared__ unsigned long long scan_sm[kScanSmem];
    __shared__ MomentsOut s_mom;
    __shared__ uint32_t s_out[2];
    __shared__ uint32_t s_ext[2];
    __shared__ int s_last;
    __shared__ Partial parked[kThreads];          // the threads' moments of phase A, reduced while waiting at barrier B
    const unsigned grid = gridDim.x;
    const unsigned gtid = blockIdx.x * kThreads + threadIdx.x, gthreads = grid * kThreads;
    const unsigned bar_base = __ldcg(&a.bar[1]);      // CTA 0 rewrites it behind barrier B, which needs every CTA's arrival

    SMALL_T(0);
    SMALL_TC(0);
    // ---- phase 0 (no barrier): what phase B accumulates into is zeroed now -- two grid barriers lie in between; the
    // first-digit bins and the chunk totals arrive zeroed (every call leaves the next call's arrays that way)
    for (unsigned i = gtid; i < (unsigned)a.nbins + 2u; i += gthreads) a.gout[i] = 0ull;
    if (gtid == 0) { a.sel->cand_n = 0ull; a.sel->cand_done = 0u; }
    SMALL_T(1);
    // ---- phase A: moments + first digit
    {
        MomentsF<kMomCoarse> f;
        f.sbins = smem_addr(dyn_bins);
        for (int i = threadIdx.x; i <= kDigitBins; i += kThreads) dyn_bins[i] = 0;
        if (threadIdx.x == 0) { s_ext[0] = 0xFFFFFFFFu; s_ext[1] = 0u; }
        __syncthreads();
        SMALL_TC(1);
        stream_cube<kThreads>(a.d, a.n, f);
        SMALL_T(2);
        SMALL_TC(2);
        f.unsubstitute();
        // Only the extrema are wanted before phase B (the [min, max] histogram range): they go to two global words by
        // atomics.  The threads' (n, mean, M2) are parked; their reduction over the CTA and the merge over the grid --
        // chains of dependent fp64 operations and L2 round trips -- leave the critical path: each CTA reduces its own
        // while it waits at barrier B, and the CTA that finishes last merges them all, beside CTA 0's last digit.
        {
            const Partial mine = f.partial();
            parked[threadIdx.x] = mine;
            const uint32_t wmin = __reduce_min_sync(0xffffffffu, mine.kmin), wmax = __reduce_max_sync(0xffffffffu, mine.kmax);
            if ((threadIdx.x & 31) == 0) { atomicMin(&s_ext[0], wmin); atomicMax(&s_ext[1], wmax); }
        }
        __syncthreads();
        if (threadIdx.x == 0) { atomicMin(&a.ext[0], s_ext[0]); atomicMax(&a.ext[1], s_ext[1]); }
        // flush: a warp takes chunks of 32 consecutive raw digits; their sum also goes to the chunk's total (a chunk of
        // raw digits IS a chunk of key-order digits: raw chunk r <-> key chunk r + 128 (positive) or 255 - r (negative))
        // (eight chunks per step: the loads and the warp sums of a step are independent, the loop is latency otherwise)
        constexpr int NCH = kDigitBins / 32, WARPS = kThreads / 32, STEP = 8;
        static_assert(NCH % (WARPS * STEP) == 0, "flush shape");
        const int lane = threadIdx.x & 31;
        for (int ch0 = threadIdx.x >> 5; ch0 < NCH; ch0 += WARPS * STEP) {
            uint32_t c[STEP], tot[STEP];
#pragma unroll
            for (int u = 0; u < STEP; ++u) c[u] = dyn_bins[(ch0 + u * WARPS) * 32 + lane];
#pragma unroll
            for (int u = 0; u < STEP; ++u) tot[u] = __reduce_add_sync(0xffffffffu, c[u]);
#pragma unroll
            for (int u = 0; u < STEP; ++u) {
                const int ch = ch0 + u * WARPS;
                if (c[u]) atomicAdd(&a.coarse[ch * 32 + lane], (unsigned long long)c[u]);
                if (lane == 0 && tot[u]) atomicAdd(&a.chunk_tot[ch < 128 ? ch + 128 : 255 - ch], (unsigned long long)tot[u]);
            }
        }
    }
    SMALL_TC(3);
    small_grid_sync(a.bar, bar_base + grid);
    SMALL_TC(4);

    SMALL_T(3);
    // ---- every CTA for itself: the first-digit bucket (warp 0) and the extrema (warp 1)
    {
        if (threadIdx.x < 32) small_locate0(&s_sel, a.coarse, a.chunk_tot, a.cand ? a.cand_cap : 0, a.k, a.use_median);
        if (threadIdx.x == 32) {
            s_mom.min = __uint_as_float(bits_of_key(__ldcg(&a.ext[0])));
            s_mom.max = __uint_as_float(bits_of_key(__ldcg(&a.ext[1])));
        }
        // meanwhile the other warps zero phase B's counters (phase A's are flushed: barrier A lies behind)
        if (threadIdx.x >= 64) {
            for (int i = threadIdx.x - 64; i < a.nbins + 2 + kBins1 + 1; i += kThreads - 64) dyn_bins[i] = 0;
            if (threadIdx.x < 66) s_out[threadIdx.x - 64] = 0;
        }
        __syncthreads();
        if (threadIdx.x == 0) s_mom.count = s_sel.count;     // all that hist_range() looks at: count, min, max
        __syncthreads();
    }

    SMALL_T(4);
    // ---- phase B: histogram + second digit + compaction (the cube comes from L2 now)
    {
        uint32_t* hbins = dyn_bins;
        uint32_t* sbins = dyn_bins + (a.nbins + 2);
        uint32_t* stage = sbins + (kBins1 + 1);
        float lo = a.lo, hi = a.hi, scale = a.scale;
        const bool range_ok = a.nbins == 0 || hist_range(a.minmax ? &s_mom : nullptr, a.nbins, lo, hi, scale);
        if (!range_ok) { lo = INFINITY; hi = -INFINITY; }   // nothing is in range: every counter stays 0
        SelView sv;
        sv.invalid = s_sel.invalid; sv.prefix = s_sel.prefix; sv.cand_n = &a.sel->cand_n; sv.cand_cap = a.cand ? a.cand_cap : 0;
        uint32_t below = 0, above = 0;
        if (a.nbins == 0) {                    // cube_median / cube_stats without a histogram: the select pass alone
            if (!sv.invalid) {
                SelectF<1, false> f;
                f.base = sv.prefix << kShift0; f.rawbase = raw_of_digit(sv.prefix) << kShift0; f.sbins = sbins;
                f.init_stage(stage, a.cand, sv.cand_n, sv.cand_cap);
                stream_cube<kThreads>(a.d, a.n, f);
                f.finish();
            }
        } else if (hist_use_fast(a.nbins, lo, hi, scale)) {
            HistFastF h;
            h.setup(lo, hi, scale, a.nbins, hbins, s_out);
            hist_select_run(a.d, a.n, h, sv, sbins, stage, a.cand, below, above);
        } else {
            HistF h;
            h.lo = lo; h.hi = hi; h.scale = scale; h.top = a.nbins - 1; h.sbins = hbins;
            hist_select_run(a.d, a.n, h, sv, sbins, stage, a.cand, below, above);
        }
        __syncthreads();
        SMALL_T(5);
        SMALL_TC(5);
        hist_flush_bins(hbins, a.nbins, a.gout + 2);
        for (int i = threadIdx.x; i < kBins1; i += kThreads) {
            const uint32_t c = sbins[i];
            if (c) atomicAdd(&a.gdigits[i], (unsigned long long)c);
        }
        if (range_ok) {
            if (below) atomicAdd(&s_out[0], below);
            if (above) atomicAdd(&s_out[1], above);
            __syncthreads();
            if (threadIdx.x < 2 && s_out[threadIdx.x]) atomicAdd(&a.gout[threadIdx.x], (unsigned long long)s_out[threadIdx.x]);
        } else if (blockIdx.x == 0 && threadIdx.x < 2) {
            a.gout[threadIdx.x] = ~0ull;  // marker: the [min,max] range was unusable
        }
    }
    SMALL_TC(6);
    small_grid_arrive(a.bar);
    {   // between arriving and being released: this CTA's moments, and -- for the CTA that is last -- the whole cube's
        const Partial p = partial_block_reduce(parked[threadIdx.x], scratch);
        if (threadIdx.x == 0) {
            a.partials[blockIdx.x] = p;
            __threadfence();
            s_last = atomicAdd(&a.ext[2], 1u) == grid - 1u;
        }
        __syncthreads();
        if (s_last) {
            __threadfence();
            const Partial m = partials_merge_block(a.partials, grid, scratch);
            if (threadIdx.x == 0) {
                MomentsOut o;
                moments_finalize(m, a.n, a.flags, &o);
                *a.acc = m; *a.nvox_acc = a.n; *a.mom_out = o;
                if (a.out_user) *a.out_user = o;
                a.ext[0] = 0xFFFFFFFFu; a.ext[1] = 0u; a.ext[2] = 0u;     // every CTA has read them: as the next call wants them
            }
        }
    }
    small_grid_wait(a.bar, bar_base + 2 * grid);
    SMALL_TC(7);

    SMALL_T(6);
    // ---- last digit
    const unsigned long long cn = __ldcg(&a.sel->cand_n);      // final: every CTA's appends precede its arrival
    const bool fits = a.cand != nullptr && cn <= a.cand_cap;   // the same on every CTA
    // housekeeping nobody waits for -- the first-digit counts (every CTA has read what it needed of them before barrier
    // B) move to where CUBE_REUSE_COARSE finds them and their array is zeroed for the next call; the histogram, complete
    // now, goes straight into the caller's buffers -- is left to the CTAs other than 0, whose chain of dependent round
    // trips ends the call
    if (grid == 1 || blockIdx.x != 0) {
        const unsigned hthreads = (grid == 1 ? 1u : grid - 1u) * kThreads;
        const unsigned htid = (grid == 1 ? 0u : blockIdx.x - 1u) * kThreads + threadIdx.x;
        for (unsigned i = htid; i < (unsigned)kDigitBins; i += hthreads) {
            a.coarse_keep[i] = __ldcg(&a.coarse[i]);
            a.coarse[i] = 0ull;
        }
        if (a.bins_user) {
            for (unsigned i = htid; i < (unsigned)a.nbins; i += hthreads) a.bins_user[i] = __ldcg(&a.gout[2 + i]);
            if (htid < 2) a.outside_user[htid] = __ldcg(&a.gout[htid]);
        }
    }
    if (fits && blockIdx.x != 0) { small_grid_arrive(a.bar); return; }
    SelectInit none;
    none.k = 0; none.cand_cap = 0; none.result_out = nullptr; none.use_median = 0; none.enabled = 0;
    select_scan_body<1, kThreads>(&s_sel, a.gdigits, 0, none, scan_sm);     // every remaining CTA: second-digit bucket
    __syncthreads();
    unsigned long long* g2 = a.gdigits + kSmallDigit2Off;
    {
        uint32_t* sbins = dyn_bins;
        for (int i = threadIdx.x; i <= kBins2; i += kThreads) sbins[i] = 0;
        __syncthreads();
        if (!s_sel.invalid) {
            if (fits) {
                SelectF<2, false> f;
                f.base = s_sel.prefix << kBits2; f.sbins = sbins;
                for (uint64_t i0 = 0; i0 < cn; i0 += 8 * kThreads) {      // eight loads in flight per thread
                    uint32_t key[8];
#pragma unroll
                    for (int u = 0; u < 8; ++u) {
                        const uint64_t i = i0 + (uint64_t)u * kThreads + threadIdx.x;
                        key[u] = i < cn ? __ldcg(a.cand + i) : 0u;
                    }
#pragma unroll
                    for (int u = 0; u < 8; ++u)
                        if (i0 + (uint64_t)u * kThreads + threadIdx.x < cn) f.key(key[u]);
                }
            } else {   // the bucket did not fit the candidate buffer: the cube once more, all CTAs
                const uint32_t top = s_sel.prefix >> kBits1;
                if (digit_may_hold_nan(top)) {
                    SelectF<2, true> f; f.base = s_sel.prefix << kBits2; f.sbins = sbins;
                    stream_cube<kThreads>(a.d, a.n, f);
                } else {
                    SelectF<2, false> f; f.base = s_sel.prefix << kBits2; f.sbins = sbins;
                    stream_cube<kThreads>(a.d, a.n, f);
                }
            }
        }
        __syncthreads();
        if (!fits) {
            for (int i = threadIdx.x; i < kBins2; i += kThreads) {
                const uint32_t c = sbins[i];
                if (c) atomicAdd(&g2[i], (unsigned long long)c);
            }
        }
    }
    if (!fits) {
        small_grid_sync(a.bar, bar_base + 3 * grid);
        if (blockIdx.x != 0) return;
    } else {
        small_grid_arrive(a.bar);
        __syncthreads();
    }
    SMALL_T(7);
    // ---- CTA 0: the key is complete (candidates: CTA 0 alone counted them, its shared-memory counters are the counts)
    SelectInit fin = none;
    fin.result_out = a.result_out;
    select_scan_body<2, kThreads>(&s_sel, g2, 0, fin, scan_sm, fits ? dyn_bins : nullptr);
    __syncthreads();
    for (int i = threadIdx.x; i < kDigitBins; i += kThreads) a.gdigits[i] = 0ull;   // as the general path leaves them
    for (int i = threadIdx.x; i < kDigitBins / 32; i += kThreads) a.chunk_tot[i] = 0ull;
    if (threadIdx.x == 0) {
        SelectState* g = a.sel;          // the state a later CUBE_REUSE_COARSE selection or a reader of the context finds
        g->k = s_sel.k; g->count = s_sel.count; g->prefix = s_sel.prefix; g->invalid = s_sel.invalid;
        SMALL_T(8);
        g->use_median = a.use_median ? 1u : 0u; g->result = s_sel.result; g->bucket_n = s_sel.bucket_n; g->cand_cap = a.cand ? a.cand_cap : 0; g->cand_done = fits ? 1u : 0u;
        a.bar[1] = bar_base + kSmallBarriers * grid;   // every CTA arrives kSmallBarriers times per launch
    }
}

}  // namespace cube
