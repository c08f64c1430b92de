// cube_fused_big.cuh -- pass B of cube_stats() for histograms with more than 16384 bins: the windowed histogram
// (cube_hist_big.cuh) + second select digit + candidate compaction in ONE read of the cube, so that cube_stats()
// takes two reads for 65536 bins as well (configs 3 and 4 of BASELINE.json; steps 4-6 and 8 of SURVEY.md sec. 8(a)).
//
// One CTA of 896 threads per SM (73 registers per thread: under the 64-register cap of 1024 threads ptxas rematerialised
// the loop state every tile).  Dynamic shared memory (192 KiB of the 227 KiB):
//     [32768 + 1 window counters][1024 + 1 digit counters][28 warps x WarpGather (96-row queue + 160 staged keys)]
// The select side is cube_gather.cuh: flagged rows are pushed onto the warp's queue two rows per lane at a time and
// taken off 32 at a time, so neither the queue nor the key stage has to hold a whole tile share.
// It only runs when the sampled plan chose the window (BigHistPlan::use_window); otherwise it returns at once
// and the packed histogram + select_pass_kernel<1> (both enqueued behind it) do the work in two reads.
#pragma once
#include "cube_kernels.cuh"
#include "cube_gather.cuh"

namespace cube {

#ifndef CUBE_FUSED_THREADS
#define CUBE_FUSED_THREADS 896
#endif
constexpr int kFusedThreads = CUBE_FUSED_THREADS;   // threads of the one CTA per SM (65536 / threads registers each)
constexpr int kBigWarps = kFusedThreads / 32;
// [window counters + trash][digit counters + trash], padded to 16 bytes, then one WarpGather per warp
constexpr int kBigFusedHead = ((kBigWords + 1 + kBins1 + 1) * (int)sizeof(uint32_t) + 15) / 16 * 16;
constexpr int kBigFusedSmem = kBigFusedHead + kBigWarps * (int)sizeof(WarpGather);

struct HistWinSelectF {
    HistWinFT<kFusedThreads> h;
    uint32_t negbase;              // 0 - (raw_of_digit(prefix) << 19)
    bool select;                   // false: nothing to select (k >= count)
    WarpGather* wq;                // this warp's queue
    const GatherShared* sh;

    // Single voxels (head / tail / ragged last tile) never go through the warp's queue or key stage.
    __device__ __forceinline__ void operator()(float x) {
        h(x);
        if (select) gather_single(sh, x);
    }
    __device__ __forceinline__ void batch(const float4 (&r)[kUnroll], const float4* __restrict__ p) {
        h.batch(r, p);
        if (select) gather_batch<kFusedThreads>(r, p, negbase, wq, sh);
    }
};

__global__ void __launch_bounds__(kFusedThreads, 1)
hist_win_select_kernel(const float* __restrict__ d, uint64_t n, int nbins, float lo, float hi, float scale,
                       const float* __restrict__ range3, const BigHistPlan* __restrict__ plan,
                       unsigned long long* __restrict__ gbins, unsigned long long* __restrict__ goutside,
                       SelectState* __restrict__ st, unsigned long long* __restrict__ gdigits,
                       uint32_t* __restrict__ cand, unsigned int* __restrict__ scan_ticket) {
    extern __shared__ __align__(16) uint32_t dyn_bins[];
    __shared__ uint32_t s_out[2];
    __shared__ GatherShared sh;
    if (!plan->use_window) return;          // the packed histogram + select_pass_kernel<1> do this pass
    uint32_t* wbins = dyn_bins;                               // kBigWords + 1
    uint32_t* sbins = dyn_bins + (kBigWords + 1);             // kBins1 + 1
    WarpGather* wgs = reinterpret_cast<WarpGather*>(reinterpret_cast<unsigned char*>(dyn_bins) + kBigFusedHead);
    for (int i = threadIdx.x; i < kBigWords + 1 + kBins1 + 1; i += kFusedThreads) dyn_bins[i] = 0;
    if (threadIdx.x < kBigWarps) {
        wgs[threadIdx.x].nrows = 0; wgs[threadIdx.x].nkeys = 0;
        wgs[threadIdx.x].compacting = (cand && st->cand_cap) ? 1u : 0u;
    }
    if (threadIdx.x < 2) s_out[threadIdx.x] = 0;
    if (threadIdx.x == 0) {
        sh.base = st->prefix << kShift0; sh.sbins = sbins; sh.cand = cand;
        sh.cand_n = &st->cand_n; sh.cand_cap = st->cand_cap;
    }
    __syncthreads();
    if (range3) { lo = range3[0]; hi = range3[1]; scale = range3[2]; }
    HistWinSelectF f;
    f.h.setup(lo, hi, scale, nbins, plan->w0, wbins, s_out, gbins);
    f.negbase = 0u - (raw_of_digit(st->prefix) << kShift0);
    f.select = st->invalid == 0;
    f.wq = wgs + (threadIdx.x >> 5);
    f.sh = &sh;
    stream_cube<kFusedThreads>(d, n, f);
    if (f.select) gather_finish(f.wq, &sh);                   // rows still queued, keys still staged
    __syncthreads();
    const uint32_t w0 = plan->w0;
    for (int i = threadIdx.x; i < kBigWords; i += kFusedThreads) {
        const uint32_t c = wbins[i];
        if (c && w0 + i < (uint32_t)nbins) atomicAdd(&gbins[w0 + i], (unsigned long long)c);
    }
    for (int i = threadIdx.x; i < kBins1; i += kFusedThreads) {
        const uint32_t c = sbins[i];
        if (c) atomicAdd(&gdigits[i], (unsigned long long)c);
    }
    if (!(lo > hi) && threadIdx.x < 2 && s_out[threadIdx.x])
        atomicAdd(&goutside[threadIdx.x], (unsigned long long)s_out[threadIdx.x]);
    if (scan_ticket) {   // the last CTA locates the second-digit bucket
        __shared__ unsigned long long scan_sm[kScanSmem];
        SelectInit none;
        none.k = 0; none.cand_cap = 0; none.result_out = nullptr; none.use_median = 0; none.enabled = 0;
        select_scan_if_last_n<1, kFusedThreads>(st, gdigits, 1, none, scan_ticket, scan_sm);
    }
}

}  // namespace cube
