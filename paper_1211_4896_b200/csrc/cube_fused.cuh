// cube_fused.cuh -- pass B of cube_stats(): histogram + second select digit + candidate compaction in ONE read
// of the cube (steps 4-6 and 8 of SURVEY.md sec. 8(a) fused).
//
// cube_stats() needs every statistic of the paper's path at once, so it reads the cube
// exactly twice -- the minimum for an exact selection with O(bins) memory:
//   pass A  moments_kernel<COARSE>: count, min, max, pivoted fp64 sums + first radix digit (8192 bins);
//           1-CTA scan picks the median's bucket;
//   pass B  this kernel: intensity histogram (range given, or [min,max] read from pass A's result on the
//           device) + second digit of the voxels in the bucket + their keys staged into the candidate buffer;
//   pass C  last digit on the candidates (a few MB, L2-resident).
// Issue budget: the histogram costs ~9 instructions per voxel and the bucket test ~4, which together still fit
// under the ~16 per voxel that the SMs can issue at the DRAM rate.
#pragma once
#include "cube_kernels.cuh"

namespace cube {

template <class H>
struct HistSelectF {
    H h;
    SelectF<1, false> s;
    __device__ __forceinline__ void operator()(float x) { h(x); s(x); }
    __device__ __forceinline__ void batch(const float4 (&r)[kUnroll], const float4* __restrict__ p) {
        h.batch(r, p);
        s.batch(r, p);
    }
};

// What pass B needs to know of the selection: the first-digit bucket (or "nothing to select") and where the
// candidates go.  Read from the SelectState in device memory, or -- cube_small.cuh -- from a CTA's own copy.
struct SelView {
    uint32_t invalid, prefix;
    unsigned long long* cand_n;
    unsigned long long cand_cap;
};
__device__ __forceinline__ SelView sel_view(SelectState* __restrict__ st) {
    SelView v;
    v.invalid = st->invalid; v.prefix = st->prefix; v.cand_n = &st->cand_n; v.cand_cap = st->cand_cap;
    return v;
}

template <class H>
__device__ __forceinline__ void hist_select_run(const float* __restrict__ d, uint64_t n, const H& h,
                                                const SelView& sv, uint32_t* sbins, uint32_t* stage,
                                                uint32_t* __restrict__ cand, uint32_t& below, uint32_t& above) {
    if (sv.invalid) {  // nothing to select (k >= count): histogram only
        H f = h;
        stream_cube<kThreads>(d, n, f);
        below = f.below; above = f.above;
        return;
    }
    HistSelectF<H> f;
    f.h = h;
    const uint32_t top = sv.prefix;
    f.s.base = top << kShift0; f.s.rawbase = raw_of_digit(top) << kShift0; f.s.sbins = sbins;
    f.s.init_stage(stage, cand, sv.cand_n, sv.cand_cap);
    stream_cube<kThreads>(d, n, f);
    f.s.finish();
    below = f.h.below; above = f.h.above;
}

// Histogram range of pass B.  range_from != nullptr: [min, max] of the moments record written by pass A
// (same stream); the scale is formed exactly as the host forms it in cube_histogram (R10, R13).
// Returns false when the range is unusable (no voxel, infinite extremum, overflowing width or scale; R19).
__device__ __forceinline__ bool hist_range(const MomentsOut* __restrict__ range_from, int nbins, float& lo,
                                           float& hi, float& scale) {
    if (range_from == nullptr) return true;
    const float mn = range_from->min, mx = range_from->max;
    lo = mn; hi = mx; scale = 0.0f;
    if (range_from->count == 0) { lo = hi = 0.0f; return false; }
    if (isinf(mn) || isinf(mx)) return false;
    if (mx == mn) return true;
    const float width = __fsub_rn(mx, mn);
    scale = __fdiv_rn((float)nbins, width);
    return !(isinf(width) || isinf(scale));
}

// Dynamic shared memory: [nbins + 2 histogram slots][kBins1 + 1 digit counters][stage slices + counters].
__global__ void __launch_bounds__(kThreads, 3)
hist_select_kernel(const float* __restrict__ d, uint64_t n, int nbins, float lo, float hi, float scale,
                   const MomentsOut* __restrict__ range_from, unsigned long long* __restrict__ gbins,
                   unsigned long long* __restrict__ goutside, SelectState* __restrict__ st,
                   unsigned long long* __restrict__ gdigits, uint32_t* __restrict__ cand,
                   unsigned int* __restrict__ scan_ticket) {
    extern __shared__ uint32_t dyn_bins[];
    __shared__ uint32_t s_out[2];
    uint32_t* hbins = dyn_bins;
    uint32_t* sbins = dyn_bins + (nbins + 2);
    uint32_t* stage = sbins + (kBins1 + 1);
    for (int i = threadIdx.x; i < nbins + 2 + kBins1 + 1; i += kThreads) dyn_bins[i] = 0;
    if (threadIdx.x < 2) s_out[threadIdx.x] = 0;
    __syncthreads();
    const bool range_ok = hist_range(range_from, nbins, lo, hi, scale);
    if (!range_ok) { lo = INFINITY; hi = -INFINITY; }  // nothing is in range: every counter stays 0
    uint32_t below = 0, above = 0;
    if (hist_use_fast(nbins, lo, hi, scale)) {
        HistFastF h;
        h.setup(lo, hi, scale, nbins, hbins, s_out);
        hist_select_run(d, n, h, sel_view(st), sbins, stage, cand, below, above);
    } else {
        HistF h;
        h.lo = lo; h.hi = hi; h.scale = scale; h.top = nbins - 1; h.sbins = hbins;
        hist_select_run(d, n, h, sel_view(st), sbins, stage, cand, below, above);
    }
    __syncthreads();
    hist_flush_bins(hbins, nbins, gbins);
    for (int i = threadIdx.x; i < kBins1; i += kThreads) {
        const uint32_t c = sbins[i];
        if (c) atomicAdd(&gdigits[i], (unsigned long long)c);
    }
    if (range_ok) {
        if (below) atomicAdd(&s_out[0], below);
        if (above) atomicAdd(&s_out[1], above);
        __syncthreads();
        if (threadIdx.x < 2 && s_out[threadIdx.x]) atomicAdd(&goutside[threadIdx.x], (unsigned long long)s_out[threadIdx.x]);
    } else if (blockIdx.x == 0 && threadIdx.x < 2) {
        goutside[threadIdx.x] = ~0ull;  // marker: the [min,max] range was unusable
    }
    if (scan_ticket) {   // the last CTA locates the second-digit bucket (no separate scan launch)
        __shared__ unsigned long long scan_sm[kScanSmem];
        SelectInit none;
        none.k = 0; none.cand_cap = 0; none.result_out = nullptr; none.use_median = 0; none.enabled = 0;
        select_scan_if_last<1>(st, gdigits, 1, none, scan_ticket, scan_sm);
    }
}

// Same range logic for a histogram-only pass B (no median requested, or more than kSmemHistMaxBins bins):
// resolves [min,max] on the device into the (lo, hi, scale) triple the histogram kernels take.
__global__ void hist_range_kernel(const MomentsOut* __restrict__ range_from, int nbins, float* __restrict__ out3,
                                  unsigned long long* __restrict__ goutside) {
    float lo = 0.f, hi = 0.f, scale = 0.f;
    const bool ok = hist_range(range_from, nbins, lo, hi, scale);
    if (!ok) { lo = INFINITY; hi = -INFINITY; scale = 0.f; goutside[0] = goutside[1] = ~0ull; }
    out3[0] = lo; out3[1] = hi; out3[2] = scale;
}

}  // namespace cube
