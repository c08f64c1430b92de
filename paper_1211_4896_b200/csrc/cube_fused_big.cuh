// cube_fused_big.cuh -- pass B of cube_stats() for histograms with more than 16384 bins: the windowed histogram
// (cube_hist_big.cuh) + second select digit + candidate compaction in ONE read of the cube, so that cube_stats()
// takes two reads for 65536 bins as well (configs 3 and 4 of BASELINE.json; steps 4-6 and 8 of SURVEY.md sec. 8(a)).
//
// One CTA of 1024 threads per SM.  Dynamic shared memory (205 KiB of the 227 KiB):
//     [32768 + 1 window counters][1024 + 1 digit counters][32 warps x (544 staged keys + 1 fill counter)]
// The per-warp stage slice must hold the flush threshold plus everything a warp can add between two checks; with
// 32 warps there is no room for a whole tile share (1024 keys), so the bucket test and the fill check are made
// per HALF tile share (4 rows of 4 voxels per lane: at most 512 keys): kBigStageThresh + 512 slots per warp.
// It only runs when the sampled plan chose the window (BigHistPlan::use_window); otherwise it returns at once
// and the packed histogram + select_pass_kernel<1> (both enqueued behind it) do the work in two reads.
#pragma once
#include "cube_kernels.cuh"

namespace cube {

constexpr uint32_t kBigStageThresh = 32;
constexpr uint32_t kBigStageCap = kBigStageThresh + 32u * 4u * (kUnroll / 2);   // 544 keys
constexpr int kBigWarps = kBigThreads / 32;
constexpr int kBigFusedSmem = (kBigWords + 1 + kBins1 + 1 + kBigWarps * ((int)kBigStageCap + 1)) * (int)sizeof(uint32_t);

// What the cold paths of the select need; kept in shared memory so that the hot loop carries none of it in registers.
struct BigSelShared {
    uint32_t base;                 // prefix << 19
    uint32_t* sbins;               // kBins1 + 1 digit counters
    uint32_t* stage;               // kBigWarps slices of kBigStageCap keys, then kBigWarps fill counters
    uint32_t* cand;
    unsigned long long* cand_n;
    unsigned long long cand_cap;
    uint32_t compacting[kBigWarps];   // per warp: 0 once the candidate buffer is known to be too small
};

struct HistWinSelectF {
    HistWinF h;
    uint32_t negbase;              // 0 - (raw_of_digit(prefix) << 19)
    bool select;                   // false: nothing to select (k >= count)
    BigSelShared* sh;

    // Single voxels (head / tail / ragged last tile: up to 8 rows x 4 voxels per lane with no fill check in between)
    // never go through the warp's stage slice, which only holds what HALF a tile share can add: their keys are
    // appended straight to the candidate buffer, one global atomic each (at most one ragged tile per launch).
    __device__ __forceinline__ void operator()(float x) {
        h(x);
        if (select) {
            const uint32_t kk = key_of(x) - sh->base;
            if (kk < SelectF<1, false>::kSpan && x == x) {
                atomicAdd(&sh->sbins[kk >> kBits2], 1u);
                if (sh->cand && sh->cand_cap) {
                    const unsigned long long pos = atomicAdd(sh->cand_n, 1ull);   // beyond the capacity: cand_n says so
                    if (pos < sh->cand_cap) sh->cand[pos] = kk + sh->base;
                }
            }
        }
    }
    // rows `rows` (bit j = row j0 + j) of this lane hold a voxel of the bucket: count its digit, stage its key
    static __device__ __noinline__ void cold(uint32_t rows, const float4* __restrict__ p, BigSelShared* sh) {
        const int warp = threadIdx.x >> 5;
        uint32_t* s_buf = sh->stage + warp * kBigStageCap;
        uint32_t* s_cnt = sh->compacting[warp] ? sh->stage + kBigWarps * kBigStageCap + warp : nullptr;
        const uint32_t base = sh->base;
        uint32_t* sbins = sh->sbins;
        do {
            const int j = __ffs(rows) - 1;
            rows &= rows - 1;
            const float4 q = __ldcg(p + j * kBigThreads);   // L2 hit: the line has just been streamed
            SelectF<1, false>::take1(q.x, base, sbins, s_cnt, s_buf);
            SelectF<1, false>::take1(q.y, base, sbins, s_cnt, s_buf);
            SelectF<1, false>::take1(q.z, base, sbins, s_cnt, s_buf);
            SelectF<1, false>::take1(q.w, base, sbins, s_cnt, s_buf);
        } while (rows);
    }
    // all lanes of the warp: move the staged keys to the candidate buffer when more than `thresh` wait
    static __device__ __noinline__ void flush_if(uint32_t thresh, BigSelShared* sh) {
        const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
        if (!sh->compacting[warp]) return;
        uint32_t* s_buf = sh->stage + warp * kBigStageCap;
        uint32_t* s_cnt = sh->stage + kBigWarps * kBigStageCap + warp;
        __syncwarp();
        const uint32_t c = *reinterpret_cast<volatile uint32_t*>(s_cnt);
        if (c <= thresh) return;
        unsigned long long pos = 0;
        if (lane == 0) pos = atomicAdd(sh->cand_n, (unsigned long long)c);
        pos = __shfl_sync(0xffffffffu, pos, 0);
        if (pos + c <= sh->cand_cap) {
            for (uint32_t i = lane; i < c; i += 32) sh->cand[pos + i] = s_buf[i];
        } else if (lane == 0) {
            sh->compacting[warp] = 0;   // the bucket does not fit: pass C will stream the cube, stop staging
        }
        __syncwarp();
        if (lane == 0) *s_cnt = 0;
        __syncwarp();
    }
    __device__ __forceinline__ void batch(const float4 (&r)[kUnroll], const float4* __restrict__ p) {
        h.batch(r, p);
        if (!select) return;
#pragma unroll
        for (int half = 0; half < 2; ++half) {
            uint32_t rm[kUnroll / 2];
#pragma unroll
            for (int j = 0; j < kUnroll / 2; ++j) {
                const float4& v = r[half * (kUnroll / 2) + j];
                rm[j] = min(min(SelectF<1, false>::sub_fma(v.x, negbase), SelectF<1, false>::sub_fma(v.y, negbase)),
                            min(SelectF<1, false>::sub_fma(v.z, negbase), SelectF<1, false>::sub_fma(v.w, negbase)));
            }
            uint32_t tmin = rm[0];
#pragma unroll
            for (int j = 1; j < kUnroll / 2; ++j) tmin = min(tmin, rm[j]);
            const bool hit = tmin < SelectF<1, false>::kSpan;
            if (hit) {
                uint32_t rows = 0;
#pragma unroll
                for (int j = 0; j < kUnroll / 2; ++j) rows |= (rm[j] < SelectF<1, false>::kSpan ? 1u : 0u) << j;
                cold(rows, p + half * (kUnroll / 2) * kBigThreads, sh);
            }
            if (__any_sync(0xffffffffu, hit)) flush_if(kBigStageThresh, sh);   // warp-uniform
        }
    }
};

__global__ void __launch_bounds__(kBigThreads, 1)
hist_win_select_kernel(const float* __restrict__ d, uint64_t n, int nbins, float lo, float hi, float scale,
                       const float* __restrict__ range3, const BigHistPlan* __restrict__ plan,
                       unsigned long long* __restrict__ gbins, unsigned long long* __restrict__ goutside,
                       SelectState* __restrict__ st, unsigned long long* __restrict__ gdigits,
                       uint32_t* __restrict__ cand, unsigned int* __restrict__ scan_ticket) {
    extern __shared__ uint32_t dyn_bins[];
    __shared__ uint32_t s_out[2];
    __shared__ BigSelShared sh;
    if (!plan->use_window) return;          // the packed histogram + select_pass_kernel<1> do this pass
    uint32_t* wbins = dyn_bins;                               // kBigWords + 1
    uint32_t* sbins = dyn_bins + (kBigWords + 1);             // kBins1 + 1
    uint32_t* stage = sbins + (kBins1 + 1);
    for (int i = threadIdx.x; i < kBigWords + 1 + kBins1 + 1; i += kBigThreads) dyn_bins[i] = 0;
    if (threadIdx.x < kBigWarps) { stage[kBigWarps * kBigStageCap + threadIdx.x] = 0; sh.compacting[threadIdx.x] = (cand && st->cand_cap) ? 1u : 0u; }
    if (threadIdx.x < 2) s_out[threadIdx.x] = 0;
    if (threadIdx.x == 0) {
        sh.base = st->prefix << kShift0; sh.sbins = sbins; sh.stage = stage; sh.cand = cand;
        sh.cand_n = &st->cand_n; sh.cand_cap = st->cand_cap;
    }
    __syncthreads();
    if (range3) { lo = range3[0]; hi = range3[1]; scale = range3[2]; }
    HistWinSelectF f;
    f.h.setup(lo, hi, scale, nbins, plan->w0, wbins, s_out, gbins);
    f.negbase = 0u - (raw_of_digit(st->prefix) << kShift0);
    f.select = st->invalid == 0;
    f.sh = &sh;
    stream_cube<kBigThreads>(d, n, f);
    if (f.select) HistWinSelectF::flush_if(0u, &sh);          // what is still staged
    __syncthreads();
    const uint32_t w0 = plan->w0;
    for (int i = threadIdx.x; i < kBigWords; i += kBigThreads) {
        const uint32_t c = wbins[i];
        if (c && w0 + i < (uint32_t)nbins) atomicAdd(&gbins[w0 + i], (unsigned long long)c);
    }
    for (int i = threadIdx.x; i < kBins1; i += kBigThreads) {
        const uint32_t c = sbins[i];
        if (c) atomicAdd(&gdigits[i], (unsigned long long)c);
    }
    if (!(lo > hi) && threadIdx.x < 2 && s_out[threadIdx.x])
        atomicAdd(&goutside[threadIdx.x], (unsigned long long)s_out[threadIdx.x]);
    if (scan_ticket) {   // the last CTA locates the second-digit bucket
        __shared__ unsigned long long scan_sm[kScanSmem];
        SelectInit none;
        none.k = 0; none.cand_cap = 0; none.result_out = nullptr; none.use_median = 0; none.enabled = 0;
        select_scan_if_last_n<1, kBigThreads>(st, gdigits, 1, none, scan_ticket, scan_sm);
    }
}

}  // namespace cube
