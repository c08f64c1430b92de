// cube_hist_big.cuh -- histogram with 16385..65536 bins (steps 4-5 of SURVEY.md sec. 8(a)).
//
// 65536 x 4 B = 256 KiB of 32-bit counters do not fit the 227 KiB of shared memory of an SM, so one CTA of 1024
// threads per SM keeps TWO 16-bit counters per 32-bit word (128 KiB): bin b < 32768 is the low half of word b,
// bin b >= 32768 the high half of word b - 32768.  Neighbouring bins -- the hot ones of a noise-dominated cube --
// therefore sit in neighbouring banks.  The low halves are incremented with +1, which compiles to ATOMS.POPC.INC
// (lanes that hit the same word are merged by the hardware; measured on B200: 5.9 increments per clock per SM with
// 37 % of the lanes on one word, against 2.6 for ATOMS.ADD of any other constant or for an atomic that returns the
// old value -- DESIGN.md sec. 4).  ptxas turns a predicated shared atomic into a branch, so the hot path issues ONE
// unconditional +1 per voxel: voxels of the "hot" half of the bin range go to their word, all others to a trash
// word, and the rows that hold such a voxel are revisited by a cold path (+65536 on the high half, closed top bin,
// outside counts).  Which half is hot is sampled before the launch (hist_window_kernel): `flip` swaps the halves.
//
// No increment returns a value, so a 16-bit field must never be allowed to wrap.  That is guaranteed without
// looking at the data: every kScanEvery tiles (a tile = 16384 voxels of the CTA) all threads meet at a barrier, each
// scans 32 words, moves the part >= 8192 of every field to the 64-bit global bin, and a second barrier ends the
// scan.  A field is < 8192 after a scan and receives at most 3 x 16384 (+ 6 head/tail voxels) increments before
// the next one, i.e. stays <= 57349 < 65536 -- even when every voxel of the cube falls into one bin.
// The scan costs 8 LDS.128 + ~25 ALU instructions per thread per 48 voxels (~0.7 per voxel); the loads of the next
// tile are issued before the current one is binned, so the barrier does not drain the memory pipeline.
// (v1 detected wraps from the value returned by atomicAdd: ~20 instructions per voxel and same-address
// serialisation; 2.7 TB/s on config 4, 3.9 TB/s on config 3 -- round-1 ncu capture.)
#pragma once
#include "cube_kernels.cuh"

namespace cube {

constexpr int kBigUnroll = 4;                              // float4 per thread per tile
constexpr int kBigTile = kBigThreads * kBigUnroll;         // float4 per tile (16384 voxels)
constexpr int kBigScanEvery = 3;                           // tiles between two scans
constexpr uint32_t kBigFlushMask = 0xE000E000u;            // some field of the word is >= 8192
constexpr int kBigWords = 32768;
static_assert(8191 + kBigScanEvery * kBigTile * 4 + 6 < 65536, "a 16-bit field could wrap between two scans");

struct HistBigF {
    float lo, hi, scale;
    int top;
    uint32_t flip;      // 0: bins < 32768 are the +1 (hot-path) halves; 0x8000: bins >= 32768 are
    float off;          // 0 or -32768: v + off is the position inside the hot half
    uint32_t limitbits; // bits of the first v + off that the hot path does not count
    uint32_t sbase;     // shared-window address of word 0
    uint32_t* sw;       // kBigWords packed words + 1 trash word
    uint32_t* s_out;    // shared {below, above}
    bool fast;          // hist_use_fast(): the one-compare hot path is valid

    __device__ __forceinline__ void setup(float lo_, float hi_, float scale_, int nbins, uint32_t flip_,
                                          uint32_t* sw_, uint32_t* s_out_) {
        lo = lo_; hi = hi_; scale = scale_; top = nbins - 1; flip = flip_;
        sw = sw_; sbase = smem_addr(sw_); s_out = s_out_;
        fast = hist_use_fast(nbins, lo, hi, scale);
        off = flip ? -32768.0f : 0.0f;
        // hot half: bins [0, min(32768, top)) or [32768, top); the top bin is closed (R11) and stays on the cold path
        const int lim = flip ? top - kBigWords : min(kBigWords, top);
        limitbits = __float_as_uint((float)max(lim, 0));
    }
    __device__ __forceinline__ void add_bin(int b) const {   // cold paths only
        const uint32_t pb = (uint32_t)b ^ flip;               // physical slot
        if (pb < (uint32_t)kBigWords) atomicAdd(&sw[pb], 1u);
        else atomicAdd(&sw[pb - kBigWords], 65536u);
    }
    // Hot path: v = (x - lo) * scale (R10), vh = v + off (exact: v >= 32768 when it matters).  The voxel is counted
    // here iff +0 <= vh < limit -- ONE unsigned compare on the bits of vh, false for negative vh (sign bit), NaN and
    // everything from the limit upwards (HistFastF has the argument why lo <= x <= hi then holds and no clamp is
    // needed).  Every other voxel increments the trash word and is left to exact().  The increment is always +1
    // => ATOMS.POPC.INC.  Returns vh.
    __device__ __forceinline__ float inc(float x) const {
        const float vh = __fadd_rn(__fmul_rn(__fsub_rn(x, lo), scale), off);
        smem_inc(sbase, __float_as_uint(vh) < limitbits ? (uint32_t)__float2int_rd(vh) : (uint32_t)kBigWords);
        return vh;
    }
    __device__ __forceinline__ bool counted(float x) const {
        return __float_as_uint(__fadd_rn(__fmul_rn(__fsub_rn(x, lo), scale), off)) < limitbits;
    }
    // Exact definition (R10-R13) for a voxel the hot path did not count: x < lo, x > hi, NaN, the other half of the
    // bins, the closed top bin (v >= nbins - 1) and v == -0.0.
    __device__ __forceinline__ void exact(float x) const {
        if (x < lo) atomicAdd(&s_out[0], 1u);
        else if (x > hi) atomicAdd(&s_out[1], 1u);
        else if (x == x) add_bin(min(max(__float2int_rd(__fmul_rn(__fsub_rn(x, lo), scale)), 0), top));
    }
    __device__ __forceinline__ void single(float x) const {   // head / tail / ragged tile / degenerate ranges
        if (fast) { if (!(__float_as_uint(inc(x)) < limitbits)) exact(x); }
        else exact(x);
    }
    __device__ __noinline__ void cold(uint32_t rows, const float4* __restrict__ p) const {
        do {
            const int j = __ffs(rows) - 1;
            rows &= rows - 1;
            const float4 q = __ldcg(p + j * kBigThreads);   // L2 hit: the line has just been streamed
            if (!counted(q.x)) exact(q.x);
            if (!counted(q.y)) exact(q.y);
            if (!counted(q.z)) exact(q.z);
            if (!counted(q.w)) exact(q.w);
        } while (rows);
    }
    // thread's share of one FULL tile: r[j] was loaded from p[j * kBigThreads]
    __device__ __forceinline__ void tile(const float4 (&r)[kBigUnroll], const float4* __restrict__ p) const {
        if (!fast) {
#pragma unroll
            for (int j = 0; j < kBigUnroll; ++j) { exact(r[j].x); exact(r[j].y); exact(r[j].z); exact(r[j].w); }
            return;
        }
        // A row needs the cold path iff it holds a voxel with vh >= limit or vh < 0 (sign bit: also -0.0).  The row
        // maximum / minimum are taken with FMNMX, which ignores NaN operands: blanked voxels count nowhere, so a
        // row is NOT revisited because of them (config 3 scatters a NaN into 2 % of the rows).
        const float limf = __uint_as_float(limitbits);
        uint32_t rows = 0;
#pragma unroll
        for (int j = 0; j < kBigUnroll; ++j) {
            const float a = inc(r[j].x), b = inc(r[j].y), c = inc(r[j].z), e = inc(r[j].w);
            const float mx = fmaxf(fmaxf(a, b), fmaxf(c, e)), mn = fminf(fminf(a, b), fminf(c, e));
            rows |= ((mx >= limf || __float_as_int(mn) < 0) ? 1u : 0u) << j;
        }
        if (rows) cold(rows, p);
    }
};

// Between the two barriers of a scan no other thread touches the counters, so plain loads and stores do.
// uint4 q of thread i = words 4 * (q * 1024 + i) .. + 3: consecutive lanes read consecutive 16 bytes.
// Physical slot s (low half of word s, or high half of word s - 32768) holds bin s ^ flip.
__device__ __forceinline__ void big_flush_word(uint32_t& w, uint32_t word, uint32_t flip, int nbins,
                                               unsigned long long* __restrict__ gbins) {
    const uint32_t l = w & 0xE000u, h = (w >> 16) & 0xE000u;
    const uint32_t bl = word ^ flip, bh = (word + kBigWords) ^ flip;
    if (l && bl < (uint32_t)nbins) atomicAdd(&gbins[bl], (unsigned long long)l);
    if (h && bh < (uint32_t)nbins) atomicAdd(&gbins[bh], (unsigned long long)h);
    w &= ~kBigFlushMask;
}
__device__ __forceinline__ void big_scan(uint32_t* sw, uint32_t flip, int nbins, unsigned long long* __restrict__ gbins) {
    uint4* p = reinterpret_cast<uint4*>(sw);
#pragma unroll
    for (int q = 0; q < kBigWords / 4 / kBigThreads; ++q) {
        const uint32_t i = q * kBigThreads + threadIdx.x;
        uint4 w = p[i];
        if ((w.x | w.y | w.z | w.w) & kBigFlushMask) {
            big_flush_word(w.x, 4 * i + 0, flip, nbins, gbins);
            big_flush_word(w.y, 4 * i + 1, flip, nbins, gbins);
            big_flush_word(w.z, 4 * i + 2, flip, nbins, gbins);
            big_flush_word(w.w, 4 * i + 3, flip, nbins, gbins);
            p[i] = w;
        }
    }
    if (threadIdx.x == 0) sw[kBigWords] = 0;   // trash word
}

__global__ void __launch_bounds__(kBigThreads, 1)
hist_packed_kernel(const float* __restrict__ d, uint64_t n, int nbins, float lo, float hi, float scale,
                   const float* __restrict__ range3, const uint32_t* __restrict__ flip_in,
                   const uint32_t* __restrict__ skip_if_set,
                   unsigned long long* __restrict__ gbins, unsigned long long* __restrict__ goutside) {
    extern __shared__ uint32_t dyn_bins[];  // kBigWords words + trash word
    __shared__ uint32_t s_out[2];
    if (skip_if_set && *skip_if_set) return;   // hist_win_kernel has done this histogram (BigHistPlan::use_window)
    for (int i = threadIdx.x; i <= kBigWords; i += kBigThreads) dyn_bins[i] = 0;
    if (threadIdx.x < 2) s_out[threadIdx.x] = 0;
    __syncthreads();
    if (range3) { lo = range3[0]; hi = range3[1]; scale = range3[2]; }  // resolved on the device (cube_stats)
    const uint32_t flip = (flip_in && nbins > kBigWords) ? (*flip_in & 0x8000u) : 0u;
    HistBigF f;
    f.setup(lo, hi, scale, nbins, flip, dyn_bins, s_out);

    // same peeling as stream_cube: <= 3 head and <= 3 tail voxels go to CTA 0
    uint64_t head = ((16u - (uint32_t)((uintptr_t)d & 15u)) & 15u) >> 2;
    if (head > n) head = n;
    const float4* __restrict__ v = reinterpret_cast<const float4*>(d + head);
    const uint64_t nvec = (n - head) >> 2;
    const uint64_t tail0 = head + (nvec << 2);
    if (blockIdx.x == 0) {
        if (threadIdx.x < head) f.single(d[threadIdx.x]);
        if (threadIdx.x >= 32 && threadIdx.x < 35) {
            const uint64_t t = tail0 + (threadIdx.x - 32);
            if (t < n) f.single(d[t]);
        }
    }
    const uint64_t nfull = nvec / kBigTile;   // full tiles, dealt round-robin to the CTAs
    uint64_t t = blockIdx.x;
    bool have = t < nfull;                    // CTA-uniform
    float4 cur[kBigUnroll], nxt[kBigUnroll];
    if (have) {
#pragma unroll
        for (int j = 0; j < kBigUnroll; ++j) cur[j] = ld_stream(v + t * kBigTile + threadIdx.x + j * kBigThreads);
    }
    int since = 0;
    while (have) {
        const uint64_t tn = t + gridDim.x;
        const bool have_n = tn < nfull;
        if (have_n) {                          // next tile's loads are in flight while this one is binned
#pragma unroll
            for (int j = 0; j < kBigUnroll; ++j) nxt[j] = ld_stream(v + tn * kBigTile + threadIdx.x + j * kBigThreads);
        }
        f.tile(cur, v + t * kBigTile + threadIdx.x);
        if (++since == kBigScanEvery) {
            since = 0;
            __syncthreads();
            big_scan(dyn_bins, flip, nbins, gbins);
            __syncthreads();
        }
#pragma unroll
        for (int j = 0; j < kBigUnroll; ++j) cur[j] = nxt[j];
        t = tn;
        have = have_n;
    }
    // ragged last tile (< 16384 voxels: `since` <= 2 full tiles are pending, so the bound above still holds)
    if (nvec % kBigTile != 0 && (nfull % gridDim.x) == blockIdx.x) {
        for (uint64_t i = nfull * kBigTile + threadIdx.x; i < nvec; i += kBigThreads) {
            const float4 r = ld_stream(v + i);
            f.single(r.x); f.single(r.y); f.single(r.z); f.single(r.w);
        }
    }
    __syncthreads();
    for (int i = threadIdx.x; i < kBigWords; i += kBigThreads) {
        const uint32_t w = dyn_bins[i];
        const uint32_t bl = (uint32_t)i ^ flip, bh = (uint32_t)(i + kBigWords) ^ flip;
        if ((w & 0xFFFFu) && bl < (uint32_t)nbins) atomicAdd(&gbins[bl], (unsigned long long)(w & 0xFFFFu));
        if ((w >> 16) && bh < (uint32_t)nbins) atomicAdd(&gbins[bh], (unsigned long long)(w >> 16));
    }
    if (lo > hi) return;  // unusable device-side [min,max] range: hist_range_kernel has left the marker
    if (threadIdx.x < 2 && s_out[threadIdx.x]) atomicAdd(&goutside[threadIdx.x], (unsigned long long)s_out[threadIdx.x]);
}

// ------------------------------------------------------------------------------------------------
// Windowed variant (the default when it applies): 32-bit counters for a WINDOW of 32768 consecutive bins
// [w0, w0 + 32768) in shared memory (128 KiB, one CTA of 1024 threads per SM), everything else straight to the
// 64-bit global bins with a RED.  Real cubes put almost all voxels into a narrow part of a 65536-bin range (noise
// around zero, sparse sources above -- PAPER.md:294: median +0.0036 in a range -1.04 ... 0.82), so the global REDs
// are rare; a 32-bit counter cannot wrap (a CTA sees < 2^32 voxels), so there is no scan, no barrier and no
// second increment flavour: the hot path is HistFastF's (FADD, FMUL, FADD, ISETP, F2I, SEL, IMAD, ATOMS.POPC.INC).
// hist_window_kernel (1 CTA) samples 16384 voxels, picks w0 (a multiple of 4096) and decides: when more than
// 1/32 of the sampled in-range voxels fall outside the best window (e.g. uniformly distributed data) the packed
// kernel above runs instead -- both kernels are always enqueued and the one not chosen returns at once, so the
// choice never leaves the device.  For nbins <= 32768 the window holds every bin and no sampling is needed.
// ------------------------------------------------------------------------------------------------
struct BigHistPlan {
    uint32_t flip;       // packed kernel: which half gets the +1 increments
    uint32_t w0;         // window kernel: first bin of the shared-memory window
    uint32_t use_window; // 1: hist_win_kernel does the work, 0: hist_packed_kernel
    uint32_t pad;
};

template <int THREADS>   // threads per CTA: the stride between a thread's rows of a tile
struct HistWinFT {
    float lo, hi, scale, off;
    int top;
    uint32_t w0, limitbits, sbase;
    uint32_t* sbins;                 // kBigWords counters + trash
    uint32_t* s_out;                 // shared {below, above}
    unsigned long long* gbins;
    __device__ __forceinline__ void setup(float lo_, float hi_, float scale_, int nbins, uint32_t w0_, uint32_t* sbins_,
                                          uint32_t* s_out_, unsigned long long* gbins_) {
        lo = lo_; hi = hi_; scale = scale_; top = nbins - 1; w0 = w0_; off = -(float)w0_;
        sbins = sbins_; sbase = smem_addr(sbins_); s_out = s_out_; gbins = gbins_;
        // hot path: window bins below the closed top bin (R11), i.e. 0 <= v - w0 < min(32768, top - w0)
        const int lim = min(kBigWords, top - (int)w0_);
        limitbits = __float_as_uint((float)max(lim, 0));
    }
    // v - w0 is exact for w0 <= v < 65536 (a multiple of ulp(v), smaller than v), negative below the window
    __device__ __forceinline__ float inc(float x) const {
        const float vh = __fadd_rn(__fmul_rn(__fsub_rn(x, lo), scale), off);
        smem_inc(sbase, __float_as_uint(vh) < limitbits ? (uint32_t)__float2int_rd(vh) : (uint32_t)kBigWords);
        return vh;
    }
    __device__ __forceinline__ bool counted(float x) const {
        return __float_as_uint(__fadd_rn(__fmul_rn(__fsub_rn(x, lo), scale), off)) < limitbits;
    }
    __device__ __forceinline__ void exact(float x) const {   // a voxel the hot path did not count
        if (x < lo) atomicAdd(&s_out[0], 1u);
        else if (x > hi) atomicAdd(&s_out[1], 1u);
        else if (x == x) {
            const uint32_t b = (uint32_t)min(max(__float2int_rd(__fmul_rn(__fsub_rn(x, lo), scale)), 0), top);
            const uint32_t pb = b - w0;
            if (pb < (uint32_t)kBigWords) atomicAdd(&sbins[pb], 1u);
            else atomicAdd(&gbins[b], 1ull);
        }
    }
    __device__ __forceinline__ void operator()(float x) const {   // head / tail / ragged tile
        if (counted(x)) inc(x); else exact(x);
    }
    __device__ __noinline__ void cold(uint32_t rows, const float4* __restrict__ p) const {
        do {
            const int j = __ffs(rows) - 1;
            rows &= rows - 1;
            const float4 q = __ldcg(p + j * THREADS);   // L2 hit: the line has just been streamed
            if (!counted(q.x)) exact(q.x);
            if (!counted(q.y)) exact(q.y);
            if (!counted(q.z)) exact(q.z);
            if (!counted(q.w)) exact(q.w);
        } while (rows);
    }
    __device__ __forceinline__ void batch(const float4 (&r)[kUnroll], const float4* __restrict__ p) const {
        const float limf = __uint_as_float(limitbits);
        uint32_t rows = 0;
#pragma unroll
        for (int j = 0; j < kUnroll; ++j) {
            const float a = inc(r[j].x), b = inc(r[j].y), c = inc(r[j].z), e = inc(r[j].w);
            const float mx = fmaxf(fmaxf(a, b), fmaxf(c, e)), mn = fminf(fminf(a, b), fminf(c, e));
            rows |= ((mx >= limf || __float_as_int(mn) < 0) ? 1u : 0u) << j;   // FMNMX: NaN voxels flag nothing
        }
        if (rows) cold(rows, p);
    }
};

using HistWinF = HistWinFT<kBigThreads>;

// 1 CTA: sample 16384 voxels spread over the cube; block histogram (16 blocks of 4096 bins); best window of 8
// consecutive blocks; also the packed kernel's flip hint.  A performance plan only: every choice is exact.
__global__ void __launch_bounds__(kBigThreads)
hist_window_kernel(const float* __restrict__ d, uint64_t n, int nbins, float lo, float hi, float scale,
                   const float* __restrict__ range3, BigHistPlan* __restrict__ plan) {
    __shared__ int blk[16];
    if (threadIdx.x < 16) blk[threadIdx.x] = 0;
    __syncthreads();
    if (range3) { lo = range3[0]; hi = range3[1]; scale = range3[2]; }
    const uint64_t stride = n / (16 * kBigThreads) + 1;
    for (int j = 0; j < 16; ++j) {
        const uint64_t i = ((uint64_t)j * kBigThreads + threadIdx.x) * stride;
        if (i < n) {
            const float x = d[i];
            if (x >= lo && x <= hi) {
                const int b = min(max(__float2int_rd(__fmul_rn(__fsub_rn(x, lo), scale)), 0), nbins - 1);
                atomicAdd(&blk[b >> 12], 1);
            }
        }
    }
    __syncthreads();
    if (threadIdx.x == 0) {
        int total = 0, best = -1, bestj = 0, lower = 0;
        for (int j = 0; j < 16; ++j) { total += blk[j]; if (j < 8) lower += blk[j]; }
        for (int j = 0; j <= 8; ++j) {
            int sum = 0;
            for (int q = 0; q < 8; ++q) sum += blk[j + q];
            if (sum > best) { best = sum; bestj = j; }
        }
        BigHistPlan pl;
        pl.flip = (total - lower > lower) ? 0x8000u : 0u;
        pl.w0 = (uint32_t)bestj << 12;
        pl.use_window = (hist_use_fast(nbins, lo, hi, scale) && (total - best) * 32 <= total) ? 1u : 0u;
        pl.pad = 0;
        if (nbins <= kBigWords) { pl.w0 = 0; pl.flip = 0; }
        *plan = pl;
    }
}

__global__ void __launch_bounds__(kBigThreads, 1)
hist_win_kernel(const float* __restrict__ d, uint64_t n, int nbins, float lo, float hi, float scale,
                const float* __restrict__ range3, const BigHistPlan* __restrict__ plan,
                unsigned long long* __restrict__ gbins, unsigned long long* __restrict__ goutside) {
    extern __shared__ uint32_t dyn_bins[];  // kBigWords counters + trash
    __shared__ uint32_t s_out[2];
    if (!plan->use_window) return;          // the packed kernel does this histogram
    for (int i = threadIdx.x; i <= kBigWords; i += kBigThreads) dyn_bins[i] = 0;
    if (threadIdx.x < 2) s_out[threadIdx.x] = 0;
    __syncthreads();
    if (range3) { lo = range3[0]; hi = range3[1]; scale = range3[2]; }
    const uint32_t w0 = plan->w0;
    HistWinF f;
    f.setup(lo, hi, scale, nbins, w0, dyn_bins, s_out, gbins);
    stream_cube<kBigThreads>(d, n, f);
    __syncthreads();
    for (int i = threadIdx.x; i < kBigWords; i += kBigThreads) {
        const uint32_t c = dyn_bins[i];
        if (c && w0 + i < (uint32_t)nbins) atomicAdd(&gbins[w0 + i], (unsigned long long)c);
    }
    if (lo > hi) return;  // unusable device-side [min,max] range: hist_range_kernel has left the marker
    if (threadIdx.x < 2 && s_out[threadIdx.x]) atomicAdd(&goutside[threadIdx.x], (unsigned long long)s_out[threadIdx.x]);
}

}  // namespace cube
