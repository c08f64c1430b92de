// cube_kernels.cuh -- the sm_100a kernels of libcube.  See DESIGN.md sec. 4 for the roofline of each.
#pragma once
#include "cube_common.cuh"

namespace cube {

// Result record as laid out by include/cube.h (cube_moments_t).
struct MomentsOut {
    uint64_t count, nan_count;
    float min, max;
    double mean, std;
};

// State of one exact selection (radix select).  Lives in device memory so that the
// bucket choice after each digit pass never crosses to the host (the paper's server round trip per
// iteration, becomes a 1-CTA kernel).
struct SelectState {
    unsigned long long k;       // residual rank inside the current prefix bucket
    unsigned long long count;   // non-NaN voxels (sum of the pass-0 digit histogram)
    uint32_t prefix;            // key bits fixed so far (right aligned)
    uint32_t invalid;           // 1 when k >= count (result NaN)
    uint32_t use_median;        // 1: k = (count-1)/2 is set by the pass-0 scan
    float result;
    unsigned long long cand_n;  // candidates written by the compacting pass
    uint32_t cand_ok;           // 1 when all candidates fitted into the buffer
    uint32_t pad;
};

constexpr int kDigitBins = 2048;  // 11-bit digits (passes 0, 1); pass 2 uses the low 10 bits

// ------------------------------------------------------------------------------------------------
// Moments: steps 1-3 of SURVEY.md sec. 8(a) (+ 3b when COARSE): count, min, max, pivoted fp64 sums.
// PAPER.md:265 "local summation and summation of squares and count of the non-null data values".
// The paper's float32-per-slice partial sums are replaced by per-thread fp64
// accumulators about a per-thread pivot (R17).
// ------------------------------------------------------------------------------------------------
template <bool COARSE>
struct MomentsF {
    uint32_t n = 0, kmin = 0xFFFFFFFFu, kmax = 0u;
    bool have = false;
    double pivot = 0.0, s = 0.0, q = 0.0;
    uint32_t* sbins;  // COARSE: kDigitBins shared counters
    __device__ __forceinline__ void operator()(float x) {
        const bool ok = (x == x);  // NaN == blanked voxel
        const uint32_t key = key_of(x);
        kmin = min(kmin, ok ? key : 0xFFFFFFFFu);
        kmax = max(kmax, ok ? key : 0u);
        if (!have) { have = ok; pivot = ok ? (double)x : 0.0; }
        const double dlt = ok ? (double)x - pivot : 0.0;
        s += dlt;
        q = fma(dlt, dlt, q);
        n += ok ? 1u : 0u;
        if (COARSE) { if (ok) atomicAdd(&sbins[key >> 21], 1u); }
    }
    __device__ __forceinline__ Partial partial() const {
        Partial p = partial_empty();
        if (n) {
            const double nn = (double)n, ms = s / nn;
            p.n = n; p.mean = pivot + ms; p.m2 = fmax(q - s * ms, 0.0);
            p.kmin = kmin; p.kmax = kmax;
        }
        return p;
    }
};

__device__ __forceinline__ void moments_finalize(const Partial& t, uint64_t nvox_total, unsigned flags,
                                                 MomentsOut* out) {
    MomentsOut o;
    o.count = t.n;
    o.nan_count = nvox_total - t.n;
    const float qnan = __int_as_float(0x7fc00000);
    if (t.n == 0) {
        o.min = o.max = qnan;
        o.mean = o.std = (double)qnan;
    } else {
        o.min = __uint_as_float(bits_of_key(t.kmin));
        o.max = __uint_as_float(bits_of_key(t.kmax));
        o.mean = t.mean;
        const double den = (flags & 1u) ? (double)t.n - 1.0 : (double)t.n;
        o.std = (den > 0.0) ? sqrt(fmax(t.m2, 0.0) / den) : (double)qnan;
    }
    *out = o;
}

// acc : running Partial across calls (out-of-core bricks); merged in call order => deterministic.
// nvox_acc : running voxel total.  When `accumulate` is 0 both are overwritten.
template <bool COARSE>
__global__ void __launch_bounds__(kThreads)
moments_kernel(const float* __restrict__ d, uint64_t n, Partial* __restrict__ partials,
               unsigned int* __restrict__ ticket, Partial* __restrict__ acc,
               unsigned long long* __restrict__ nvox_acc, int accumulate, unsigned flags,
               MomentsOut* __restrict__ out, unsigned long long* __restrict__ gdigits) {
    __shared__ Partial scratch[kThreads / 32];
    __shared__ uint32_t sbins[COARSE ? kDigitBins : 1];
    __shared__ bool is_last;
    MomentsF<COARSE> f;
    f.sbins = sbins;
    if (COARSE) {
        for (int i = threadIdx.x; i < kDigitBins; i += kThreads) sbins[i] = 0;
        __syncthreads();
    }
    stream_cube(d, n, f);
    Partial p = partial_block_reduce(f.partial(), scratch);
    if (COARSE) {
        __syncthreads();
        for (int i = threadIdx.x; i < kDigitBins; i += kThreads) {
            uint32_t c = sbins[i];
            if (c) atomicAdd(&gdigits[i], (unsigned long long)c);
        }
    }
    if (threadIdx.x == 0) {
        partials[blockIdx.x] = p;
        __threadfence();
        unsigned int t = atomicAdd(ticket, 1u);
        is_last = (t == gridDim.x - 1);
    }
    __syncthreads();
    if (!is_last) return;
    // last CTA: fixed-order merge of the per-CTA partials (thread i takes i, i+256, ...; then the tree)
    __threadfence();
    Partial m = partial_empty();
    for (unsigned i = threadIdx.x; i < gridDim.x; i += kThreads) {
        Partial b;  // written by other CTAs: read through L2
        b.n = __ldcg(&partials[i].n); b.mean = __ldcg(&partials[i].mean); b.m2 = __ldcg(&partials[i].m2);
        b.kmin = __ldcg(&partials[i].kmin); b.kmax = __ldcg(&partials[i].kmax);
        m = partial_merge(m, b);
    }
    __syncthreads();
    m = partial_block_reduce(m, scratch);
    if (threadIdx.x == 0) {
        unsigned long long tot = n;
        if (accumulate) { m = partial_merge(*acc, m); tot += *nvox_acc; }
        *acc = m;
        *nvox_acc = tot;
        moments_finalize(m, tot, flags, out);
        *ticket = 0u;
    }
}

// Re-evaluate mean/std of the running partial with other flags (sample std) -- O(1).
__global__ void moments_refinalize_kernel(const Partial* __restrict__ acc, const unsigned long long* __restrict__ nvox,
                                          unsigned flags, MomentsOut* __restrict__ out) {
    moments_finalize(*acc, *nvox, flags, out);
}

// ------------------------------------------------------------------------------------------------
// Histogram: steps 4-5.  PAPER.md:259-261; bin formula DESIGN.md R10-R13 (float32, no contraction).
// Shared-memory privatised 32-bit counters per CTA, merged into the 64-bit global bins by atomics
// ("summation ... associative and commutative, any arbitrary data composition order is valid").
// ------------------------------------------------------------------------------------------------
struct HistF {
    float lo, hi, scale;
    int top;  // nbins-1
    uint32_t* sbins;
    uint32_t below = 0, above = 0;
    __device__ __forceinline__ void operator()(float x) {
        if (x >= lo && x <= hi) {  // false for NaN
            const float v = __fmul_rn(__fsub_rn(x, lo), scale);
            int b = __float2int_rd(v);  // floor; v >= 0
            b = min(b, top);            // closed top bin (R11)
            atomicAdd(&sbins[b], 1u);
        } else {
            below += (x < lo) ? 1u : 0u;
            above += (x > hi) ? 1u : 0u;
        }
    }
};

__global__ void __launch_bounds__(kThreads)
hist_smem_kernel(const float* __restrict__ d, uint64_t n, int nbins, float lo, float hi, float scale,
                 unsigned long long* __restrict__ gbins, unsigned long long* __restrict__ goutside) {
    extern __shared__ uint32_t dyn_bins[];
    __shared__ uint32_t s_out[2];
    for (int i = threadIdx.x; i < nbins; i += kThreads) dyn_bins[i] = 0;
    if (threadIdx.x < 2) s_out[threadIdx.x] = 0;
    __syncthreads();
    HistF f;
    f.lo = lo; f.hi = hi; f.scale = scale; f.top = nbins - 1; f.sbins = dyn_bins;
    stream_cube(d, n, f);
    if (f.below) atomicAdd(&s_out[0], f.below);
    if (f.above) atomicAdd(&s_out[1], f.above);
    __syncthreads();
    for (int i = threadIdx.x; i < nbins; i += kThreads) {
        uint32_t c = dyn_bins[i];
        if (c) atomicAdd(&gbins[i], (unsigned long long)c);
    }
    if (threadIdx.x < 2 && s_out[threadIdx.x]) atomicAdd(&goutside[threadIdx.x], (unsigned long long)s_out[threadIdx.x]);
}

// Large-nbins variant: counters do not fit one CTA's shared memory as 32-bit words; v1 counts straight
// into the global 64-bit bins (L2 atomics).
struct HistGlobalF {
    float lo, hi, scale;
    int top;
    unsigned long long* gbins;
    uint32_t below = 0, above = 0;
    __device__ __forceinline__ void operator()(float x) {
        if (x >= lo && x <= hi) {
            const float v = __fmul_rn(__fsub_rn(x, lo), scale);
            int b = min(__float2int_rd(v), top);
            atomicAdd(&gbins[b], 1ull);
        } else {
            below += (x < lo) ? 1u : 0u;
            above += (x > hi) ? 1u : 0u;
        }
    }
};

__global__ void __launch_bounds__(kThreads)
hist_global_kernel(const float* __restrict__ d, uint64_t n, int nbins, float lo, float hi, float scale,
                   unsigned long long* __restrict__ gbins, unsigned long long* __restrict__ goutside) {
    __shared__ uint32_t s_out[2];
    if (threadIdx.x < 2) s_out[threadIdx.x] = 0;
    __syncthreads();
    HistGlobalF f;
    f.lo = lo; f.hi = hi; f.scale = scale; f.top = nbins - 1; f.gbins = gbins;
    stream_cube(d, n, f);
    if (f.below) atomicAdd(&s_out[0], f.below);
    if (f.above) atomicAdd(&s_out[1], f.above);
    __syncthreads();
    if (threadIdx.x < 2 && s_out[threadIdx.x]) atomicAdd(&goutside[threadIdx.x], (unsigned long long)s_out[threadIdx.x]);
}

// ------------------------------------------------------------------------------------------------
// Exact k-th value: steps 6-8.  The paper's Torben bisection (Alg. 1) counts voxels
// below/above/equal to a guess, ~31 passes; here each pass counts 2048 (1024) sub-ranges at once on the
// order-preserving key, so three passes fix all 32 bits.  PASS 0: digit = key>>21 (all voxels);
// PASS 1: voxels with key>>21 == prefix, digit = (key>>10)&2047; PASS 2: key>>10 == prefix,
// digit = key&1023.
// ------------------------------------------------------------------------------------------------
template <int PASS>
struct SelectF {
    uint32_t prefix;
    uint32_t* sbins;
    __device__ __forceinline__ void operator()(float x) {
        const uint32_t key = key_of(x);
        if (PASS == 0) {
            if (x == x) atomicAdd(&sbins[key >> 21], 1u);
        } else if (PASS == 1) {
            if (x == x && (key >> 21) == prefix) atomicAdd(&sbins[(key >> 10) & 2047u], 1u);
        } else {
            if (x == x && (key >> 10) == prefix) atomicAdd(&sbins[key & 1023u], 1u);
        }
    }
};

template <int PASS>
__global__ void __launch_bounds__(kThreads)
select_pass_kernel(const float* __restrict__ d, uint64_t n, const SelectState* __restrict__ st,
                   unsigned long long* __restrict__ gdigits) {
    __shared__ uint32_t sbins[kDigitBins];
    for (int i = threadIdx.x; i < kDigitBins; i += kThreads) sbins[i] = 0;
    __syncthreads();
    SelectF<PASS> f;
    f.prefix = (PASS == 0) ? 0u : st->prefix;
    f.sbins = sbins;
    if (PASS == 0 || !st->invalid) stream_cube(d, n, f);
    __syncthreads();
    for (int i = threadIdx.x; i < kDigitBins; i += kThreads) {
        uint32_t c = sbins[i];
        if (c) atomicAdd(&gdigits[i], (unsigned long long)c);
    }
}

// One CTA of 1024 threads: exclusive scan of the digit histogram, pick the bucket holding rank k,
// update (prefix, k), clear the histogram for the next pass.  After PASS 2 the 32-bit key is complete
// and is mapped back to the float.
template <int PASS>
__global__ void __launch_bounds__(1024)
select_scan_kernel(SelectState* __restrict__ st, unsigned long long* __restrict__ gdigits, int clear) {
    constexpr int NB = (PASS == 2) ? 1024 : kDigitBins;
    constexpr int BITS = (PASS == 2) ? 10 : 11;
    __shared__ unsigned long long warp_tot[32];
    __shared__ unsigned long long s_k;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    // thread t owns bins [t*PER, t*PER+PER)
    constexpr int PER = NB / 1024;
    unsigned long long c[PER > 0 ? PER : 1];
    unsigned long long mine = 0;
#pragma unroll
    for (int j = 0; j < PER; ++j) { c[j] = gdigits[tid * PER + j]; mine += c[j]; }
    unsigned long long incl = mine;
#pragma unroll
    for (int off = 1; off < 32; off <<= 1) {
        unsigned long long v = __shfl_up_sync(0xffffffffu, incl, off);
        if (lane >= off) incl += v;
    }
    if (lane == 31) warp_tot[warp] = incl;
    __syncthreads();
    if (warp == 0) {
        unsigned long long w = warp_tot[lane], wi = w;
#pragma unroll
        for (int off = 1; off < 32; off <<= 1) {
            unsigned long long v = __shfl_up_sync(0xffffffffu, wi, off);
            if (lane >= off) wi += v;
        }
        warp_tot[lane] = wi - w;  // exclusive prefix of warp totals
        if (lane == 31 && tid == 31) {
            // total over all bins
            unsigned long long total = wi;
            if (PASS == 0) {
                st->count = total;
                if (st->use_median) st->k = total ? (total - 1) / 2 : 0;
                st->invalid = (st->k >= total) ? 1u : 0u;
            }
            s_k = st->k;
        }
    }
    __syncthreads();
    const unsigned long long k = s_k;
    unsigned long long excl = warp_tot[warp] + (incl - mine);
    const bool invalid = st->invalid != 0;
    __syncthreads();
    if (!invalid) {
#pragma unroll
        for (int j = 0; j < PER; ++j) {
            if (c[j] && excl <= k && k < excl + c[j]) {  // exactly one (thread, j) satisfies this
                const uint32_t b = (uint32_t)(tid * PER + j);
                const uint32_t pre = (PASS == 0) ? b : ((st->prefix << BITS) | b);
                st->prefix = pre;
                st->k = k - excl;
                if (PASS == 2) st->result = __uint_as_float(bits_of_key(pre));
            }
            excl += c[j];
        }
    } else if (tid == 0) {
        st->result = __int_as_float(0x7fc00000);
    }
    if (clear) {  // leave the digit bins zeroed for the next pass
#pragma unroll
        for (int j = 0; j < PER; ++j) gdigits[tid * PER + j] = 0ull;
        if (PASS == 2) gdigits[1024 + tid] = 0ull;
    }
}

}  // namespace cube
