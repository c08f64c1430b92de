// cube_select_multi.cuh -- several exact ranks of one cube in TWO reads (cube_kth_multi; config 3 of BASELINE.json
// asks for the median and the values at n/100 and 99n/100).
//
// The radix select of cube_select.cuh (which replaces the ~31 passes of the paper's Alg. 1)
// fixes one rank per selection.  Here up to kMultiGroup ranks share both reads of the cube:
//   read 1  first digit of every voxel (select_pass_kernel<0>, counts kept in the context);
//           multi_locate_kernel: the first-digit bucket and the residual rank of EVERY requested rank;
//   read 2  multi_gather_kernel: the keys of the voxels of ANY of those buckets go to the candidate buffer;
//   then, on the candidates only (a few per cent of the cube): per rank the second digit (multi_cand_kernel<1>,
//   multi_scan_kernel<1>) and the third (multi_cand_kernel<2>, multi_scan_kernel<2>), all ranks in one launch.
// If the buckets together do not fit the candidate buffer, MultiState::ok stays 0 and the caller's per-rank
// selections (enqueued behind, skipped when ok == 1) store the results into the same record: the decision never leaves the device.
// The cube is never written.
#pragma once
#include "cube_select.cuh"

namespace cube {

constexpr int kMultiGroup = 4;   // ranks per gather read (the bucket test is unrolled over them)

struct MultiState {
    unsigned long long k[kMultiGroup];       // residual rank inside the current prefix bucket
    unsigned long long count;                // non-NaN voxels
    unsigned long long cand_n, cand_cap;     // keys gathered / capacity of the candidate buffer
    uint32_t prefix[kMultiGroup];            // key bits fixed so far (right aligned)
    uint32_t rawbase[kMultiGroup];           // raw_of_digit(first digit) << kShift0 of the nb DISTINCT buckets
    uint32_t nb;                             // distinct first-digit buckets of the valid ranks (0: idle)
    uint32_t invalid[kMultiGroup];           // 1: k >= count, result NaN
    uint32_t nk;
    uint32_t ok;                             // 1: every result of this group was found on the candidates
    uint32_t idle;                           // 1: no rank of the group is below count (every result is NaN)
    float result[kMultiGroup];
};

struct MultiRanks { unsigned long long k[kMultiGroup]; uint32_t nk; };

// Bucket location for every rank of the group on the first-digit counts (raw-indexed, as select_pass_kernel<0>
// leaves them): one CTA of 1024 threads, thread t owns the kBins0/1024 consecutive digits in KEY order.
__global__ void __launch_bounds__(1024)
multi_locate_kernel(MultiState* __restrict__ ms, const unsigned long long* __restrict__ coarse, MultiRanks req,
                    unsigned long long cand_cap) {
    constexpr int PER = kBins0 / 1024;
    static_assert(kBins0 % 1024 == 0, "first digit bins per thread");
    static_assert(kMultiGroup == 4, "multi_gather_kernel dispatches on 1...4 distinct buckets");
    __shared__ unsigned long long wtot[32];
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    unsigned long long v[PER], mine = 0;
#pragma unroll
    for (int j = 0; j < PER; ++j) { v[j] = __ldcg(&coarse[raw_of_digit((uint32_t)(tid * PER + j))]); mine += v[j]; }
    unsigned long long incl = mine;
#pragma unroll
    for (int off = 1; off < 32; off <<= 1) {
        const unsigned long long u = __shfl_up_sync(0xffffffffu, incl, off);
        if (lane >= off) incl += u;
    }
    if (lane == 31) wtot[warp] = incl;
    __syncthreads();
    unsigned long long before = 0, total = 0;
    for (int w = 0; w < 32; ++w) { const unsigned long long t = wtot[w]; if (w < warp) before += t; total += t; }
    unsigned long long excl = before + incl - mine;
    // owners leave (bucket, residual rank) in shared memory; thread 0 then writes the whole record once (no global
    // read-backs in this one-CTA latency chain)
    __shared__ uint32_t s_b[kMultiGroup];
    __shared__ unsigned long long s_k[kMultiGroup];
#pragma unroll
    for (int j = 0; j < PER; ++j) {
        for (int i = 0; i < (int)req.nk; ++i) {
            const unsigned long long k = req.k[i];
            if (v[j] && excl <= k && k < excl + v[j]) {          // exactly one (thread, j) per valid rank
                s_b[i] = (uint32_t)(tid * PER + j);
                s_k[i] = k - excl;
            }
        }
        excl += v[j];
    }
    __syncthreads();
    if (tid == 0) {
        uint32_t ub[kMultiGroup], nb = 0;   // the distinct buckets of the valid ranks (the gather tests exactly nb)
        for (int i = 0; i < kMultiGroup; ++i) {
            const bool valid = i < (int)req.nk && req.k[i] < total;
            ms->invalid[i] = valid ? 0u : 1u;
            ms->result[i] = __int_as_float(0x7fc00000);
            ms->k[i] = valid ? s_k[i] : 0ull;
            ms->prefix[i] = valid ? s_b[i] : 0u;
            if (!valid) continue;
            const uint32_t b = raw_of_digit(s_b[i]) << kShift0;
            bool seen = false;
            for (uint32_t j = 0; j < nb; ++j) seen = seen || ub[j] == b;
            if (!seen) ub[nb++] = b;
        }
        for (uint32_t j = 0; j < (uint32_t)kMultiGroup; ++j) ms->rawbase[j] = j < nb ? ub[j] : 0u;
        ms->count = total; ms->cand_n = 0; ms->cand_cap = cand_cap; ms->nk = req.nk; ms->ok = 0;
        ms->nb = nb;
        ms->idle = nb == 0 ? 1u : 0u;   // no rank below count: the gather returns at once, every result is NaN
    }
}

// Read 2: append the key of every non-NaN voxel whose first digit is one of the group's buckets.
// Hot path per voxel: NB IMAD (bits - rawbase < 2^19 <=> the raw top bits match) + minima (NB = the number of
// DISTINCT buckets, 1...kMultiGroup: compiled for each); one test per thread per tile; the flagged rows are
// revisited from the registers.  Staging per warp as in SelectF (PASS 1).
template <int NB>
struct GatherF {
    static constexpr uint32_t kSpan = 1u << kShift0;
    uint32_t rb[NB];
    uint32_t* s_cnt; uint32_t* s_buf;
    uint32_t* cand; unsigned long long* cand_n; unsigned long long cand_cap;
    bool compacting;
    // bits - rawbase < 2^19 (mod 2^32) <=> the raw top bits match; the subtraction is issued as IMAD on the FMA pipe
    // (multiplier 1 from constant memory, as in SelectF), so only the minima use the ALU pipe; rb[] holds -rawbase
    __device__ __forceinline__ uint32_t dist(float x) const {
        uint32_t m = SelectF<1, false>::sub_fma(x, rb[0]);
#pragma unroll
        for (int i = 1; i < NB; ++i) m = min(m, SelectF<1, false>::sub_fma(x, rb[i]));
        return m;
    }
    __device__ __forceinline__ void take(float x) {
        if (dist(x) < kSpan && x == x && compacting) {
            const uint32_t slot = atomicAdd(s_cnt, 1u);
            CUBE_CHECK(slot < kStageCap);
            s_buf[slot] = key_of(x);
        }
    }
    __device__ __forceinline__ void operator()(float x) {   // head / tail / ragged last tile: straight to the buffer
        if (dist(x) < kSpan && x == x) {
            const unsigned long long pos = atomicAdd(cand_n, 1ull);
            if (pos < cand_cap) cand[pos] = key_of(x);
        }
    }
    __device__ __forceinline__ void flush(uint32_t c) {
        const uint32_t lane = threadIdx.x & 31;
        unsigned long long pos = 0;
        if (lane == 0) pos = atomicAdd(cand_n, (unsigned long long)c);
        pos = __shfl_sync(0xffffffffu, pos, 0);
        if (pos + c <= cand_cap) {
            for (uint32_t i = lane; i < c; i += 32) cand[pos + i] = s_buf[i];
        } else {
            compacting = false;   // does not fit: cand_n > cand_cap tells the scan kernels, stop staging
        }
        __syncwarp();
        if (lane == 0) *s_cnt = 0;
        __syncwarp();
    }
    __device__ __forceinline__ void batch(const float4 (&r)[kUnroll], const float4*) {
        uint32_t rm[kUnroll];
#pragma unroll
        for (int j = 0; j < kUnroll; ++j)
            rm[j] = min(min(dist(r[j].x), dist(r[j].y)), min(dist(r[j].z), dist(r[j].w)));
        uint32_t tmin = rm[0];
#pragma unroll
        for (int j = 1; j < kUnroll; ++j) tmin = min(tmin, rm[j]);
        if (tmin < kSpan) {
#pragma unroll
            for (int j = 0; j < kUnroll; ++j)
                if (rm[j] < kSpan) { take(r[j].x); take(r[j].y); take(r[j].z); take(r[j].w); }
        }
        if (compacting) {   // warp-uniform
            __syncwarp();
            const uint32_t c = *reinterpret_cast<volatile uint32_t*>(s_cnt);
            if (c > kStageThresh) flush(c);
        }
    }
};

template <int NB>
__device__ __forceinline__ void gather_run(const float* __restrict__ d, uint64_t n, MultiState* __restrict__ ms,
                                           uint32_t* __restrict__ cand, unsigned long long cap, uint32_t* s_buf,
                                           uint32_t* s_cnt) {
    GatherF<NB> f;
#pragma unroll
    for (int i = 0; i < NB; ++i) f.rb[i] = 0u - ms->rawbase[i];
    f.s_buf = s_buf; f.s_cnt = s_cnt;
    f.cand = cand; f.cand_n = &ms->cand_n; f.cand_cap = cap; f.compacting = true;
    stream_cube<kThreads>(d, n, f);
    __syncwarp();
    const uint32_t c = *reinterpret_cast<volatile uint32_t*>(s_cnt);
    if (c) f.flush(c);
}

__global__ void __launch_bounds__(kThreads, 3)
multi_gather_kernel(const float* __restrict__ d, uint64_t n, MultiState* __restrict__ ms, uint32_t* __restrict__ cand) {
    __shared__ uint32_t stage[(kThreads / 32) * (kStageCap + 1)];
    const unsigned long long cap = ms->cand_cap;
    if (ms->idle) return;
    if (cap == 0 || cand == nullptr) {   // no candidate buffer: cand_n says "does not fit"
        if (blockIdx.x == 0 && threadIdx.x == 0) ms->cand_n = ~0ull;
        return;
    }
    const uint32_t warp = threadIdx.x >> 5;
    uint32_t* s_buf = stage + warp * kStageCap;
    uint32_t* s_cnt = stage + (kThreads / 32) * kStageCap + warp;
    if ((threadIdx.x & 31) == 0) *s_cnt = 0;
    __syncwarp();
    switch (ms->nb) {   // uniform over the grid
        case 1: gather_run<1>(d, n, ms, cand, cap, s_buf, s_cnt); break;
        case 2: gather_run<2>(d, n, ms, cand, cap, s_buf, s_cnt); break;
        case 3: gather_run<3>(d, n, ms, cand, cap, s_buf, s_cnt); break;
        default: gather_run<kMultiGroup>(d, n, ms, cand, cap, s_buf, s_cnt); break;
    }
}

// Digit counts of every rank of the group over the candidates, ONE read of the buffer (two 128-bit loads in flight
// per thread): PASS 1 = second digit of the keys of a rank's first-digit bucket, PASS 2 = third digit of the keys of
// its (first, second) prefix.  Counts go to gdigits[rank * kBins1 ...].  A key outside a rank's bucket touches no
// counter (a trash counter would be one hot address).
template <int PASS>
__global__ void __launch_bounds__(kThreads)
multi_cand_kernel(const MultiState* __restrict__ ms, unsigned long long* __restrict__ gdigits,
                  const uint32_t* __restrict__ cand) {
    constexpr int NB = (PASS == 1) ? kBins1 : kBins2;
    static_assert(kMultiGroup * kBins1 <= kDigitBins && kBins2 <= kBins1, "per-rank digit slots");
    __shared__ uint32_t sbins[kMultiGroup][NB];
    const unsigned long long m = ms->cand_n;
    if (m > ms->cand_cap) return;
    uint32_t base[kMultiGroup];
    bool live[kMultiGroup];
#pragma unroll
    for (int r = 0; r < kMultiGroup; ++r) {
        live[r] = r < (int)ms->nk && !ms->invalid[r];
        base[r] = (PASS == 1) ? (ms->prefix[r] << kShift0) : (ms->prefix[r] << kBits2);
    }
    for (int i = threadIdx.x; i < kMultiGroup * NB; i += kThreads) (&sbins[0][0])[i] = 0;
    __syncthreads();
    auto one = [&](uint32_t key) {
#pragma unroll
        for (int r = 0; r < kMultiGroup; ++r) {
            const uint32_t t = key - base[r];
            const uint32_t idx = (PASS == 1) ? (t >> kBits2) : t;    // outside the bucket: >= NB
            if (live[r] && idx < (uint32_t)NB) atomicAdd(&sbins[r][idx], 1u);
        }
    };
    const uint4* __restrict__ c4 = reinterpret_cast<const uint4*>(cand);   // cudaMalloc'ed: 16-byte aligned
    const uint64_t m4 = m >> 2, stride = (uint64_t)gridDim.x * kThreads, g = (uint64_t)blockIdx.x * kThreads + threadIdx.x;
    for (uint64_t i = g; i < m4; i += 2 * stride) {
        const uint4 a = __ldg(c4 + i);
        const bool two = i + stride < m4;
        const uint4 b = two ? __ldg(c4 + i + stride) : make_uint4(0, 0, 0, 0);
        one(a.x); one(a.y); one(a.z); one(a.w);
        if (two) { one(b.x); one(b.y); one(b.z); one(b.w); }
    }
    if (g < (m & 3ull)) one(__ldg(cand + (m4 << 2) + g));
    __syncthreads();
#pragma unroll
    for (int r = 0; r < kMultiGroup; ++r) {
        if (!live[r]) continue;
        unsigned long long* gd = gdigits + (size_t)r * kBins1;
        for (int i = threadIdx.x; i < NB; i += kThreads) {
            const uint32_t c = sbins[r][i];
            if (c) atomicAdd(&gd[i], (unsigned long long)c);
        }
    }
}

// Bucket location of one rank (blockIdx.x) on its PASS digit counts; clears them.  After PASS 2 the key is complete.
template <int PASS>
__global__ void __launch_bounds__(kBins1)
multi_scan_kernel(MultiState* __restrict__ ms, unsigned long long* __restrict__ gdigits) {
    constexpr int NB = (PASS == 1) ? kBins1 : kBins2;
    constexpr int BITS = (PASS == 1) ? kBits1 : kBits2;
    __shared__ unsigned long long wtot[32];
    const int r = blockIdx.x, tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const bool fits = ms->cand_n <= ms->cand_cap;
    unsigned long long* g = gdigits + (size_t)r * kBins1;
    const unsigned long long v = (tid < NB) ? __ldcg(&g[tid]) : 0ull;
    if (tid < NB && v) g[tid] = 0ull;
    unsigned long long incl = v;
#pragma unroll
    for (int off = 1; off < 32; off <<= 1) {
        const unsigned long long u = __shfl_up_sync(0xffffffffu, incl, off);
        if (lane >= off) incl += u;
    }
    if (lane == 31) wtot[warp] = incl;
    __syncthreads();
    unsigned long long before = 0;
    for (int w = 0; w < warp; ++w) before += wtot[w];
    const unsigned long long excl = before + incl - v, k = ms->k[r];
    const bool live = fits && r < (int)ms->nk && !ms->invalid[r];
    __syncthreads();   // every thread has read k before the owner replaces it
    if (live && v && excl <= k && k < excl + v) {   // exactly one thread
        const uint32_t pre = (ms->prefix[r] << BITS) | (uint32_t)tid;
        ms->prefix[r] = pre;
        ms->k[r] = k - excl;
        if (PASS == 2) ms->result[r] = __uint_as_float(bits_of_key(pre));
    }
}

// After the PASS 2 scans: the group is done iff the candidates fitted (ok is read by LATER launches only: the
// per-rank selections enqueued behind skip themselves when it is set).
__global__ void multi_done_kernel(MultiState* __restrict__ ms) {
    if (ms->cand_n <= ms->cand_cap) ms->ok = 1;
}

}  // namespace cube
