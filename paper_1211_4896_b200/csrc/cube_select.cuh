// cube_select.cuh -- exact k-th value / median by radix select (steps 6-8 of SURVEY.md sec. 8(a)).
//
// The paper's Torben bisection (Alg. 1) counts the voxels below / above /
// equal to one guess per pass, ~31 passes over the cube.  Here each pass counts 2048 (1024) sub-ranges of
// the order-preserving uint32 key at once, so three digits (11/11/10 bits) fix all 32 bits exactly:
//   PASS 0: digit = key>>21 over all non-NaN voxels;
//   PASS 1: voxels with key>>21 == prefix: digit = (key>>10)&2047, and their keys are appended to the
//           candidate buffer (step 8, "compaction");
//   PASS 2: key>>10 == prefix: digit = key&1023, read from the candidate buffer -- so the cube is read
//           twice, not three times.  If the bucket did not fit the buffer, PASS 2 streams the cube again.
// Like the paper's choice the cube itself is never written.
#pragma once
#include "cube_common.cuh"

namespace cube {

constexpr uint32_t kCandChunk = 256;  // keys reserved per global atomic by one warp

// Per-voxel work, written to stay at ~8 instructions with no branch:
//   PASS 0:  idx = NaN ? trash : key >> 21
//   PASS 1/2: kk = key - (prefix << S) (S = 21 / 10); the voxel is in the prefix bucket iff kk < 2^S
//            (unsigned), and then its digit is kk >> 10 (PASS 1) or kk (PASS 2); so
//            idx = min(kk >> 10, 2048) resp. min(kk, 1024) sends every other voxel to the trash counter
//            without a compare.  NaN keys can only fall into the buckets next to +-inf (top digit 0-3 or
//            2044-2047); only then (NANCHK) is the x == x test compiled in.
// The counter increment is an unconditional ATOMS.POPC.INC (hardware-aggregated over equal addresses).
template <int PASS, bool NANCHK>
struct SelectF {
    static constexpr uint32_t kSpan = (PASS == 1) ? (1u << 21) : (1u << 10);
    static constexpr int kDShift = (PASS == 1) ? 10 : 0;
    static constexpr uint32_t kTrash = (PASS == 2) ? 1024u : (uint32_t)kDigitBins;
    uint32_t base;     // prefix << 21 (PASS 1) or prefix << 10 (PASS 2)
    uint32_t* sbins;   // kDigitBins + 1 counters
    // PASS 1 compaction: each warp appends into a private reservation [w_pos, w_end) of the candidate
    // buffer and takes a new one of kCandChunk keys with ONE global atomic when it runs out (an atomic per
    // warp per tile on the single counter serialises in L2: 1 M atomics cost ~1 ms on config 2).  What is
    // left of the last reservation is filled with a key that cannot match, so the buffer has no stale slot.
    uint32_t* cand;
    unsigned long long* cand_n;
    unsigned long long cand_cap;
    unsigned long long w_pos = 0, w_end = 0;  // warp-uniform

    __device__ __forceinline__ uint32_t kk_of(float x) const {
        uint32_t kk = key_of(x) - base;
        if (NANCHK) kk = (x == x) ? kk : 0xFFFFFFFFu;
        return kk;
    }
    __device__ __forceinline__ void count(float x, uint32_t kk) {
        if (PASS == 0) atomicAdd(&sbins[(x == x) ? (key_of(x) >> 21) : kTrash], 1u);
        else atomicAdd(&sbins[min(kk >> kDShift, kTrash)], 1u);
    }
    __device__ __forceinline__ void key(uint32_t k) {  // PASS 2 over the candidate buffer (no NaN in it)
        atomicAdd(&sbins[min(k - base, kTrash)], 1u);
    }
    __device__ __forceinline__ void operator()(float x) {  // single voxels: head / tail / ragged last tile
        const uint32_t kk = (PASS == 0) ? 0u : kk_of(x);
        count(x, kk);
        if (PASS == 1 && kk < kSpan) {
            const unsigned long long pos = atomicAdd(cand_n, 1ull);
            if (pos < cand_cap) cand[pos] = kk + base;
        }
    }
    __device__ __forceinline__ void batch(const float4 (&r)[kUnroll]) {
        if (PASS != 1) {
#pragma unroll
            for (int j = 0; j < kUnroll; ++j) {
                const float v[4] = {r[j].x, r[j].y, r[j].z, r[j].w};
#pragma unroll
                for (int c = 0; c < 4; ++c) count(v[c], (PASS == 0) ? 0u : kk_of(v[c]));
            }
            return;
        }
        uint32_t mask = 0;
#pragma unroll
        for (int j = 0; j < kUnroll; ++j) {
            const float v[4] = {r[j].x, r[j].y, r[j].z, r[j].w};
#pragma unroll
            for (int c = 0; c < 4; ++c) {
                const uint32_t kk = kk_of(v[c]);
                count(v[c], kk);
                mask |= (kk < kSpan ? 1u : 0u) << (j * 4 + c);
            }
        }
        if (__any_sync(0xffffffffu, mask != 0)) {  // the bucket is ~0.1-3 % of the cube on the configs
            const uint32_t lane = threadIdx.x & 31;
            const uint32_t cnt = __popc(mask);
            uint32_t incl = cnt;
#pragma unroll
            for (int off = 1; off < 32; off <<= 1) {
                const uint32_t t = __shfl_up_sync(0xffffffffu, incl, off);
                if (lane >= off) incl += t;
            }
            const uint32_t total = __shfl_sync(0xffffffffu, incl, 31);
            const unsigned long long rem = w_end - w_pos;
            unsigned long long nb = 0;
            uint32_t size = 0;
            if (total > rem) {  // warp-uniform
                const uint32_t need = total - (uint32_t)rem;
                size = need > kCandChunk ? need : kCandChunk;
                if (lane == 0) nb = atomicAdd(cand_n, (unsigned long long)size);
                nb = __shfl_sync(0xffffffffu, nb, 0);
            }
            if (mask) {
                uint32_t slot = incl - cnt;
#pragma unroll
                for (int j = 0; j < kUnroll; ++j) {
                    const float v[4] = {r[j].x, r[j].y, r[j].z, r[j].w};
#pragma unroll
                    for (int c = 0; c < 4; ++c) {
                        if (mask & (1u << (j * 4 + c))) {
                            const unsigned long long idx = (slot < rem) ? w_pos + slot : nb + (slot - rem);
                            if (idx < cand_cap) cand[idx] = key_of(v[c]);
                            ++slot;
                        }
                    }
                }
            }
            if (total > rem) { w_pos = nb + (total - rem); w_end = nb + size; }
            else w_pos += total;
        }
    }
    // all lanes of every warp, after the streaming loop
    __device__ __forceinline__ void finish() {
        if (PASS != 1) return;
        const uint32_t sentinel = base ^ (1u << 21);  // top digit != prefix: never matches in PASS 2
        for (unsigned long long i = w_pos + (threadIdx.x & 31); i < w_end; i += 32)
            if (i < cand_cap) cand[i] = sentinel;
    }
};

template <int PASS, bool NANCHK>
__device__ __forceinline__ void select_run(const float* __restrict__ d, uint64_t n, SelectState* __restrict__ st,
                                           uint32_t* sbins, uint32_t* __restrict__ cand) {
    SelectF<PASS, NANCHK> f;
    f.base = (PASS == 0) ? 0u : (PASS == 1) ? (st->prefix << 21) : (st->prefix << 10);
    f.sbins = sbins;
    f.cand = cand;
    f.cand_n = &st->cand_n;
    f.cand_cap = (PASS == 1 && cand) ? st->cand_cap : 0ull;
    // cand_n is final when PASS 2 runs: it follows PASS 1 on the same stream
    if (PASS == 2 && cand && st->cand_n <= st->cand_cap) stream_keys<kThreads>(cand, st->cand_n, f);
    else stream_cube<kThreads>(d, n, f);
    f.finish();
}

template <int PASS>
__global__ void __launch_bounds__(kThreads)
select_pass_kernel(const float* __restrict__ d, uint64_t n, SelectState* __restrict__ st,
                   unsigned long long* __restrict__ gdigits, uint32_t* __restrict__ cand) {
    __shared__ uint32_t sbins[kDigitBins + 1];  // + trash counter
    for (int i = threadIdx.x; i <= kDigitBins; i += kThreads) sbins[i] = 0;
    __syncthreads();
    if (PASS == 0) {
        select_run<0, true>(d, n, st, sbins, cand);
    } else if (!st->invalid) {
        const uint32_t top = (PASS == 1) ? st->prefix : (st->prefix >> 11);  // first digit of the bucket
        if (top <= 3u || top >= 2044u) select_run<PASS, true>(d, n, st, sbins, cand);
        else select_run<PASS, false>(d, n, st, sbins, cand);
    }
    __syncthreads();
    constexpr int NB = (PASS == 2) ? 1024 : kDigitBins;
    for (int i = threadIdx.x; i < NB; i += kThreads) {
        uint32_t c = sbins[i];
        if (c) atomicAdd(&gdigits[i], (unsigned long long)c);
    }
}

// PASS 2 over the candidate buffer only (out-of-core: no third sweep over the host link).  The caller has
// checked cand_n <= cand_cap on the host.
__global__ void __launch_bounds__(kThreads)
select_cand_kernel(SelectState* __restrict__ st, unsigned long long* __restrict__ gdigits,
                   const uint32_t* __restrict__ cand) {
    __shared__ uint32_t sbins[kDigitBins + 1];
    for (int i = threadIdx.x; i <= kDigitBins; i += kThreads) sbins[i] = 0;
    __syncthreads();
    SelectF<2, false> f;
    f.base = st->prefix << 10;
    f.sbins = sbins;
    if (!st->invalid) stream_keys<kThreads>(cand, st->cand_n, f);
    __syncthreads();
    for (int i = threadIdx.x; i < 1024; i += kThreads) {
        uint32_t c = sbins[i];
        if (c) atomicAdd(&gdigits[i], (unsigned long long)c);
    }
}

// One CTA of 1024 threads: exclusive scan of the digit histogram, pick the bucket holding rank k,
// update (prefix, k), clear the histogram for the next pass (step 7: the paper's server-side "determine
// the next guess").  After PASS 2 the 32-bit key is complete and is mapped back to the float.
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
        if (lane == 31) {
            const unsigned long long total = wi;  // over all bins
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
