// cube_select.cuh -- exact k-th value / median by radix select (steps 6-8 of SURVEY.md sec. 8(a)).
//
// The paper's Torben bisection (Alg. 1) counts the voxels below / above /
// equal to one guess per pass, ~31 passes over the cube.  Here each pass counts 8192 (1024, 512) sub-ranges of
// the order-preserving uint32 key at once, so three digits (13/10/9 bits) fix all 32 bits exactly:
//   PASS 0: digit = key>>19 over all non-NaN voxels;
//   PASS 1: voxels with key>>19 == prefix: digit = (key>>9)&1023, and their keys are appended to the
//           candidate buffer (step 8, "compaction");
//   PASS 2: key>>9 == prefix: digit = key&511, read from the candidate buffer -- so the cube is read
//           twice, not three times.  If the bucket did not fit the buffer, PASS 2 streams the cube again.
// Like the paper's choice the cube itself is never written.
#pragma once
#include "cube_common.cuh"

namespace cube {

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
    unsigned long long cand_n;  // keys of the pass-0 bucket seen by the compacting pass 1
    unsigned long long cand_cap;  // capacity of the candidate buffer, in keys
    uint32_t cand_done;         // 1: the last digit has been counted on the candidates (select_cand_kernel), so the
    uint32_t pad_;              //    per-brick PASS 2 launches of a brick-streamed / sharded run return at once
    unsigned long long bucket_n;  // voxels in the bucket chosen by the last bucket location
};
// A first-digit bucket holding more than 1/8 of the voxels (tie-heavy data: 30 % of config 4's voxels are one value)
// cannot be compacted into a candidate buffer of 1/16 of the cube and would keep PASS 1's cold path busy on nearly
// every row: PASS 1 then counts the second digit of every voxel in its hot loop instead (as PASS 0 and PASS 2 do) and
// PASS 2 reads the cube a third time.  Decided on the device from the counts.
__device__ __forceinline__ bool select_dense(const SelectState* st) { return st->bucket_n * 8ull > st->count; }

// PASS 1 compaction ("step 8"): every warp stages the keys of the prefix bucket in its own slice of shared
// memory and moves them to the candidate buffer in coalesced runs, reserving the space with ONE global atomic
// per flush.  A warp checks its fill level once per tile (1024 voxels per warp), so a slice holds the flush
// threshold plus one whole tile and can never overflow -- also on a constant cube, where every voxel is a
// candidate.  (v2 reserved space by ballot + warp scan per tile: at the 0.3 % bucket density of config 2
// ~95 % of the warp tiles took that path to place ~3 keys, 564 M instructions, 5.1 TB/s;
// round-1 ncu capture.)
constexpr uint32_t kStageThresh = 128;                                 // flush when more keys than this wait
constexpr uint32_t kStageCap = kStageThresh + 32u * 4u * kUnroll;      // + one tile of a warp: 1152 keys
constexpr int kStageBytes = (kThreads / 32) * (int)kStageCap * 4;      // 36 KiB per CTA

// Per-voxel work, branch-free:
//   PASS 0:  idx = NaN ? trash : bits >> 19 (the RAW top 13 bits; the scan kernel reads the bins in key order
//            through raw_of_digit(), so the key transform is not paid per voxel); ATOMS.POPC.INC
//            (hardware-aggregated over equal addresses).  SHF, FSETP, SEL, LEA, ATOMS.
//   PASS 1:  the voxel is in the prefix bucket iff bits - rawbase < 2^19 (mod 2^32): IMAD per voxel, row minima,
//            one test per tile share of 32 voxels (1.7 issue slots per voxel, NO shared-memory traffic).
//            Only the rows that hold a voxel of the bucket (the bucket is 0.05-3 % of the cube on the
//            configs) are visited again by a cold path that re-loads the row (an L2 hit: its line has just been
//            streamed), counts the digit (kk >> 9) and stages the key.  So pass 1 costs less issue bandwidth
//            than pass 0.
//   PASS 2 over the cube (only when the candidates did not fit): idx = min(key - (prefix << 9), 512) sends every
//            voxel outside the bucket to the trash counter without a compare.
//   NaN keys can only fall into the buckets beyond +-inf (digit_may_hold_nan); only then (NANCHK)
//   is the x == x test compiled in.
//   DEV (NEXT-1, median absolute deviation): the value that is ranked is y = |fl32(x - center)|
//   instead of x (one FADD; the absolute value folds into the consumer as an operand modifier or a LOP).
//   y is NaN exactly when x is (or for Inf - Inf), so the NaN handling carries over unchanged.
template <int PASS, bool NANCHK, bool DEV = false>
struct SelectF {
    static constexpr uint32_t kSpan = 1u << kShift0;
    static constexpr uint32_t kTrash = (PASS == 2) ? (uint32_t)kBins2 : (uint32_t)kBins0;
    uint32_t base;     // prefix << 19 (PASS 1) or prefix << 9 (PASS 2)
    uint32_t* sbins;   // bins of this pass + 1 trash counter
    // PASS 1 compaction state
    bool compacting = false;    // false once the candidate buffer is known to be too small (or absent)
    uint32_t* s_cnt = nullptr;  // this warp's fill counter (shared memory)
    uint32_t* s_buf = nullptr;  // this warp's kStageCap slots (shared memory)
    uint32_t* cand = nullptr;
    unsigned long long* cand_n = nullptr;
    unsigned long long cand_cap = 0;

    // PASS 1 hot path: key >> 19 == prefix  <=>  bits >> 19 == raw_of_digit(prefix)  <=>  (bits ^ rawbase) < 2^19
    // (LOP3), reduced over each 4-voxel row with VIMNMX3; NaN voxels may flag a row, the cold path drops them.
    uint32_t rawbase = 0;  // raw_of_digit(prefix) << 19
    float center = 0.0f;   // DEV
    static __device__ __forceinline__ float xf(float x, float center_) {
        return DEV ? fabsf(__fsub_rn(x, center_)) : x;
    }
    static __device__ __forceinline__ uint32_t sub_fma(float y, uint32_t negbase) {   // bits(y) - rawbase on the FMA pipe
        uint32_t t;
        asm("mad.lo.u32 %0, %1, %2, %3;" : "=r"(t) : "r"(__float_as_uint(y)), "r"(c_one), "r"(negbase));
        return t;
    }
    __device__ __forceinline__ uint32_t kk_of(float x) const {
        uint32_t kk = key_of(x) - base;
        if (NANCHK) kk = (x == x) ? kk : 0xFFFFFFFFu;
        return kk;
    }
    __device__ __forceinline__ void count(float x) {  // PASS 0 / PASS 2: every voxel increments a counter
        x = xf(x, center);
        if (PASS == 0) smem_inc(smem_addr(sbins), (x == x) ? raw_digit(x) : kTrash);
        else atomicAdd(&sbins[min(kk_of(x), kTrash)], 1u);
    }
    __device__ __forceinline__ void key(uint32_t k) {  // PASS 2 over the candidate buffer (no NaN in it)
        atomicAdd(&sbins[min(k - base, kTrash)], 1u);
    }
    __device__ __forceinline__ void operator()(float x) {  // single voxels: head / tail / ragged last tile
        if (PASS != 1) { count(x); return; }
        take1(xf(x, center), base, sbins, compacting ? s_cnt : nullptr, s_buf);
    }
    // Cold path of PASS 1 (static, arguments by value: the functor itself stays in registers): revisit the
    // flagged 4-voxel rows, count the second digit of the voxels of the bucket and stage their keys.
    static __device__ __forceinline__ void take1(float x, uint32_t base_, uint32_t* sbins_, uint32_t* s_cnt_,
                                                 uint32_t* s_buf_) {
        const uint32_t kk = key_of(x) - base_;
        if (kk < kSpan && x == x) {
            atomicAdd(&sbins_[kk >> kBits2], 1u);
            if (s_cnt_) {
                const uint32_t slot = atomicAdd(s_cnt_, 1u);
                CUBE_CHECK(slot < kStageCap);
                s_buf_[slot] = kk + base_;
            }
        }
    }
    static __device__ __noinline__ void cold(uint32_t rows, const float4* __restrict__ p, uint32_t base_,
                                             uint32_t* sbins_, uint32_t* s_cnt_, uint32_t* s_buf_, float center_) {
        do {
            const int j = __ffs(rows) - 1;
            rows &= rows - 1;
            const float4 q = __ldcg(p + j * kThreads);  // L2 hit: the line has just been streamed
            take1(xf(q.x, center_), base_, sbins_, s_cnt_, s_buf_);
            take1(xf(q.y, center_), base_, sbins_, s_cnt_, s_buf_);
            take1(xf(q.z, center_), base_, sbins_, s_cnt_, s_buf_);
            take1(xf(q.w, center_), base_, sbins_, s_cnt_, s_buf_);
        } while (rows);
    }
    // all lanes of the warp: move the c staged keys to the candidate buffer
    __device__ __forceinline__ void flush(uint32_t c) {
        const uint32_t lane = threadIdx.x & 31;
        unsigned long long pos = 0;
        if (lane == 0) pos = atomicAdd(cand_n, (unsigned long long)c);
        pos = __shfl_sync(0xffffffffu, pos, 0);
        CUBE_CHECK(c <= kStageCap);
        if (pos + c <= cand_cap) {
            for (uint32_t i = lane; i < c; i += 32) cand[pos + i] = s_buf[i];
        } else {
            compacting = false;  // the bucket does not fit: PASS 2 will stream the cube, stop staging
        }
        __syncwarp();
        if (lane == 0) *s_cnt = 0;
        __syncwarp();
    }
    __device__ __forceinline__ uint32_t staged() const {
        __syncwarp();
        return *reinterpret_cast<volatile uint32_t*>(s_cnt);
    }
    __device__ __forceinline__ void batch(const float4 (&r)[kUnroll], const float4* __restrict__ p) {
        if (PASS != 1) {
#pragma unroll
            for (int j = 0; j < kUnroll; ++j) { count(r[j].x); count(r[j].y); count(r[j].z); count(r[j].w); }
            return;
        }
        // Does this thread's share of the tile (8 rows of 4 voxels) hold a voxel of the bucket?  bits - rawbase <
        // 2^19 (mod 2^32) <=> the top 13 raw bits match; the subtraction is issued as IMAD on the FMA pipe
        // (multiplier 1 from constant memory), each row's minimum takes a VIMNMX3 + VIMNMX, the tile minimum four
        // more VIMNMX3, then ONE test per tile share: 1.7 issue slots per voxel, 0.7 of them on the ALU pipe (v3:
        // LOP3 per voxel and a test per row, 2.7 / 2.7).  The row flags are only formed behind the branch.
        // NaN voxels may flag a row, the cold path drops them.
        uint32_t rm[kUnroll];
        const uint32_t negbase = 0u - rawbase;
#pragma unroll
        for (int j = 0; j < kUnroll; ++j)
            rm[j] = min(min(sub_fma(xf(r[j].x, center), negbase), sub_fma(xf(r[j].y, center), negbase)),
                        min(sub_fma(xf(r[j].z, center), negbase), sub_fma(xf(r[j].w, center), negbase)));
        uint32_t tmin = rm[0];
#pragma unroll
        for (int j = 1; j < kUnroll; ++j) tmin = min(tmin, rm[j]);
        if (tmin < kSpan) {
            uint32_t rows = 0;
#pragma unroll
            for (int j = 0; j < kUnroll; ++j) rows |= (rm[j] < kSpan ? 1u : 0u) << j;
            cold(rows, p, base, sbins, compacting ? s_cnt : nullptr, s_buf, center);
        }
        if (compacting) {               // warp-uniform
            const uint32_t c = staged();
            if (c > kStageThresh) flush(c);
        }
    }
    // all lanes of every warp, after the streaming loop
    __device__ __forceinline__ void finish() {
        if (PASS != 1 || s_cnt == nullptr) return;
        const uint32_t c = staged();
        if (c) flush(c);
    }
    // PASS 1 set-up: `stage` = kThreads/32 slices of kStageCap keys + kThreads/32 counters (shared memory)
    __device__ __forceinline__ void init_stage(uint32_t* stage, uint32_t* cand_, unsigned long long* cand_n_,
                                               unsigned long long cap) {
        const uint32_t warp = threadIdx.x >> 5;
        s_buf = stage + warp * kStageCap;
        s_cnt = stage + (kThreads / 32) * kStageCap + warp;
        if ((threadIdx.x & 31) == 0) *s_cnt = 0;
        __syncwarp();
        cand = cand_; cand_n = cand_n_; cand_cap = cap;
        compacting = (cand_ != nullptr) && cap != 0;
    }
};

// PASS 1 on a dense bucket: digit (key - base) >> 9 of every voxel, everything outside the bucket to the trash counter.
template <bool NANCHK, bool DEV>
struct SelectDense1F {
    uint32_t base;
    uint32_t* sbins;   // kBins1 + 1
    float center;
    __device__ __forceinline__ void operator()(float x) {
        const float y = SelectF<1, NANCHK, DEV>::xf(x, center);
        uint32_t idx = min((key_of(y) - base) >> kBits2, (uint32_t)kBins1);
        if (NANCHK) idx = (y == y) ? idx : (uint32_t)kBins1;
        atomicAdd(&sbins[idx], 1u);
    }
    CUBE_DEFAULT_BATCH()
};

template <int PASS, bool NANCHK, bool DEV>
__device__ __forceinline__ void select_run(const float* __restrict__ d, uint64_t n, SelectState* __restrict__ st,
                                           uint32_t* sbins, uint32_t* stage, uint32_t* __restrict__ cand,
                                           float center) {
    if (PASS == 1 && select_dense(st)) {   // uniform over the grid
        SelectDense1F<NANCHK, DEV> g;
        g.base = st->prefix << kShift0; g.sbins = sbins; g.center = center;
        stream_cube<kThreads>(d, n, g);
        if (blockIdx.x == 0 && threadIdx.x == 0) st->cand_n = st->cand_cap + 1ull;   // "did not fit": PASS 2 streams the cube
        return;
    }
    SelectF<PASS, NANCHK, DEV> f;
    f.base = (PASS == 0) ? 0u : (PASS == 1) ? (st->prefix << kShift0) : (st->prefix << kBits2);
    f.rawbase = (PASS == 1) ? (raw_of_digit(st->prefix) << kShift0) : 0u;
    f.sbins = sbins;
    f.center = center;
    if (PASS == 1) f.init_stage(stage, cand, &st->cand_n, st->cand_cap);
    // cand_n is final when PASS 2 runs: it follows PASS 1 on the same stream
    if (PASS == 2 && cand && st->cand_n <= st->cand_cap) stream_keys<kThreads>(cand, st->cand_n, f);
    else stream_cube<kThreads>(d, n, f);
    f.finish();
}

// Bucket location (step 7: the paper's server-side "determine the next guess"): exclusive scan of
// the digit histogram, pick the bucket holding rank k, update (prefix, k), clear the histogram for the next pass.
// After PASS 2 the 32-bit key is complete and is mapped back to the float.  Run by ONE CTA of THREADS threads:
// either the stand-alone select_scan_kernel (brick-streamed and sharded runs, CUBE_REUSE_COARSE) or -- fused -- the
// last CTA to finish the pass kernel that produced the counts (in-core calls: three launches fewer per selection).
// With init.enabled (PASS 0) the whole SelectState is initialised here from kernel arguments, so no host-to-device
// copy precedes a selection.  `sm` = kScanSmem words of shared memory.
struct SelectInit {
    unsigned long long k, cand_cap;
    float* result_out;   // PASS 2: also write the result here (the caller's buffer when the device can reach it), or null
    uint32_t use_median, enabled;
};

constexpr int kScanSmem = 256 + 4;   // words (u64) of shared memory select_scan_body needs

// Sum of a 64-bit value over the warp, every lane gets it: three REDUX.SUM on 24-bit limbs (32 x 2^24 < 2^32, so no
// limb sum wraps) instead of five 64-bit shuffle-and-add steps -- 3 instructions per chunk, not ~25; the bucket
// location is ONE CTA's instruction and latency chain at the tail of every pass.
__device__ __forceinline__ unsigned long long warp_sum_u64(unsigned long long v) {
    const uint32_t a = (uint32_t)v & 0xFFFFFFu, b = (uint32_t)(v >> 24) & 0xFFFFFFu, c = (uint32_t)(v >> 48);
    return (unsigned long long)__reduce_add_sync(0xffffffffu, a) +
           ((unsigned long long)__reduce_add_sync(0xffffffffu, b) << 24) +
           ((unsigned long long)__reduce_add_sync(0xffffffffu, c) << 48);
}

// Two levels, every global load coalesced and independent of the others: (1) each warp sums chunks of 32 consecutive
// bins (one load per lane per chunk, up to 8 chunks in flight) into shared memory; (2) warp 0 scans the <= 256 chunk
// totals and finds the chunk holding rank k; (3) the warp that loaded that chunk finds the bin in its registers (when
// a warp's chunks did not all fit one round -- 8192 bins on 256 threads -- it loads the chunk once more).  The scan
// is a chain of dependent L2 round trips run by ONE CTA at the tail of a pass (~0.5 us each), so everything that
// does not depend on the counts (the rank asked for, the prefix so far) is loaded before the bins.
template <int PASS, int THREADS>
__device__ __forceinline__ void select_scan_body(SelectState* __restrict__ st, unsigned long long* __restrict__ gdigits,
                                                 int clear, const SelectInit& init, unsigned long long* sm,
                                                 const uint32_t* local_bins = nullptr) {
    constexpr int NB = (PASS == 0) ? kBins0 : (PASS == 1) ? kBins1 : kBins2;
    constexpr int BITS = (PASS == 0) ? kBits0 : (PASS == 1) ? kBits1 : kBits2;
    constexpr int CHUNKS = NB / 32, NW = THREADS / 32;
    constexpr int CPL = (CHUNKS + 31) / 32;               // chunk totals per lane of warp 0
    constexpr int CPW = (CHUNKS + NW - 1) / NW;           // chunks per warp
    constexpr int INFL = CPW < 8 ? CPW : 8;               // loads in flight per lane
    constexpr bool KEEP = (CPW <= INFL);                  // a warp's chunks stay in registers
    static_assert(CHUNKS <= 256, "chunk totals must fit the shared array");
    unsigned long long* ctot = sm;              // [256]
    unsigned long long& s_excl = sm[256];       // rank of the first element of the chosen chunk
    unsigned long long& s_k = sm[257];
    unsigned long long& s_flags = sm[258];      // invalid | chunk << 1 | prefix << 32
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    // the request: the same values in every thread, in flight together with the bins
    const bool fresh = (PASS == 0) && init.enabled;
    unsigned long long k = fresh ? init.k : st->k;
    uint32_t invalid = (PASS == 0) ? 0u : st->invalid;
    const uint32_t prefix = (PASS == 0) ? 0u : st->prefix;
    const bool med = (PASS == 0) && (fresh ? init.use_median != 0 : st->use_median != 0);
    auto bin = [&](uint32_t b) -> unsigned long long {   // PASS 0 bins are indexed by the raw top bits of the float
        if (local_bins) return (unsigned long long)local_bins[b];   // one CTA counted everything: its shared-memory counters
        return __ldcg(&gdigits[PASS == 0 ? raw_of_digit(b) : b]);
    };
    unsigned long long v[INFL];
#pragma unroll 1
    for (int c0 = 0; c0 < CPW; c0 += INFL) {
#pragma unroll
        for (int j = 0; j < INFL; ++j) {
            const int ch = warp + (c0 + j) * NW;
            v[j] = (c0 + j < CPW && ch < CHUNKS) ? bin((uint32_t)(ch * 32 + lane)) : 0ull;
        }
#pragma unroll
        for (int j = 0; j < INFL; ++j) {
            const int ch = warp + (c0 + j) * NW;
            const unsigned long long t = warp_sum_u64(v[j]);
            if (lane == 0 && c0 + j < CPW && ch < CHUNKS) ctot[ch] = t;
        }
    }
    __syncthreads();
    if (warp == 0) {
        unsigned long long c[CPL], mine = 0;
#pragma unroll
        for (int j = 0; j < CPL; ++j) { c[j] = (lane * CPL + j < CHUNKS) ? ctot[lane * CPL + j] : 0ull; mine += c[j]; }
        unsigned long long incl = mine;
#pragma unroll
        for (int off = 1; off < 32; off <<= 1) {
            unsigned long long u = __shfl_up_sync(0xffffffffu, incl, off);
            if (lane >= off) incl += u;
        }
        const unsigned long long total = __shfl_sync(0xffffffffu, incl, 31);
        if (PASS == 0) {
            if (med) k = total ? (total - 1) / 2 : 0;
            invalid = (k >= total) ? 1u : 0u;
        }
        if (lane == 0) {
            if (PASS == 0) {
                st->count = total; st->invalid = invalid;
                if (init.enabled) {
                    st->use_median = init.use_median; st->cand_n = 0; st->cand_cap = init.cand_cap; st->cand_done = 0;
                }
            }
            if (PASS == 0 || invalid) { st->k = k; st->prefix = prefix; st->result = __int_as_float(0x7fc00000); }
            if (PASS == 2 && invalid && init.result_out) *init.result_out = __int_as_float(0x7fc00000);
            s_k = k;
            s_flags = (unsigned long long)invalid | ((unsigned long long)prefix << 32);
        }
        __syncwarp();
        if (!invalid) {
            unsigned long long excl = incl - mine;
#pragma unroll
            for (int j = 0; j < CPL; ++j) {
                if (c[j] && excl <= k && k < excl + c[j]) {   // exactly one (lane, j)
                    s_excl = excl;
                    s_flags |= (unsigned long long)(lane * CPL + j) << 1;
                }
                excl += c[j];
            }
        }
    }
    __syncthreads();   // the chosen chunk, its first rank and k are in shared memory; lane 0's record is written
    {
        const unsigned long long fl = s_flags;
        const uint32_t ch = (uint32_t)((fl >> 1) & 0x7FFFFFFFu);
        const bool bad = (fl & 1ull) != 0;
        const int owner = KEEP ? (int)(ch % NW) : 0;
        if (!bad && warp == owner) {
            const unsigned long long kk = s_k - s_excl;           // rank inside the chunk
            unsigned long long x = 0;
            if (KEEP) {
#pragma unroll
                for (int j = 0; j < INFL; ++j)
                    if ((int)(ch / NW) == j) x = v[j];
            } else {
                x = bin(ch * 32 + lane);
            }
            unsigned long long inc2 = x;
#pragma unroll
            for (int off = 1; off < 32; off <<= 1) {
                unsigned long long u = __shfl_up_sync(0xffffffffu, inc2, off);
                if (lane >= off) inc2 += u;
            }
            const unsigned long long ex2 = inc2 - x;
            if (x && ex2 <= kk && kk < inc2) {                    // exactly one lane
                const uint32_t b = ch * 32 + lane;
                const uint32_t pfx = (uint32_t)(fl >> 32);
                const uint32_t pre = (PASS == 0) ? b : ((pfx << BITS) | b);
                st->prefix = pre;
                st->k = kk - ex2;
                st->bucket_n = x;
                if (PASS == 2) {
                    const float r = __uint_as_float(bits_of_key(pre));
                    st->result = r;
                    if (init.result_out) *init.result_out = r;
                }
            }
        }
    }
    if (clear) {  // leave the digit bins zeroed for the next pass
        __syncthreads();   // the owner has read its chunk
        for (int i = tid; i < kDigitBins; i += THREADS) gdigits[i] = 0ull;
    }
}

template <int PASS>
__global__ void __launch_bounds__(1024)
select_scan_kernel(SelectState* __restrict__ st, unsigned long long* __restrict__ gdigits, int clear, SelectInit init,
                   const uint32_t* __restrict__ skip_if_set) {
    __shared__ unsigned long long sm[kScanSmem];
    if (skip_if_set && *skip_if_set) return;   // cube_kth_multi's fallback selection is not needed
    select_scan_body<PASS, 1024>(st, gdigits, clear, init, sm);
}

// Fused form: called by every thread of every CTA at the end of a pass kernel, after the CTA's counters have gone
// to gdigits.  The last CTA to arrive (ticket) runs the scan; returns true in that CTA.
template <int PASS, int THREADS>
__device__ __forceinline__ bool select_scan_if_last_n(SelectState* __restrict__ st, unsigned long long* __restrict__ gdigits,
                                                      int clear, const SelectInit& init, unsigned int* __restrict__ ticket,
                                                      unsigned long long* sm) {
    __shared__ bool last;
    __threadfence();      // this thread's REDs to gdigits
    __syncthreads();
    if (threadIdx.x == 0) {
        const unsigned int t = atomicAdd(ticket, 1u);
        last = (t == gridDim.x - 1);
    }
    __syncthreads();
    if (!last) return false;
    __threadfence();
    select_scan_body<PASS, THREADS>(st, gdigits, clear, init, sm);
    if (threadIdx.x == 0) *ticket = 0u;
    return true;
}
template <int PASS>
__device__ __forceinline__ bool select_scan_if_last(SelectState* __restrict__ st, unsigned long long* __restrict__ gdigits,
                                                    int clear, const SelectInit& init, unsigned int* __restrict__ ticket,
                                                    unsigned long long* sm) {
    return select_scan_if_last_n<PASS, kThreads>(st, gdigits, clear, init, ticket, sm);
}

// DEV: rank y = |fl32(x - *center)| (cube_mad); center is a device pointer (the median found just before).
template <int PASS, bool DEV>
__global__ void __launch_bounds__(kThreads, 4)
select_pass_kernel(const float* __restrict__ d, uint64_t n, SelectState* __restrict__ st,
                   unsigned long long* __restrict__ gdigits, uint32_t* __restrict__ cand,
                   const float* __restrict__ center, unsigned int* __restrict__ scan_ticket, SelectInit init,
                   const uint32_t* __restrict__ skip_if_set) {
    constexpr int NB = (PASS == 0) ? kBins0 : (PASS == 1) ? kBins1 : kBins2;
    if (skip_if_set && *skip_if_set) return;   // hist_win_select_kernel has done this pass (BigHistPlan::use_window)
    __shared__ uint32_t sbins[NB + 1];  // + trash counter
    __shared__ uint32_t stage[(PASS == 1) ? (kThreads / 32) * (kStageCap + 1) : 1];
    for (int i = threadIdx.x; i <= NB; i += kThreads) sbins[i] = 0;
    __syncthreads();
    const float ctr = DEV ? *center : 0.0f;
    if (PASS == 0) {
        select_run<0, true, DEV>(d, n, st, sbins, stage, cand, ctr);
    } else if (!st->invalid) {
        const uint32_t top = (PASS == 1) ? st->prefix : (st->prefix >> kBits1);  // first digit of the bucket
        if (digit_may_hold_nan(top)) select_run<PASS, true, DEV>(d, n, st, sbins, stage, cand, ctr);
        else select_run<PASS, false, DEV>(d, n, st, sbins, stage, cand, ctr);
    }
    __syncthreads();
    for (int i = threadIdx.x; i < NB; i += kThreads) {
        uint32_t c = sbins[i];
        if (c) atomicAdd(&gdigits[i], (unsigned long long)c);
    }
    if (scan_ticket) {   // in-core selection: the last CTA locates the bucket (no separate scan launch)
        __shared__ unsigned long long scan_sm[kScanSmem];
        select_scan_if_last<PASS>(st, gdigits, 1, init, scan_ticket, scan_sm);
    }
}

// PASS 2 over the candidate buffer only (out-of-core: no third sweep over the host link; sharded: every rank counts
// its own candidates ONCE, however many bricks its slab is presented in).  Runs iff the bucket fitted the buffer
// (cand_n <= cand_cap, decided here on the device) and then sets cand_done, which makes the per-brick PASS 2
// launches that may follow return at once.
__global__ void __launch_bounds__(kThreads)
select_cand_kernel(SelectState* __restrict__ st, unsigned long long* __restrict__ gdigits,
                   const uint32_t* __restrict__ cand) {
    __shared__ uint32_t sbins[kBins2 + 1];
    if (st->cand_n > st->cand_cap) return;   // uniform over the grid: the bricks are streamed again instead
    if (blockIdx.x == 0 && threadIdx.x == 0) st->cand_done = 1u;   // read by LATER launches only
    for (int i = threadIdx.x; i <= kBins2; i += kThreads) sbins[i] = 0;
    __syncthreads();
    SelectF<2, false> f;
    f.base = st->prefix << kBits2;
    f.sbins = sbins;
    if (!st->invalid) stream_keys<kThreads>(cand, st->cand_n, f);
    __syncthreads();
    for (int i = threadIdx.x; i < kBins2; i += kThreads) {
        uint32_t c = sbins[i];
        if (c) atomicAdd(&gdigits[i], (unsigned long long)c);
    }
}

}  // namespace cube
