// cube_gather.cuh -- warp-cooperative cold path of the compacting select pass (step 8 of SURVEY.md sec. 8(a) fused
// into pass B of cube_stats): the voxels of the median's first-digit bucket have their second digit counted and their
// keys appended to the candidate buffer.
//
// The hot loop only finds out, per 4-voxel row, WHETHER the row holds a voxel of the bucket (row minimum of
// bits - rawbase, cube_select.cuh).  Before, every lane then revisited its own flagged rows one after the other
// (re-loaded through L2), so a warp ran that code as often as its busiest lane had flagged rows, with most lanes idle:
// on config 4 (the bucket holds 2.2 % of the voxels, 8.5 % of the rows) a third of pass B's instructions were issued
// with 11 of 32 lanes active and the pass ran at 0.58 of the HBM rate (profiles/r2_c3.md).  Now a lane PUSHES its flagged
// rows onto a per-warp queue in shared memory, two at a time (re-loaded through L2, both loads in flight together:
// keeping the 32 data registers alive across the cold code made ptxas spill in the hot loop), and the warp takes them
// off 32 at a time -- one row per lane, every lane busy: the work per flagged row no longer depends on how the rows
// are spread over the lanes, and rows left over at the end of a tile simply wait for the next one.
#pragma once
#include "cube_select.cuh"

namespace cube {

constexpr int kRowQRound = 2;                                   // rows per lane between two looks at the queue
constexpr int kRowQCap = 31 + 32 * kRowQRound + 1;              // 96 rows: what can wait + one round of a warp
constexpr uint32_t kKeyThresh = 32;                             // flush the staged keys when more than this wait
constexpr int kKeyCap = (int)kKeyThresh + 128;                  // + the keys of one batch of 32 rows

struct alignas(16) WarpGather {      // per warp, shared memory
    float4 rows[kRowQCap];
    uint32_t keys[kKeyCap];
    uint32_t nrows, nkeys, compacting, pad;
};

struct GatherShared {                // per CTA, shared memory
    uint32_t base;                   // prefix << 19: key - base < 2^19 <=> the voxel is in the bucket
    uint32_t* sbins;                 // kBins1 (+ 1) second-digit counters
    uint32_t* cand;
    unsigned long long* cand_n;
    unsigned long long cand_cap;
};

// all lanes: move the staged keys to the candidate buffer when more than `thresh` wait
static __device__ __forceinline__ void gather_flush(WarpGather* w, const GatherShared* sh, uint32_t thresh) {
    const uint32_t lane = threadIdx.x & 31;
    const uint32_t c = *reinterpret_cast<volatile uint32_t*>(&w->nkeys);
    if (c <= thresh) return;
    unsigned long long pos = 0;
    if (lane == 0) pos = atomicAdd(sh->cand_n, (unsigned long long)c);
    pos = __shfl_sync(0xffffffffu, pos, 0);
    if (pos + c <= sh->cand_cap) {
        CUBE_CHECK(c <= (uint32_t)kKeyCap);
        for (uint32_t i = lane; i < c; i += 32) sh->cand[pos + i] = w->keys[i];
    } else if (lane == 0) {
        w->compacting = 0;           // the bucket does not fit: the last digit will be counted over the cube
    }
    __syncwarp();
    if (lane == 0) w->nkeys = 0;
    __syncwarp();
}

// all lanes: rows [first, first + n) of the queue, one per lane (n <= 32)
static __device__ __noinline__ void gather_rows(WarpGather* w, const GatherShared* sh, uint32_t first, uint32_t n) {
    constexpr uint32_t kSpan = 1u << kShift0;
    const uint32_t lane = threadIdx.x & 31;
    const bool act = lane < n;
    CUBE_CHECK(first + n <= (uint32_t)kRowQCap && n <= 32u);
    const float4 v = w->rows[first + (act ? lane : 0)];
    const uint32_t base = sh->base;
    const float x[4] = {v.x, v.y, v.z, v.w};
    uint32_t kk[4], nh = 0;
    bool hit[4];
#pragma unroll
    for (int i = 0; i < 4; ++i) {
        kk[i] = key_of(x[i]) - base;
        hit[i] = act && kk[i] < kSpan && x[i] == x[i];          // a NaN may have flagged the row: dropped here
        nh += hit[i] ? 1u : 0u;
        if (hit[i]) atomicAdd(&sh->sbins[kk[i] >> kBits2], 1u);
    }
    if (w->compacting) {             // warp-uniform
        uint32_t pos = nh ? atomicAdd(&w->nkeys, nh) : 0u;
        CUBE_CHECK(pos + nh <= (uint32_t)kKeyCap);
#pragma unroll
        for (int i = 0; i < 4; ++i)
            if (hit[i]) w->keys[pos++] = kk[i] + base;
        __syncwarp();
        gather_flush(w, sh, kKeyThresh);
    }
}

// all lanes, after a round of pushes: take rows off the queue while a full batch of 32 waits
static __device__ __forceinline__ void gather_drain_full(WarpGather* w, const GatherShared* sh) {
    __syncwarp();
    uint32_t n = *reinterpret_cast<volatile uint32_t*>(&w->nrows);
    if (n < 32) return;
    do {
        n -= 32;
        gather_rows(w, sh, n, 32);
    } while (n >= 32);
    __syncwarp();
    if ((threadIdx.x & 31) == 0) w->nrows = n;
    __syncwarp();
}

// Cold path of a tile share, called by ALL lanes of the warp when any lane has a flagged row: bit j of `rows` = row j
// of this lane (p[j * THREADS]) holds a voxel of the bucket.  Every lane re-loads up to two of its flagged rows per
// turn (L2 hits: the lines have just been streamed) and pushes them; the queue is drained whenever 32 rows wait.
template <int THREADS>
static __device__ __noinline__ void gather_cold(uint32_t rows, const float4* __restrict__ p, WarpGather* w,
                                                const GatherShared* sh) {
    do {
        const int j0 = __ffs(rows) - 1;                 // -1: none
        rows &= rows - 1;
        const int j1 = __ffs(rows) - 1;
        rows &= rows - 1;
        float4 a = make_float4(0.f, 0.f, 0.f, 0.f), b = a;
        if (j0 >= 0) a = __ldcg(p + j0 * THREADS);
        if (j1 >= 0) b = __ldcg(p + j1 * THREADS);
        const uint32_t cnt = (j0 >= 0 ? 1u : 0u) + (j1 >= 0 ? 1u : 0u);
        if (cnt) {
            uint32_t slot = atomicAdd(&w->nrows, cnt);
            CUBE_CHECK(slot + cnt <= (uint32_t)kRowQCap);
            w->rows[slot] = a;
            if (j1 >= 0) w->rows[slot + 1] = b;
        }
        gather_drain_full(w, sh);
    } while (__any_sync(0xffffffffu, rows != 0));
}

// all lanes, after the streaming loop: what is left on the queue, then the staged keys
static __device__ __forceinline__ void gather_finish(WarpGather* w, const GatherShared* sh) {
    __syncwarp();
    const uint32_t n = *reinterpret_cast<volatile uint32_t*>(&w->nrows);
    if (n) gather_rows(w, sh, 0, n);
    __syncwarp();
    if ((threadIdx.x & 31) == 0) w->nrows = 0;
    __syncwarp();
    if (w->compacting) gather_flush(w, sh, 0u);
}

// Single voxels (head / tail / ragged last tile): counted at once, key straight to the candidate buffer.
static __device__ __forceinline__ void gather_single(const GatherShared* sh, float x) {
    const uint32_t kk = key_of(x) - sh->base;
    if (kk < (1u << kShift0) && x == x) {
        atomicAdd(&sh->sbins[kk >> kBits2], 1u);
        if (sh->cand && sh->cand_cap) {
            const unsigned long long pos = atomicAdd(sh->cand_n, 1ull);   // beyond the capacity: cand_n says so
            if (pos < sh->cand_cap) sh->cand[pos] = kk + sh->base;
        }
    }
}

// The hot-path side: does this thread's share of the tile (8 rows of 4 voxels) hold a voxel of the bucket?
// bits - rawbase < 2^19 (mod 2^32) <=> the top 13 raw bits match; the subtraction is issued as IMAD on the FMA pipe,
// each row's minimum takes a VIMNMX3 + VIMNMX, the tile minimum four more VIMNMX3, then ONE vote per warp tile: 1.7
// issue slots per voxel and NO shared-memory traffic.  The row flags are only formed behind the branch.
// NaN voxels may flag a row, gather_rows drops them.  negbase = 0 - rawbase.
template <int THREADS>
static __device__ __forceinline__ void gather_batch(const float4 (&r)[kUnroll], const float4* __restrict__ p,
                                                    uint32_t negbase, WarpGather* w, const GatherShared* sh) {
    constexpr uint32_t kSpan = 1u << kShift0;
    uint32_t rm[kUnroll];
#pragma unroll
    for (int j = 0; j < kUnroll; ++j)
        rm[j] = min(min(SelectF<1, false>::sub_fma(r[j].x, negbase), SelectF<1, false>::sub_fma(r[j].y, negbase)),
                    min(SelectF<1, false>::sub_fma(r[j].z, negbase), SelectF<1, false>::sub_fma(r[j].w, negbase)));
    uint32_t tmin = rm[0];
#pragma unroll
    for (int j = 1; j < kUnroll; ++j) tmin = min(tmin, rm[j]);
    if (!__any_sync(0xffffffffu, tmin < kSpan)) return;          // no voxel of the bucket in this warp's tile
    uint32_t rows = 0;
#pragma unroll
    for (int j = 0; j < kUnroll; ++j) rows |= (rm[j] < kSpan ? 1u : 0u) << j;
    gather_cold<THREADS>(rows, p, w, sh);
}

}  // namespace cube
