// cube_kernels.cuh -- the sm_100a kernels of libcube.  See DESIGN.md sec. 4 for the roofline of each.
//
// All of them are HBM-read-bound scans (4 B per voxel per pass, no dense contraction => no tensor cores).
// At the measured ~7.3 TB/s read ceiling an SM must retire ~6 voxels per clock, i.e. the per-voxel budget
// is ~21 issue slots, ~10 of them on the half-rate ALU pipe -- so the functors below are written to be
// branch-free and light on integer/compare instructions (ncu: profiles/r1_*.md).
#pragma once
#include <math.h>

#include "cube_common.cuh"
#include "cube_select.cuh"

namespace cube {

// Result record as laid out by include/cube.h (cube_moments_t).
struct MomentsOut {
    uint64_t count, nan_count;
    float min, max;
    double mean, std;
};

// ------------------------------------------------------------------------------------------------
// Moments: steps 1-3 of SURVEY.md sec. 8(a) (+ 3b when COARSE): count, min, max, pivoted fp64 sums.
// PAPER.md:265 "local summation and summation of squares and count of the non-null data values".
// The paper's float32-per-slice partial sums are replaced by per-thread fp64
// accumulators about a per-thread pivot (R17): d = x - pivot is exact in fp64, so a constant
// cube gives std == 0 exactly and sum(d^2) - sum(d)^2/n does not cancel catastrophically.
// Per voxel: FSETP, FSEL, 2 FMNMX (alu pipe), F2F (xu), 2 DADD + DFMA (fp64), 1 predicated IADD.
// min/max use FMNMX, which ignores NaN operands and orders -0.0 < +0.0.
// ------------------------------------------------------------------------------------------------
// MODE: kMomPlain, kMomCoarse (+ first select digit, step 3b) or kMomWindow (NEXT-1, clipped moments: only
// voxels with wlo <= x <= whi take part -- the test is made on x itself and fails for NaN; one more FSETP + FSEL).
constexpr int kMomPlain = 0, kMomCoarse = 1, kMomWindow = 2;
template <int MODE>
struct MomentsF {
    static constexpr bool COARSE = (MODE == kMomCoarse);
    float mn = INFINITY, mx = -INFINITY;
    float pivf = 0.0f;
    bool have = false;
    uint32_t n = 0;
    double pivot = 0.0, s = 0.0, q = 0.0;
    uint32_t sbins;   // COARSE: shared-window address of kDigitBins + 1 counters
    float wlo = -INFINITY, whi = INFINITY;  // kMomWindow
    __device__ __forceinline__ bool taken(float x) const {
        return (MODE == kMomWindow) ? (x >= wlo && x <= whi) : (x == x);  // NaN == blanked voxel
    }
    template <bool MINMAX = true>
    __device__ __forceinline__ void core(float x) {
        const bool ok = taken(x);
        if (MODE == kMomWindow) {  // FMNMX ignores NaN operands: a voxel outside the window is fed as NaN
            const float xw = ok ? x : __int_as_float(0x7fc00000);
            mn = fminf(mn, xw);
            mx = fmaxf(mx, xw);
        } else if (MINMAX) {
            mn = fminf(mn, x);
            mx = fmaxf(mx, x);
        }
        const float xs = ok ? x : pivf;  // a voxel that is left out contributes d == 0
        const double dlt = (double)xs - pivot;
        s += dlt;
        q = fma(dlt, dlt, q);
        n += ok ? 1u : 0u;
        // COARSE: the digit of xs -- a NULL voxel is counted in the PIVOT's bin (no select per voxel) and taken back
        // out once per thread after the streaming loop (nsub0 / nsub1: NULL voxels met before / after the pivot was
        // found; the pivot changes only once, from the initial +0.0f)
        if (COARSE) smem_inc(sbins, raw_digit(xs));
    }
    uint32_t nsub0 = 0, nsub1 = 0;
    __device__ __forceinline__ void note_subst(uint32_t k) { if (have) nsub1 += k; else nsub0 += k; }
    // after the streaming loop: take the substituted NULL voxels back out of the pivot's digit bins
    __device__ __forceinline__ void unsubstitute() const {
        if (!COARSE) return;
        if (nsub0) asm volatile("red.shared.add.u32 [%0], %1;" :: "r"(sbins + 4u * raw_digit(0.0f)), "r"(0u - nsub0) : "memory");
        if (nsub1) asm volatile("red.shared.add.u32 [%0], %1;" :: "r"(sbins + 4u * raw_digit(pivf)), "r"(0u - nsub1) : "memory");
    }
    // The pivot is the first FINITE voxel that takes part: about an infinite pivot every deviation would be
    // infinite or NaN.  (A cube with +-Inf voxels has mean = std = NaN whatever the summation order: reading R8,
    // applied in moments_finalize.)
    __device__ __forceinline__ void take_pivot(float x) {
        if (!have && taken(x) && fabsf(x) < INFINITY) { have = true; pivf = x; pivot = (double)x; }
    }
    __device__ __forceinline__ void operator()(float x) {
        take_pivot(x);
        core(x);
        if (COARSE && !taken(x)) note_subst(1u);
    }

    // A tile share (kUnroll rows of 4 voxels) whose sum of deviations came out NaN holds a NaN voxel (or +Inf and
    // -Inf): the hot path has left it out of s, q and n, and has counted every one of its voxels in the digit bins.
    // Revisit it (the lines are L2 hits): add the non-NaN voxels one by one and take the NaN voxels back out of
    // the bins.
    struct TileFix { double s, q; uint32_t n; };
    static __device__ __noinline__ TileFix cold_tile(const float4* __restrict__ p, double pivot_, uint32_t sbins_) {
        TileFix f;
        f.s = 0.0; f.q = 0.0; f.n = 0;
#pragma unroll 1
        for (int j = 0; j < kUnroll; ++j) {
            const float4 v = __ldcg(p + j * kThreads);
            const float x[4] = {v.x, v.y, v.z, v.w};
#pragma unroll
            for (int i = 0; i < 4; ++i) {
                if (x[i] == x[i]) {
                    const double dlt = (double)x[i] - pivot_;
                    f.s += dlt; f.q = fma(dlt, dlt, f.q); f.n += 1;
                } else if (COARSE) {
                    asm volatile("red.shared.add.u32 [%0], -1;" :: "r"(sbins_ + 4u * raw_digit(x[i])) : "memory");
                }
            }
        }
        return f;
    }
    // Full tile (all 32 lanes of the warp are here: stream_cube calls batch() CTA-uniformly).  Two ways through:
    //  HOT (kMomPlain / kMomCoarse), per row of 4 voxels: d_i = (double)x_i - pivot (exact); ts += (d0+d1)+(d2+d3);
    //   tq += d0^2+d1^2+d2^2+d3^2 (DFMA chain); the tile share joins s, q, n when ts is not NaN -- no per-voxel NaN
    //   test, select or count (FMNMX ignores NaN operands; the digit increment is unconditional): ~8.5 issue slots
    //   per voxel.  A lane whose ts is NaN (a NaN voxel, or +Inf and -Inf) repairs its share in cold_tile().
    //  SAFE: the branch-free per-voxel form (core(): FSETP, FSEL, count; extrema per row; the digit of a NULL voxel is
    //   the pivot's, put right once per thread: ~11 slots per voxel), which costs the same whatever the NaN density.
    // The warp runs HOT until a tile with a NaN shows up and SAFE until a tile without one has gone by (one vote
    // per tile), so cubes with scattered NULL voxels (config 3: 0.5 %, i.e. some lane of every warp tile) never
    // pay the divergent repair, and NaN-free stretches never pay the per-voxel tests (profiles/: the fused passes
    // are issue/power bound once the SM clock drops under a sustained load).
    bool safe = true;   // warp-uniform
    __device__ __forceinline__ void batch(const float4 (&r)[kUnroll], const float4* __restrict__ p) {
        if (MODE == kMomWindow || safe) {
            if (!have) {  // only until this thread has met its first voxel that takes part
#pragma unroll
                for (int j = 0; j < kUnroll; ++j) { take_pivot(r[j].x); take_pivot(r[j].y); take_pivot(r[j].z); take_pivot(r[j].w); }
            }
            const uint32_t n0 = n;
#pragma unroll
            for (int j = 0; j < kUnroll; ++j) {
                if (MODE != kMomWindow) {   // extrema per row of 4 (FMNMX3, NaN-blind) instead of 2 FMNMX per voxel
                    mn = fminf(fminf(mn, r[j].x), fminf(r[j].y, fminf(r[j].z, r[j].w)));
                    mx = fmaxf(fmaxf(mx, r[j].x), fmaxf(r[j].y, fmaxf(r[j].z, r[j].w)));
                }
                core<false>(r[j].x); core<false>(r[j].y); core<false>(r[j].z); core<false>(r[j].w);
            }
            if (COARSE) note_subst(4u * kUnroll - (n - n0));
            if (MODE != kMomWindow) safe = __any_sync(0xffffffffu, n - n0 != 4u * kUnroll);  // every lane has a pivot then
            return;
        }
        double ts[2] = {0.0, 0.0}, tq[2] = {0.0, 0.0};  // two chains for instruction-level parallelism
#pragma unroll
        for (int j = 0; j < kUnroll; ++j) {
            const double d0 = (double)r[j].x - pivot, d1 = (double)r[j].y - pivot;
            const double d2 = (double)r[j].z - pivot, d3 = (double)r[j].w - pivot;
            ts[j & 1] += (d0 + d1) + (d2 + d3);
            tq[j & 1] = fma(d3, d3, fma(d2, d2, fma(d1, d1, fma(d0, d0, tq[j & 1]))));
            mn = fminf(fminf(mn, r[j].x), fminf(r[j].y, fminf(r[j].z, r[j].w)));
            mx = fmaxf(fmaxf(mx, r[j].x), fmaxf(r[j].y, fmaxf(r[j].z, r[j].w)));
            if (COARSE) {
                smem_inc(sbins, raw_digit(r[j].x)); smem_inc(sbins, raw_digit(r[j].y));
                smem_inc(sbins, raw_digit(r[j].z)); smem_inc(sbins, raw_digit(r[j].w));
            }
        }
        const double tsum = ts[0] + ts[1];
        const bool bad = !(tsum == tsum);
        if (!bad) {
            s += tsum; q += tq[0] + tq[1]; n += 4u * kUnroll;
        } else {
            const TileFix f = cold_tile(p, pivot, sbins);
            s += f.s; q += f.q; n += f.n;
        }
        safe = __any_sync(0xffffffffu, bad);
    }
    __device__ __forceinline__ Partial partial() const {
        Partial p = partial_empty();
        if (n) {
            const double nn = (double)n, ms = s / nn;
            const double m2 = q - s * ms;
            p.n = n; p.mean = pivot + ms; p.m2 = (m2 < 0.0) ? 0.0 : m2;   // rounding only; a NaN (Inf voxels) stays
            p.kmin = key_of(mn); p.kmax = key_of(mx);
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
        // reading R8: a set with an infinite member has no finite mean or deviation -- both are NaN, decided on the
        // extrema so that the answer depends neither on the summation order nor on the grid
        if (isinf(o.min) || isinf(o.max)) o.mean = o.std = (double)qnan;
    }
    *out = o;
}

// State of an iterated sigma clip (NEXT-1), kept on the device so that the loop
// "statistics -> window -> clipped statistics" never crosses to the host.
struct ClipState {
    float lo, hi;                   // window of the pass about to run / last run (NaN before the first)
    uint32_t done;                  // 1: converged or degenerate -- the remaining passes return at once
    int iters;                      // clipped passes made
    unsigned long long prev_count;  // count of the statistics the window was formed from
};

// Fixed-order merge of `nparts` per-CTA partials by ONE CTA of kThreads threads (all of them call; the result is valid
// in thread 0).  `scratch`: kThreads / 32 Partials of shared memory, free on entry.
__device__ __forceinline__ Partial partials_merge_block(const Partial* __restrict__ partials, unsigned nparts, Partial* scratch) {
    // last CTA: fixed-order merge of the per-CTA partials.  A tree of Chan merges is a chain of ~13 dependent fp64
    // divisions (5 us of tail on a cube that streams in 10 us: profiles/r1_v11_c2.md), so the partials are first
    // re-expressed as sums about ONE pivot P -- the mean of the lowest-indexed non-empty partial: s_i = n_i (mean_i -
    // P), q_i = M2_i + n_i (mean_i - P)^2 -- which merge by plain additions (thread i takes i, i+256, ...; then
    // shuffles).  P is the mean of a CTA whose tiles are spread over the whole cube, so |P - mean| << std and
    // q - s^2/n loses nothing; a constant cube gives mean_i == P, s = q = 0 and std = 0 exactly.
    __shared__ unsigned int first_live;
    __shared__ double pivot_sm;
    __shared__ int again_sm;
    unsigned int first = 0;   // block-uniform: partial 0 unless CTA 0 saw only NULL voxels (then the search below)
    if (__ldcg(&partials[0].n) == 0) {
        if (threadIdx.x == 0) first_live = 0xFFFFFFFFu;
        __syncthreads();
        unsigned int mine = 0xFFFFFFFFu;
        for (unsigned i = threadIdx.x; i < nparts; i += kThreads)
            if (mine == 0xFFFFFFFFu && __ldcg(&partials[i].n) != 0) mine = i;
        if (mine != 0xFFFFFFFFu) atomicMin(&first_live, mine);
        __syncthreads();
        first = first_live;
    }
    Partial m = partial_empty();
    if (first != 0xFFFFFFFFu) {
        if (threadIdx.x == 0) again_sm = 0;
        double P = __ldcg(&partials[first].mean);
        // Second round only if the pivot turned out to be far from the mean (more than 16 standard deviations: data
        // arranged so that CTA first_live saw something else than the rest): q - s^2/n would then cancel ~2^8 or more
        // of the 2^53; the refined pivot P + s/n is as good as the mean itself.
#pragma unroll 1
        for (int round = 0; round < 2; ++round) {
            unsigned long long cn = 0;
            double cs = 0.0, cq = 0.0;
            uint32_t kmin = 0xFFFFFFFFu, kmax = 0u;
            for (unsigned i = threadIdx.x; i < nparts; i += kThreads) {   // written by other CTAs: read through L2
                const unsigned long long bn = __ldcg(&partials[i].n);
                const double bmean = __ldcg(&partials[i].mean), bm2 = __ldcg(&partials[i].m2);
                kmin = min(kmin, __ldcg(&partials[i].kmin));
                kmax = max(kmax, __ldcg(&partials[i].kmax));
                if (bn) {
                    const double nb = (double)bn, dm = bmean - P, nd = nb * dm;
                    cn += bn; cs += nd; cq += bm2 + nd * dm;
                }
            }
#pragma unroll
            for (int off = 16; off > 0; off >>= 1) {
                cn += __shfl_down_sync(0xffffffffu, cn, off);
                cs += __shfl_down_sync(0xffffffffu, cs, off);
                cq += __shfl_down_sync(0xffffffffu, cq, off);
                kmin = min(kmin, __shfl_down_sync(0xffffffffu, kmin, off));
                kmax = max(kmax, __shfl_down_sync(0xffffffffu, kmax, off));
            }
            const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
            __syncthreads();   // scratch is free (the CTA's own block reduce / the round before is over)
            if (lane == 0) { scratch[warp].n = cn; scratch[warp].mean = cs; scratch[warp].m2 = cq; scratch[warp].kmin = kmin; scratch[warp].kmax = kmax; }
            __syncthreads();
            if (threadIdx.x == 0) {
                cn = 0; cs = 0.0; cq = 0.0; kmin = 0xFFFFFFFFu; kmax = 0u;
#pragma unroll
                for (int w = 0; w < kThreads / 32; ++w) {
                    cn += scratch[w].n; cs += scratch[w].mean; cq += scratch[w].m2;
                    kmin = min(kmin, scratch[w].kmin); kmax = max(kmax, scratch[w].kmax);
                }
                const double nn = (double)cn, shift = cs / nn;
                const double m2 = cq - cs * shift;
                m.n = cn; m.mean = P + shift; m.m2 = (m2 < 0.0) ? 0.0 : m2;   // rounding only; a NaN (Inf voxels) stays
                m.kmin = kmin; m.kmax = kmax;
                const bool far = round == 0 && shift * shift * nn > 256.0 * m.m2 && isfinite(m.mean);
                again_sm = far ? 1 : 0;
                if (far) pivot_sm = m.mean;
            }
            __syncthreads();
            if (!again_sm) break;
            P = pivot_sm;
        }
    }
    return m;
}

// acc : running Partial across calls (out-of-core bricks); merged in call order => deterministic.
// nvox_acc : running voxel total.  When `accumulate` is 0 both are overwritten.
// kMomWindow: the window is (wlo, whi), or *clip when clip != nullptr (then a finished clip makes the kernel a no-op).
#ifndef CUBE_MOM_CTAS
#define CUBE_MOM_CTAS 4
#endif
template <int MODE>
__global__ void __launch_bounds__(kThreads, CUBE_MOM_CTAS)
moments_kernel(const float* __restrict__ d, uint64_t n, Partial* __restrict__ partials,
               unsigned int* __restrict__ ticket, Partial* __restrict__ acc,
               unsigned long long* __restrict__ nvox_acc, int accumulate, unsigned flags,
               MomentsOut* __restrict__ out, unsigned long long* __restrict__ gdigits,
               float wlo, float whi, const ClipState* __restrict__ clip,
               SelectState* __restrict__ sel, unsigned int* __restrict__ scan_ticket, SelectInit init,
               MomentsOut* __restrict__ out_user) {
    constexpr bool COARSE = (MODE == kMomCoarse);
    __shared__ Partial scratch[kThreads / 32];
    __shared__ uint32_t sbins[COARSE ? kDigitBins + 1 : 1];
    __shared__ bool is_last;
    MomentsF<MODE> f;
    f.sbins = smem_addr(sbins);
    if (MODE == kMomWindow) {
        if (clip) {
            if (clip->done) return;  // uniform over the grid
            wlo = clip->lo; whi = clip->hi;
        }
        f.wlo = wlo; f.whi = whi;
    }
    if (COARSE) {
        for (int i = threadIdx.x; i <= kDigitBins; i += kThreads) sbins[i] = 0;
        __syncthreads();
    }
    stream_cube<kThreads>(d, n, f);
    f.unsubstitute();
    Partial p = partial_block_reduce(f.partial(), scratch);
    if (COARSE) {
        __syncthreads();
        for (int i = threadIdx.x; i < kDigitBins; i += kThreads) {
            uint32_t c = sbins[i];
            if (c) atomicAdd(&gdigits[i], (unsigned long long)c);
        }
        if (scan_ticket) {   // cube_stats: the last CTA locates the median's first-digit bucket (no scan launch)
            __shared__ unsigned long long scan_sm[kScanSmem];
            select_scan_if_last<0>(sel, gdigits, 0, init, scan_ticket, scan_sm);
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
    // last CTA: fixed-order merge of the per-CTA partials (partials_merge_block)
    __threadfence();
    Partial m = partials_merge_block(partials, gridDim.x, scratch);
    if (threadIdx.x == 0) {
        unsigned long long tot = n;
        if (accumulate) { m = partial_merge(*acc, m); tot += *nvox_acc; }
        *acc = m;
        *nvox_acc = tot;
        moments_finalize(m, tot, flags, out);
        if (out_user) *out_user = *out;   // the caller's record, when the device can reach it (no copy is enqueued then)
        *ticket = 0u;
    }
}

// One step of the sigma-clip loop, between two passes over the cube (1 thread): has the last pass
// reproduced the count its window was formed from (converged)?  Otherwise form the next window
//   lo = fl32(mean - kappa * std), hi = fl32(mean + kappa * std)
// from the statistics of the last pass -- product and sum rounded to double separately (no FMA), one rounding
// to float32 (R23).
__global__ void clip_step_kernel(const MomentsOut* __restrict__ m, ClipState* __restrict__ st, double kappa) {
    if (st->done) return;
    const unsigned long long cnt = m->count;
    if (st->iters > 0 && cnt == st->prev_count) { st->done = 1u; return; }
    const double mean = m->mean, sd = m->std;
    if (cnt == 0 || !isfinite(sd) || !isfinite(mean)) { st->done = 1u; return; }
    const double w = __dmul_rn(kappa, sd);
    st->lo = __double2float_rn(__dsub_rn(mean, w));
    st->hi = __double2float_rn(__dadd_rn(mean, w));
    st->prev_count = cnt;
    st->iters += 1;
}

// NEXT-3 (z-slab sharding over GPUs): merge the all-gathered per-rank records {Partial, voxel total} in rank
// order -- the paper's server-side O(1) combination of (count, sum, sum of squares) ("any
// arbitrary data composition order is valid"), in Chan's cancellation-free form -- into the running record of this
// rank and re-finalise.  Every rank does the same merge in the same order, so all ranks hold identical bits.
__global__ void shard_merge_kernel(const unsigned char* __restrict__ gathered, int world, int rec_bytes, unsigned flags,
                                   Partial* __restrict__ acc, unsigned long long* __restrict__ nvox,
                                   MomentsOut* __restrict__ out) {
    Partial m = partial_empty();
    unsigned long long tot = 0;
    for (int r = 0; r < world; ++r) {
        const Partial* p = reinterpret_cast<const Partial*>(gathered + (size_t)r * rec_bytes);
        tot += *reinterpret_cast<const unsigned long long*>(gathered + (size_t)r * rec_bytes + sizeof(Partial));
        m = partial_merge(m, *p);
    }
    *acc = m;
    *nvox = tot;
    moments_finalize(m, tot, flags, out);
}

// Start of a brick-streamed / sharded accumulation: the running record is the empty one (a rank whose slab holds no
// voxel contributes exactly that to the all-gather), the voxel total 0, the finalised record that of an empty cube.
__global__ void moments_reset_kernel(Partial* __restrict__ acc, unsigned long long* __restrict__ nvox,
                                     MomentsOut* __restrict__ out) {
    *acc = partial_empty();
    *nvox = 0ull;
    moments_finalize(*acc, 0ull, 0u, out);
}

// Re-evaluate mean/std of the running partial with other flags (sample std) -- O(1).
__global__ void moments_refinalize_kernel(const Partial* __restrict__ acc, const unsigned long long* __restrict__ nvox,
                                          unsigned flags, MomentsOut* __restrict__ out) {
    moments_finalize(*acc, *nvox, flags, out);
}

// ------------------------------------------------------------------------------------------------
// Histogram: steps 4-5.  PAPER.md:259-261; bin formula DESIGN.md R10-R13 (float32, no contraction).
// Shared-memory privatised counters per CTA, merged into the 64-bit global bins by atomics
// ("summation ... associative and commutative, any arbitrary data composition order is valid").
// The shared-memory increment compiles to ATOMS.POPC.INC, which the hardware aggregates over lanes that
// hit the same address -- hot bins (config 4: 30 % of the voxels in one bin) cost no serialisation.
// ------------------------------------------------------------------------------------------------
struct HistBase {
    float lo, hi, scale;
    int top;  // nbins-1
    uint32_t below = 0, above = 0;
    // bin of an in-range voxel; garbage (never used) otherwise
    __device__ __forceinline__ int bin_of(float x) const {
        const float v = __fmul_rn(__fsub_rn(x, lo), scale);
        return min(__float2int_rd(v), top);  // floor (v >= 0), closed top bin (R11)
    }
    __device__ __forceinline__ void outside(float x) {  // rare path: NaN, x < lo, x > hi
        below += (x < lo) ? 1u : 0u;
        above += (x > hi) ? 1u : 0u;
    }
};

// Shared-memory layout of the <= 16384-bin kernels: slots 0 .. top-1 hold bins 0 .. top-1 (top = nbins-1), slot
// `top` is a TRASH counter (never read) and slot top+1 holds the closed top bin.  So the hot path of the fast
// functor can clamp with one unsigned minimum: everything at or beyond `top` -- the top bin, voxels above the
// range, and negative positions (huge as unsigned) -- lands on the trash slot and is put right by a cold path.
__device__ __forceinline__ uint32_t hist_slot(int b, int top) { return (uint32_t)(b + (b >= top ? 1 : 0)); }

// General functor (hi == lo, fewer than 8 bins, subnormal scale): per voxel 2 FSETP (range test on x itself, false
// for NaN), FADD, FMUL (__fsub_rn / __fmul_rn: never contracted), F2I.FLOOR, VIMNMX (closed top bin), SEL,
// ATOMS.POPC.INC.  The increment is unconditional: voxels that are NaN or outside [lo,hi] go to the trash slot.
// Voxels outside [lo,hi] are found per batch from the batch min/max (FMNMX3, NaN-blind) and counted in a cold path.
struct HistF : HistBase {
    uint32_t* sbins;  // nbins + 2 slots (layout above)
    __device__ __forceinline__ void inc(float x) const {
        const bool in = (x >= lo) && (x <= hi);
        const uint32_t slot = in ? hist_slot(bin_of(x), top) : (uint32_t)top;
        atomicAdd(&sbins[slot], 1u);
    }
    __device__ __forceinline__ void operator()(float x) {
        inc(x);
        outside(x);
    }
    __device__ __forceinline__ void batch(const float4 (&r)[kUnroll], const float4*) {
        float bmin = INFINITY, bmax = -INFINITY;
#pragma unroll
        for (int j = 0; j < kUnroll; ++j) {
            inc(r[j].x); inc(r[j].y); inc(r[j].z); inc(r[j].w);
            bmin = fminf(fminf(bmin, r[j].x), fminf(r[j].y, fminf(r[j].z, r[j].w)));
            bmax = fmaxf(fmaxf(bmax, r[j].x), fmaxf(r[j].y, fmaxf(r[j].z, r[j].w)));
        }
        if (bmin < lo || bmax > hi) {
#pragma unroll
            for (int j = 0; j < kUnroll; ++j) { outside(r[j].x); outside(r[j].y); outside(r[j].z); outside(r[j].w); }
        }
    }
};

// Fast functor (the default).  With v = fl(fl(x - lo) * scale) (R10) the hot path does
//     i = floor(max(v, -1));  counter[min((unsigned)i, top)] += 1;  tmax = max(tmax, i);  xmin = min(xmin, x)
// i.e. per voxel FADD, FMUL, FMNMX, F2I.FLOOR, VIMNMX.U32, IMAD, ATOMS.POPC.INC and half a VIMNMX3 + half an FMNMX3
// -- no compare, no select, no branch (8 issue slots; v3 had ISETP + SEL + FMNMX row flags: 8.7 and one more on the
// half-rate ALU pipe).  FMNMX returns the other operand for a NaN, so a NULL voxel becomes i = -1 like any voxel
// below the range, and min((unsigned)-1, top) sends both to the trash slot: NaN voxels need no further attention.
// 0 <= i < top is exactly the case "+0 <= v < nbins-1", for which lo <= x <= hi is guaranteed (t = x - lo has
// the sign of the exact difference, and x > hi implies v >= fl(fl(hi-lo) * scale) > nbins - 1 whenever hi > lo and
// scale is a normal number, nbins <= 65536) and the bin is floor(v), no clamp.  What is left -- the closed top bin
// (R11), x > hi (both: i >= top, signed) and x < lo (xmin < lo; FMNMX3 ignores NaN; such a voxel is i = -1, or i = 0
// when the product underflows to -0.0, which the cold path takes back out of bin 0) -- is rare and detected per
// tile share (32 voxels); a cold path reloads the 8 rows (L2 hits), finds the rows concerned and applies the exact
// definition to their voxels.  Not valid for hi == lo (scale 0), fewer than 8 bins or a subnormal scale.
__host__ __device__ __forceinline__ bool hist_use_fast(int nbins, float lo, float hi, float scale) {
    return hi > lo && nbins >= 8 && scale >= 1.17549435e-38f;
}
struct HistFastF {
    float lo, hi, scale;
    int top;
    uint32_t* sbins;   // nbins + 2 slots (layout above)
    uint32_t sbase;    // shared-window address of sbins
    uint32_t* s_out;   // shared {below, above}
    uint32_t below = 0, above = 0;  // unused (kept for hist_flush_outside); the cold path counts in s_out
    __device__ __forceinline__ void setup(float lo_, float hi_, float scale_, int nbins, uint32_t* sbins_,
                                          uint32_t* s_out_) {
        lo = lo_; hi = hi_; scale = scale_; top = nbins - 1;
        sbins = sbins_; sbase = smem_addr(sbins_); s_out = s_out_;
    }
    static __device__ __forceinline__ int pos(float x, float lo, float scale) {   // i of the hot path
        return __float2int_rd(fmaxf(__fmul_rn(__fsub_rn(x, lo), scale), -1.0f));
    }
    // exact definition for a voxel the hot path sent to the trash slot (NaN: nothing to do)
    static __device__ __forceinline__ void fix(float x, float lo, float hi, float scale, int top, uint32_t* sbins,
                                               uint32_t* s_out) {
        const int i = pos(x, lo, scale);
        if (x < lo || x > hi) {
            atomicAdd(&s_out[x < lo ? 0 : 1], 1u);
            // (x - lo) * scale can underflow to -0.0 for x just below lo (scale < 1): the hot path has then
            // counted the voxel in bin 0 -- take it back out
            if ((uint32_t)i < (uint32_t)top) atomicSub(&sbins[i], 1u);
        } else if (x == x) {
            if ((uint32_t)i >= (uint32_t)top) atomicAdd(&sbins[hist_slot(min(max(i, 0), top), top)], 1u);
        }
    }
    static __device__ __noinline__ void cold(const float4* __restrict__ p, float lo, float hi, float scale, int top,
                                             uint32_t* sbins, uint32_t* s_out) {
#pragma unroll 1
        for (int j = 0; j < kUnroll; ++j) {
            const float4 q = __ldcg(p + j * kThreads);  // L2 hit: the line has just been streamed
            const int im = max(max(pos(q.x, lo, scale), pos(q.y, lo, scale)), max(pos(q.z, lo, scale), pos(q.w, lo, scale)));
            const float xm = fminf(fminf(q.x, q.y), fminf(q.z, q.w));
            if (im >= top || xm < lo) {
                fix(q.x, lo, hi, scale, top, sbins, s_out);
                fix(q.y, lo, hi, scale, top, sbins, s_out);
                fix(q.z, lo, hi, scale, top, sbins, s_out);
                fix(q.w, lo, hi, scale, top, sbins, s_out);
            }
        }
    }
    __device__ __forceinline__ void operator()(float x) {   // head / tail / ragged last tile
        const int i = pos(x, lo, scale);
        if ((uint32_t)i < (uint32_t)top && x >= lo) atomicAdd(&sbins[i], 1u);
        else if ((uint32_t)i < (uint32_t)top) atomicAdd(&s_out[0], 1u);   // x < lo with a product that underflowed to -0.0
        else fix(x, lo, hi, scale, top, sbins, s_out);
    }
    __device__ __forceinline__ void batch(const float4 (&r)[kUnroll], const float4* __restrict__ p) {
        int tmax = -1;
        float xmin = INFINITY;
#pragma unroll
        for (int j = 0; j < kUnroll; ++j) {
            const int i0 = pos(r[j].x, lo, scale), i1 = pos(r[j].y, lo, scale);
            const int i2 = pos(r[j].z, lo, scale), i3 = pos(r[j].w, lo, scale);
            smem_inc(sbase, min((uint32_t)i0, (uint32_t)top));
            smem_inc(sbase, min((uint32_t)i1, (uint32_t)top));
            smem_inc(sbase, min((uint32_t)i2, (uint32_t)top));
            smem_inc(sbase, min((uint32_t)i3, (uint32_t)top));
            tmax = max(max(tmax, max(i0, i1)), max(i2, i3));
            xmin = fminf(fminf(xmin, fminf(r[j].x, r[j].y)), fminf(r[j].z, r[j].w));
        }
        if (tmax >= top || xmin < lo) cold(p, lo, hi, scale, top, sbins, s_out);
    }
};

template <class F>
__device__ __forceinline__ void hist_flush_outside(F& f, uint32_t* s_out, unsigned long long* goutside) {
    if (f.lo > f.hi) return;  // unusable device-side [min,max] range: hist_range_kernel has left the marker
    if (f.below) atomicAdd(&s_out[0], f.below);
    if (f.above) atomicAdd(&s_out[1], f.above);
    __syncthreads();
    if (threadIdx.x < 2 && s_out[threadIdx.x]) atomicAdd(&goutside[threadIdx.x], (unsigned long long)s_out[threadIdx.x]);
}

// Flush of the per-CTA counters (layout above) into the 64-bit global bins.
__device__ __forceinline__ void hist_flush_bins(const uint32_t* sbins, int nbins, unsigned long long* __restrict__ gbins) {
    const int top = nbins - 1;
    for (int i = threadIdx.x; i < nbins; i += kThreads) {
        const uint32_t c = sbins[i < top ? i : top + 1];
        if (c) atomicAdd(&gbins[i], (unsigned long long)c);
    }
}

// nbins <= 16384: 32-bit counters, several CTAs per SM.
__global__ void __launch_bounds__(kThreads)
hist_smem_kernel(const float* __restrict__ d, uint64_t n, int nbins, float lo, float hi, float scale,
                 const float* __restrict__ range3,
                 unsigned long long* __restrict__ gbins, unsigned long long* __restrict__ goutside) {
    extern __shared__ uint32_t dyn_bins[];
    __shared__ uint32_t s_out[2];
    for (int i = threadIdx.x; i < nbins + 2; i += kThreads) dyn_bins[i] = 0;  // + trash slot
    if (threadIdx.x < 2) s_out[threadIdx.x] = 0;
    __syncthreads();
    if (range3) { lo = range3[0]; hi = range3[1]; scale = range3[2]; }  // resolved on the device (cube_stats)
    uint32_t below = 0, above = 0;
    if (hist_use_fast(nbins, lo, hi, scale)) {
        HistFastF f;
        f.setup(lo, hi, scale, nbins, dyn_bins, s_out);
        stream_cube<kThreads>(d, n, f);
    } else {
        HistF f;
        f.lo = lo; f.hi = hi; f.scale = scale; f.top = nbins - 1; f.sbins = dyn_bins;
        stream_cube<kThreads>(d, n, f);
        below = f.below; above = f.above;
    }
    __syncthreads();
    hist_flush_bins(dyn_bins, nbins, gbins);
    if (lo > hi) return;  // unusable device-side [min,max] range: hist_range_kernel has left the marker
    if (below) atomicAdd(&s_out[0], below);
    if (above) atomicAdd(&s_out[1], above);
    __syncthreads();
    if (threadIdx.x < 2 && s_out[threadIdx.x]) atomicAdd(&goutside[threadIdx.x], (unsigned long long)s_out[threadIdx.x]);
}

constexpr int kBigThreads = 1024;

// Alternative for 16384 < nbins <= 65536 (north_star (2)): a thread-block cluster of two CTAs on two SMs
// holds the whole histogram as 32-bit counters in DISTRIBUTED shared memory -- bin b lives in CTA (b & 1)
// of the pair at index b >> 1 (interleaved, so a narrow hot range loads both SMs equally) -- and every
// voxel does one red.shared::cluster.add to the owner.  Half of the increments cross the SM-to-SM
// network.  Selected with cube_set_knob(CUBE_KNOB_BIGHIST, 1); DESIGN.md sec. 4 records which variant
// is faster on B200 and why.
struct HistDsmF : HistBase {
    uint32_t base_local;  // shared::cta address of this CTA's counters
    __device__ __forceinline__ void inc(float x) const {
        const bool in = (x >= lo) && (x <= hi);
        const int b = in ? bin_of(x) : 2 * 32768;            // trash: index 32768 of CTA 0
        const uint32_t local = base_local + (((uint32_t)b >> 1) << 2);
        uint32_t remote;
        asm volatile("mapa.shared::cluster.u32 %0, %1, %2;" : "=r"(remote) : "r"(local), "r"((uint32_t)b & 1u));
        asm volatile("red.relaxed.cluster.shared::cluster.add.u32 [%0], 1;" :: "r"(remote) : "memory");
    }
    __device__ __forceinline__ void operator()(float x) {
        inc(x);
        outside(x);
    }
    __device__ __forceinline__ void batch(const float4 (&r)[kUnroll], const float4*) {
        float bmin = INFINITY, bmax = -INFINITY;
#pragma unroll
        for (int j = 0; j < kUnroll; ++j) {
            inc(r[j].x); inc(r[j].y); inc(r[j].z); inc(r[j].w);
            bmin = fminf(fminf(bmin, r[j].x), fminf(r[j].y, fminf(r[j].z, r[j].w)));
            bmax = fmaxf(fmaxf(bmax, r[j].x), fmaxf(r[j].y, fmaxf(r[j].z, r[j].w)));
        }
        if (bmin < lo || bmax > hi) {
#pragma unroll
            for (int j = 0; j < kUnroll; ++j) { outside(r[j].x); outside(r[j].y); outside(r[j].z); outside(r[j].w); }
        }
    }
};

__device__ __forceinline__ void cluster_sync_all() {
    asm volatile("barrier.cluster.arrive.release.aligned;\n\tbarrier.cluster.wait.acquire.aligned;" ::: "memory");
}

__global__ void __cluster_dims__(2, 1, 1) __launch_bounds__(kBigThreads)
hist_dsm_kernel(const float* __restrict__ d, uint64_t n, int nbins, float lo, float hi, float scale,
                const float* __restrict__ range3,
                unsigned long long* __restrict__ gbins, unsigned long long* __restrict__ goutside) {
    extern __shared__ uint32_t dyn_bins[];  // 32768 + 1 counters per CTA
    __shared__ uint32_t s_out[2];
    uint32_t rank;
    asm volatile("mov.u32 %0, %%cluster_ctarank;" : "=r"(rank));
    for (int i = threadIdx.x; i <= 32768; i += kBigThreads) dyn_bins[i] = 0;
    if (threadIdx.x < 2) s_out[threadIdx.x] = 0;
    cluster_sync_all();  // both CTAs zeroed before any remote increment
    if (range3) { lo = range3[0]; hi = range3[1]; scale = range3[2]; }
    HistDsmF f;
    f.lo = lo; f.hi = hi; f.scale = scale; f.top = nbins - 1; f.base_local = smem_addr(dyn_bins);
    stream_cube<kBigThreads>(d, n, f);
    cluster_sync_all();  // all remote increments have landed
    for (int i = threadIdx.x; i < 32768; i += kBigThreads) {
        const uint32_t c = dyn_bins[i];
        const int b = 2 * i + (int)rank;
        if (c && b < nbins) atomicAdd(&gbins[b], (unsigned long long)c);
    }
    hist_flush_outside(f, s_out, goutside);
}

// Read-only STREAM probe: the same streaming loop with the lightest possible functor (one FADD per voxel).
// Its rate is the measured read ceiling the statistics kernels are compared with (north_star: "a measured
// STREAM-style read peak").
struct ProbeF {
    float acc = 0.f;
    __device__ __forceinline__ void operator()(float x) { acc += x; }
    CUBE_DEFAULT_BATCH()
};
__global__ void __launch_bounds__(kThreads)
probe_read_kernel(const float* __restrict__ d, uint64_t n, float* __restrict__ out) {
    ProbeF f;
    stream_cube<kThreads>(d, n, f);
    if (f.acc == 123.456f) *out = f.acc;  // keeps the loads alive; practically never true
}

}  // namespace cube

#include "cube_hist_big.cuh"
#include "cube_fused.cuh"
#include "cube_fused_big.cuh"
#include "cube_minimap.cuh"
#include "cube_torben.cuh"
