// cube_minimap_median.cuh -- per-cell lower median of the statistical mini-map (SURVEY.md sec. 8(f) NEXT-2 "mean/std
// (then median) per user partition"; "each data point represents the data statistics of a bigger region").
//
// The exact selection of cube_select.cuh, segmented: one group of threads owns one cell at a time.
//   * cells of >= 1024 voxels, default: minimap_median_two_reads_kernel -- a CTA of 256 threads reads the cell from
//     HBM counting an 11-bit first digit, reads it again from L2 keeping the median bucket's voxels in shared memory,
//     and fixes the other 21 bits on those (8 B per voxel through the SM, 4 B from HBM when the cell's lines stay in
//     L2; 24 KiB of shared memory whatever the cell size);
//   * CUBE_KNOB_MAPMEDIAN = 1 (and cells whose offsets do not fit 32 bits): minimap_median_cta_kernel -- 512 threads
//     read the cell ONCE and keep all its keys in shared memory (a 30^3 cell is 105 KiB; NULL voxels become the key
//     0xFFFFFFFF, above every value), four 8-bit digit histograms over the staged keys; cells of more than
//     kMedStageKeys voxels are re-read from global memory for each digit instead;
//   * cells below 1024 voxels: minimap_median_warp_kernel, one warp per cell, keys staged in shared memory.
// The paper's Alg. 1 would take ~31 passes per cell.
#pragma once
#include <type_traits>

#include "cube_common.cuh"

namespace cube {

struct MedGeom { long long nx, ny, nz, px, py, pz, mx, my, mz; };

constexpr int kMedCtaThreads = 512;
constexpr int kMedStageKeys = 56000;                 // most keys a CTA can stage (219 KiB: one CTA per SM; a 30^3 cell
                                                     // takes 105 KiB: two CTAs per SM)
constexpr int kMedWarpKeys = 1024;                   // cells below this many voxels: one warp per cell
constexpr int kMedCtaExtra = (264 + 40) * 4;         // histogram + reduction words behind the staged keys
constexpr int kMedWarpSmemPerWarp = (kMedWarpKeys + 264 + 8) * 4;

template <int GROUP> __device__ __forceinline__ void med_sync() {
    if (GROUP == 32) __syncwarp(); else __syncthreads();
}

// Sum of v over the group; every thread gets it.  `red` = 8 words of the group's shared memory.
template <int GROUP>
__device__ __forceinline__ uint32_t med_sum(uint32_t v, uint32_t* red, int tid) {
    v = __reduce_add_sync(0xffffffffu, v);
    if (GROUP == 32) return v;
    med_sync<GROUP>();                               // red is free
    if ((tid & 31) == 0) red[tid >> 5] = v;
    med_sync<GROUP>();
    uint32_t t = 0;
#pragma unroll
    for (int w = 0; w < GROUP / 32; ++w) t += red[w];
    return t;
}

// The bin holding rank k in hist[BINS] (counts of the keys still in play) and the rank left inside it; every thread
// gets both.  Thread t < OWNERS = min(GROUP, BINS) owns the BINS / OWNERS bins from t * PER on.
template <int GROUP, int BINS = 256>
__device__ __forceinline__ void med_locate(const uint32_t* hist, uint32_t k, uint32_t* red, int tid, uint32_t& bin, uint32_t& krem) {
    constexpr int OWNERS = GROUP < BINS ? GROUP : BINS;   // threads that own bins
    constexpr int PER = BINS / OWNERS;
    const bool owner = tid < OWNERS;
    uint32_t c[PER], mine = 0;
    if (PER % 4 == 0) {
#pragma unroll
        for (int j = 0; j < PER; j += 4) {
            const uint4 q = owner ? *reinterpret_cast<const uint4*>(hist + tid * PER + j) : make_uint4(0u, 0u, 0u, 0u);
            c[j] = q.x; c[j + 1] = q.y; c[j + 2] = q.z; c[j + 3] = q.w;
        }
    } else {
#pragma unroll
        for (int j = 0; j < PER; ++j) c[j] = owner ? hist[tid * PER + j] : 0u;
    }
#pragma unroll
    for (int j = 0; j < PER; ++j) mine += c[j];
    uint32_t incl = mine;
    const int lane = tid & 31;
#pragma unroll
    for (int off = 1; off < 32; off <<= 1) {
        const uint32_t u = __shfl_up_sync(0xffffffffu, incl, off);
        if (lane >= off) incl += u;
    }
    uint32_t before = 0;
    if (GROUP > 32) {
        med_sync<GROUP>();
        if (lane == 31 && owner) red[tid >> 5] = incl;
        med_sync<GROUP>();
        if (owner) for (int w = 0; w < (tid >> 5); ++w) before += red[w];
    }
    uint32_t excl = before + incl - mine;
    med_sync<GROUP>();                               // red[0..1] become the answer
    if (excl <= k && k < excl + mine) {              // exactly one owner
#pragma unroll
        for (int j = 0; j < PER; ++j) {
            if (c[j] && excl <= k && k < excl + c[j]) { red[0] = (uint32_t)(tid * PER + j); red[1] = k - excl; }
            excl += c[j];
        }
    }
    med_sync<GROUP>();
    bin = red[0]; krem = red[1];
}

// The voxels of one cell: `rows` rows of w contiguous voxels.
struct MedCell {
    const float* base;
    int w, h, rows, dep;             // dep: planes (rows = h * dep)
    uint32_t nvox, magic;            // magic = floor(2^32 / h) + 1: r / h == umulhi(r, magic) while r * h < 2^32
    int lpr_log1, lpr_log2;          // log2 of the lanes a row takes, read as floats / as float2 (-1: not eligible)
    long long row_step, plane_step;
};

__device__ __forceinline__ MedCell med_cell_of(const float* __restrict__ d, const MedGeom& g, long long cell) {
    const long long cx = cell % g.mx, cy = (cell / g.mx) % g.my, cz = cell / (g.mx * g.my);
    const long long x0 = cx * g.px, y0 = cy * g.py, z0 = cz * g.pz;
    MedCell c;
    c.w = (int)min(g.px, g.nx - x0);
    c.h = (int)min(g.py, g.ny - y0);
    c.rows = c.h * (int)min(g.pz, g.nz - z0);
    c.nvox = (uint32_t)c.w * (uint32_t)c.rows;
    c.base = d + ((z0 * g.ny + y0) * g.nx + x0);
    c.row_step = g.nx;
    c.plane_step = g.ny * g.nx;
    c.dep = c.rows / c.h;
    if (c.h == 1) { c.h = c.rows; c.row_step = c.plane_step; c.dep = 1; }   // one line per plane: the planes are the rows
    c.magic = c.h == 1 ? 0u : (uint32_t)(0x100000000ull / (uint32_t)c.h) + 1u;   // h == 1: a single row, r = 0
    auto lanes_log = [](int n) { int l = 0; while ((1 << l) < n && l < 5) ++l; return l; };
    c.lpr_log1 = lanes_log(c.w);
    const bool pairs = (c.w & 1) == 0 && (reinterpret_cast<uintptr_t>(c.base) & 7u) == 0 && (c.row_step & 1) == 0 &&
                       (c.plane_step & 1) == 0;
    c.lpr_log2 = pairs ? lanes_log(c.w / 2) : -1;
    return c;
}

// fn(v) for every voxel of the cell: a warp takes rows, kMedInFlight at a time (that many loads per lane in flight:
// the read of a cell is a chain of dependent round trips otherwise); the (y, z) of a warp's row advances by
// additions; offsets from the cell's first voxel fit 32 bits (checked by the caller).
#ifndef CUBE_MED_INFLIGHT
#define CUBE_MED_INFLIGHT 8
#endif
constexpr int kMedInFlight = CUBE_MED_INFLIGHT;

// A row of the cell takes LPR = 2^lpr_log lanes (the smallest power of two holding w / VEC elements, at most 32), so a
// warp load covers 32 / LPR rows: a 30-voxel row read as 15 float2 (VEC = 2: rows 8-byte aligned, w even) shares its
// load with a second row, a 16-voxel row with three more.  What a load costs in address arithmetic (the division of
// the row number by the cell's height is a multiplication by c.magic, exact while r * h < 2^32; the byte offset three
// IMADs; base + 32-bit offset) is spent once per load, hence the packing.
// L2 eviction hints of the two reads: the lines of a cell are wanted again (read 2) by the same CTA a few
// microseconds later and never after that.  Load POLICY 0: plain read-only loads; 1: evict_last; 2: evict_first.
// CUBE_MED_POLICY 1 (default): read 2 marks its lines evict_first (their last use); 2: read 1 evict_last as well
// (measured: 1.58 vs 1.62 ms without hints on c2 30^3; the two settings tie).
#ifndef CUBE_MED_POLICY
#define CUBE_MED_POLICY 1
#endif
template <int POLICY> __device__ __forceinline__ uint64_t med_policy() {
    uint64_t p = 0;
    if (POLICY == 1) asm("createpolicy.fractional.L2::evict_last.b64 %0, 1.0;" : "=l"(p));
    if (POLICY == 2) asm("createpolicy.fractional.L2::evict_first.b64 %0, 1.0;" : "=l"(p));
    return p;
}
template <int POLICY> __device__ __forceinline__ float med_ld(const float* p, uint64_t pol) {
    if (POLICY == 0) return __ldg(p);
    float v;
    asm volatile("ld.global.nc.L2::cache_hint.f32 %0, [%1], %2;" : "=f"(v) : "l"(p), "l"(pol));
    return v;
}
template <int POLICY> __device__ __forceinline__ float2 med_ld(const float2* p, uint64_t pol) {
    if (POLICY == 0) return __ldg(p);
    float2 v;
    asm volatile("ld.global.nc.L2::cache_hint.v2.f32 {%0, %1}, [%2], %3;" : "=f"(v.x), "=f"(v.y) : "l"(p), "l"(pol));
    return v;
}

template <int GROUP, int VEC, int POLICY, class F>
__device__ __forceinline__ void med_for_each_voxel_v(const MedCell& c, int tid, F&& fn) {
    const uint64_t pol = med_policy<POLICY>();
    constexpr int NW = GROUP / 32, U = kMedInFlight;
    const int lane = tid & 31, wid = tid >> 5;
    const int lpr_log = VEC == 2 ? c.lpr_log2 : c.lpr_log1, rpw_log = 5 - lpr_log;
    const uint32_t sub = (uint32_t)lane >> lpr_log, col = ((uint32_t)lane & ((1u << lpr_log) - 1u)) * VEC;
    const uint32_t rstep = (uint32_t)NW << rpw_log;                          // rows per step of the whole CTA
    const uint32_t xstep = (uint32_t)VEC << lpr_log;
    const uint32_t hh = (uint32_t)c.h, magic = c.magic, rows = (uint32_t)c.rows, w = (uint32_t)c.w;
    const uint32_t row_bytes = (uint32_t)c.row_step * 4u, plane_bytes = (uint32_t)c.plane_step * 4u;
    const char* __restrict__ base = reinterpret_cast<const char*>(c.base);
    for (uint32_t rw = (uint32_t)wid << rpw_log; rw < rows; rw += rstep * U) {   // rw: the warp's first row of the batch
        uint32_t o[U];
#pragma unroll
        for (int u = 0; u < U; ++u) {
            const uint32_t r = rw + sub + (uint32_t)u * rstep;
            const uint32_t z = __umulhi(r, magic), y = r - z * hh;
            o[u] = z * plane_bytes + y * row_bytes + col * 4u;
        }
        const bool full = rw + ((1u << rpw_log) - 1u) + (U - 1) * rstep < rows;   // warp-uniform
        for (uint32_t x0 = 0; x0 < w; x0 += xstep) {
            const char* __restrict__ q = base + x0 * 4u;                     // warp-uniform
            if (col + x0 < w) {
                float a[U], b[U];
                if (full) {
#pragma unroll
                    for (int u = 0; u < U; ++u) {
                        if (VEC == 2) {
                            const float2 t = med_ld<POLICY>(reinterpret_cast<const float2*>(q + o[u]), pol);
                            a[u] = t.x; b[u] = t.y;
                        } else {
                            a[u] = med_ld<POLICY>(reinterpret_cast<const float*>(q + o[u]), pol);
                        }
                    }
#pragma unroll
                    for (int u = 0; u < U; ++u) { fn(a[u]); if (VEC == 2) fn(b[u]); }
                } else {
#pragma unroll
                    for (int u = 0; u < U; ++u) {
                        if (rw + sub + (uint32_t)u * rstep < rows) {
                            if (VEC == 2) {
                                const float2 t = med_ld<POLICY>(reinterpret_cast<const float2*>(q + o[u]), pol);
                                fn(t.x); fn(t.y);
                            } else {
                                fn(med_ld<POLICY>(reinterpret_cast<const float*>(q + o[u]), pol));
                            }
                        }
                    }
                }
            }
        }
    }
}

// The same visit for cells that are deep enough (c.dep >= kMedDeep planes): a warp keeps its rows' y and walks along z,
// kMedInFlight planes per batch -- the address of a load is the previous one plus the plane stride (one 64-bit add),
// where the row-major order above pays a division and three multiplications per load (ncu on 30^3 cells: 11 IMAD per
// LDG, a third of all instructions).  The warps share the ng = ceil(h / rows-per-load) groups of rows; when there are
// fewer groups than warps, several warps take the same group and interleave its planes.
constexpr int kMedDeep = 16;

template <int GROUP, int VEC, int POLICY, class F>
__device__ __forceinline__ void med_for_each_voxel_z(const MedCell& c, int tid, F&& fn) {
    const uint64_t pol = med_policy<POLICY>();
    constexpr uint32_t NW = GROUP / 32, U = kMedInFlight;
    const int lane = tid & 31;
    const uint32_t wid = (uint32_t)tid >> 5;
    const int lpr_log = VEC == 2 ? c.lpr_log2 : c.lpr_log1, rpw_log = 5 - lpr_log;
    const uint32_t sub = (uint32_t)lane >> lpr_log, col = ((uint32_t)lane & ((1u << lpr_log) - 1u)) * VEC;
    const uint32_t xstep = (uint32_t)VEC << lpr_log;
    const uint32_t h = (uint32_t)c.h, w = (uint32_t)c.w, dep = (uint32_t)c.dep;
    const uint32_t ng = (h + (1u << rpw_log) - 1u) >> rpw_log;
    const uint32_t G = ng < NW ? ng : NW, ZS = NW / G;          // warps per plane sweep, sweeps interleaved along z
    const uint32_t g0 = wid % G, z0 = wid / G;
    if (z0 >= ZS) return;                                        // NW is not a multiple of G: the left-over warps
    const uint64_t row_bytes = (uint64_t)c.row_step * 4u, zs_bytes = (uint64_t)c.plane_step * 4u * ZS;
    using V = typename std::conditional<VEC == 2, float2, float>::type;
    for (uint32_t g = g0; g < ng; g += G) {
        const uint32_t y = (g << rpw_log) + sub;
        for (uint32_t x0 = 0; x0 < w; x0 += xstep) {
            if (!(y < h && col + x0 < w)) continue;              // lane-constant over the z walk
            const char* __restrict__ q = reinterpret_cast<const char*>(c.base) + y * row_bytes + (uint64_t)(col + x0) * 4u +
                                         (uint64_t)z0 * (uint64_t)c.plane_step * 4u;
            uint32_t z = z0;
            for (; z + (U - 1) * ZS < dep; z += U * ZS, q += U * zs_bytes) {
                float a[U], b[U];
#pragma unroll
                for (uint32_t u = 0; u < U; ++u) {
                    if (VEC == 2) {
                        const float2 t = med_ld<POLICY>(reinterpret_cast<const float2*>(q + u * zs_bytes), pol);
                        a[u] = t.x; b[u] = t.y;
                    } else {
                        a[u] = med_ld<POLICY>(reinterpret_cast<const float*>(q + u * zs_bytes), pol);
                    }
                }
#pragma unroll
                for (uint32_t u = 0; u < U; ++u) { fn(a[u]); if (VEC == 2) fn(b[u]); }
            }
            if (z < dep) {                                       // the last, partial batch
                float a[U], b[U];
#pragma unroll
                for (uint32_t u = 0; u < U; ++u) {
                    a[u] = b[u] = 0.0f;
                    if (z + u * ZS < dep) {
                        if (VEC == 2) {
                            const float2 t = med_ld<POLICY>(reinterpret_cast<const float2*>(q + u * zs_bytes), pol);
                            a[u] = t.x; b[u] = t.y;
                        } else {
                            a[u] = med_ld<POLICY>(reinterpret_cast<const float*>(q + u * zs_bytes), pol);
                        }
                    }
                }
#pragma unroll
                for (uint32_t u = 0; u < U; ++u)
                    if (z + u * ZS < dep) { fn(a[u]); if (VEC == 2) fn(b[u]); }
            }
        }
    }
}

#ifndef CUBE_MED_ZWALK
#define CUBE_MED_ZWALK 1
#endif
template <int GROUP, int POLICY = 0, class F>
__device__ __forceinline__ void med_for_each_voxel(const MedCell& c, int tid, F&& fn) {
    // z walk: deep cells with at least one group of rows per warp (measured on c2: 30 x 30 x 16 cells 2.09 -> 1.66 ms,
    // 64 x 16 x 64 1.23 -> 1.11, 64^3 1.40 -> 1.33, 30^3 unchanged at 1.58; 16^3 cells -- four groups for eight warps --
    // are 7 % faster in row order)
    const int lpr = c.lpr_log2 >= 0 ? c.lpr_log2 : c.lpr_log1;
    const int ng = (c.h + (1 << (5 - lpr)) - 1) >> (5 - lpr);
    if (CUBE_MED_ZWALK && c.dep >= kMedDeep && ng >= GROUP / 32) {                   // all uniform over the CTA
        if (c.lpr_log2 >= 0) med_for_each_voxel_z<GROUP, 2, POLICY>(c, tid, fn);
        else med_for_each_voxel_z<GROUP, 1, POLICY>(c, tid, fn);
    } else {
        if (c.lpr_log2 >= 0) med_for_each_voxel_v<GROUP, 2, POLICY>(c, tid, fn);
        else med_for_each_voxel_v<GROUP, 1, POLICY>(c, tid, fn);
    }
}

// Two-read selection of one cell by one CTA (cells of any size).
//   read 1 (HBM): the 11-bit first digit counted in shared memory.  The digit is taken from the RAW bits (sign, exponent,
//       two mantissa bits) -- no key conversion per voxel; NULL voxels are left out by a predicate (5 instructions per
//       voxel: LDG, FSETP, SHF, LOP3, predicated RED) and the buckets are only put in key order when they are
//       scanned: key-order bucket j is raw bucket 2047 - j (negative values, descending) or j - 1024.
//   read 2 (the cell's lines are in L2: a 30^3 cell is 105 KiB): the voxels of the median's bucket -- a few per cent
//       of the cell -- are appended to a buffer in shared memory (bits - rawbase < 2^21, predicated ATOMS + STS); the
//       remaining 11 + 10 key bits are fixed on those.
// A bucket that does not fit kMed2Cand keys (constant cells, heavy ties) has its digits counted by further reads of
// the cell instead.  24.1 KiB of shared memory per CTA whatever the cell size.
#ifndef CUBE_MED2_THREADS
#define CUBE_MED2_THREADS 256
#endif
constexpr int kMed2Threads = CUBE_MED2_THREADS;
constexpr int kMed2Bins = 2048;
constexpr int kMed2Per = kMed2Bins / kMed2Threads;            // buckets a thread scans
constexpr int kMed2Cand = 4096;
constexpr int kMed2Smem = (kMed2Bins + kMed2Cand + 32) * 4;
static_assert(kMed2Per >= 4 && kMed2Per % 4 == 0 && kMed2Threads % 64 == 0, "four +-Inf / NaN buckets per end thread");

// counts of key-order buckets PER * tid .. PER * tid + PER - 1 from the raw-order histogram
__device__ __forceinline__ void med_load_raw_order(const uint32_t* hist, int tid, uint32_t (&c)[kMed2Per]) {
    constexpr int PER = kMed2Per;
    const bool neg = tid < kMed2Threads / 2;
    const int base = neg ? kMed2Bins - PER * (tid + 1) : PER * tid - kMed2Bins / 2;
    uint32_t r[PER];
#pragma unroll
    for (int j = 0; j < PER; j += 4) {
        const uint4 a = *reinterpret_cast<const uint4*>(hist + base + j);
        r[j] = a.x; r[j + 1] = a.y; r[j + 2] = a.z; r[j + 3] = a.w;
    }
#pragma unroll
    for (int j = 0; j < PER; ++j) c[j] = neg ? r[PER - 1 - j] : r[j];
}

// as med_locate, on bucket counts already in registers (bucket index = PER * tid + j); k = 0xFFFFFFFF: the lower
// median of what was counted.  red[0..2] = bucket, rank inside it, its count.
__device__ __forceinline__ void med_locate_regs(const uint32_t (&c)[kMed2Per], uint32_t k, uint32_t* red, int tid, uint32_t& bin,
                                                uint32_t& krem, uint32_t& total) {
    constexpr int PER = kMed2Per, NWARP = kMed2Threads / 32;
    uint32_t mine = 0;
#pragma unroll
    for (int j = 0; j < PER; ++j) mine += c[j];
    uint32_t incl = mine;
    const int lane = tid & 31;
#pragma unroll
    for (int off = 1; off < 32; off <<= 1) {
        const uint32_t u = __shfl_up_sync(0xffffffffu, incl, off);
        if (lane >= off) incl += u;
    }
    __syncthreads();
    if (lane == 31) red[12 + (tid >> 5)] = incl;
    __syncthreads();
    uint32_t before = 0, all = 0;
#pragma unroll
    for (int w = 0; w < NWARP; ++w) { const uint32_t t = red[12 + w]; all += t; before += w < (tid >> 5) ? t : 0u; }
    total = all;
    if (k == 0xFFFFFFFFu) k = all ? (all - 1) / 2 : 0;
    uint32_t excl = before + incl - mine;
    if (excl <= k && k < excl + mine) {                      // exactly one thread (none when all == 0)
#pragma unroll
        for (int j = 0; j < PER; ++j) {
            if (c[j] && excl <= k && k < excl + c[j]) { red[0] = (uint32_t)(tid * PER + j); red[1] = k - excl; red[2] = c[j]; }
            excl += c[j];
        }
    }
    __syncthreads();
    bin = red[0]; krem = red[1];
}

__device__ __forceinline__ float med_cell_two_reads(const MedCell& c, uint32_t* hist, uint32_t* cand, uint32_t* red, int tid) {
    constexpr int GROUP = kMed2Threads;
    const uint32_t hist_s = (uint32_t)__cvta_generic_to_shared(hist);
    const uint32_t cand_s = (uint32_t)__cvta_generic_to_shared(cand);
    const uint32_t ncand_s = (uint32_t)__cvta_generic_to_shared(red + 8);
    auto zero_hist = [&]() {
        uint4* h4 = reinterpret_cast<uint4*>(hist);
        for (int i = tid; i < kMed2Bins / 4; i += GROUP) h4[i] = make_uint4(0u, 0u, 0u, 0u);
        if (tid == 0) red[8] = 0;                    // the candidate counter
    };
    zero_hist();
    __syncthreads();
    // read 1: every voxel counted by its raw top 11 bits, NULL voxels included (SHF, LEA, ATOMS per voxel).  The raw
    // buckets 0x3FD-0x3FF / 0x7FD-0x7FF hold nothing but NaN patterns and are dropped when the buckets are scanned;
    // 0x3FC / 0x7FC hold +-Inf AND the NaN patterns with a payload below 2^21: a cell with anything in those two is
    // counted again with the NULL test per voxel (rare: cells holding infinities).
    med_for_each_voxel<GROUP, (CUBE_MED_POLICY >= 2 ? 1 : 0)>(c, tid, [&](float v) {
        const uint32_t a = hist_s + (__float_as_uint(v) >> 21) * 4u;
        asm volatile("red.shared.add.u32 [%0], 1;" ::"r"(a) : "memory");
    });
    __syncthreads();
    constexpr int PER = kMed2Per;
    uint32_t cnt[PER], k, b0, b1, b2, count;
    auto load_counts = [&]() {
        med_load_raw_order(hist, tid, cnt);
        if (tid == 0) cnt[0] = cnt[1] = cnt[2] = 0;            // key-order buckets 0-2 and 2045-2047: NaN patterns only
        if (tid == GROUP - 1) cnt[PER - 3] = cnt[PER - 2] = cnt[PER - 1] = 0;
    };
    load_counts();
    if (tid == 0) red[9] = cnt[3];                             // -Inf and negative NaNs of small payload
    if (tid == GROUP - 1) red[10] = cnt[PER - 4];              // +Inf and positive NaNs of small payload
    __syncthreads();
    const bool careful = (red[9] | red[10]) != 0;              // uniform over the CTA
    if (careful) {
        __syncthreads();
        zero_hist();
        __syncthreads();
        med_for_each_voxel<GROUP>(c, tid, [&](float v) {
            if (v == v) atomicAdd(&hist[__float_as_uint(v) >> 21], 1u);
        });
        __syncthreads();
        load_counts();
    }
    med_locate_regs(cnt, 0xFFFFFFFFu, red, tid, b0, k, count);
    if (count == 0) return __int_as_float(0x7fc00000);       // uniform over the CTA: no non-NULL voxel
    const uint32_t c0 = red[2];
    const uint32_t rawbase = (b0 >= 1024u ? b0 - 1024u : 2047u - b0) << 21;
    __syncthreads();
    zero_hist();
    __syncthreads();
    if (c0 <= (uint32_t)kMed2Cand) {
        // read 2: the voxels of the bucket (bits - rawbase < 2^21; a NULL voxel can only pass in a `careful` cell)
        if (!careful) {
            med_for_each_voxel<GROUP, (CUBE_MED_POLICY >= 1 ? 2 : 0)>(c, tid, [&](float v) {
                const uint32_t bits = __float_as_uint(v);
                if (bits - rawbase < 0x200000u) {
                    uint32_t pos;
                    asm volatile("atom.shared.add.u32 %0, [%1], 1;" : "=r"(pos) : "r"(ncand_s) : "memory");
                    CUBE_CHECK(pos < (uint32_t)kMed2Cand);
                    asm volatile("st.shared.u32 [%0], %1;" ::"r"(cand_s + pos * 4u), "r"(bits) : "memory");
                }
            });
        } else {
            med_for_each_voxel<GROUP>(c, tid, [&](float v) {
                const uint32_t bits = __float_as_uint(v);
                if (bits - rawbase < 0x200000u && v == v) {
                    const uint32_t pos = atomicAdd(&red[8], 1u);
                    CUBE_CHECK(pos < (uint32_t)kMed2Cand);
                    cand[pos] = bits;
                }
            });
        }
        __syncthreads();
        CUBE_CHECK(red[8] == c0);
        for (uint32_t i = tid; i < c0; i += GROUP) atomicAdd(&hist[(key_of(__uint_as_float(cand[i])) >> 10) & 2047u], 1u);
        __syncthreads();
        med_locate<GROUP, kMed2Bins>(hist, k, red + 12, tid, b1, k);
        __syncthreads();
        zero_hist();
        __syncthreads();
        for (uint32_t i = tid; i < c0; i += GROUP) {
            const uint32_t key = key_of(__uint_as_float(cand[i]));
            if (((key >> 10) & 2047u) == b1) atomicAdd(&hist[key & 1023u], 1u);
        }
    } else {
        med_for_each_voxel<GROUP>(c, tid, [&](float v) {
            const uint32_t key = key_of(v);
            if ((key >> 21) == b0 && v == v) atomicAdd(&hist[(key >> 10) & 2047u], 1u);
        });
        __syncthreads();
        med_locate<GROUP, kMed2Bins>(hist, k, red + 12, tid, b1, k);
        __syncthreads();
        zero_hist();
        __syncthreads();
        const uint32_t top = (b0 << 11) | b1;
        med_for_each_voxel<GROUP>(c, tid, [&](float v) {
            const uint32_t key = key_of(v);
            if ((key >> 10) == top && v == v) atomicAdd(&hist[key & 1023u], 1u);
        });
    }
    __syncthreads();
    med_locate<GROUP, kMed2Bins>(hist, k, red + 12, tid, b2, k);
    return __uint_as_float(bits_of_key((b0 << 21) | (b1 << 10) | b2));
}

#ifndef CUBE_MED2_CTAS
#define CUBE_MED2_CTAS 5
#endif
__global__ void __launch_bounds__(kMed2Threads, CUBE_MED2_CTAS)
minimap_median_two_reads_kernel(const float* __restrict__ d, MedGeom g, float* __restrict__ med) {
    extern __shared__ __align__(16) uint32_t med_smem[];
    uint32_t* hist = med_smem;
    uint32_t* cand = med_smem + kMed2Bins;
    uint32_t* red = cand + kMed2Cand;
    const long long ncell = g.mx * g.my * g.mz;
    for (long long cell = blockIdx.x; cell < ncell; cell += gridDim.x) {
        const MedCell c = med_cell_of(d, g, cell);
        const float r = med_cell_two_reads(c, hist, cand, red, threadIdx.x);
        if (threadIdx.x == 0) med[cell] = r;
        __syncthreads();
    }
}

// One group, one cell.  keys: the group's stage (STAGED) ; hist: 256 counters; red: 8 words.
template <int GROUP, bool STAGED>
__device__ __forceinline__ float med_cell(const float* __restrict__ d, const MedGeom& g, long long cell, uint32_t* keys,
                                          uint32_t* hist, uint32_t* red, int tid) {
    const long long cx = cell % g.mx, cy = (cell / g.mx) % g.my, cz = cell / (g.mx * g.my);
    const long long x0 = cx * g.px, y0 = cy * g.py, z0 = cz * g.pz;
    const int w = (int)min(g.px, g.nx - x0), h = (int)min(g.py, g.ny - y0), dep = (int)min(g.pz, g.nz - z0);
    const int rows = h * dep;
    const uint32_t nvox = (uint32_t)w * (uint32_t)rows;
    const float* __restrict__ base = d + ((z0 * g.ny + y0) * g.nx + x0);
    const int lane = tid & 31, wid = tid >> 5;
    constexpr int NW = GROUP / 32;
    // visit every voxel of the cell: a warp takes rows (a row is px contiguous voxels), eight rows at a time so that
    // eight loads per lane are in flight (one load at a time left the read of a 30^3 cell at the latency of 113
    // dependent L2 / HBM round trips per warp); the (y, z) of a warp's row advances by additions, no division per row,
    // and a full batch of eight rows carries no per-row bounds test
    const long long row_step = g.nx, plane_step = g.ny * g.nx;
    auto for_each_key = [&](auto&& fn) {
        int yy = wid % h, zz = wid / h;
        for (int r0 = wid; r0 < rows; r0 += NW * 8) {
            const float* p[8];
#pragma unroll
            for (int u = 0; u < 8; ++u) {
                p[u] = base + (long long)zz * plane_step + (long long)yy * row_step;
                yy += NW;
                while (yy >= h) { yy -= h; ++zz; }
            }
            const bool full = r0 + 7 * NW < rows;            // warp-uniform
            uint32_t idx0 = (uint32_t)r0 * (uint32_t)w + (uint32_t)lane;
            for (int xc = 0; xc < w; xc += 32, idx0 += 32) {
                if (xc + lane < w) {
                    float v[8];
                    if (full) {
#pragma unroll
                        for (int u = 0; u < 8; ++u) v[u] = __ldg(p[u] + xc + lane);
#pragma unroll
                        for (int u = 0; u < 8; ++u)
                            fn(v[u] == v[u] ? key_of(v[u]) : 0xFFFFFFFFu, idx0 + (uint32_t)(u * NW) * (uint32_t)w);
                    } else {
#pragma unroll
                        for (int u = 0; u < 8; ++u) v[u] = (r0 + u * NW < rows) ? __ldg(p[u] + xc + lane) : 0.0f;
#pragma unroll
                        for (int u = 0; u < 8; ++u)
                            if (r0 + u * NW < rows)
                                fn(v[u] == v[u] ? key_of(v[u]) : 0xFFFFFFFFu, idx0 + (uint32_t)(u * NW) * (uint32_t)w);
                    }
                }
            }
        }
    };
    uint32_t nan = 0;
    uint32_t prefix = 0, k = 0;
    float result = __int_as_float(0x7fc00000);
#pragma unroll 1
    for (int pass = 0; pass < 4; ++pass) {
        const int shift = 24 - 8 * pass;
        for (int i = tid; i < 256; i += GROUP) hist[i] = 0;
        med_sync<GROUP>();
        const uint32_t hi_mask = pass == 0 ? 0u : (0xFFFFFFFFu << (shift + 8));   // bits fixed so far
        if (pass == 0 || !STAGED) {
            for_each_key([&](uint32_t key, uint32_t idx) {
                if (pass == 0) { nan += key == 0xFFFFFFFFu ? 1u : 0u; if (STAGED) { CUBE_CHECK(idx < nvox); keys[idx] = key; } }
                if ((key & hi_mask) == prefix) atomicAdd(&hist[(key >> shift) & 255u], 1u);
            });
        } else {
            // the staged keys, four per load (the stage is 16-byte aligned; nvox4 * 4 <= nvox)
            const uint32_t nvox4 = nvox >> 2;
            const uint4* __restrict__ k4 = reinterpret_cast<const uint4*>(keys);
            for (uint32_t i = tid; i < nvox4; i += GROUP) {
                const uint4 q = k4[i];
                if ((q.x & hi_mask) == prefix) atomicAdd(&hist[(q.x >> shift) & 255u], 1u);
                if ((q.y & hi_mask) == prefix) atomicAdd(&hist[(q.y >> shift) & 255u], 1u);
                if ((q.z & hi_mask) == prefix) atomicAdd(&hist[(q.z >> shift) & 255u], 1u);
                if ((q.w & hi_mask) == prefix) atomicAdd(&hist[(q.w >> shift) & 255u], 1u);
            }
            for (uint32_t i = (nvox4 << 2) + tid; i < nvox; i += GROUP) {
                const uint32_t key = keys[i];
                if ((key & hi_mask) == prefix) atomicAdd(&hist[(key >> shift) & 255u], 1u);
            }
        }
        med_sync<GROUP>();
        if (pass == 0) {
            const uint32_t count = nvox - med_sum<GROUP>(nan, red, tid);
            if (count == 0) return result;           // uniform over the group: no non-NULL voxel
            k = (count - 1) / 2;
        }
        uint32_t bin;
        med_locate<GROUP>(hist, k, red, tid, bin, k);
        prefix |= bin << shift;
        med_sync<GROUP>();
    }
    return __uint_as_float(bits_of_key(prefix));
}

// Cells of >= kMedWarpKeys voxels: one CTA per cell at a time (grid-stride over the cells).
__global__ void __launch_bounds__(kMedCtaThreads, 2)
minimap_median_cta_kernel(const float* __restrict__ d, MedGeom g, int stage_keys, float* __restrict__ med) {
    extern __shared__ __align__(16) uint32_t med_smem[];
    uint32_t* keys = med_smem;
    uint32_t* hist = med_smem + stage_keys;          // stage_keys = 0: the cell is re-read for every digit
    const bool staged = stage_keys > 0;
    uint32_t* red = hist + 264;
    const long long ncell = g.mx * g.my * g.mz;
    for (long long cell = blockIdx.x; cell < ncell; cell += gridDim.x) {
        const float r = staged ? med_cell<kMedCtaThreads, true>(d, g, cell, keys, hist, red, threadIdx.x)
                               : med_cell<kMedCtaThreads, false>(d, g, cell, keys, hist, red, threadIdx.x);
        if (threadIdx.x == 0) med[cell] = r;
        __syncthreads();
    }
}

// Smaller cells: one warp per cell, eight cells in flight per CTA.
__global__ void __launch_bounds__(kMedCtaThreads)
minimap_median_warp_kernel(const float* __restrict__ d, MedGeom g, float* __restrict__ med) {
    extern __shared__ __align__(16) uint32_t med_smem[];
    const int wid = threadIdx.x >> 5, lane = threadIdx.x & 31;
    uint32_t* keys = med_smem + wid * (kMedWarpSmemPerWarp / 4);
    uint32_t* hist = keys + kMedWarpKeys;
    uint32_t* red = hist + 264;
    const long long ncell = g.mx * g.my * g.mz;
    const long long nwarps = (long long)gridDim.x * (kMedCtaThreads / 32);
    for (long long cell = (long long)blockIdx.x * (kMedCtaThreads / 32) + wid; cell < ncell; cell += nwarps) {
        const float r = med_cell<32, true>(d, g, cell, keys, hist, red, lane);
        if (lane == 0) med[cell] = r;
        __syncwarp();
    }
}

}  // namespace cube
