// cube_minimap_median.cuh -- per-cell lower median of the statistical mini-map (SURVEY.md sec. 8(f) NEXT-2 "mean/std
// (then median) per user partition"; "each data point represents the data statistics of a bigger region").
//
// The exact selection of cube_select.cuh, segmented: one GROUP of threads (a CTA of 512 for cells of >= 1024 voxels,
// a warp otherwise) owns one cell at a time, reads its px x py x pz voxels ONCE (4 B per voxel, rows of px voxels),
// keeps their order-preserving keys in shared memory (a 30^3 cell is 27000 keys = 105 KiB; NULL voxels become the key
// 0xFFFFFFFF, above every value, and are counted) and fixes the key of rank k = (count - 1) / 2 with four 8-bit digit
// histograms over the staged keys -- no second read of the cube.  Cells too large for shared memory (more than
// kMedStageKeys voxels) are re-read from global memory for each digit instead (L2 / HBM: 16 B per voxel).
// The paper's Alg. 1 would take ~31 passes per cell.
#pragma once
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

// The bin holding rank k in hist[256] (counts of the keys still in play) and the rank left inside it; every thread
// gets both.  GROUP >= 256: thread t < 256 owns bin t; GROUP = 32: lane l owns bins 8l .. 8l+7.
template <int GROUP>
__device__ __forceinline__ void med_locate(const uint32_t* hist, uint32_t k, uint32_t* red, int tid, uint32_t& bin, uint32_t& krem) {
    constexpr int OWNERS = GROUP < 256 ? GROUP : 256;   // threads that own bins
    constexpr int PER = 256 / OWNERS;
    const bool owner = tid < OWNERS;
    uint32_t c[PER], mine = 0;
#pragma unroll
    for (int j = 0; j < PER; ++j) { c[j] = owner ? hist[tid * PER + j] : 0u; mine += c[j]; }
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
#pragma unroll
    for (int j = 0; j < PER; ++j) {
        if (c[j] && excl <= k && k < excl + c[j]) { red[0] = (uint32_t)(tid * PER + j); red[1] = k - excl; }   // exactly one
        excl += c[j];
    }
    med_sync<GROUP>();
    bin = red[0]; krem = red[1];
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
