// cube_minimap.cuh -- the statistical mini-map (Fig. 7): "a
// scaled-down version of the data cube [where] each data point represents the data statistics of a bigger region
// in the real dataset", regions of px x py x pz voxels ("30x30x30 pixel").  One record (count, nan_count, min,
// max, mean, std) per cell, cell (cx,cy,cz) covering x in [cx*px, min((cx+1)*px, nx)) and likewise in y, z
// (R25); it is the segmented form of the global moments pass, so it is HBM-read-bound as well:
// 4 B per voxel in, 40 B per cell out.
//
// Work decomposition.  A CTA owns a SEGMENT of whole cells along x (as many as fit kMapThreads voxels) for one
// (cy, cz): thread t reads column x0 + t of every one of the py*pz lines of those cells -- each line a contiguous,
// coalesced run of up to 2 KiB -- and keeps ONE accumulator set (count, min, max, fp64 sums about its own pivot),
// because a column never leaves its cell.  kMapUnroll lines are loaded before the first is used and, when none of
// them holds a NaN, accumulated without any per-voxel test (MapColF).  The columns of
// a cell are then merged in x order by one thread per cell (Chan's pairwise update; fixed order => deterministic)
// and the finished record goes straight to the output.  Cells wider than kMapThreads voxels get a CTA of their
// own whose threads stride over the columns and merge through the block tree.
#pragma once
#include "cube_kernels.cuh"

namespace cube {

constexpr int kMapThreads = 512;
constexpr int kMapUnroll = 8;

struct MapGeom {
    long long nx, ny, nz, px, py, pz, mx, my, mz;
    long long cells_per_seg;   // whole cells per CTA along x (1 when px > kMapThreads)
    long long nseg;            // segments per cell row
    long long main_threads;    // 128-bit kernel: threads that own a float4 slot (the rest own cell boundaries)
};

__device__ __forceinline__ float ld_stream1(const float* p) {
    float r;
    asm volatile("ld.global.nc.L1::no_allocate.f32 %0, [%1];" : "=f"(r) : "l"(p));
    return r;
}

// One column of a cell row: the same two ways through as MomentsF::batch.  Groups of kMapUnroll
// lines take the HOT path -- d = (double)x - pivot, tree sum, DFMA chain, FMNMX3, n += 8, valid iff the sum is not
// NaN -- unless the warp is in SAFE mode (a NaN was seen in its last group) or the thread has no pivot yet; the
// y-remainder of every plane (py mod 8 lines) takes the per-voxel form.
struct MapColF : MomentsF<kMomPlain> {
    __device__ __forceinline__ void group(const float (&v)[kMapUnroll], bool& safe_mode) {
        if (safe_mode) {
            const uint32_t n0 = n;
            if (!have) {   // only until this column has met its first voxel that takes part
#pragma unroll
                for (int k = 0; k < kMapUnroll; ++k) take_pivot(v[k]);
            }
            // extrema of the eight lines at once (FMNMX3, NaN-blind) instead of two FMNMX per voxel
            mn = fminf(fminf(fminf(mn, v[0]), fminf(v[1], v[2])), fminf(fminf(v[3], v[4]), fminf(v[5], fminf(v[6], v[7]))));
            mx = fmaxf(fmaxf(fmaxf(mx, v[0]), fmaxf(v[1], v[2])), fmaxf(fmaxf(v[3], v[4]), fmaxf(v[5], fmaxf(v[6], v[7]))));
#pragma unroll
            for (int k = 0; k < kMapUnroll; ++k) core<false>(v[k]);
            safe_mode = __any_sync(__activemask(), n - n0 != (uint32_t)kMapUnroll);
            return;
        }
        double d[kMapUnroll];
#pragma unroll
        for (int k = 0; k < kMapUnroll; ++k) d[k] = (double)v[k] - pivot;
        const double ts = ((d[0] + d[1]) + (d[2] + d[3])) + ((d[4] + d[5]) + (d[6] + d[7]));
        double tq = d[0] * d[0];
#pragma unroll
        for (int k = 1; k < kMapUnroll; ++k) tq = fma(d[k], d[k], tq);
        mn = fminf(fminf(fminf(mn, v[0]), fminf(v[1], v[2])), fminf(fminf(v[3], v[4]), fminf(v[5], fminf(v[6], v[7]))));
        mx = fmaxf(fmaxf(fmaxf(mx, v[0]), fmaxf(v[1], v[2])), fmaxf(fmaxf(v[3], v[4]), fmaxf(v[5], fmaxf(v[6], v[7]))));
        const bool bad = !(ts == ts);
        if (!bad) { s += ts; q += tq; n += kMapUnroll; }
        else {
#pragma unroll
            for (int k = 0; k < kMapUnroll; ++k) {   // rare: redo the group voxel by voxel (min/max are already in)
                const float x = v[k];
                if (x == x) { const double dl = (double)x - pivot; s += dl; q = fma(dl, dl, q); n += 1; }
            }
        }
        safe_mode = __any_sync(__activemask(), bad);
    }
};
static_assert(kMapUnroll == 8, "MapColF::group is written for 8 lines");

__global__ void __launch_bounds__(kMapThreads, 2)
minimap_kernel(const float* __restrict__ d, MapGeom g, unsigned flags, MomentsOut* __restrict__ cells) {
    __shared__ Partial cols[kMapThreads];
    __shared__ Partial scratch[kMapThreads / 32];
    // CTA -> (segment, cy, cz)
    const long long b = blockIdx.x;
    const long long seg = b % g.nseg, cy = (b / g.nseg) % g.my, cz = b / (g.nseg * g.my);
    const long long c0 = seg * g.cells_per_seg;                                  // first cell of the segment
    const long long x0 = c0 * g.px;
    const long long x1 = min((c0 + g.cells_per_seg) * g.px, g.nx);               // end of the segment
    const long long y0 = cy * g.py, y1 = min(y0 + g.py, g.ny);
    const long long z0 = cz * g.pz, z1 = min(z0 + g.pz, g.nz);
    const bool wide = g.px > kMapThreads;   // one cell per CTA, threads stride over its columns

    MapColF f;
    bool safe_mode = true;   // uniform over the active lanes of the warp (they run the same loops)
    const long long yfull = y0 + ((y1 - y0) / kMapUnroll) * kMapUnroll;
    for (long long x = x0 + threadIdx.x; x < x1; x += kMapThreads) {
        for (long long z = z0; z < z1; ++z) {
            const float* __restrict__ p = d + ((z * g.ny + y0) * g.nx + x);
            for (long long y = y0; y < yfull; y += kMapUnroll) {
                float v[kMapUnroll];
#pragma unroll
                for (int k = 0; k < kMapUnroll; ++k) v[k] = ld_stream1(p + (long long)k * g.nx);
                f.group(v, safe_mode);
                p += (long long)kMapUnroll * g.nx;
            }
            for (long long y = yfull; y < y1; ++y) {   // py mod 8 lines: per-voxel form
                f(ld_stream1(p));
                p += g.nx;
            }
        }
    }
    const unsigned long long lines = (unsigned long long)((y1 - y0) * (z1 - z0));
    if (wide) {
        Partial m = partial_block_reduce_n<kMapThreads>(f.partial(), scratch);
        if (threadIdx.x == 0) moments_finalize(m, lines * (unsigned long long)(x1 - x0), flags, &cells[(cz * g.my + cy) * g.mx + c0]);
        return;
    }
    cols[threadIdx.x] = f.partial();
    __syncthreads();
    const long long ncell = min(g.cells_per_seg, g.mx - c0);
    if (threadIdx.x < ncell) {
        const long long cb = (long long)threadIdx.x * g.px;                      // first column of my cell
        const long long w = min(g.px, (x1 - x0) - cb);                           // ragged last cell of the row
        Partial m = partial_empty();
        for (long long i = 0; i < w; ++i) m = partial_merge(m, cols[cb + i]);
        moments_finalize(m, lines * (unsigned long long)w, flags, &cells[(cz * g.my + cy) * g.mx + c0 + threadIdx.x]);
    }
}

// ------------------------------------------------------------------------------------------------
// 128-bit variant (the default when nx is a multiple of 4, px >= 4 and the cube is 16-byte aligned).  The scalar
// kernel above keeps only 32-64 KiB per SM in flight and is latency-bound at 2.8-4.2 TB/s; here every thread reads one
// float4 of every line with LDG.128, 8 lines in flight (128 B per thread, as in stream_cube), and still keeps ONE
// accumulator set: it owns only the columns of its float4 that lie in the cell of ... its first owned column.  A
// float4 that straddles a cell boundary (px = 30: every 7th or 8th) is read by two threads -- the "main" thread of
// the slot owns the columns before the boundary, an extra "boundary" thread (one per cell boundary of the segment,
// threads 256..) owns the rest (its load is an L1/L2 hit).  Columns a thread does not own are replaced by its
// pivot value (d = 0, no effect on min / max; one FSEL per voxel) and left out of n.
// A CTA covers up to 1024 columns = whole cells, the segment start a multiple of 4 voxels.  Hot / safe paths as in
// MomentsF::batch, one NaN test per group of 8 lines.
// ------------------------------------------------------------------------------------------------
constexpr int kMap4Threads = 256;                 // main threads = float4 slots of a segment
constexpr int kMap4Cols = 4 * kMap4Threads;
constexpr int kMap4MaxThreads = 2 * kMap4Threads; // + boundary threads (px >= 4 => at most 255)

// Cursor over the py x pz lines of a cell row taken as ONE sequence: the pointer steps by a row, and by the rest of
// the plane after the last row of a plane.
struct MapLines {
    const float4* p;
    long long nx4, plane_skip;
    int yy, pyn;
    __device__ __forceinline__ void step() {
        p += nx4;
        if (++yy == pyn) { yy = 0; p += plane_skip; }
    }
    __device__ __forceinline__ void load(float4 (&v)[kMapUnroll]) {
#pragma unroll
        for (int k = 0; k < kMapUnroll; ++k) { v[k] = ld_stream(p); step(); }
    }
};

struct MapV4F : MomentsF<kMomPlain> {
    bool own[4];       // thread constants: which columns of the float4 are mine
    uint32_t nown;     // how many
    __device__ __forceinline__ void line(const float4& v) {   // per-voxel form; a column that is not mine is fed as NaN
        const float qnan = __int_as_float(0x7fc00000);
        const float x[4] = {v.x, v.y, v.z, v.w};
#pragma unroll
        for (int c = 0; c < 4; ++c) { const float xm = own[c] ? x[c] : qnan; take_pivot(xm); core(xm); }
    }
    // repair of a HOT group whose sum came out NaN: reload the lines (L2 hits), add the owned non-NaN voxels.
    // Static, arguments and result by value: the functor itself stays in registers (a member function taking
    // `this` put it on the stack -- 116 M local-memory sectors per pass in a round-1 ncu capture).
    struct GroupFix { double s, q; uint32_t n; };
    static __device__ __noinline__ GroupFix redo_group(MapLines at, double pivot_, uint32_t ownmask) {
        GroupFix f;
        f.s = 0.0; f.q = 0.0; f.n = 0;
#pragma unroll 1
        for (int k = 0; k < kMapUnroll; ++k) {
            const float4 v = __ldcg(at.p);
            at.step();
            const float x[4] = {v.x, v.y, v.z, v.w};
#pragma unroll
            for (int c = 0; c < 4; ++c)
                if (((ownmask >> c) & 1u) && x[c] == x[c]) {
                    const double dl = (double)x[c] - pivot_;
                    f.s += dl; f.q = fma(dl, dl, f.q); f.n += 1;
                }
        }
        return f;
    }
    // HOT mode.  -> true when the group held a NaN (or +Inf and -Inf) in an owned column.
    __device__ __forceinline__ bool hot_group(const float4 (&v)[kMapUnroll], const MapLines& at) {
        double ts[2] = {0.0, 0.0}, tq[2] = {0.0, 0.0};
#pragma unroll
        for (int k = 0; k < kMapUnroll; ++k) {
            const float x0 = own[0] ? v[k].x : pivf, x1 = own[1] ? v[k].y : pivf;
            const float x2 = own[2] ? v[k].z : pivf, x3 = own[3] ? v[k].w : pivf;
            const double d0 = (double)x0 - pivot, d1 = (double)x1 - pivot, d2 = (double)x2 - pivot, d3 = (double)x3 - pivot;
            ts[k & 1] += (d0 + d1) + (d2 + d3);
            tq[k & 1] = fma(d3, d3, fma(d2, d2, fma(d1, d1, fma(d0, d0, tq[k & 1]))));
            mn = fminf(fminf(mn, x0), fminf(x1, fminf(x2, x3)));
            mx = fmaxf(fmaxf(mx, x0), fmaxf(x1, fmaxf(x2, x3)));
        }
        const double tsum = ts[0] + ts[1];
        const bool bad = !(tsum == tsum);
        if (!bad) { s += tsum; q += tq[0] + tq[1]; n += nown * kMapUnroll; }
        else {   // min/max are already in (FMNMX ignores NaN)
            const uint32_t ownmask = (own[0] ? 1u : 0u) | (own[1] ? 2u : 0u) | (own[2] ? 4u : 0u) | (own[3] ? 8u : 0u);
            const GroupFix f = redo_group(at, pivot, ownmask);
            s += f.s; q += f.q; n += f.n;
        }
        return bad;
    }
};

// g.cells_per_seg * g.px is a multiple of 4 and <= kMap4Cols; g.px >= 4; g.nx % 4 == 0; d is 16-byte aligned.
// blockDim.x = kMap4Threads + boundary threads (a multiple of 32, >= cells_per_seg - 1).
__global__ void __launch_bounds__(kMap4MaxThreads, 2)
minimap_v4_kernel(const float* __restrict__ d, MapGeom g, unsigned flags, MomentsOut* __restrict__ cells) {
    __shared__ Partial cols[kMap4MaxThreads];
    const long long b = blockIdx.x;
    const long long seg = b % g.nseg, cy = (b / g.nseg) % g.my, cz = b / (g.nseg * g.my);
    const long long c0 = seg * g.cells_per_seg;
    const long long x0 = c0 * g.px;
    const long long x1 = min((c0 + g.cells_per_seg) * g.px, g.nx);
    const long long y0 = cy * g.py, y1 = min(y0 + g.py, g.ny);
    const long long z0 = cz * g.pz, z1 = min(z0 + g.pz, g.nz);
    const long long width = x1 - x0, nx4 = g.nx >> 2;
    const int px = (int)g.px;

    // role of this thread: float4 slot `slot`, owned columns [lo, hi) of it
    const int tid = threadIdx.x;
    int slot, lo, hi;
    bool active;
    const int nmain = (int)g.main_threads;   // float4 slots of a full segment, rounded up to a warp
    if (tid < nmain) {
        slot = tid; lo = 0;
        const int first = 4 * slot;
        hi = min(4, (first / px + 1) * px - first);                 // up to the end of the first column's cell
        active = first < width;
    } else {
        const int bnd = (tid - nmain + 1) * px;                     // cell boundary (column, relative to the segment)
        slot = bnd >> 2; lo = bnd & 3; hi = 4;
        active = bnd < width && lo != 0;
    }
    MapV4F f;
    f.nown = 0;
#pragma unroll
    for (int c = 0; c < 4; ++c) { f.own[c] = (c >= lo && c < hi); f.nown += f.own[c] ? 1u : 0u; }
    bool safe_mode = true;
    if (active) {
        // the py x pz lines of the cell row as ONE sequence, 8 at a time (only the last group of the whole cell can
        // be short)
        MapLines at;
        at.p = reinterpret_cast<const float4*>(d + ((z0 * g.ny + y0) * g.nx + x0)) + slot;
        at.nx4 = nx4; at.pyn = (int)(y1 - y0); at.yy = 0;
        at.plane_skip = (g.ny - (y1 - y0)) * nx4;
        const long long total = (y1 - y0) * (z1 - z0);
        long long l = 0;
        for (; l + kMapUnroll <= total; l += kMapUnroll) {
            bool nan_seen;
            if (safe_mode) {
                float4 v[kMapUnroll];
                at.load(v);
                const uint32_t n0 = f.n;
#pragma unroll
                for (int k = 0; k < kMapUnroll; ++k) f.line(v[k]);
                nan_seen = f.n - n0 != f.nown * kMapUnroll;
            } else {
                const MapLines start = at;
                float4 v[kMapUnroll];
                at.load(v);
                nan_seen = f.hot_group(v, start);
            }
            safe_mode = __any_sync(__activemask(), nan_seen);
        }
        for (; l < total; ++l) {   // the last (py * pz) mod 8 lines of the cell: per-voxel form
            f.line(ld_stream(at.p));
            at.step();
        }
    }
    cols[tid] = active ? f.partial() : partial_empty();
    __syncthreads();
    const unsigned long long lines = (unsigned long long)((y1 - y0) * (z1 - z0));
    const long long ncell = min(g.cells_per_seg, g.mx - c0);
    if (tid < ncell) {   // merge, in x order: the boundary thread of my left edge, then the main slots that start in my cell
        const long long cb = (long long)tid * g.px;
        const long long w = min(g.px, width - cb);
        Partial m = (tid > 0) ? cols[nmain + tid - 1] : partial_empty();
        const int s0 = (int)((cb + 3) >> 2), s1 = (int)((cb + w - 1) >> 2);
        for (int i = s0; i <= s1; ++i) m = partial_merge(m, cols[i]);
        moments_finalize(m, lines * (unsigned long long)w, flags, &cells[(cz * g.my + cy) * g.mx + c0 + tid]);
    }
}

}  // namespace cube
