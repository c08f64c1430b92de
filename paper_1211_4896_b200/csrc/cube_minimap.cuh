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
// because a column never leaves its cell.  kMapUnroll lines are loaded before the first is used.  The columns of
// a cell are then merged in x order by one thread per cell (Chan's pairwise update; fixed order => deterministic)
// and the finished record goes straight to the output.  Cells wider than kMapThreads voxels get a CTA of their
// own whose threads stride over the columns and merge through the block tree.
#pragma once
#include "cube_kernels.cuh"

namespace cube {

constexpr int kMapThreads = 512;
constexpr int kMapUnroll = 16;

struct MapGeom {
    long long nx, ny, nz, px, py, pz, mx, my, mz;
    long long cells_per_seg;   // whole cells per CTA along x (1 when px > kMapThreads)
    long long nseg;            // segments per cell row
};

__device__ __forceinline__ float ld_stream1(const float* p) {
    float r;
    asm volatile("ld.global.nc.L1::no_allocate.f32 %0, [%1];" : "=f"(r) : "l"(p));
    return r;
}

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

    MomentsF<kMomPlain> f;
    const float qnan = __int_as_float(0x7fc00000);
    for (long long x = x0 + threadIdx.x; x < x1; x += kMapThreads) {
        for (long long z = z0; z < z1; ++z) {
            const float* __restrict__ p = d + ((z * g.ny + y0) * g.nx + x);
            for (long long y = y0; y < y1; y += kMapUnroll) {
                float v[kMapUnroll];
#pragma unroll
                for (int k = 0; k < kMapUnroll; ++k)   // lines past the cell are fed as NaN: they count nowhere
                    v[k] = (y + k < y1) ? ld_stream1(p + (long long)k * g.nx) : qnan;
                if (!f.have) {
#pragma unroll
                    for (int k = 0; k < kMapUnroll; ++k) f.take_pivot(v[k]);
                }
#pragma unroll
                for (int k = 0; k < kMapUnroll; ++k) f.core(v[k]);
                p += (long long)kMapUnroll * g.nx;
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

}  // namespace cube
