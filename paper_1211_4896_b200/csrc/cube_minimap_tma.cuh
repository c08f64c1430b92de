// cube_minimap_tma.cuh -- the statistical mini-map (DESIGN.md sec. 11 NEXT-2) with the lines of
// a cell row staged through a shared-memory ring by TMA bulk copies (cp.async.bulk + mbarrier).
//
// Why a ring here and not in the global passes: a cell row of 30-voxel cells has no 128-bit register tiling that
// respects the cell boundaries (minimap_v4_kernel masks columns, reads straddling float4s twice and spends 16.7
// instructions per voxel).  With the lines in shared memory a thread simply owns ONE COLUMN of the segment -- a
// conflict-free LDS.32 per voxel, one accumulator set, no masks -- and the copy engine keeps ~96 KiB per CTA in
// flight whatever the consumers are doing.
//
// CTA = (segment of whole cells along x, cy, cz), exactly as in minimap_kernel.  Warps 0..W-1 own the columns,
// the last warp is the producer: for every group of kMapUnroll lines it waits for the stage to be released
// (`empty` barrier: one arrival per consumer warp), posts the byte count on the stage's `full` barrier and lets 8
// lanes issue one bulk copy each (a line of the segment is contiguous, 16-byte aligned, a multiple of 16 bytes).
// Consumers wait on `full`, take their column of the 8 lines into registers, release the stage at once and then
// run MapColF::group (the hot / safe paths of the moments pass).  The per-cell merge is the scalar kernel's.
#pragma once
#include "cube_minimap.cuh"

namespace cube {

constexpr int kMapTmaCols = 480;                       // most columns (consumer threads) per segment: 15 warps + producer
constexpr int kMapTmaMaxThreads = kMapTmaCols + 32;    // + the producer warp
constexpr int kMapTmaLine = kMapTmaCols * 4;           // bytes between lines of a stage (compile time: LDS [R + imm])
constexpr int kMapTmaStageLines = 2 * kMapUnroll;      // lines per stage = two MapColF groups per barrier wait
constexpr int kMapTmaStage = kMapTmaStageLines * kMapTmaLine;
constexpr int kMapTmaStages = 3;
constexpr int kMapTmaBarBytes = 128;                   // full[3], empty[3] in front of the ring
constexpr int kMapTmaSmem = kMapTmaBarBytes + kMapTmaStages * kMapTmaStage + kMapTmaCols * 32;   // + column records: 107648 B, 2 CTAs per SM

__device__ __forceinline__ void mbar_init(uint32_t bar, uint32_t count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" :: "r"(bar), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint32_t bar) {
    asm volatile("{\n\t.reg .b64 st;\n\tmbarrier.arrive.shared::cta.b64 st, [%0];\n\t}" :: "r"(bar) : "memory");
}
__device__ __forceinline__ void mbar_arrive_expect_tx(uint32_t bar, uint32_t bytes) {
    asm volatile("{\n\t.reg .b64 st;\n\tmbarrier.arrive.expect_tx.shared::cta.b64 st, [%0], %1;\n\t}"
                 :: "r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint32_t bar, uint32_t parity) {
    uint32_t done;
    do {
        asm volatile("{\n\t.reg .pred p;\n\tmbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2, %3;\n\t"
                     "selp.u32 %0, 1, 0, p;\n\t}" : "=r"(done) : "r"(bar), "r"(parity), "r"(20000u) : "memory");
    } while (!done);
}
// 1-D bulk copy global -> shared, completion counted in bytes on `bar` (TMA without a tensor map).
__device__ __forceinline__ void bulk_load(uint32_t dst, const void* src, uint32_t bytes, uint32_t bar) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                 :: "r"(dst), "l"(src), "r"(bytes), "r"(bar) : "memory");
}


// column value k of the current stage: `base` = shared address of this thread's column in line 0 of the stage
template <int K>
__device__ __forceinline__ float lds_line(uint32_t base) {
    float v;
    asm volatile("ld.shared.f32 %0, [%1+%2];" : "=f"(v) : "r"(base), "n"(K * kMapTmaLine) : "memory");
    return v;
}
template <int K0>
__device__ __forceinline__ void lds_group(uint32_t base, float (&v)[kMapUnroll]) {
    v[0] = lds_line<K0 + 0>(base); v[1] = lds_line<K0 + 1>(base); v[2] = lds_line<K0 + 2>(base); v[3] = lds_line<K0 + 3>(base);
    v[4] = lds_line<K0 + 4>(base); v[5] = lds_line<K0 + 5>(base); v[6] = lds_line<K0 + 6>(base); v[7] = lds_line<K0 + 7>(base);
}

// Per-cell merge of the column records cols[0..w) in x order (one thread per cell): sums about the mean of the
// first non-empty column, plain additions -- a chain of Chan merges would put w fp64 divisions behind one another
// while the other warps of the CTA are already consuming the next cell row.
__device__ __forceinline__ Partial map_merge_columns(const Partial* __restrict__ cols, int w) {
    Partial m = partial_empty();
    bool have = false;
    double P = 0.0;
    for (int i = 0; i < w && !have; ++i)
        if (cols[i].n) { have = true; P = cols[i].mean; }
    if (!have) return m;
#pragma unroll 1
    for (int round = 0; round < 2; ++round) {   // a second round only if the first column was far from the cell's mean
        double cs = 0.0, cq = 0.0;
        unsigned long long cn = 0;
        m.kmin = 0xFFFFFFFFu; m.kmax = 0u;
        for (int i = 0; i < w; ++i) {
            const Partial c = cols[i];
            m.kmin = min(m.kmin, c.kmin);
            m.kmax = max(m.kmax, c.kmax);
            if (c.n) {
                const double nb = (double)c.n, dm = c.mean - P, nd = nb * dm;
                cn += c.n; cs += nd; cq += c.m2 + nd * dm;
            }
        }
        const double nn = (double)cn, shift = cs / nn, m2 = cq - cs * shift;
        m.n = cn; m.mean = P + shift; m.m2 = (m2 < 0.0) ? 0.0 : m2;   // rounding only; a NaN (Inf voxels) stays
        if (!(shift * shift * nn > 256.0 * m.m2 && isfinite(m.mean))) break;   // else q - s^2/n cancelled: refine P
        P = m.mean;
    }
    return m;
}

// barrier among the consumer warps that own columns (the producer warp and idle warps take no part)
__device__ __forceinline__ void map_consumer_sync(int nthreads) {
    asm volatile("bar.sync 1, %0;" :: "r"(nthreads) : "memory");
}

// g.cells_per_seg * g.px is a multiple of 4 and <= kMapTmaCols; g.nx % 4 == 0; d is 16-byte aligned; py * pz < 2^31.
// blockDim.x = 32 * (warps that cover the widest segment + 1); kMapTmaSmem bytes of dynamic shared memory.
// A CTA takes `rows` consecutive cell rows (cy) of one (segment, cz): the producer runs straight on into the next
// cell row while the consumers merge and store the cells of the one they have finished, so the ring is filled and
// drained once per CTA, not once per cell row (16^3 cells: 256 lines per cell row against a ring of 48 lines).
__global__ void __launch_bounds__(kMapTmaMaxThreads, 2)
minimap_tma_kernel(const float* __restrict__ d, MapGeom g, unsigned flags, int rows, MomentsOut* __restrict__ cells) {
    extern __shared__ __align__(128) unsigned char smem[];
    const long long b = blockIdx.x;
    const long long myg = (g.my + rows - 1) / rows;                // groups of cell rows
    const long long seg = b % g.nseg, cyg = (b / g.nseg) % myg, cz = b / (g.nseg * myg);
    const long long c0 = seg * g.cells_per_seg;
    const long long x0 = c0 * g.px;
    const long long x1 = min((c0 + g.cells_per_seg) * g.px, g.nx);
    const long long z0 = cz * g.pz, z1 = min(z0 + g.pz, g.nz);
    const int cy0 = (int)(cyg * rows), cy1 = (int)min((long long)cy0 + rows, g.my);
    const int width = (int)(x1 - x0), nz = (int)(z1 - z0);
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int producer = (int)(blockDim.x >> 5) - 1;               // the last warp
    const int nactive = (width + 31) >> 5;                         // consumer warps that own a column
    const uint32_t full0 = smem_addr(smem), empty0 = full0 + 8u * kMapTmaStages, ring0 = full0 + kMapTmaBarBytes;
    Partial* const cols = reinterpret_cast<Partial*>(smem + kMapTmaBarBytes + kMapTmaStages * kMapTmaStage);

    if (tid == 0) {
#pragma unroll
        for (int s = 0; s < kMapTmaStages; ++s) { mbar_init(full0 + 8u * s, 1u); mbar_init(empty0 + 8u * s, (uint32_t)nactive); }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();

    if (warp == producer) {
        // ---- producer warp: lane k copies line k of every stage; a cell row starts on a fresh stage
        const uint32_t lbytes = (uint32_t)width * 4u;
        const long long plane = g.ny * g.nx;
        int st = 0;
        uint32_t par = 1;   // parity to wait for on `empty`: the first round passes at once
        for (int cy = cy0; cy < cy1; ++cy) {
            const long long y0 = (long long)cy * g.py;
            const int pyn = (int)(min(y0 + g.py, g.ny) - y0);
            const int total = pyn * nz;                            // lines of the cell row, taken as one sequence
            const float* const base = d + ((z0 * g.ny + y0) * g.nx + x0);
            for (int l0 = 0; l0 < total; l0 += kMapTmaStageLines) {
                mbar_wait(empty0 + 8u * st, par);
                const int cnt = min(kMapTmaStageLines, total - l0);
                if (lane == 0) mbar_arrive_expect_tx(full0 + 8u * st, lbytes * (uint32_t)cnt);
                __syncwarp();
                if (lane < cnt) {
                    const int l = l0 + lane;
                    const int zz = l / pyn, yy = l - zz * pyn;
                    bulk_load(ring0 + (uint32_t)(st * kMapTmaStage + lane * kMapTmaLine), base + zz * plane + yy * g.nx,
                              lbytes, full0 + 8u * st);
                }
                if (++st == kMapTmaStages) { st = 0; par ^= 1u; }
            }
        }
    } else if (warp < nactive) {
        // ---- consumers: thread t owns column x0 + t (warps beyond the segment's width have nothing to do)
        const bool active = tid < width;
        int st = 0;
        uint32_t par = 0;
        const uint32_t mycol = ring0 + 4u * (uint32_t)tid;
#pragma unroll 1
        for (int cy = cy0; cy < cy1; ++cy) {
            const long long y0 = (long long)cy * g.py;
            const int total = (int)(min(y0 + g.py, g.ny) - y0) * nz;
            MapColF f;
            bool safe_mode = true;
            for (int l0 = 0; l0 < total; l0 += kMapTmaStageLines) {
                const uint32_t col = mycol + (uint32_t)(st * kMapTmaStage);
                mbar_wait(full0 + 8u * st, par);
                const int cnt = total - l0;
                if (cnt >= kMapTmaStageLines) {
                    float v0[kMapUnroll], v1[kMapUnroll];
                    lds_group<0>(col, v0);
                    lds_group<kMapUnroll>(col, v1);
                    __syncwarp();
                    if (lane == 0) mbar_arrive(empty0 + 8u * st);  // values are in registers: release the stage
                    if (active) { f.group(v0, safe_mode); f.group(v1, safe_mode); }
                } else {                                           // the last (py * pz) mod 16 lines of the cell row
                    if (active)
                        for (int k = 0; k < cnt; ++k) {
                            float x;
                            asm volatile("ld.shared.f32 %0, [%1];" : "=f"(x) : "r"(col + (uint32_t)(k * kMapTmaLine)) : "memory");
                            f(x);
                        }
                    __syncwarp();
                    if (lane == 0) mbar_arrive(empty0 + 8u * st);
                }
                if (++st == kMapTmaStages) { st = 0; par ^= 1u; }
            }
            map_consumer_sync(nactive * 32);   // the cells of the cell row before this one have been merged and stored
            if (active) cols[tid] = f.partial();
            map_consumer_sync(nactive * 32);
            if (tid < (int)min(g.cells_per_seg, g.mx - c0)) {
                const int cb = tid * (int)g.px;
                const int w = min((int)g.px, width - cb);          // ragged last cell of the row
                const Partial m = map_merge_columns(cols + cb, w);
                moments_finalize(m, (unsigned long long)total * (unsigned long long)w, flags,
                                 &cells[(cz * g.my + cy) * g.mx + c0 + tid]);
            }
        }
    }
}

}  // namespace cube
