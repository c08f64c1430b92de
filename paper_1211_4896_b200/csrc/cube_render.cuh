// cube_render.cuh -- NEXT-4: the paper's volume ray casting and 3-D spectrum tool as CUDA compute
// kernels writing into headless device buffers (no graphics API, no window).
//
//   maximum intensity projection       PAPER.md:166-172  "only the value of the maximum voxel through each cast ray"
//   generic transfer function          PAPER.md:174-180  "The data values' range is partitioned into discrete levels.
//                                      Each data level is assigned a colour and opacity value", ordered compositing
//   sigma-clipping transfer function   PAPER.md:352-358, Fig. 7, Fig. 9: the generic one applied to (sample - local
//                                      mean) / local std, "two trilinear interpolation operations" per sample
//   3-D spectrum tool                  PAPER.md:298-306, Fig. 6: the profile along an arbitrary line of sight, "a
//                                      constant sampling step ... trilinear interpolation"
//
// The paper keeps the cube in 3-D texture memory; texture filtering interpolates with 9-bit fixed-point
// weights, which no CPU restatement can match bit for bit, and a 64 GiB cube would have to be copied into a CUDA
// array first.  Here the cube stays the caller's plain float32 array, read through the read-only L1 path (LDG.NC).
// Two families of kernels, chosen per view by the host (csrc/cube.cu, render_along): one ray per THREAD -- the 32 rays
// of a warp are a compact block of the image, so their eight-voxel neighbourhoods overlap and most loads hit L1/L2 --
// and one ray per WARP with the lanes on consecutive samples, for rays that run along the cube's x axis, where
// neighbouring samples are neighbouring voxels of a line.  Both give the same images bit for bit.
// Every floating-point operation is an explicitly rounded float32 operation (__fadd_rn / __fmul_rn / __fsub_rn, never
// contracted), in the order DESIGN.md R27-R31 state, so the images equal the oracle's bit for bit.
#pragma once
#include <math.h>

#include "cube_common.cuh"

namespace cube {

struct RenderView {          // == cube_view_t (include/cube.h)
    float origin[3], du[3], dv[3], step[3];
    int32_t width, height, nsteps;
};

struct RenderGeom {
    long long nx, ny, nz;
    float xmax, ymax, zmax;  // (float)(n - 1)
};

struct RayF {
    float o[3];
    int i0, i1;              // samples outside [i0, i1] are certainly outside the cube (conservative clip)
};

// First sample of pixel (u, v) (R27) and the conservative range of samples that can be inside the cube: the exact
// inside test below is still made on every sample of that range, so clipping changes no result -- it only skips the
// empty space between the bounding sphere the rays start on and the cube.
__device__ __forceinline__ RayF ray_setup(const RenderView& vw, const RenderGeom& g, int u, int v) {
    RayF r;
#pragma unroll
    for (int c = 0; c < 3; ++c)
        r.o[c] = __fadd_rn(__fadd_rn(vw.origin[c], __fmul_rn((float)u, vw.du[c])), __fmul_rn((float)v, vw.dv[c]));
    const double hi[3] = {(double)g.xmax, (double)g.ymax, (double)g.zmax};
    double enter = 0.0, exit_ = (double)(vw.nsteps - 1);
    bool empty = false;
#pragma unroll
    for (int c = 0; c < 3; ++c) {
        const double o = (double)r.o[c], s = (double)vw.step[c];
        // float32 evaluation of o + i * s is within `err` of the exact value for every sample of the ray
        const double err = 1e-6 * (fabs(o) + (double)vw.nsteps * fabs(s) + 1.0);
        if (s == 0.0) {
            if (o < -err || o > hi[c] + err) empty = true;
        } else {
            const double t0 = (-err - o) / s, t1 = (hi[c] + err - o) / s;
            enter = fmax(enter, fmin(t0, t1) - 2.0);
            exit_ = fmin(exit_, fmax(t0, t1) + 2.0);
        }
    }
    if (empty || !(enter <= exit_)) { r.i0 = 0; r.i1 = -1; return r; }
    r.i0 = (int)fmax(0.0, floor(enter));
    r.i1 = (int)fmin((double)(vw.nsteps - 1), ceil(exit_));
    return r;
}

// Sample i of the ray (R27): p = o + (float)i * step.
__device__ __forceinline__ void ray_point(const RenderView& vw, const float (&o)[3], int i, float (&p)[3]) {
    const float fi = (float)i;
#pragma unroll
    for (int c = 0; c < 3; ++c) p[c] = __fadd_rn(o[c], __fmul_rn(fi, vw.step[c]));
}

__device__ __forceinline__ float lerp_rn(float a, float b, float f) { return __fadd_rn(a, __fmul_rn(f, __fsub_rn(b, a))); }

// Trilinear sample at the data point p (R28).  false: outside the cube.
__device__ __forceinline__ bool sample_at(const float* __restrict__ d, const RenderGeom& g, const float (&pt)[3], float& out) {
    const float px = pt[0], py = pt[1], pz = pt[2];
    if (!(px >= 0.0f && px <= g.xmax && py >= 0.0f && py <= g.ymax && pz >= 0.0f && pz <= g.zmax)) return false;
    const float flx = floorf(px), fly = floorf(py), flz = floorf(pz);
    const float fx = __fsub_rn(px, flx), fy = __fsub_rn(py, fly), fz = __fsub_rn(pz, flz);
    const long long x0 = (long long)flx, y0 = (long long)fly, z0 = (long long)flz;
    // a neighbour of weight zero does not take part (R28): its offset is 0 then
    const long long dx = fx > 0.0f ? 1 : 0, dy = fy > 0.0f ? g.nx : 0, dz = fz > 0.0f ? g.nx * g.ny : 0;
    const float* __restrict__ p = d + ((z0 * g.ny + y0) * g.nx + x0);
    const float v000 = __ldg(p), v100 = __ldg(p + dx), v010 = __ldg(p + dy), v110 = __ldg(p + dy + dx);
    const float v001 = __ldg(p + dz), v101 = __ldg(p + dz + dx), v011 = __ldg(p + dz + dy), v111 = __ldg(p + dz + dy + dx);
    const float c00 = lerp_rn(v000, v100, fx), c10 = lerp_rn(v010, v110, fx);
    const float c01 = lerp_rn(v001, v101, fx), c11 = lerp_rn(v011, v111, fx);
    out = lerp_rn(lerp_rn(c00, c10, fy), lerp_rn(c01, c11, fy), fz);
    return true;
}

__device__ __forceinline__ bool ray_sample(const float* __restrict__ d, const RenderGeom& g, const RenderView& vw,
                                           const float (&o)[3], int i, float& out) {
    float p[3];
    ray_point(vw, o, i, p);
    return sample_at(d, g, p, out);
}

// The same sample in two halves, so that the loads of several samples of a ray are in flight together (the march is
// a chain of dependent L1 / L2 / HBM round trips otherwise: ncu showed 14 % of the issue slots used and 35 stalled
// warps per issued instruction): tap_load issues the eight loads -- for a sample outside the cube from voxel 0, so
// that they need no branch --, tap_value interpolates.  Same operations, same order, same bits as sample_at.
// Samples of a ray fetched before the first is consumed.  MIP: 1 (the branch-free loads alone took c2 at yaw 30 deg
// from 9.6 to 7.7 ms; larger groups cost occupancy and gain nothing: a sample is consumed by one compare).  Transfer
// functions: 6 (each sample ends in a dependent table load and five dependent float operations: 8.0 -> 5.2 ms at
// 128 registers per thread).
#ifndef CUBE_RENDER_GROUP_MIP
#define CUBE_RENDER_GROUP_MIP 1
#endif
#ifndef CUBE_RENDER_GROUP_TF
#define CUBE_RENDER_GROUP_TF 6
#endif

struct Tap {
    float v[8];
    float fx, fy, fz;
    bool in;
};

__device__ __forceinline__ void tap_load(const float* __restrict__ d, const RenderGeom& g, const float (&pt)[3], bool wanted, Tap& t) {
    t.in = wanted && pt[0] >= 0.0f && pt[0] <= g.xmax && pt[1] >= 0.0f && pt[1] <= g.ymax && pt[2] >= 0.0f && pt[2] <= g.zmax;
    const float px = t.in ? pt[0] : 0.0f, py = t.in ? pt[1] : 0.0f, pz = t.in ? pt[2] : 0.0f;
    const float flx = floorf(px), fly = floorf(py), flz = floorf(pz);
    t.fx = __fsub_rn(px, flx); t.fy = __fsub_rn(py, fly); t.fz = __fsub_rn(pz, flz);
    const long long x0 = (long long)flx, y0 = (long long)fly, z0 = (long long)flz;
    const long long dx = t.fx > 0.0f ? 1 : 0, dy = t.fy > 0.0f ? g.nx : 0, dz = t.fz > 0.0f ? g.nx * g.ny : 0;
    const float* __restrict__ p = d + ((z0 * g.ny + y0) * g.nx + x0);
    t.v[0] = __ldg(p); t.v[1] = __ldg(p + dx); t.v[2] = __ldg(p + dy); t.v[3] = __ldg(p + dy + dx);
    t.v[4] = __ldg(p + dz); t.v[5] = __ldg(p + dz + dx); t.v[6] = __ldg(p + dz + dy); t.v[7] = __ldg(p + dz + dy + dx);
}

__device__ __forceinline__ float tap_value(const Tap& t) {
    const float c00 = lerp_rn(t.v[0], t.v[1], t.fx), c10 = lerp_rn(t.v[2], t.v[3], t.fx);
    const float c01 = lerp_rn(t.v[4], t.v[5], t.fx), c11 = lerp_rn(t.v[6], t.v[7], t.fx);
    return lerp_rn(lerp_rn(c00, c10, t.fy), lerp_rn(c01, c11, t.fy), t.fz);
}

// The statistical mini-map as the second lookup of the sigma-clipping transfer function (R34): cell
// (cx, cy, cz) sits at the centre of its nominal block, data coordinate cx * px + (px - 1) / 2.
struct MapLookupGeom {
    long long mx, my, mz;
    float part[3], off[3], top[3];       // (float)px ..., (px - 1) / 2 ..., (float)(mx - 1) ...
};

// map: (mean, std) of every cell rounded to float32 -- what R34 interpolates --, written by map_compact_kernel from the
// records of cube_minimap before the rays are cast (8 bytes per cell instead of two doubles in a 40-byte record: 8
// loads per lookup instead of 16 loads and 16 conversions).
__global__ void __launch_bounds__(256)
map_compact_kernel(const double* __restrict__ cells, long long ncell, float2* __restrict__ map) {
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i < ncell) map[i] = make_float2((float)cells[i * 5 + 3], (float)cells[i * 5 + 4]);   // record: count, nan_count, min|max, mean, std
}

__device__ __forceinline__ void map_lookup(const float2* __restrict__ map, const MapLookupGeom& m, const float (&pt)[3],
                                           float& mean, float& sd) {
    long long i0[3], st[3];
    float f[3];
    const long long stride[3] = {1, m.mx, m.mx * m.my};
#pragma unroll
    for (int c = 0; c < 3; ++c) {
        float q = __fdiv_rn(__fsub_rn(pt[c], m.off[c]), m.part[c]);
        if (!(q >= 0.0f)) q = 0.0f;
        if (q > m.top[c]) q = m.top[c];
        const float fl = floorf(q);
        i0[c] = (long long)fl;
        f[c] = __fsub_rn(q, fl);
        st[c] = f[c] > 0.0f ? stride[c] : 0;
    }
    const float2* __restrict__ p = map + ((i0[2] * m.my + i0[1]) * m.mx + i0[0]);
    const float2 v000 = __ldg(p), v100 = __ldg(p + st[0]), v010 = __ldg(p + st[1]), v110 = __ldg(p + st[1] + st[0]);
    const float2 v001 = __ldg(p + st[2]), v101 = __ldg(p + st[2] + st[0]), v011 = __ldg(p + st[2] + st[1]),
                 v111 = __ldg(p + st[2] + st[1] + st[0]);
    {
        const float c00 = lerp_rn(v000.x, v100.x, f[0]), c10 = lerp_rn(v010.x, v110.x, f[0]);
        const float c01 = lerp_rn(v001.x, v101.x, f[0]), c11 = lerp_rn(v011.x, v111.x, f[0]);
        mean = lerp_rn(lerp_rn(c00, c10, f[1]), lerp_rn(c01, c11, f[1]), f[2]);
    }
    {
        const float c00 = lerp_rn(v000.y, v100.y, f[0]), c10 = lerp_rn(v010.y, v110.y, f[0]);
        const float c01 = lerp_rn(v001.y, v101.y, f[0]), c11 = lerp_rn(v011.y, v111.y, f[0]);
        sd = lerp_rn(lerp_rn(c00, c10, f[1]), lerp_rn(c01, c11, f[1]), f[2]);
    }
}

constexpr int kRenderTileU = 32, kRenderTileV = 8;

// Pixel of a thread in the CTA's tile of 32 x 8 pixels.  A warp's 32 pixels form a block of 2^fw_log x 2^(5 - fw_log):
// 16 x 2 when the image rows run nearly along the cube's x axis (the lanes then read neighbouring voxels), 8 x 4 for
// oblique views -- the rays of a compact block stay close together in y and z as well, so a warp's loads touch fewer
// planes and lines of the cube than those of 32 pixels in a row (c2, yaw 45 pitch 20: MIP 10.3 -> 7.2 ms).  The host
// chooses (csrc/cube.cu, render_footprint).
__device__ __forceinline__ void render_pixel(int fw_log, int& u, int& v) {
    const int lane = threadIdx.x, warp = threadIdx.y;            // blockDim = (32, 8)
    const int across_log = 5 - fw_log;                            // blocks across the tile: 2^across_log
    u = blockIdx.x * kRenderTileU + ((warp & ((1 << across_log) - 1)) << fw_log) + (lane & ((1 << fw_log) - 1));
    v = blockIdx.y * kRenderTileV + ((warp >> across_log) << across_log) + (lane >> fw_log);
}   // a warp = 32 neighbouring pixels of one image row

// MIP (R29): the largest sample >= vmin in march order; NaN when the ray has none.
__global__ void __launch_bounds__(kRenderTileU * kRenderTileV)
render_mip_kernel(const float* __restrict__ d, RenderGeom g, RenderView vw, float vmin, int fw_log, float* __restrict__ image) {
    int u, v;
    render_pixel(fw_log, u, v);
    if (u >= vw.width || v >= vw.height) return;
    const RayF r = ray_setup(vw, g, u, v);
    float m = 0.0f;
    bool have = false;
#pragma unroll 1
    for (int i = r.i0; i <= r.i1; i += CUBE_RENDER_GROUP_MIP) {
        Tap t[CUBE_RENDER_GROUP_MIP];
#pragma unroll
        for (int j = 0; j < CUBE_RENDER_GROUP_MIP; ++j) {
            float p[3];
            ray_point(vw, r.o, i + j, p);
            tap_load(d, g, p, i + j <= r.i1, t[j]);
        }
#pragma unroll
        for (int j = 0; j < CUBE_RENDER_GROUP_MIP; ++j) {
            const float s = tap_value(t[j]);
            if (t[j].in && s >= vmin && (!have || s > m)) { m = s; have = true; }   // NULL samples fail the comparison
        }
    }
    image[(size_t)v * vw.width + u] = have ? m : __int_as_float(0x7fc00000);
}

// MIP for views whose rays run along the cube's x axis (an orbit camera towards yaw 90 / 270 degrees): there the 32 rays
// of a ray-per-thread warp read up to 32 different planes per load (32 sectors per request, none shared), so a warp
// takes ONE ray instead and its lanes consecutive samples -- the eight loads of a warp then cover
// neighbouring voxels of the same lines.  The maximum does not depend on the order of the samples, except between
// equal maxima (-0.0 and +0.0 compare equal): the sequential march keeps the first, so lanes and the reduction carry
// the sample index and a tie goes to the smaller one -- the images stay bit-identical to render_mip_kernel's.
constexpr int kRenderRaysPerCta = 8;

// The ray of a warp: the CTA's kRenderRaysPerCta = 8 rays are a block of 2^rw_log x 2^(3 - rw_log) pixels (blockIdx.x
// runs over the blocks row by row).
__device__ __forceinline__ bool render_ray_of_warp(const RenderView& vw, int rw_log, int& u, int& v) {
    const int warp = threadIdx.x >> 5;
    const unsigned across = ((unsigned)vw.width + (1u << rw_log) - 1u) >> rw_log;     // blocks per row of blocks
    u = (int)((blockIdx.x % across) << rw_log) + (warp & ((1 << rw_log) - 1));
    v = (int)((blockIdx.x / across) << (3 - rw_log)) + (warp >> rw_log);
    return u < vw.width && v < vw.height;
}

__global__ void __launch_bounds__(32 * kRenderRaysPerCta)
render_mip_along_kernel(const float* __restrict__ d, RenderGeom g, RenderView vw, float vmin, int rw_log, float* __restrict__ image) {
    const int lane = threadIdx.x & 31;
    int u, v;
    if (!render_ray_of_warp(vw, rw_log, u, v)) return;                   // warp-uniform
    const long long pix = (long long)v * vw.width + u;
    const RayF r = ray_setup(vw, g, u, v);
    float m = 0.0f;
    int mi = 0x7fffffff;
    bool have = false;
#pragma unroll 1
    for (int i = r.i0 + lane; i <= r.i1; i += 64) {                      // two samples per lane in flight
        Tap t[2];
#pragma unroll
        for (int j = 0; j < 2; ++j) {
            float p[3];
            ray_point(vw, r.o, i + 32 * j, p);
            tap_load(d, g, p, i + 32 * j <= r.i1, t[j]);
        }
#pragma unroll
        for (int j = 0; j < 2; ++j) {
            const float s = tap_value(t[j]);
            if (t[j].in && s >= vmin && (!have || s > m)) { m = s; mi = i + 32 * j; have = true; }
        }
    }
#pragma unroll
    for (int off = 16; off >= 1; off >>= 1) {
        const float om = __shfl_xor_sync(0xffffffffu, m, off);
        const int oi = __shfl_xor_sync(0xffffffffu, mi, off);
        const bool oh = __shfl_xor_sync(0xffffffffu, have ? 1 : 0, off) != 0;
        if (oh && (!have || om > m || (om == m && oi < mi))) { m = om; mi = oi; have = true; }
    }
    if (lane == 0) image[pix] = have ? m : __int_as_float(0x7fc00000);
}

// Generic transfer function (R30, R31): level of the sample by the histogram's bin formula, front-to-back compositing
//   w = (1 - A) * a;  C = C + w * c;  A = A + w;  stop when A >= opacity_cut.
// table: nlevels x (r, g, b, opacity), device memory.
// SIGMA: the sigma-clipping transfer function (R34) -- the looked-up value is the sample's distance
// from the LOCAL mean in units of the LOCAL standard deviation, both interpolated in the mini-map; `lo` is then the
// clipping threshold ("3 sigma").  Samples where the map has no statistics (std not > 0, NaN) are skipped.
template <bool SIGMA>
__global__ void __launch_bounds__(kRenderTileU * kRenderTileV)
render_tf_kernel(const float* __restrict__ d, RenderGeom g, RenderView vw, int nlevels, float lo, float scale,
                 const float4* __restrict__ table, float opacity_cut, const float2* __restrict__ cells, MapLookupGeom mg,
                 int fw_log, float4* __restrict__ rgba) {
    int u, v;
    render_pixel(fw_log, u, v);
    if (u >= vw.width || v >= vw.height) return;
    const RayF r = ray_setup(vw, g, u, v);
    float cr = 0.0f, cg = 0.0f, cb = 0.0f, A = 0.0f;
    const float top = (float)(nlevels - 1);
    bool done = false;
#pragma unroll 1
    for (int i0 = r.i0; i0 <= r.i1 && !done; i0 += CUBE_RENDER_GROUP_TF) {
      Tap t[CUBE_RENDER_GROUP_TF];
      float pts[CUBE_RENDER_GROUP_TF][3];
#pragma unroll
      for (int j = 0; j < CUBE_RENDER_GROUP_TF; ++j) {
          ray_point(vw, r.o, i0 + j, pts[j]);
          tap_load(d, g, pts[j], i0 + j <= r.i1, t[j]);
      }
#pragma unroll
      for (int j = 0; j < CUBE_RENDER_GROUP_TF; ++j) {
        if (done || !t[j].in) continue;
        float s = tap_value(t[j]);
        const float (&p)[3] = pts[j];
        if (SIGMA) {
            if (s != s) continue;            // NULL sample: no need to look at the map
            float mean, sd;
            map_lookup(cells, mg, p, mean, sd);
            if (!(sd > 0.0f)) continue;
            s = __fdiv_rn(__fsub_rn(s, mean), sd);
        }
        if (!(s >= lo)) continue;            // below the range (the global threshold) or NULL
        const float fl = floorf(__fmul_rn(__fsub_rn(s, lo), scale));
        const int L = (fl >= top) ? nlevels - 1 : (int)fl;
        const float4 e = __ldg(table + L);
        const float w = __fmul_rn(__fsub_rn(1.0f, A), e.w);
        cr = __fadd_rn(cr, __fmul_rn(w, e.x));
        cg = __fadd_rn(cg, __fmul_rn(w, e.y));
        cb = __fadd_rn(cb, __fmul_rn(w, e.z));
        A = __fadd_rn(A, w);
        if (A >= opacity_cut) done = true;
      }
    }
    rgba[(size_t)v * vw.width + u] = make_float4(cr, cg, cb, A);
}

// The transfer functions with one ray per warp (see render_mip_along_kernel for when).  Compositing is ordered, so
// only the part of a sample that does not depend on the samples before it is done by its lane -- the trilinear value,
// the mini-map lookup, the level, the table entry --; the recurrence itself is then run by the whole warp, uniformly,
// over the lanes whose sample contributes, in march order (ballot + shuffles): the same float32 operations in the same
// order as the sequential march, hence the same bits.  A transfer function skips what lies below its threshold --
// nearly every sample of a noise-dominated cube -- so that loop is short.
template <bool SIGMA>
__global__ void __launch_bounds__(32 * kRenderRaysPerCta)
render_tf_along_kernel(const float* __restrict__ d, RenderGeom g, RenderView vw, int nlevels, float lo, float scale,
                       const float4* __restrict__ table, float opacity_cut, const float2* __restrict__ cells,
                       MapLookupGeom mg, int rw_log, float4* __restrict__ rgba) {
    const int lane = threadIdx.x & 31;
    int u, v;
    if (!render_ray_of_warp(vw, rw_log, u, v)) return;                   // warp-uniform
    const long long pix = (long long)v * vw.width + u;
    const RayF r = ray_setup(vw, g, u, v);
    float cr = 0.0f, cg = 0.0f, cb = 0.0f, A = 0.0f;
    const float top = (float)(nlevels - 1);
    bool done = false;
#pragma unroll 1
    for (int i0 = r.i0; i0 <= r.i1 && !done; i0 += 64) {                 // two samples per lane in flight
        Tap t[2];
        float pts[2][3];
#pragma unroll
        for (int j = 0; j < 2; ++j) {
            ray_point(vw, r.o, i0 + 32 * j + lane, pts[j]);
            tap_load(d, g, pts[j], i0 + 32 * j + lane <= r.i1, t[j]);
        }
#pragma unroll
        for (int j = 0; j < 2; ++j) {
            float s = tap_value(t[j]);
            bool c = t[j].in;
            if (SIGMA && c) {
                c = s == s;                                              // NULL sample: no need to look at the map
                if (c) {
                    float mean, sd;
                    map_lookup(cells, mg, pts[j], mean, sd);
                    c = sd > 0.0f;
                    if (c) s = __fdiv_rn(__fsub_rn(s, mean), sd);
                }
            }
            c = c && s >= lo;                                            // below the range (the threshold) or NULL
            float4 e = make_float4(0.0f, 0.0f, 0.0f, 0.0f);
            if (c) {
                const float fl = floorf(__fmul_rn(__fsub_rn(s, lo), scale));
                e = __ldg(table + ((fl >= top) ? nlevels - 1 : (int)fl));
            }
            unsigned mask = done ? 0u : __ballot_sync(0xffffffffu, c);   // done is warp-uniform
            while (mask) {
                const int src = __ffs(mask) - 1;
                mask &= mask - 1;
                const float ex = __shfl_sync(0xffffffffu, e.x, src), ey = __shfl_sync(0xffffffffu, e.y, src);
                const float ez = __shfl_sync(0xffffffffu, e.z, src), ew = __shfl_sync(0xffffffffu, e.w, src);
                const float w = __fmul_rn(__fsub_rn(1.0f, A), ew);
                cr = __fadd_rn(cr, __fmul_rn(w, ex));
                cg = __fadd_rn(cg, __fmul_rn(w, ey));
                cb = __fadd_rn(cb, __fmul_rn(w, ez));
                A = __fadd_rn(A, w);
                if (A >= opacity_cut) { done = true; break; }
            }
        }
    }
    if (lane == 0) rgba[pix] = make_float4(cr, cg, cb, A);
}

// 3-D spectrum tool: sample i of pixel (u, v)'s ray, NaN outside the cube; one thread per sample.
__global__ void __launch_bounds__(256)
spectrum_kernel(const float* __restrict__ d, RenderGeom g, RenderView vw, int u, int v, float* __restrict__ out) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= vw.nsteps) return;
    float o[3];
#pragma unroll
    for (int c = 0; c < 3; ++c)
        o[c] = __fadd_rn(__fadd_rn(vw.origin[c], __fmul_rn((float)u, vw.du[c])), __fmul_rn((float)v, vw.dv[c]));
    float s;
    out[i] = ray_sample(d, g, vw, o, i, s) ? s : __int_as_float(0x7fc00000);
}

}  // namespace cube
