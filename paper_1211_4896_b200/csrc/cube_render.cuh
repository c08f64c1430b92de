// cube_render.cuh -- NEXT-4: the paper's volume ray casting and 3-D spectrum tool as CUDA compute
// kernels writing into headless device buffers (no graphics API, no window).
//
//   maximum intensity projection       PAPER.md:166-172  "only the value of the maximum voxel through each cast ray"
//   generic transfer function          PAPER.md:174-180  "The data values' range is partitioned into discrete levels.
//                                      Each data level is assigned a colour and opacity value", ordered compositing
//   3-D spectrum tool                  PAPER.md:298-306, Fig. 6: the profile along an arbitrary line of sight, "a
//                                      constant sampling step ... trilinear interpolation"
//
// The paper keeps the cube in 3-D texture memory; texture filtering interpolates with 9-bit fixed-point
// weights, which no CPU restatement can match bit for bit, and a 64 GiB cube would have to be copied into a CUDA
// array first.  Here the cube stays the caller's plain float32 array, read through the read-only L1 path (LDG.NC): the
// 32 rays of a warp are neighbours in the image, so their eight-voxel neighbourhoods overlap and most loads hit L1/L2.
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

// Trilinear sample at sample i of the ray (R28).  false: outside the cube.
__device__ __forceinline__ bool ray_sample(const float* __restrict__ d, const RenderGeom& g, const RenderView& vw,
                                           const float (&o)[3], int i, float& out) {
    const float fi = (float)i;
    const float px = __fadd_rn(o[0], __fmul_rn(fi, vw.step[0]));
    const float py = __fadd_rn(o[1], __fmul_rn(fi, vw.step[1]));
    const float pz = __fadd_rn(o[2], __fmul_rn(fi, vw.step[2]));
    if (!(px >= 0.0f && px <= g.xmax && py >= 0.0f && py <= g.ymax && pz >= 0.0f && pz <= g.zmax)) return false;
    const float flx = floorf(px), fly = floorf(py), flz = floorf(pz);
    const float fx = __fsub_rn(px, flx), fy = __fsub_rn(py, fly), fz = __fsub_rn(pz, flz);
    const long long x0 = (long long)flx, y0 = (long long)fly, z0 = (long long)flz;
    // a neighbour of weight zero does not take part (R28): its offset is 0 then
    const long long dx = fx > 0.0f ? 1 : 0, dy = fy > 0.0f ? g.nx : 0, dz = fz > 0.0f ? g.nx * g.ny : 0;
    const float* __restrict__ p = d + ((z0 * g.ny + y0) * g.nx + x0);
    const float v000 = __ldg(p), v100 = __ldg(p + dx), v010 = __ldg(p + dy), v110 = __ldg(p + dy + dx);
    const float v001 = __ldg(p + dz), v101 = __ldg(p + dz + dx), v011 = __ldg(p + dz + dy), v111 = __ldg(p + dz + dy + dx);
    auto lerp = [](float a, float b, float f) { return __fadd_rn(a, __fmul_rn(f, __fsub_rn(b, a))); };
    const float c00 = lerp(v000, v100, fx), c10 = lerp(v010, v110, fx);
    const float c01 = lerp(v001, v101, fx), c11 = lerp(v011, v111, fx);
    out = lerp(lerp(c00, c10, fy), lerp(c01, c11, fy), fz);
    return true;
}

constexpr int kRenderTileU = 32, kRenderTileV = 8;   // a warp = 32 neighbouring pixels of one image row

// MIP (R29): the largest sample >= vmin in march order; NaN when the ray has none.
__global__ void __launch_bounds__(kRenderTileU * kRenderTileV)
render_mip_kernel(const float* __restrict__ d, RenderGeom g, RenderView vw, float vmin, float* __restrict__ image) {
    const int u = blockIdx.x * kRenderTileU + threadIdx.x, v = blockIdx.y * kRenderTileV + threadIdx.y;
    if (u >= vw.width || v >= vw.height) return;
    const RayF r = ray_setup(vw, g, u, v);
    float m = 0.0f;
    bool have = false;
#pragma unroll 4
    for (int i = r.i0; i <= r.i1; ++i) {
        float s;
        if (!ray_sample(d, g, vw, r.o, i, s)) continue;
        if (!(s >= vmin)) continue;          // NULL samples fail the comparison
        if (!have || s > m) { m = s; have = true; }
    }
    image[(size_t)v * vw.width + u] = have ? m : __int_as_float(0x7fc00000);
}

// Generic transfer function (R30, R31): level of the sample by the histogram's bin formula, front-to-back compositing
//   w = (1 - A) * a;  C = C + w * c;  A = A + w;  stop when A >= opacity_cut.
// table: nlevels x (r, g, b, opacity), device memory.
__global__ void __launch_bounds__(kRenderTileU * kRenderTileV)
render_tf_kernel(const float* __restrict__ d, RenderGeom g, RenderView vw, int nlevels, float lo, float scale,
                 const float4* __restrict__ table, float opacity_cut, float4* __restrict__ rgba) {
    const int u = blockIdx.x * kRenderTileU + threadIdx.x, v = blockIdx.y * kRenderTileV + threadIdx.y;
    if (u >= vw.width || v >= vw.height) return;
    const RayF r = ray_setup(vw, g, u, v);
    float cr = 0.0f, cg = 0.0f, cb = 0.0f, A = 0.0f;
    const float top = (float)(nlevels - 1);
    for (int i = r.i0; i <= r.i1; ++i) {
        float s;
        if (!ray_sample(d, g, vw, r.o, i, s)) continue;
        if (!(s >= lo)) continue;            // below the range (the global threshold) or NULL
        const float fl = floorf(__fmul_rn(__fsub_rn(s, lo), scale));
        const int L = (fl >= top) ? nlevels - 1 : (int)fl;
        const float4 e = __ldg(table + L);
        const float w = __fmul_rn(__fsub_rn(1.0f, A), e.w);
        cr = __fadd_rn(cr, __fmul_rn(w, e.x));
        cg = __fadd_rn(cg, __fmul_rn(w, e.y));
        cb = __fadd_rn(cb, __fmul_rn(w, e.z));
        A = __fadd_rn(A, w);
        if (A >= opacity_cut) break;
    }
    rgba[(size_t)v * vw.width + u] = make_float4(cr, cg, cb, A);
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
