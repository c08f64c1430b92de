// cubegen.cu -- seeded synthetic spectral-cube generator, CUDA implementation.
//
// INPUTS ONLY: this file holds none of the method's arithmetic (no moments, no binning, no
// key transform, no selection).  It is shared by the oracle-side and the CUDA-side tests in the
// only way the build contract allows: both consume the bytes it writes.  The recipe is stated in
// cubegen/__init__.py and DESIGN.md section 5; the cubes stand in for the paper's HI cubes
// which are not available.
//
// C ABI (device pointers, caller-owned; all work enqueued on the given stream; returns the
// cudaError_t of the launch, 0 = OK).
#include <cuda_runtime.h>
#include <stdint.h>

namespace {

struct Words { uint32_t r0, r1, r2, r3; };

__host__ __device__ inline uint32_t mulhi32(uint32_t a, uint32_t b) {
    return (uint32_t)(((uint64_t)a * (uint64_t)b) >> 32);
}

// Philox4x32-10 (Salmon, Moraes, Dror, Shaw 2011).
__host__ __device__ inline Words philox4x32_10(uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3,
                                               uint32_t k0, uint32_t k1) {
    const uint32_t M0 = 0xD2511F53u, M1 = 0xCD9E8D57u, W0 = 0x9E3779B9u, W1 = 0xBB67AE85u;
#pragma unroll
    for (int r = 0; r < 10; ++r) {
        uint32_t hi0 = mulhi32(M0, c0), lo0 = M0 * c0;
        uint32_t hi1 = mulhi32(M1, c2), lo1 = M1 * c2;
        uint32_t n0 = hi1 ^ c1 ^ k0, n2 = hi0 ^ c3 ^ k1;
        c0 = n0; c1 = lo1; c2 = n2; c3 = lo0;
        k0 += W0; k1 += W1;
    }
    Words w = {c0, c1, c2, c3};
    return w;
}

__device__ inline float u01(uint32_t r) { return ((float)(r >> 8) + 0.5f) * 5.9604644775390625e-08f; }

__global__ void fill_kernel(float* __restrict__ d, int64_t gx, int64_t gy, int64_t gz,
                            int64_t ox, int64_t oy, int64_t oz, int64_t bx, int64_t by, int64_t bz,
                            uint32_t seed, float sigma0, float sigma1, int lognormal,
                            uint32_t thr_nan, uint32_t thr_zero) {
    const int64_t n = bx * by * bz;
    const float zden = (float)(gz > 1 ? gz - 1 : 1);
    for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n;
         i += (int64_t)gridDim.x * blockDim.x) {
        int64_t x = i % bx, t = i / bx, y = t % by, z = t / by;
        uint64_t g = ((uint64_t)(z + oz) * (uint64_t)gy + (uint64_t)(y + oy)) * (uint64_t)gx + (uint64_t)(x + ox);
        Words w = philox4x32_10((uint32_t)g, (uint32_t)(g >> 32), 0u, 0u, seed, 0u);
        float zn = sqrtf(-2.0f * logf(u01(w.r0))) * cosf(6.283185307179586f * u01(w.r1));
        float v;
        if (lognormal) {
            const float step = 16.0f / 4096.0f;
            float lvl = rintf((2.0f * zn + 8.0f) / step);
            lvl = fminf(fmaxf(lvl, 0.0f), 4095.0f);
            v = expf(lvl * step - 8.0f);
        } else {
            float zf = (float)(z + oz) / zden;
            v = zn * (sigma0 + (sigma1 - sigma0) * zf);
        }
        if (w.r3 < thr_zero) v = 0.0f;
        if (w.r2 < thr_nan) v = __int_as_float(0x7fc00000);
        d[i] = v;
    }
}

// One Gaussian source added over its clipped bounding box [x0,x1) x [y0,y1) x [z0,z1) (brick
// coordinates).  Launches for successive sources are serialised on the stream, so overlapping
// sources are added in source-index order.
__global__ void source_kernel(float* __restrict__ d, int64_t bx, int64_t by, int64_t bz,
                              int64_t ox, int64_t oy, int64_t oz,
                              int64_t x0, int64_t y0, int64_t z0, int64_t x1, int64_t y1, int64_t z1,
                              float cx, float cy, float cz, float sxy, float sz, float peak) {
    const int64_t wx = x1 - x0, wy = y1 - y0, wz = z1 - z0, n = wx * wy * wz;
    for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n;
         i += (int64_t)gridDim.x * blockDim.x) {
        int64_t x = x0 + i % wx, t = i / wx, y = y0 + t % wy, z = z0 + t / wy;
        float dx = ((float)(x + ox) - cx) / sxy;
        float dy = ((float)(y + oy) - cy) / sxy;
        float dz = ((float)(z + oz) - cz) / sz;
        float q = dz * dz + dy * dy + dx * dx;
        d[(z * by + y) * bx + x] += peak * expf(-0.5f * q);
    }
}

__global__ void nan_plane_kernel(float* __restrict__ d, int64_t plane, int64_t z) {
    float* p = d + z * plane;
    for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < plane;
         i += (int64_t)gridDim.x * blockDim.x)
        p[i] = __int_as_float(0x7fc00000);
}

inline int grid_for(int64_t n, int threads, int cap) {
    int64_t g = (n + threads - 1) / threads;
    if (g < 1) g = 1;
    if (g > cap) g = cap;
    return (int)g;
}

}  // namespace

extern "C" {

int cubegen_fill(float* d, int64_t gx, int64_t gy, int64_t gz, int64_t ox, int64_t oy, int64_t oz,
                 int64_t bx, int64_t by, int64_t bz, uint32_t seed, float sigma0, float sigma1,
                 int lognormal, uint32_t thr_nan, uint32_t thr_zero, cudaStream_t stream) {
    int64_t n = bx * by * bz;
    if (n <= 0) return 0;
    fill_kernel<<<grid_for(n, 256, 148 * 32), 256, 0, stream>>>(d, gx, gy, gz, ox, oy, oz, bx, by, bz, seed,
                                                                 sigma0, sigma1, lognormal, thr_nan, thr_zero);
    return (int)cudaGetLastError();
}

int cubegen_add_source(float* d, int64_t bx, int64_t by, int64_t bz, int64_t ox, int64_t oy, int64_t oz,
                       int64_t x0, int64_t y0, int64_t z0, int64_t x1, int64_t y1, int64_t z1,
                       float cx, float cy, float cz, float sxy, float sz, float peak, cudaStream_t stream) {
    int64_t n = (x1 - x0) * (y1 - y0) * (z1 - z0);
    if (n <= 0) return 0;
    source_kernel<<<grid_for(n, 256, 148 * 8), 256, 0, stream>>>(d, bx, by, bz, ox, oy, oz, x0, y0, z0,
                                                                x1, y1, z1, cx, cy, cz, sxy, sz, peak);
    return (int)cudaGetLastError();
}

int cubegen_nan_plane(float* d, int64_t bx, int64_t by, int64_t z, cudaStream_t stream) {
    int64_t plane = bx * by;
    nan_plane_kernel<<<grid_for(plane, 256, 148 * 8), 256, 0, stream>>>(d, plane, z);
    return (int)cudaGetLastError();
}

// Copy a generated brick from its device buffer into (pinned) host memory on the stream -- used when the
// consumer wants the cube in host memory (out-of-core configuration).
int cubegen_to_host(float* h_dst, const float* d_src, uint64_t nvox, cudaStream_t stream) {
    return (int)cudaMemcpyAsync(h_dst, d_src, nvox * sizeof(float), cudaMemcpyDeviceToHost, stream);
}

// Host evaluation of the same Philox source, to pin the integers against the numpy restatement.
int cubegen_philox(uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3, uint32_t k0, uint32_t k1,
                   uint32_t* out4) {
    Words w = philox4x32_10(c0, c1, c2, c3, k0, k1);
    out4[0] = w.r0; out4[1] = w.r1; out4[2] = w.r2; out4[3] = w.r3;
    return 0;
}

}  // extern "C"
