// cube_common.cuh -- shared device helpers of libcube (CUDA path only; the CPU oracle under
// oracle/ shares nothing with this file).
//
// Streaming model: every operation of the paper's statistics path visits each
// voxel once per pass ("visiting each data value once"; "visiting each data
// point and classifying it").  On B200 that is an HBM-read-bound scan, so all kernels share one
// persistent, coalesced, 128-bit streaming loop and differ only in the per-voxel functor.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

// -DCUBE_CHECKED: every index into a per-warp queue, key stage or the candidate buffer is checked against its
// capacity and a violation traps (the launch fails with cudaErrorLaunchFailure and every test that runs it fails).
// compute-sanitizer is not available on the GPU pool this library is developed on; the checked build run over the
// GPU test suite stands in for its memcheck on the hand-rolled staging structures (profiles/r2_checks.md).
#ifdef CUBE_CHECKED
#define CUBE_CHECK(cond) do { if (!(cond)) __trap(); } while (0)
#else
#define CUBE_CHECK(cond) do { } while (0)
#endif

namespace cube {

constexpr int kThreads = 256;  // threads per CTA (8 warps)
constexpr int kUnroll = 8;     // independent 128-bit loads in flight per thread per tile

// 128-bit read-only load that does not allocate in L1 (each voxel is used once per pass).  L2 policy is
// left at the default so that cubes smaller than the 126 MB L2 (config 1) are re-read from L2 by the
// later select passes.
__device__ __forceinline__ float4 ld_stream(const float4* p) {
    float4 r;
    asm volatile("ld.global.nc.L1::no_allocate.v4.f32 {%0,%1,%2,%3}, [%4];"
                 : "=f"(r.x), "=f"(r.y), "=f"(r.z), "=f"(r.w)
                 : "l"(p));
    return r;
}

// Order-preserving map float32 bits -> uint32 (IEEE total order on non-NaN: -0.0 < +0.0; R7).
// Negative values: flip all bits; non-negative: set the sign bit.
__device__ __forceinline__ uint32_t key_of(float x) {
    uint32_t u = __float_as_uint(x);
    return u ^ ((uint32_t)((int32_t)u >> 31) | 0x80000000u);
}
// Radix digits of the exact select: 13 + 10 + 9 bits of the order-preserving key.  A wide first
// digit makes the median's bucket small (sign + exponent + 4 mantissa bits: ~0.08 % of config 2), which is what
// the second pass has to revisit and compact.
#ifndef CUBE_BITS0      // build-time override for digit-width experiments
#define CUBE_BITS0 13
#define CUBE_BITS1 10
#endif
constexpr int kBits0 = CUBE_BITS0, kBits1 = CUBE_BITS1, kBits2 = 32 - CUBE_BITS0 - CUBE_BITS1;
constexpr int kShift0 = 32 - kBits0;          // 19: key >> kShift0 is the first digit
constexpr int kBins0 = 1 << kBits0, kBins1 = 1 << kBits1, kBins2 = 1 << kBits2;
constexpr int kDigitBins = kBins0;            // size of the global digit arrays
static_assert(kBits0 + kBits1 + kBits2 == 32, "digits must cover the key");
// First digit (key >> 19) <-> raw top 13 bits of the float (bits >> 19): a bijection (raw_of_digit maps
// digit -> raw), so a histogram indexed by the raw bits holds the same counts in permuted order.
__device__ __forceinline__ uint32_t raw_digit(float x) { return __float_as_uint(x) >> kShift0; }
__host__ __device__ __forceinline__ uint32_t raw_of_digit(uint32_t digit) {
    constexpr uint32_t sign = 1u << (kBits0 - 1), all = (1u << kBits0) - 1u;
    return (digit & sign) ? (digit ^ sign) : (~digit & all);
}
// NaN keys lie beyond +-inf, i.e. only in first-digit buckets whose raw exponent field is all ones.
__host__ __device__ __forceinline__ bool digit_may_hold_nan(uint32_t digit) {
    return ((raw_of_digit(digit) >> (kBits0 - 9)) & 0xFFu) == 0xFFu;
}
__host__ __device__ __forceinline__ uint32_t bits_of_key(uint32_t k) {
    return (k & 0x80000000u) ? (k ^ 0x80000000u) : ~k;
}

// Visit all n voxels of d exactly once across the grid.  F provides `void operator()(float)` for single
// voxels and `void batch(const float4 (&r)[kUnroll], const float4* p)` for a thread's share of a full tile
// (r[j] was loaded from p[j * THREADS]).
// Tiles of THREADS*kUnroll float4 are dealt round-robin to the CTAs, so concurrently running CTAs read
// adjacent tiles (DRAM page locality) and the assignment is static => per-CTA results are deterministic.
// The <= 3 voxels before the first 16-byte boundary and the <= 3 after the last full float4 are visited
// by CTA 0.
template <int THREADS, class F>
__device__ __forceinline__ void stream_cube(const float* __restrict__ d, uint64_t n, F& f) {
    constexpr int TILE = THREADS * kUnroll;
    uint64_t head = ((16u - (uint32_t)((uintptr_t)d & 15u)) & 15u) >> 2;
    if (head > n) head = n;
    const float4* __restrict__ v = reinterpret_cast<const float4*>(d + head);
    const uint64_t nvec = (n - head) >> 2;
    const uint64_t tail0 = head + (nvec << 2);
    if (blockIdx.x == 0) {
        if (threadIdx.x < head) f(d[threadIdx.x]);
        if (threadIdx.x >= 32 && threadIdx.x < 35) {
            uint64_t t = tail0 + (threadIdx.x - 32);
            if (t < n) f(d[t]);
        }
    }
    // Full tiles: a 32-bit tile counter (n <= 2^37 voxels: fewer than 2^23 tiles) and one running pointer, so that
    // the loop carries three registers of state and nothing is recomputed per tile (with the 64-bit tile index and
    // the in-loop "whole tile?" test ptxas rematerialised head / nvec / ntiles every iteration under the 64-register
    // cap of the 1024-thread kernels: ~85 of ~510 instructions per warp tile, profiles/r2_c3.md).
    const uint32_t nfull = (uint32_t)(nvec / TILE);
    const float4* __restrict__ q = v + (uint64_t)blockIdx.x * TILE + threadIdx.x;
    const uint64_t stride = (uint64_t)gridDim.x * TILE;
    for (uint32_t t = blockIdx.x; t < nfull; t += gridDim.x, q += stride) {   // CTA-uniform: batch() may use warp collectives
        float4 r[kUnroll];
#pragma unroll
        for (int j = 0; j < kUnroll; ++j) r[j] = ld_stream(q + j * THREADS);
        asm volatile("" ::: "memory");  // all kUnroll loads are issued before the first counter update
        f.batch(r, q);
    }
    // the ragged last tile goes to the CTA whose turn it would be, voxel by voxel
    if (nvec % TILE != 0 && nfull % gridDim.x == blockIdx.x) {
        const uint64_t base = (uint64_t)nfull * TILE + threadIdx.x;
#pragma unroll 1
        for (int j = 0; j < kUnroll; ++j) {
            const uint64_t i = base + (uint64_t)j * THREADS;
            if (i < nvec) {
                const float4 r = ld_stream(v + i);
                f(r.x); f(r.y); f(r.z); f(r.w);
            }
        }
    }
}

// Default batch: the single-voxel functor applied to the 4*kUnroll values.
#define CUBE_DEFAULT_BATCH()                                                        \
    __device__ __forceinline__ void batch(const float4 (&r)[kUnroll], const float4*) { \
        _Pragma("unroll") for (int j = 0; j < kUnroll; ++j) {                       \
            (*this)(r[j].x); (*this)(r[j].y); (*this)(r[j].z); (*this)(r[j].w);     \
        }                                                                           \
    }

// 32-bit shared-window address of a shared-memory pointer (what ATOMS/RED take), computed once per kernel
// instead of once per voxel.
__device__ __forceinline__ uint32_t smem_addr(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }

// Shared-memory counter increment, counter[idx] += 1 with `saddr` the shared-window address of counter[0].
// The byte offset is formed as idx * c_four + saddr with the 4 read from constant memory, so that ptxas emits one
// IMAD (FMA pipe) instead of a LEA: the kernels are limited by the half-rate ALU pipe (ncu:
// sm__inst_executed_pipe_alu 60-70 %, profiles/), and the FMA pipe is idle.  The RED compiles to
// ATOMS.POPC.INC, which the hardware aggregates over lanes that hit the same address.
__constant__ uint32_t c_four = 4u;
__constant__ uint32_t c_one = 1u;
__device__ __forceinline__ void smem_inc(uint32_t saddr, uint32_t idx) {
    asm volatile("{\n\t.reg .u32 a;\n\tmad.lo.u32 a, %0, %1, %2;\n\tred.shared.add.u32 [a], 1;\n\t}"
                 :: "r"(idx), "r"(c_four), "r"(saddr) : "memory");
}

// Same static tiling over an array of 32-bit keys (the select's candidate buffer, 16-byte aligned).
template <int THREADS, class F>
__device__ __forceinline__ void stream_keys(const uint32_t* __restrict__ k, uint64_t n, F& f) {
    for (uint64_t i = (uint64_t)blockIdx.x * THREADS + threadIdx.x; i < n; i += (uint64_t)gridDim.x * THREADS)
        f.key(__ldg(k + i));
}

// ---------------------------------------------------------------- (n, mean, M2, min, max) partials
// Pairwise update of Chan, Golub & LeVeque for merging two (n, mean, M2) summaries; what the paper's
// server does with (count, sum, sum of squares) in O(1), in a cancellation-free form.
struct Partial {
    uint64_t n;
    double mean, m2;
    uint32_t kmin, kmax;  // order-preserving keys; kmin=0xFFFFFFFF / kmax=0 when n == 0
};

__device__ __forceinline__ Partial partial_empty() {
    Partial p;
    p.n = 0; p.mean = 0.0; p.m2 = 0.0; p.kmin = 0xFFFFFFFFu; p.kmax = 0u;
    return p;
}

__device__ __forceinline__ Partial partial_merge(const Partial& a, const Partial& b) {
    Partial r;
    r.kmin = min(a.kmin, b.kmin);
    r.kmax = max(a.kmax, b.kmax);
    r.n = a.n + b.n;
    if (b.n == 0) { r.mean = a.mean; r.m2 = a.m2; return r; }
    if (a.n == 0) { r.mean = b.mean; r.m2 = b.m2; return r; }
    const double na = (double)a.n, nb = (double)b.n, nn = (double)r.n;
    const double delta = b.mean - a.mean;
    r.mean = a.mean + delta * (nb / nn);
    r.m2 = a.m2 + b.m2 + delta * delta * (na * (nb / nn));
    return r;
}

__device__ __forceinline__ Partial partial_shfl_down(const Partial& p, int off) {
    Partial q;
    q.n = __shfl_down_sync(0xffffffffu, p.n, off);
    q.mean = __shfl_down_sync(0xffffffffu, p.mean, off);
    q.m2 = __shfl_down_sync(0xffffffffu, p.m2, off);
    q.kmin = __shfl_down_sync(0xffffffffu, p.kmin, off);
    q.kmax = __shfl_down_sync(0xffffffffu, p.kmax, off);
    return q;
}

// Fixed-shape tree over the CTA: lanes (shuffle, offsets 16..1) then warps (first warp).  Result valid
// in thread 0.  `scratch` holds THREADS/32 Partials of shared memory.
template <int THREADS>
__device__ __forceinline__ Partial partial_block_reduce_n(Partial p, Partial* scratch) {
#pragma unroll
    for (int off = 16; off > 0; off >>= 1) p = partial_merge(p, partial_shfl_down(p, off));
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    if (lane == 0) scratch[warp] = p;
    __syncthreads();
    if (warp == 0) {
        p = (lane < THREADS / 32) ? scratch[lane] : partial_empty();
#pragma unroll
        for (int off = 16; off > 0; off >>= 1) p = partial_merge(p, partial_shfl_down(p, off));
    }
    return p;
}
__device__ __forceinline__ Partial partial_block_reduce(Partial p, Partial* scratch) {
    return partial_block_reduce_n<kThreads>(p, scratch);
}

}  // namespace cube
