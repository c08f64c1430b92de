// cube_torben.cuh -- the paper's own median method on the GPU: Torben's bisection, Alg. 1 (sec. 4.3
// PAPER.md:286-296), one pass over the cube per guess.  SURVEY.md sec. 8(f) NEXT-3: "Torben-on-GPU as the
// paper-faithful comparison and early-stop approximate median" ("if a median approximation is accepted,
// the number of iterations could have been reduced to 20 with an error of order 1e-6").
//
// A pass classifies every non-NULL voxel against the current guess and returns the paper's five values -- counts
// less / greater / equal, the largest voxel below and the smallest voxel above the guess.  Here the
// "server" that turns them into the next guess is a 1-thread kernel between two passes, so the whole
// loop stays on the device: max_iter passes are enqueued, those after the stop test has fired return at once.
// It reads the cube ~30 times where the radix select reads it twice; it exists for the comparison, and for callers
// who want the paper's early-stop approximation.
#pragma once
#include "cube_kernels.cuh"

namespace cube {

struct TorbenState {
    unsigned long long less, greater;   // of the pass just made
    unsigned long long n;               // non-NaN voxels
    uint32_t kmaxlt, kmingt;            // order-preserving keys of max{x < guess}, min{x > guess}; 0 / ~0 when none
    float mn, mx, guess;                // Min, Max, Guess of Alg. 1
    float result;
    int iters;                          // passes made
    uint32_t done, converged;
};

// Per voxel: 2 FSETP, 2 FSEL, 2 FMNMX, 2 predicated counts; a NaN fails both comparisons and is counted nowhere
// (equal = n - less - greater with n the non-NaN count).
struct TorbenF {
    float g;
    uint32_t less = 0, greater = 0;
    float maxlt = -INFINITY, mingt = INFINITY;
    __device__ __forceinline__ void operator()(float x) {
        const bool lt = x < g, gt = x > g;
        less += lt ? 1u : 0u;
        greater += gt ? 1u : 0u;
        maxlt = fmaxf(maxlt, lt ? x : -INFINITY);
        mingt = fminf(mingt, gt ? x : INFINITY);
    }
    CUBE_DEFAULT_BATCH()
};

__global__ void __launch_bounds__(kThreads, 4)
torben_pass_kernel(const float* __restrict__ d, uint64_t n, TorbenState* __restrict__ st) {
    __shared__ unsigned long long s_less, s_greater;
    __shared__ uint32_t s_kmaxlt, s_kmingt;
    if (st->done) return;   // uniform over the grid
    if (threadIdx.x == 0) { s_less = 0; s_greater = 0; s_kmaxlt = 0u; s_kmingt = 0xFFFFFFFFu; }
    __syncthreads();
    TorbenF f;
    f.g = st->guess;
    stream_cube<kThreads>(d, n, f);
    uint32_t less = f.less, greater = f.greater;
    float maxlt = f.maxlt, mingt = f.mingt;
#pragma unroll
    for (int off = 16; off > 0; off >>= 1) {
        less += __shfl_xor_sync(0xffffffffu, less, off);
        greater += __shfl_xor_sync(0xffffffffu, greater, off);
        maxlt = fmaxf(maxlt, __shfl_xor_sync(0xffffffffu, maxlt, off));
        mingt = fminf(mingt, __shfl_xor_sync(0xffffffffu, mingt, off));
    }
    if ((threadIdx.x & 31) == 0) {
        atomicAdd(&s_less, (unsigned long long)less);
        atomicAdd(&s_greater, (unsigned long long)greater);
        // a voxel equal to the sentinel (-Inf below / +Inf above the guess) is the data minimum / maximum itself,
        // which is what the step kernel falls back to when no key has been recorded
        if (maxlt != -INFINITY) atomicMax(&s_kmaxlt, key_of(maxlt));
        if (mingt != INFINITY) atomicMin(&s_kmingt, key_of(mingt));
    }
    __syncthreads();
    if (threadIdx.x == 0) {
        if (s_less) atomicAdd(&st->less, s_less);
        if (s_greater) atomicAdd(&st->greater, s_greater);
        if (s_kmaxlt != 0u) atomicMax(&st->kmaxlt, s_kmaxlt);
        if (s_kmingt != 0xFFFFFFFFu) atomicMin(&st->kmingt, s_kmingt);
    }
}

// Alg. 1 between two passes (and after the last one with `final` set).  Restored lines as in DESIGN.md R1-R4:
// Guess = (Min+Max)/2 in float32; stop when Less <= (n+1)/2 and Greater <= (n+1)/2 (integer division).
__global__ void torben_step_kernel(const MomentsOut* __restrict__ m, TorbenState* __restrict__ st, int final) {
    if (st->done) return;
    const float qnan = __int_as_float(0x7fc00000);
    if (st->iters == 0) {                       // before the first pass: Min, Max, n from the moments pass
        st->n = m->count;
        st->mn = m->min; st->mx = m->max;
        if (m->count == 0 || final) { st->done = 1u; st->result = qnan; return; }
    } else {
        const unsigned long long n = st->n, half = (n + 1) / 2, less = st->less, greater = st->greater;
        const unsigned long long equal = n - less - greater;
        // MaxLt starts at Min, MinGt at Max
        const float maxlt = st->kmaxlt != 0u ? fmaxf(st->mn, __uint_as_float(bits_of_key(st->kmaxlt))) : st->mn;
        const float mingt = st->kmingt != 0xFFFFFFFFu ? fminf(st->mx, __uint_as_float(bits_of_key(st->kmingt))) : st->mx;
        const bool stop = less <= half && greater <= half;
        if (stop || final) {
            st->converged = stop ? 1u : 0u;
            st->result = (less >= half) ? maxlt : (less + equal >= half) ? st->guess : mingt;
            st->done = 1u;
            return;
        }
        if (less > greater) st->mx = maxlt;
        else st->mn = mingt;
    }
    st->guess = __fmul_rn(__fadd_rn(st->mn, st->mx), 0.5f);   // == (Min+Max)/2 in float32, no contraction
    st->less = 0; st->greater = 0; st->kmaxlt = 0u; st->kmingt = 0xFFFFFFFFu;
    st->iters += 1;
}

}  // namespace cube
