// cube.cu -- C ABI of libcube (include/cube.h) over the kernels in cube_kernels.cuh.
// No CPU fallback anywhere: every statistic is computed by the CUDA kernels; the host code only
// validates arguments, enqueues launches and copies results.
#include "../../include/cube.h"

#include <math.h>
#include <new>
#include <string.h>

#include "cube_kernels.cuh"

using namespace cube;

struct cube_ctx {
    int device = 0;
    int num_sms = 0;
    int ctas_per_sm = 0;  // 0 = per-kernel default
    int last_cuda = 0;
    uint64_t launches = 0;
    // device scratch
    Partial* partials = nullptr;           // one per CTA
    unsigned int* ticket = nullptr;
    Partial* acc = nullptr;                // running moments (out-of-core)
    unsigned long long* nvox_acc = nullptr;
    MomentsOut* mom_out = nullptr;
    unsigned long long* gbins = nullptr;   // CUBE_MAX_BINS + 2 (outside) counters
    unsigned long long* gdigits = nullptr; // kDigitBins
    unsigned long long* coarse = nullptr;  // kDigitBins: digit histogram kept by CUBE_COARSE_HIST
    SelectState* sel = nullptr;
    // out-of-core state (host side)
    int ooc_active = 0, ooc_sweep = 0, ooc_nbins = 0, ooc_want_median = 0, ooc_bricks = 0;
    float ooc_lo = 0.f, ooc_hi = 0.f, ooc_scale = 0.f;
    // host-cube driver workspace
    float* resident = nullptr;
    size_t resident_bytes = 0;
    float* chunk[2] = {nullptr, nullptr};
    size_t chunk_bytes = 0;
    cudaStream_t copy_stream = nullptr, work_stream = nullptr;
    cudaEvent_t ev_copied[2] = {nullptr, nullptr}, ev_consumed[2] = {nullptr, nullptr};
    void* pinned_results = nullptr;  // staging for cube_stats_host results
    int max_ctas = 0;
};

namespace {

constexpr int kMaxCtasPerSm = 8;
constexpr int kSmemHistMaxBins = 16384;  // 64 KiB of 32-bit counters per CTA

#define CUBE_CUDA(ctx, call)                              \
    do {                                                  \
        cudaError_t e__ = (call);                         \
        if (e__ != cudaSuccess) {                         \
            (ctx)->last_cuda = (int)e__;                  \
            return CUBE_ECUDA;                            \
        }                                                 \
    } while (0)

inline bool dims_ok(int64_t nx, int64_t ny, int64_t nz, uint64_t* n) {
    if (nx <= 0 || ny <= 0 || nz <= 0) return false;
    const long double p = (long double)nx * (long double)ny * (long double)nz;
    if (p > 137438953472.0L) return false;  // 2^37 voxels
    *n = (uint64_t)nx * (uint64_t)ny * (uint64_t)nz;
    return true;
}

inline int grid_for(const cube_ctx* c, int default_per_sm, int occ_limit) {
    int per = c->ctas_per_sm > 0 ? c->ctas_per_sm : default_per_sm;
    if (per > occ_limit) per = occ_limit;
    if (per < 1) per = 1;
    return c->num_sms * per;
}

// scale = (float)nbins / (hi - lo), both roundings in float32 (R10); hi == lo -> 0 (R13).
inline bool hist_scale(int nbins, float lo, float hi, float* scale) {
    if (nbins < 1 || nbins > CUBE_MAX_BINS) return false;
    if (!(lo <= hi) || !isfinite(lo) || !isfinite(hi)) return false;
    if (hi == lo) { *scale = 0.0f; return true; }
    volatile float width = hi - lo;
    volatile float s = (float)nbins / width;
    if (!isfinite(width) || !isfinite(s)) return false;  // R19
    *scale = s;
    return true;
}

int launch_moments(cube_ctx* c, const float* d, uint64_t n, unsigned flags, int accumulate, cudaStream_t s) {
    const bool coarse = (flags & CUBE_COARSE_HIST) != 0;
    const int grid = grid_for(c, coarse ? 3 : 4, kMaxCtasPerSm);
    if (coarse) {
        if (!accumulate) CUBE_CUDA(c, cudaMemsetAsync(c->coarse, 0, kDigitBins * sizeof(unsigned long long), s));
        moments_kernel<true><<<grid, kThreads, 0, s>>>(d, n, c->partials, c->ticket, c->acc, c->nvox_acc,
                                                       accumulate, flags, c->mom_out, c->coarse);
    } else {
        moments_kernel<false><<<grid, kThreads, 0, s>>>(d, n, c->partials, c->ticket, c->acc, c->nvox_acc,
                                                        accumulate, flags, c->mom_out, c->coarse);
    }
    c->launches++;
    CUBE_CUDA(c, cudaGetLastError());
    return CUBE_OK;
}

int launch_hist(cube_ctx* c, const float* d, uint64_t n, int nbins, float lo, float hi, float scale,
                cudaStream_t s) {
    unsigned long long* outside = c->gbins + CUBE_MAX_BINS;
    if (nbins <= kSmemHistMaxBins) {
        const size_t smem = (size_t)nbins * sizeof(uint32_t);
        int occ = (int)((200 * 1024) / (smem + 1024));
        const int grid = grid_for(c, 4, occ < kMaxCtasPerSm ? occ : kMaxCtasPerSm);
        hist_smem_kernel<<<grid, kThreads, smem, s>>>(d, n, nbins, lo, hi, scale, c->gbins, outside);
    } else {
        const int grid = grid_for(c, 4, kMaxCtasPerSm);
        hist_global_kernel<<<grid, kThreads, 0, s>>>(d, n, nbins, lo, hi, scale, c->gbins, outside);
    }
    c->launches++;
    CUBE_CUDA(c, cudaGetLastError());
    return CUBE_OK;
}

template <int PASS>
int launch_select_pass(cube_ctx* c, const float* d, uint64_t n, cudaStream_t s) {
    const int grid = grid_for(c, 4, kMaxCtasPerSm);
    select_pass_kernel<PASS><<<grid, kThreads, 0, s>>>(d, n, c->sel, c->gdigits);
    c->launches++;
    CUBE_CUDA(c, cudaGetLastError());
    return CUBE_OK;
}

template <int PASS>
int launch_select_scan(cube_ctx* c, unsigned long long* digits, cudaStream_t s) {
    // the coarse histogram kept by CUBE_COARSE_HIST is left intact so that several k can reuse it
    select_scan_kernel<PASS><<<1, 1024, 0, s>>>(c->sel, digits, digits == c->gdigits ? 1 : 0);
    c->launches++;
    CUBE_CUDA(c, cudaGetLastError());
    return CUBE_OK;
}

int select_init(cube_ctx* c, uint64_t k, int use_median, cudaStream_t s) {
    SelectState h;
    memset(&h, 0, sizeof(h));
    h.k = k;
    h.use_median = use_median ? 1u : 0u;
    h.result = nanf("");
    // small H2D of a stack struct: cudaMemcpyAsync from pageable memory stages the bytes before returning
    CUBE_CUDA(c, cudaMemcpyAsync(c->sel, &h, sizeof(h), cudaMemcpyHostToDevice, s));
    return CUBE_OK;
}

int kth_impl(cube_ctx* c, const float* d, uint64_t n, uint64_t k, int use_median, unsigned flags, float* out,
             cudaStream_t s) {
    int rc;
    if ((rc = select_init(c, k, use_median, s))) return rc;
    if (flags & CUBE_REUSE_COARSE) {
        if ((rc = launch_select_scan<0>(c, c->coarse, s))) return rc;
    } else {
        CUBE_CUDA(c, cudaMemsetAsync(c->gdigits, 0, kDigitBins * sizeof(unsigned long long), s));
        if ((rc = launch_select_pass<0>(c, d, n, s))) return rc;
        if ((rc = launch_select_scan<0>(c, c->gdigits, s))) return rc;
    }
    if ((rc = launch_select_pass<1>(c, d, n, s))) return rc;
    if ((rc = launch_select_scan<1>(c, c->gdigits, s))) return rc;
    if ((rc = launch_select_pass<2>(c, d, n, s))) return rc;
    if ((rc = launch_select_scan<2>(c, c->gdigits, s))) return rc;
    CUBE_CUDA(c, cudaMemcpyAsync(out, &c->sel->result, sizeof(float), cudaMemcpyDefault, s));
    return CUBE_OK;
}

}  // namespace

extern "C" {

int cube_create(cube_ctx** out, size_t scratch_bytes_hint) {
    (void)scratch_bytes_hint;
    if (!out) return CUBE_EINVAL;
    *out = nullptr;
    cube_ctx* c = new (std::nothrow) cube_ctx();
    if (!c) return CUBE_ENOMEM;
    cudaError_t e = cudaGetDevice(&c->device);
    cudaDeviceProp prop;
    if (e == cudaSuccess) e = cudaGetDeviceProperties(&prop, c->device);
    if (e != cudaSuccess) { delete c; return CUBE_ECUDA; }  // no device: fail loudly, no CPU path
    c->num_sms = prop.multiProcessorCount;
    c->max_ctas = c->num_sms * kMaxCtasPerSm;
    size_t bytes_bins = (CUBE_MAX_BINS + 2) * sizeof(unsigned long long);
    bool ok = true;
    ok = ok && cudaMalloc(&c->partials, c->max_ctas * sizeof(Partial)) == cudaSuccess;
    ok = ok && cudaMalloc(&c->ticket, sizeof(unsigned int)) == cudaSuccess;
    ok = ok && cudaMalloc(&c->acc, sizeof(Partial)) == cudaSuccess;
    ok = ok && cudaMalloc(&c->nvox_acc, sizeof(unsigned long long)) == cudaSuccess;
    ok = ok && cudaMalloc(&c->mom_out, sizeof(MomentsOut)) == cudaSuccess;
    ok = ok && cudaMalloc(&c->gbins, bytes_bins) == cudaSuccess;
    ok = ok && cudaMalloc(&c->gdigits, kDigitBins * sizeof(unsigned long long)) == cudaSuccess;
    ok = ok && cudaMalloc(&c->coarse, kDigitBins * sizeof(unsigned long long)) == cudaSuccess;
    ok = ok && cudaMalloc(&c->sel, sizeof(SelectState)) == cudaSuccess;
    ok = ok && cudaMemset(c->ticket, 0, sizeof(unsigned int)) == cudaSuccess;
    ok = ok && cudaMemset(c->gdigits, 0, kDigitBins * sizeof(unsigned long long)) == cudaSuccess;
    ok = ok && cudaMemset(c->coarse, 0, kDigitBins * sizeof(unsigned long long)) == cudaSuccess;
    ok = ok && cudaFuncSetAttribute(hist_smem_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                    kSmemHistMaxBins * (int)sizeof(uint32_t)) == cudaSuccess;
    if (!ok) { cube_destroy(c); return CUBE_ENOMEM; }
    *out = c;
    return CUBE_OK;
}

int cube_destroy(cube_ctx* c) {
    if (!c) return CUBE_EINVAL;
    cudaFree(c->partials); cudaFree(c->ticket); cudaFree(c->acc); cudaFree(c->nvox_acc);
    cudaFree(c->mom_out); cudaFree(c->gbins); cudaFree(c->gdigits); cudaFree(c->coarse); cudaFree(c->sel);
    cudaFree(c->resident); cudaFree(c->chunk[0]); cudaFree(c->chunk[1]);
    if (c->pinned_results) cudaFreeHost(c->pinned_results);
    for (int i = 0; i < 2; ++i) {
        if (c->ev_copied[i]) cudaEventDestroy(c->ev_copied[i]);
        if (c->ev_consumed[i]) cudaEventDestroy(c->ev_consumed[i]);
    }
    if (c->copy_stream) cudaStreamDestroy(c->copy_stream);
    if (c->work_stream) cudaStreamDestroy(c->work_stream);
    delete c;
    return CUBE_OK;
}

int cube_moments(cube_ctx* c, const float* d, int64_t nx, int64_t ny, int64_t nz, unsigned flags,
                 cube_moments_t* out, cudaStream_t s) {
    uint64_t n;
    if (!c || !d || !out || !dims_ok(nx, ny, nz, &n)) return CUBE_EINVAL;
    static_assert(sizeof(cube_moments_t) == sizeof(MomentsOut), "layout");
    int rc = launch_moments(c, d, n, flags, 0, s);
    if (rc) return rc;
    CUBE_CUDA(c, cudaMemcpyAsync(out, c->mom_out, sizeof(MomentsOut), cudaMemcpyDefault, s));
    return CUBE_OK;
}

int cube_histogram(cube_ctx* c, const float* d, int64_t nx, int64_t ny, int64_t nz, int nbins, float lo,
                   float hi, uint64_t* bins, uint64_t* outside, cudaStream_t s) {
    uint64_t n;
    float scale;
    if (!c || !d || !bins || !outside || !dims_ok(nx, ny, nz, &n)) return CUBE_EINVAL;
    if (!hist_scale(nbins, lo, hi, &scale)) return CUBE_EINVAL;
    CUBE_CUDA(c, cudaMemsetAsync(c->gbins, 0, (size_t)nbins * sizeof(unsigned long long), s));
    CUBE_CUDA(c, cudaMemsetAsync(c->gbins + CUBE_MAX_BINS, 0, 2 * sizeof(unsigned long long), s));
    int rc = launch_hist(c, d, n, nbins, lo, hi, scale, s);
    if (rc) return rc;
    CUBE_CUDA(c, cudaMemcpyAsync(bins, c->gbins, (size_t)nbins * sizeof(uint64_t), cudaMemcpyDefault, s));
    CUBE_CUDA(c, cudaMemcpyAsync(outside, c->gbins + CUBE_MAX_BINS, 2 * sizeof(uint64_t), cudaMemcpyDefault, s));
    return CUBE_OK;
}

int cube_kth_ex(cube_ctx* c, const float* d, int64_t nx, int64_t ny, int64_t nz, uint64_t k, unsigned flags,
                float* out, cudaStream_t s) {
    uint64_t n;
    if (!c || !d || !out || !dims_ok(nx, ny, nz, &n)) return CUBE_EINVAL;
    return kth_impl(c, d, n, k, 0, flags, out, s);
}

int cube_kth(cube_ctx* c, const float* d, int64_t nx, int64_t ny, int64_t nz, uint64_t k, float* out,
             cudaStream_t s) {
    return cube_kth_ex(c, d, nx, ny, nz, k, 0u, out, s);
}

int cube_median_ex(cube_ctx* c, const float* d, int64_t nx, int64_t ny, int64_t nz, unsigned flags, float* out,
                   cudaStream_t s) {
    uint64_t n;
    if (!c || !d || !out || !dims_ok(nx, ny, nz, &n)) return CUBE_EINVAL;
    return kth_impl(c, d, n, 0, 1, flags, out, s);
}

int cube_median(cube_ctx* c, const float* d, int64_t nx, int64_t ny, int64_t nz, float* out, cudaStream_t s) {
    return cube_median_ex(c, d, nx, ny, nz, 0u, out, s);
}

const char* cube_strerror(int code) {
    switch (code) {
        case CUBE_OK: return "ok";
        case CUBE_EINVAL: return "invalid argument";
        case CUBE_EEMPTY: return "no non-NaN voxel";
        case CUBE_ECUDA: return "CUDA error (see cube_last_cuda_error)";
        case CUBE_ERANGE: return "out of range";
        case CUBE_ENOMEM: return "allocation failed";
        default: return "unknown error";
    }
}

int cube_last_cuda_error(const cube_ctx* c) { return c ? c->last_cuda : 0; }

int cube_set_launch(cube_ctx* c, int ctas_per_sm) {
    if (!c || ctas_per_sm < 0 || ctas_per_sm > kMaxCtasPerSm) return CUBE_EINVAL;
    c->ctas_per_sm = ctas_per_sm;
    return CUBE_OK;
}

uint64_t cube_launch_count(const cube_ctx* c) { return c ? c->launches : 0; }

}  // extern "C"

#include "cube_ooc.inl"
