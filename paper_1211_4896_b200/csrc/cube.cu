// cube.cu -- C ABI of libcube (include/cube.h) over the kernels in cube_kernels.cuh.
// No CPU fallback anywhere: every statistic is computed by the CUDA kernels; the host code only
// validates arguments, enqueues launches and copies results.
#include "../../include/cube.h"

#include <mutex>
#include <math.h>
#include <new>
#include <stddef.h>
#include <string.h>
#include <stdio.h>
#include <stdlib.h>
#include <algorithm>
#include <vector>

#include "cube_kernels.cuh"
#include "cube_minimap_tma.cuh"
#include "cube_render.cuh"
#include "cube_minimap_median.cuh"
#include "cube_small.cuh"
#include "cube_select_multi.cuh"

using namespace cube;

struct cube_ctx {
    int device = 0;
    int num_sms = 0;
    int ctas_per_sm = 0;  // 0 = per-kernel default
    int bighist = 0;      // CUBE_KNOB_BIGHIST: 0 = automatic (window or packed, chosen on the device), 1 = cluster DSM, 2 = packed
    int no_small = 0;     // CUBE_KNOB_SMALL: 1 = never the single cooperative launch
    int mapmedian = 0;    // CUBE_KNOB_MAPMEDIAN
    int render_variant = 0;   // CUBE_KNOB_RENDER
    float2* map32 = nullptr;  // cube_render_sigma: (mean, std) of the mini-map's cells as float32 pairs
    size_t map32_cap = 0;     // cells it holds
    int coop = 0;         // the device supports cooperative launches
    unsigned int* bar = nullptr;   // grid-barrier counter of stats_small_kernel (only grows)
    unsigned long long* coarse_next = nullptr;   // all zero between calls: the first-digit array of the single-launch cube_stats
    unsigned long long* chunk_tot = nullptr;     // kDigitBins / 32 chunk totals, all zero between calls
    unsigned int* small_ext = nullptr;           // stats_small_kernel: {min key, max key, ticket} = {~0, 0, 0} between calls
    unsigned long long* small_tstamp = nullptr;   // debug builds only (-DCUBE_SMALL_TIMING)
    int minimap_variant = 0;  // CUBE_KNOB_MINIMAP: 0 = automatic, 1 = no TMA ring, 2 = scalar kernel only, 3 = TMA ring whenever eligible
    int last_cuda = 0;
    uint64_t launches = 0;
    // device scratch
    Partial* partials = nullptr;           // one per CTA
    unsigned int* ticket = nullptr;
    unsigned int* ticket2 = nullptr;       // arrival counter of the fused bucket-location step
    Partial* acc = nullptr;                // running moments (out-of-core)
    unsigned long long* nvox_acc = nullptr;
    MomentsOut* mom_out = nullptr;
    unsigned long long* gout = nullptr;    // allocation: [outside (2)][bins (CUBE_MAX_BINS)] -- one memset clears both
    unsigned long long* gbins = nullptr;   // = gout + 2
    unsigned long long* gdigits = nullptr; // kDigitBins
    unsigned long long* coarse = nullptr;  // kDigitBins: digit histogram kept by CUBE_COARSE_HIST
    SelectState* sel = nullptr;
    MultiState* multi = nullptr;           // cube_kth_multi: the ranks of one group (cube_select_multi.cuh)
    float* range3 = nullptr;               // (lo, hi, scale) resolved on the device by cube_stats
    float* probe_out = nullptr;            // cube_probe_read sink
    BigHistPlan* plan = nullptr;           // hist_window_kernel's plan for the > 16384-bin histogram kernels
    ClipState* clip = nullptr;             // sigma-clip loop state (NEXT-1)
    TorbenState* torben = nullptr;         // Alg. 1 loop state (cube_median_torben)
    float* center = nullptr;               // cube_mad: the median the deviations are taken from
    float4* tf_table = nullptr;            // cube_render_tf: device copy of a host transfer-function table (4096 levels)
    uint32_t* cand = nullptr;              // candidate keys of the select (step 8)
    unsigned long long cand_cap = 0;       // in keys
    // out-of-core state (host side)
    int ooc_active = 0, ooc_sweep = 0, ooc_nbins = 0, ooc_want_median = 0, ooc_bricks = 0;
    float ooc_lo = 0.f, ooc_hi = 0.f, ooc_scale = 0.f;
    int ooc_minmax = 0;                    // CUBE_RANGE_MINMAX: histogram over [min, max], in sweep 1
    // host-cube driver workspace
    float* resident = nullptr;
    size_t resident_bytes = 0;
    float* chunk[2] = {nullptr, nullptr};
    size_t chunk_bytes = 0;
    cudaStream_t copy_stream = nullptr, work_stream = nullptr;
    cudaEvent_t ev_copied[2] = {nullptr, nullptr}, ev_consumed[2] = {nullptr, nullptr};
    void* pinned_results = nullptr;  // staging for cube_stats_host results
    // brick-callback driver (cube_stats_stream): pinned staging ring the callback fills
    static constexpr int kMaxStage = 8;
    float* h_stage[kMaxStage] = {};
    cudaEvent_t ev_filled[kMaxStage] = {}, ev_h2d_done[kMaxStage] = {};
    int stage_slots = 0;
    size_t stage_bytes = 0;
    cudaStream_t fill_stream = nullptr;
    uint64_t stream_h2d_bytes = 0;   // bytes that crossed the host link in the last cube_stats_stream call
    int stream_sweeps = 0;
    int max_ctas = 0;
    // occupancy of each kernel, asked once per (kernel, dynamic shared memory) instead of once per call
    struct OccEntry { const void* fn; size_t smem; int occ; };
    OccEntry occ_cache[24] = {};
    int occ_used = 0;
    // per-kernel timing (cube_profile_*)
    int prof_on = 0;
    std::vector<cudaEvent_t> prof_ev;   // pairs
    std::vector<int> prof_kind;         // kind of pair i
    size_t prof_used = 0;               // pairs in use
    double prof_ms[CUBE_K_KINDS] = {};
    uint64_t prof_n[CUBE_K_KINDS] = {};
};

namespace {

constexpr int kMaxCtasPerSm = 8;
constexpr int kSmemHistMaxBins = 16384;  // 64 KiB of 32-bit counters per CTA
// dynamic shared memory of hist_select_kernel: histogram + trash, digit bins + trash, stage slices + counters
constexpr int hist_select_smem(int nbins) {
    return (nbins + 2 + kBins1 + 1 + (kThreads / 32) * ((int)kStageCap + 1)) * (int)sizeof(uint32_t);
}

#define CUBE_CUDA(ctx, call)                              \
    do {                                                  \
        cudaError_t e__ = (call);                         \
        if (e__ != cudaSuccess) {                         \
            (ctx)->last_cuda = (int)e__;                  \
            return CUBE_ECUDA;                            \
        }                                                 \
    } while (0)

// Brackets one kernel launch with an event pair when profiling is on.
struct ProfScope {
    cube_ctx* c; cudaStream_t s; cudaEvent_t stop = nullptr;
    ProfScope(cube_ctx* c_, int kind, cudaStream_t s_) : c(c_), s(s_) {
        c->launches++;
        if (!c->prof_on) return;
        if (c->prof_used * 2 + 2 > c->prof_ev.size()) {
            cudaEvent_t a, b;
            if (cudaEventCreate(&a) != cudaSuccess || cudaEventCreate(&b) != cudaSuccess) return;
            c->prof_ev.push_back(a); c->prof_ev.push_back(b); c->prof_kind.push_back(kind);
        }
        c->prof_kind[c->prof_used] = kind;
        cudaEventRecord(c->prof_ev[c->prof_used * 2], s);
        stop = c->prof_ev[c->prof_used * 2 + 1];
        c->prof_used++;
    }
    ~ProfScope() { if (stop) cudaEventRecord(stop, s); }
};

int prof_collect(cube_ctx* c) {
    if (c->prof_used == 0) return CUBE_OK;
    CUBE_CUDA(c, cudaDeviceSynchronize());
    for (size_t i = 0; i < c->prof_used; ++i) {
        float ms = 0.f;
        if (cudaEventElapsedTime(&ms, c->prof_ev[2 * i], c->prof_ev[2 * i + 1]) == cudaSuccess) {
            c->prof_ms[c->prof_kind[i]] += ms;
            c->prof_n[c->prof_kind[i]]++;
        }
    }
    c->prof_used = 0;
    return CUBE_OK;
}

inline bool dims_ok(int64_t nx, int64_t ny, int64_t nz, uint64_t* n) {
    if (nx <= 0 || ny <= 0 || nz <= 0) return false;
    const long double p = (long double)nx * (long double)ny * (long double)nz;
    if (p > 137438953472.0L) return false;  // 2^37 voxels
    *n = (uint64_t)nx * (uint64_t)ny * (uint64_t)nz;
    return true;
}

// Device-side address of a caller's output buffer when the kernels can write it themselves (memory of this device,
// or pinned / managed host memory): small results are then stored by the producing kernel and no copy is enqueued.
// nullptr for pageable host memory or another device's memory (the cudaMemcpyAsync path).
inline void* device_reachable(const cube_ctx* c, void* p) {
    cudaPointerAttributes at;
    if (!p || cudaPointerGetAttributes(&at, p) != cudaSuccess) { cudaGetLastError(); return nullptr; }
    if (at.type == cudaMemoryTypeDevice) return at.device == c->device ? at.devicePointer : nullptr;
    if (at.type == cudaMemoryTypeHost || at.type == cudaMemoryTypeManaged) return at.devicePointer;
    return nullptr;
}

template <class K>
int occupancy_of(cube_ctx* c, K kernel, int threads, size_t smem) {
    const void* fn = reinterpret_cast<const void*>(kernel);
    for (int i = 0; i < c->occ_used; ++i)
        if (c->occ_cache[i].fn == fn && c->occ_cache[i].smem == smem) return c->occ_cache[i].occ;
    int occ = 0;
    if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, kernel, threads, smem) != cudaSuccess) { cudaGetLastError(); occ = 1; }
    if (c->occ_used < 24) c->occ_cache[c->occ_used++] = {fn, smem, occ};
    return occ;
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

// mode: kMomPlain / kMomCoarse / kMomWindow (window = (wlo, whi), or the context's ClipState when use_clip)
// digits: where kMomCoarse adds the first-digit counts (nullptr: the context's `coarse` array, zeroed first unless
// accumulating; the brick-streamed path passes gdigits, which cube_ooc_begin has zeroed)
int launch_moments(cube_ctx* c, const float* d, uint64_t n, unsigned flags, int accumulate, cudaStream_t s,
                   int mode = -1, float wlo = 0.f, float whi = 0.f, bool use_clip = false,
                   const SelectInit* fuse_scan = nullptr, MomentsOut* out_user = nullptr,
                   unsigned long long* digits = nullptr) {
    if (mode < 0) mode = (flags & CUBE_COARSE_HIST) ? kMomCoarse : kMomPlain;
    const bool coarse = mode == kMomCoarse;
    const int occ_m = mode == kMomCoarse ? occupancy_of(c, moments_kernel<kMomCoarse>, kThreads, 0)
                    : mode == kMomWindow ? occupancy_of(c, moments_kernel<kMomWindow>, kThreads, 0)
                                         : occupancy_of(c, moments_kernel<kMomPlain>, kThreads, 0);
    const int grid = grid_for(c, 4, occ_m < kMaxCtasPerSm ? occ_m : kMaxCtasPerSm);
    if (coarse && !accumulate && !digits) CUBE_CUDA(c, cudaMemsetAsync(c->coarse, 0, kDigitBins * sizeof(unsigned long long), s));
    if (!digits) digits = c->coarse;
    {
    ProfScope prof(c, coarse ? CUBE_K_MOMENTS_COARSE : mode == kMomWindow ? CUBE_K_MOMENTS_WINDOW : CUBE_K_MOMENTS, s);
    const ClipState* clip = use_clip ? c->clip : nullptr;
    SelectInit none;
    none.k = 0; none.cand_cap = 0; none.result_out = nullptr; none.use_median = 0; none.enabled = 0;
    if (coarse) {   // fuse_scan: the kernel's last CTA also locates the first-digit bucket (cube_stats)
        moments_kernel<kMomCoarse><<<grid, kThreads, 0, s>>>(d, n, c->partials, c->ticket, c->acc, c->nvox_acc,
                                                             accumulate, flags, c->mom_out, digits, 0.f, 0.f, nullptr,
                                                             c->sel, fuse_scan ? c->ticket2 : nullptr,
                                                             fuse_scan ? *fuse_scan : none, out_user);
    } else if (mode == kMomWindow) {
        moments_kernel<kMomWindow><<<grid, kThreads, 0, s>>>(d, n, c->partials, c->ticket, c->acc, c->nvox_acc,
                                                             accumulate, flags, c->mom_out, c->coarse, wlo, whi, clip,
                                                             nullptr, nullptr, none, out_user);
    } else {
        moments_kernel<kMomPlain><<<grid, kThreads, 0, s>>>(d, n, c->partials, c->ticket, c->acc, c->nvox_acc,
                                                            accumulate, flags, c->mom_out, c->coarse, 0.f, 0.f, nullptr,
                                                            nullptr, nullptr, none, out_user);
    }
    }
    CUBE_CUDA(c, cudaGetLastError());
    return CUBE_OK;
}

// fused_select: more than 16384 bins, the window histogram shares its read with the second select digit
// (hist_win_select_kernel); fused_scan: its last CTA also locates the bucket (in-core calls; the brick-streamed
// path locates it after the last brick)
int launch_hist(cube_ctx* c, const float* d, uint64_t n, int nbins, float lo, float hi, float scale,
                cudaStream_t s, const float* range3 = nullptr, bool fused_select = false, bool fused_scan = true) {
    unsigned long long* outside = c->gout;
    {
    ProfScope prof(c, fused_select ? CUBE_K_HIST_SELECT : CUBE_K_HIST, s);
    if (nbins <= kSmemHistMaxBins) {
        const size_t smem = (size_t)(nbins + 2) * sizeof(uint32_t);  // + trash slot
        const int grid = grid_for(c, 4, occupancy_of(c, hist_smem_kernel, kThreads, smem));
        hist_smem_kernel<<<grid, kThreads, smem, s>>>(d, n, nbins, lo, hi, scale, range3, c->gbins, outside);
    } else {
        // one CTA of 1024 threads per SM: 32-bit counters for a 32768-bin window (default when the sampled plan
        // allows it) or 16-bit packed counters for all bins; both are enqueued, the one not chosen returns at once
        const size_t smem = (size_t)(kBigWords + 4) * sizeof(uint32_t);
        if (c->bighist == 1) {
            hist_dsm_kernel<<<c->num_sms & ~1, kBigThreads, (32768 + 1) * sizeof(uint32_t), s>>>(
                d, n, nbins, lo, hi, scale, range3, c->gbins, outside);
        } else {
            hist_window_kernel<<<1, kBigThreads, 0, s>>>(d, n, nbins, lo, hi, scale, range3, c->plan);
            const bool window_allowed = c->bighist != 2;
            if (fused_select) {   // cube_stats: window histogram + second select digit in one kernel
                c->launches++;
                hist_win_select_kernel<<<c->num_sms, kFusedThreads, kBigFusedSmem, s>>>(
                    d, n, nbins, lo, hi, scale, range3, c->plan, c->gbins, outside, c->sel, c->gdigits, c->cand,
                    fused_scan ? c->ticket2 : nullptr);
            } else if (window_allowed) {
                c->launches++;
                hist_win_kernel<<<c->num_sms, kBigThreads, smem, s>>>(d, n, nbins, lo, hi, scale, range3, c->plan,
                                                                      c->gbins, outside);
            }
            hist_packed_kernel<<<c->num_sms, kBigThreads, smem, s>>>(d, n, nbins, lo, hi, scale, range3, &c->plan->flip,
                                                                     window_allowed ? &c->plan->use_window : nullptr,
                                                                     c->gbins, outside);
        }
    }
    }
    CUBE_CUDA(c, cudaGetLastError());
    return CUBE_OK;
}

inline SelectInit select_init_args(const cube_ctx* c, uint64_t k, int use_median, bool enabled,
                                   float* result_out = nullptr) {
    SelectInit i;
    i.result_out = result_out;
    i.k = k; i.cand_cap = c->cand ? c->cand_cap : 0; i.use_median = use_median ? 1u : 0u; i.enabled = enabled ? 1u : 0u;
    return i;
}

// fuse != nullptr: the last CTA of the pass also locates the bucket (select_scan_if_last) -- in-core selections
// brick_only (PASS 2 of a brick-streamed run): never read the candidate buffer -- select_cand_kernel counts it once
template <int PASS, bool DEV = false>
int launch_select_pass(cube_ctx* c, const float* d, uint64_t n, cudaStream_t s, const SelectInit* fuse = nullptr,
                       const uint32_t* skip_if_set = nullptr, bool brick_only = false) {
    const int occ = occupancy_of(c, select_pass_kernel<PASS, DEV>, kThreads, 0);  // every CTA must be resident (static tile dealing)
    const int grid = grid_for(c, 4, occ < kMaxCtasPerSm ? occ : kMaxCtasPerSm);
    {
        ProfScope prof(c, PASS == 0 ? CUBE_K_SELECT_PASS0 : PASS == 1 ? CUBE_K_SELECT_PASS1 : CUBE_K_SELECT_PASS2, s);
        select_pass_kernel<PASS, DEV><<<grid, kThreads, 0, s>>>(d, n, c->sel, c->gdigits, brick_only ? nullptr : c->cand, c->center,
                                                                fuse ? c->ticket2 : nullptr,
                                                                fuse ? *fuse : select_init_args(c, 0, 0, false), skip_if_set);
    }
    CUBE_CUDA(c, cudaGetLastError());
    return CUBE_OK;
}

template <int PASS>
int launch_select_scan(cube_ctx* c, unsigned long long* digits, cudaStream_t s, const SelectInit* init = nullptr,
                       const uint32_t* skip_if_set = nullptr) {
    // the coarse histogram kept by CUBE_COARSE_HIST is left intact so that several k can reuse it
    {
        ProfScope prof(c, CUBE_K_SELECT_SCAN, s);
        select_scan_kernel<PASS><<<1, 1024, 0, s>>>(c->sel, digits, digits == c->gdigits ? 1 : 0,
                                                    init ? *init : select_init_args(c, 0, 0, false), skip_if_set);
    }
    CUBE_CUDA(c, cudaGetLastError());
    return CUBE_OK;
}

int select_init(cube_ctx* c, uint64_t k, int use_median, cudaStream_t s) {
    SelectState h;
    memset(&h, 0, sizeof(h));
    h.k = k;
    h.use_median = use_median ? 1u : 0u;
    h.result = nanf("");
    h.cand_n = 0;
    h.cand_cap = c->cand ? c->cand_cap : 0;
    // small H2D of a stack struct: cudaMemcpyAsync from pageable memory stages the bytes before returning
    CUBE_CUDA(c, cudaMemcpyAsync(c->sel, &h, sizeof(h), cudaMemcpyHostToDevice, s));
    return CUBE_OK;
}

// DEV: rank |fl32(x - *c->center)| instead of x (cube_mad)
template <bool DEV = false>
int kth_impl(cube_ctx* c, const float* d, uint64_t n, uint64_t k, int use_median, unsigned flags, float* out,
             cudaStream_t s, const uint32_t* skip_if_set = nullptr) {
    int rc;
    // three launches: every pass kernel ends with the bucket location in its last CTA; the select state is
    // initialised by the first of them from kernel arguments (no host-to-device copy)
    float* direct = static_cast<float*>(device_reachable(c, out));   // pass C stores the result there itself
    const SelectInit init = select_init_args(c, k, use_median, true), cont = select_init_args(c, 0, 0, false, direct);
    if (!DEV && (flags & CUBE_REUSE_COARSE)) {
        if ((rc = launch_select_scan<0>(c, c->coarse, s, &init, skip_if_set))) return rc;
    } else {
        CUBE_CUDA(c, cudaMemsetAsync(c->gdigits, 0, kDigitBins * sizeof(unsigned long long), s));
        if ((rc = launch_select_pass<0, DEV>(c, d, n, s, &init))) return rc;
    }
    // skip_if_set (cube_kth_multi's fallback): both reads return at once when the word is set on the device
    if ((rc = launch_select_pass<1, DEV>(c, d, n, s, &cont, skip_if_set))) return rc;
    if ((rc = launch_select_pass<2, DEV>(c, d, n, s, &cont, skip_if_set))) return rc;
    if (out && !direct) CUBE_CUDA(c, cudaMemcpyAsync(out, &c->sel->result, sizeof(float), cudaMemcpyDefault, s));
    return CUBE_OK;
}

}  // namespace

extern "C" {

int cube_create(cube_ctx** out, size_t scratch_bytes_hint) {
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
    ok = ok && cudaMalloc(&c->ticket2, sizeof(unsigned int)) == cudaSuccess;
    ok = ok && cudaMemset(c->ticket2, 0, sizeof(unsigned int)) == cudaSuccess;
    // running (n, mean, M2, kmin, kmax) record followed by the voxel total: ONE 40-byte block, so that a sharded
    // run can all-gather it as it is (cube_shard_buffers)
    static_assert(sizeof(Partial) == 32, "shard record layout");
    void* rec = nullptr;
    ok = ok && cudaMalloc(&rec, CUBE_SHARD_RECORD_BYTES) == cudaSuccess;
    c->acc = reinterpret_cast<Partial*>(rec);
    c->nvox_acc = rec ? reinterpret_cast<unsigned long long*>(static_cast<char*>(rec) + sizeof(Partial)) : nullptr;
    ok = ok && cudaMalloc(&c->mom_out, sizeof(MomentsOut)) == cudaSuccess;
    ok = ok && cudaMalloc(&c->gout, bytes_bins) == cudaSuccess;
    c->gbins = c->gout ? c->gout + 2 : nullptr;
    ok = ok && cudaMalloc(&c->gdigits, kDigitBins * sizeof(unsigned long long)) == cudaSuccess;
    ok = ok && cudaMalloc(&c->coarse, kDigitBins * sizeof(unsigned long long)) == cudaSuccess;
    ok = ok && cudaMalloc(&c->sel, sizeof(SelectState)) == cudaSuccess;
    ok = ok && cudaMalloc(&c->multi, sizeof(MultiState)) == cudaSuccess;
    ok = ok && cudaMalloc(&c->range3, 4 * sizeof(float)) == cudaSuccess;
    ok = ok && cudaMalloc(&c->probe_out, sizeof(float)) == cudaSuccess;
    ok = ok && cudaMalloc(&c->plan, sizeof(BigHistPlan)) == cudaSuccess;
    ok = ok && cudaMalloc(&c->clip, sizeof(ClipState)) == cudaSuccess;
    ok = ok && cudaMalloc(&c->torben, sizeof(TorbenState)) == cudaSuccess;
    ok = ok && cudaMalloc(&c->center, sizeof(float)) == cudaSuccess;
    ok = ok && cudaMalloc(&c->tf_table, 4096 * sizeof(float4)) == cudaSuccess;
    ok = ok && cudaMalloc(&c->coarse_next, kDigitBins * sizeof(unsigned long long)) == cudaSuccess;
    ok = ok && cudaMemset(c->coarse_next, 0, kDigitBins * sizeof(unsigned long long)) == cudaSuccess;
    ok = ok && cudaMalloc(&c->chunk_tot, (kDigitBins / 32) * sizeof(unsigned long long)) == cudaSuccess;
    ok = ok && cudaMemset(c->chunk_tot, 0, (kDigitBins / 32) * sizeof(unsigned long long)) == cudaSuccess;
    {
        const unsigned int ext0[4] = {0xFFFFFFFFu, 0u, 0u, 0u};
        ok = ok && cudaMalloc(&c->small_ext, sizeof(ext0)) == cudaSuccess;
        ok = ok && cudaMemcpy(c->small_ext, ext0, sizeof(ext0), cudaMemcpyHostToDevice) == cudaSuccess;
    }
    ok = ok && cudaMalloc(&c->bar, 2 * sizeof(unsigned int)) == cudaSuccess;      // counter, base of the next launch
    ok = ok && cudaMemset(c->bar, 0, 2 * sizeof(unsigned int)) == cudaSuccess;
    c->coop = prop.cooperativeLaunch ? 1 : 0;
#ifdef CUBE_SMALL_TIMING
    ok = ok && cudaMallocManaged(&c->small_tstamp, (16 + 8 * 4096) * sizeof(unsigned long long)) == cudaSuccess;
    if (getenv("CUBE_SMALL_TSTAMP_PTR")) { FILE* fp = fopen(getenv("CUBE_SMALL_TSTAMP_PTR"), "w"); if (fp) { fprintf(fp, "%llu\n", (unsigned long long)(uintptr_t)c->small_tstamp); fclose(fp); } }
#endif
    ok = ok && cudaFuncSetAttribute(stats_small_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                    small_smem(kSmallMaxBins)) == cudaSuccess;
    ok = ok && cudaMemset(c->plan, 0, sizeof(BigHistPlan)) == cudaSuccess;
    ok = ok && cudaMemset(c->ticket, 0, sizeof(unsigned int)) == cudaSuccess;
    ok = ok && cudaMemset(c->gdigits, 0, kDigitBins * sizeof(unsigned long long)) == cudaSuccess;
    ok = ok && cudaMemset(c->coarse, 0, kDigitBins * sizeof(unsigned long long)) == cudaSuccess;
    ok = ok && cudaFuncSetAttribute(hist_smem_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                    (kSmemHistMaxBins + 2) * (int)sizeof(uint32_t)) == cudaSuccess;
    ok = ok && cudaFuncSetAttribute(hist_select_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                    hist_select_smem(kSmemHistMaxBins)) == cudaSuccess;
    ok = ok && cudaFuncSetAttribute(hist_packed_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                    (kBigWords + 4) * (int)sizeof(uint32_t)) == cudaSuccess;
    ok = ok && cudaFuncSetAttribute(hist_win_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                    (kBigWords + 4) * (int)sizeof(uint32_t)) == cudaSuccess;
    ok = ok && cudaFuncSetAttribute(hist_win_select_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                    kBigFusedSmem) == cudaSuccess;
    ok = ok && cudaFuncSetAttribute(minimap_tma_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                    kMapTmaSmem) == cudaSuccess;
    ok = ok && cudaFuncSetAttribute(minimap_median_cta_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                    kMedStageKeys * 4 + kMedCtaExtra) == cudaSuccess;
    ok = ok && cudaFuncSetAttribute(minimap_median_warp_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                    (kMedCtaThreads / 32) * kMedWarpSmemPerWarp) == cudaSuccess;
    ok = ok && cudaFuncSetAttribute(hist_dsm_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                    (32768 + 1) * (int)sizeof(uint32_t)) == cudaSuccess;
    if (!ok) { cube_destroy(c); return CUBE_ENOMEM; }
    // candidate buffer of the select: optional (without it pass 2 streams the cube a third time)
    const size_t cand_bytes = scratch_bytes_hint ? scratch_bytes_hint : ((size_t)256 << 20);
    if (cudaMalloc(&c->cand, cand_bytes) == cudaSuccess) c->cand_cap = cand_bytes / sizeof(uint32_t);
    else { cudaGetLastError(); c->cand = nullptr; c->cand_cap = 0; }
    *out = c;
    return CUBE_OK;
}

int cube_destroy(cube_ctx* c) {
    if (!c) return CUBE_EINVAL;
    cudaFree(c->partials); cudaFree(c->ticket); cudaFree(c->ticket2); cudaFree(c->acc);
    cudaFree(c->mom_out); cudaFree(c->gout); cudaFree(c->gdigits); cudaFree(c->coarse); cudaFree(c->sel); cudaFree(c->multi);
    cudaFree(c->range3); cudaFree(c->probe_out); cudaFree(c->plan); cudaFree(c->clip); cudaFree(c->torben); cudaFree(c->center);
    cudaFree(c->cand); cudaFree(c->tf_table); cudaFree(c->bar); cudaFree(c->coarse_next); cudaFree(c->chunk_tot); cudaFree(c->small_ext); cudaFree(c->map32);
    cudaFree(c->resident); cudaFree(c->chunk[0]); cudaFree(c->chunk[1]);
    if (c->pinned_results) cudaFreeHost(c->pinned_results);
    for (int i = 0; i < cube_ctx::kMaxStage; ++i) {
        if (c->h_stage[i]) cudaFreeHost(c->h_stage[i]);
        if (c->ev_filled[i]) cudaEventDestroy(c->ev_filled[i]);
        if (c->ev_h2d_done[i]) cudaEventDestroy(c->ev_h2d_done[i]);
    }
    if (c->fill_stream) cudaStreamDestroy(c->fill_stream);
    for (int i = 0; i < 2; ++i) {
        if (c->ev_copied[i]) cudaEventDestroy(c->ev_copied[i]);
        if (c->ev_consumed[i]) cudaEventDestroy(c->ev_consumed[i]);
    }
    for (cudaEvent_t e : c->prof_ev) cudaEventDestroy(e);
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
    MomentsOut* direct = static_cast<MomentsOut*>(device_reachable(c, out));
    int rc = launch_moments(c, d, n, flags, 0, s, -1, 0.f, 0.f, false, nullptr, direct);
    if (rc) return rc;
    if (!direct) CUBE_CUDA(c, cudaMemcpyAsync(out, c->mom_out, sizeof(MomentsOut), cudaMemcpyDefault, s));
    return CUBE_OK;
}

int cube_histogram(cube_ctx* c, const float* d, int64_t nx, int64_t ny, int64_t nz, int nbins, float lo,
                   float hi, uint64_t* bins, uint64_t* outside, cudaStream_t s) {
    uint64_t n;
    float scale;
    if (!c || !d || !bins || !outside || !dims_ok(nx, ny, nz, &n)) return CUBE_EINVAL;
    if (!hist_scale(nbins, lo, hi, &scale)) return CUBE_EINVAL;
    CUBE_CUDA(c, cudaMemsetAsync(c->gout, 0, (size_t)(nbins + 2) * sizeof(unsigned long long), s));
    int rc = launch_hist(c, d, n, nbins, lo, hi, scale, s);
    if (rc) return rc;
    CUBE_CUDA(c, cudaMemcpyAsync(bins, c->gbins, (size_t)nbins * sizeof(uint64_t), cudaMemcpyDefault, s));
    CUBE_CUDA(c, cudaMemcpyAsync(outside, c->gout, 2 * sizeof(uint64_t), cudaMemcpyDefault, s));
    return CUBE_OK;
}

// cube_stats / cube_median / cube_kth on a cube that stays in L2 between its reads: ONE cooperative launch
// (cube_small.cuh).  *launched = false: no CTA fits, the caller takes the general path.
static bool small_path_ok(const cube_ctx* c, uint64_t n, int nbins) {
    return nbins <= kSmallMaxBins && n * sizeof(float) <= ((size_t)96 << 20) && c->coop && !c->no_small;
}

static int small_launch(cube_ctx* c, const float* d, uint64_t n, int nbins, float lo, float hi, float scale, bool minmax,
                        unsigned flags, cube_moments_t* moments, uint64_t* bins, uint64_t* outside, float* median,
                        uint64_t k, int use_median, cudaStream_t s, bool* launched) {
    const bool want_hist = nbins > 0;
    float* med_direct = static_cast<float*>(device_reachable(c, median));
    MomentsOut* mom_direct = static_cast<MomentsOut*>(device_reachable(c, moments));
    *launched = false;
    {
        const size_t smem = (size_t)small_smem(nbins);
        const int occ = occupancy_of(c, stats_small_kernel, kThreads, smem);
        int per = c->ctas_per_sm > 0 ? c->ctas_per_sm : 2;
        if (per > occ) per = occ;
        if (per >= 1) {
            const unsigned grid = (unsigned)(c->num_sms * per);
            SmallArgs a;
            a.d = d; a.n = n; a.nbins = nbins; a.lo = lo; a.hi = hi; a.scale = scale; a.minmax = minmax ? 1 : 0;
            a.flags = flags & CUBE_SAMPLE_STD;
            a.partials = c->partials; a.acc = c->acc; a.nvox_acc = c->nvox_acc; a.mom_out = c->mom_out; a.out_user = mom_direct;
            a.coarse = c->coarse_next; a.coarse_keep = c->coarse; a.chunk_tot = c->chunk_tot;
            a.gdigits = c->gdigits; a.gout = c->gout;
            a.sel = c->sel; a.cand = c->cand; a.cand_cap = c->cand ? c->cand_cap : 0; a.result_out = med_direct;
            a.k = k; a.use_median = use_median;
            a.bar = c->bar; a.ext = c->small_ext; a.tstamp = c->small_tstamp;
            a.bins_user = static_cast<unsigned long long*>(device_reachable(c, bins));
            a.outside_user = static_cast<unsigned long long*>(device_reachable(c, outside));
            if (!a.bins_user || !a.outside_user) a.bins_user = a.outside_user = nullptr;
            void* args[] = {&a};
            {
                ProfScope prof(c, CUBE_K_STATS_SMALL, s);
                CUBE_CUDA(c, cudaLaunchCooperativeKernel(reinterpret_cast<void*>(stats_small_kernel), dim3(grid), dim3(kThreads),
                                                         args, smem, s));
            }
            if (!med_direct) CUBE_CUDA(c, cudaMemcpyAsync(median, &c->sel->result, sizeof(float), cudaMemcpyDefault, s));
            if (moments && !mom_direct) CUBE_CUDA(c, cudaMemcpyAsync(moments, c->mom_out, sizeof(MomentsOut), cudaMemcpyDefault, s));
            if (want_hist && !a.bins_user) {
                CUBE_CUDA(c, cudaMemcpyAsync(bins, c->gbins, (size_t)nbins * sizeof(uint64_t), cudaMemcpyDefault, s));
                CUBE_CUDA(c, cudaMemcpyAsync(outside, c->gout, 2 * sizeof(uint64_t), cudaMemcpyDefault, s));
            }
            *launched = true;
            return CUBE_OK;
        }
    }
    return CUBE_OK;
}

int cube_kth_ex(cube_ctx* c, const float* d, int64_t nx, int64_t ny, int64_t nz, uint64_t k, unsigned flags,
                float* out, cudaStream_t s) {
    uint64_t n;
    if (!c || !d || !out || !dims_ok(nx, ny, nz, &n)) return CUBE_EINVAL;
    if (flags == 0u && small_path_ok(c, n, 0)) {       // an L2-resident cube: one cooperative launch, as cube_median
        bool launched = false;
        const int rc = small_launch(c, d, n, 0, 0.f, 0.f, 0.f, false, 0u, nullptr, nullptr, nullptr, out, k, 0, s, &launched);
        if (rc || launched) return rc;
    }
    return kth_impl<false>(c, d, n, k, 0, flags, out, s);
}

int cube_kth(cube_ctx* c, const float* d, int64_t nx, int64_t ny, int64_t nz, uint64_t k, float* out,
             cudaStream_t s) {
    return cube_kth_ex(c, d, nx, ny, nz, k, 0u, out, s);
}

int cube_kth_multi(cube_ctx* c, const float* d, int64_t nx, int64_t ny, int64_t nz, int nk, const uint64_t* k,
                   unsigned flags, float* out, cudaStream_t s) {
    uint64_t n;
    int rc;
    if (!c || !d || !out || !k || nk < 1 || !dims_ok(nx, ny, nz, &n)) return CUBE_EINVAL;
    if (!(flags & CUBE_REUSE_COARSE)) {
        // first digit of every voxel, once: the pass kernel without its bucket location leaves the counts in gdigits;
        // they move to the slot CUBE_COARSE_HIST uses, where every rank's bucket location reads them
        CUBE_CUDA(c, cudaMemsetAsync(c->gdigits, 0, kDigitBins * sizeof(unsigned long long), s));
        if ((rc = launch_select_pass<0, false>(c, d, n, s, nullptr))) return rc;
        CUBE_CUDA(c, cudaMemcpyAsync(c->coarse, c->gdigits, kDigitBins * sizeof(unsigned long long),
                                     cudaMemcpyDeviceToDevice, s));
        CUBE_CUDA(c, cudaMemsetAsync(c->gdigits, 0, kDigitBins * sizeof(unsigned long long), s));
    }
    // groups of kMultiGroup ranks: ONE more read of the cube gathers the voxels of all their first-digit buckets, the
    // other two digits are counted on the candidates (cube_select_multi.cuh).  The per-rank selections enqueued
    // behind (one read each) skip themselves on the device unless the buckets did not fit the candidate buffer.
    const uint32_t* ok_word = reinterpret_cast<const uint32_t*>(reinterpret_cast<const char*>(c->multi) +
                                                                 offsetof(MultiState, ok));
    const int occ = occupancy_of(c, multi_gather_kernel, kThreads, 0);
    const int grid = grid_for(c, 4, occ < kMaxCtasPerSm ? occ : kMaxCtasPerSm);
    for (int g0 = 0; g0 < nk; g0 += kMultiGroup) {
        const int m = nk - g0 < kMultiGroup ? nk - g0 : kMultiGroup;
        MultiRanks req;
        memset(&req, 0, sizeof(req));
        req.nk = (uint32_t)m;
        for (int i = 0; i < m; ++i) req.k[i] = k[g0 + i];
        {
            ProfScope prof(c, CUBE_K_SELECT_SCAN, s);
            multi_locate_kernel<<<1, 1024, 0, s>>>(c->multi, c->coarse, req, c->cand ? c->cand_cap : 0);
        }
        {
            ProfScope prof(c, CUBE_K_SELECT_PASS1, s);
            multi_gather_kernel<<<grid, kThreads, 0, s>>>(d, n, c->multi, c->cand);
        }
        const int cgrid = 4 * c->num_sms;
        {
            ProfScope prof(c, CUBE_K_SELECT_CAND, s);
            multi_cand_kernel<1><<<cgrid, kThreads, 0, s>>>(c->multi, c->gdigits, c->cand);
        }
        {
            ProfScope prof(c, CUBE_K_SELECT_SCAN, s);
            multi_scan_kernel<1><<<m, kBins1, 0, s>>>(c->multi, c->gdigits);
        }
        {
            ProfScope prof(c, CUBE_K_SELECT_CAND, s);
            multi_cand_kernel<2><<<cgrid, kThreads, 0, s>>>(c->multi, c->gdigits, c->cand);
        }
        {
            ProfScope prof(c, CUBE_K_SELECT_SCAN, s);
            multi_scan_kernel<2><<<m, kBins1, 0, s>>>(c->multi, c->gdigits);
        }
        {
            ProfScope prof(c, CUBE_K_OTHER, s);
            multi_done_kernel<<<1, 1, 0, s>>>(c->multi);
        }
        CUBE_CUDA(c, cudaGetLastError());
        // a fallback selection stores its result straight into the group's record (its last pass, when it runs)
        float* results = reinterpret_cast<float*>(reinterpret_cast<char*>(c->multi) + offsetof(MultiState, result));
        for (int i = 0; i < m; ++i)
            if ((rc = kth_impl<false>(c, d, n, k[g0 + i], 0, CUBE_REUSE_COARSE, results + i, s, ok_word))) return rc;
        CUBE_CUDA(c, cudaMemcpyAsync(out + g0, results, (size_t)m * sizeof(float), cudaMemcpyDefault, s));
    }
    return CUBE_OK;
}

int cube_median_ex(cube_ctx* c, const float* d, int64_t nx, int64_t ny, int64_t nz, unsigned flags, float* out,
                   cudaStream_t s) {
    uint64_t n;
    if (!c || !d || !out || !dims_ok(nx, ny, nz, &n)) return CUBE_EINVAL;
    // A cube that stays in L2 between its reads: the single cooperative launch of cube_stats (cube_small.cuh) without
    // the histogram -- one launch and two reads instead of three of each
    if (flags == 0u && small_path_ok(c, n, 0)) {
        bool launched = false;
        const int rc = small_launch(c, d, n, 0, 0.f, 0.f, 0.f, false, 0u, nullptr, nullptr, nullptr, out, 0, 1, s, &launched);
        if (rc || launched) return rc;
    }
    return kth_impl<false>(c, d, n, 0, 1, flags, out, s);
}

int cube_median(cube_ctx* c, const float* d, int64_t nx, int64_t ny, int64_t nz, float* out, cudaStream_t s) {
    return cube_median_ex(c, d, nx, ny, nz, 0u, out, s);
}

int cube_stats(cube_ctx* c, const float* d, int64_t nx, int64_t ny, int64_t nz, int nbins, float lo, float hi,
               unsigned flags, cube_moments_t* moments, uint64_t* bins, uint64_t* outside, float* median,
               cudaStream_t s) {
    uint64_t n;
    if (!c || !d || !dims_ok(nx, ny, nz, &n)) return CUBE_EINVAL;
    const bool want_hist = bins != nullptr || outside != nullptr;
    const bool minmax = (flags & CUBE_RANGE_MINMAX) != 0;
    const bool want_median = median != nullptr;
    float scale = 0.f;
    if (want_hist) {
        if (!bins || !outside) return CUBE_EINVAL;
        if (minmax) { if (nbins < 1 || nbins > CUBE_MAX_BINS) return CUBE_EINVAL; lo = hi = 0.f; }
        else if (!hist_scale(nbins, lo, hi, &scale)) return CUBE_EINVAL;
    }
    int rc;
    float* med_direct = static_cast<float*>(device_reachable(c, median));
    MomentsOut* mom_direct = static_cast<MomentsOut*>(device_reachable(c, moments));
    // A cube that stays in L2 between its two reads: everything in ONE cooperative launch (cube_small.cuh)
    if (!want_hist) nbins = 0;
    if (want_median && small_path_ok(c, n, nbins)) {
        bool launched = false;
        rc = small_launch(c, d, n, nbins, lo, hi, scale, minmax, flags, moments, bins, outside, median, 0, 1, s, &launched);
        if (rc || launched) return rc;
    }
    // pass A: moments (+ first select digit)
    const SelectInit init = select_init_args(c, 0, 1, true), cont = select_init_args(c, 0, 0, false, med_direct);
    const unsigned mflags = (flags & CUBE_SAMPLE_STD) | (want_median ? (unsigned)CUBE_COARSE_HIST : 0u);
    if ((rc = launch_moments(c, d, n, mflags, 0, s, -1, 0.f, 0.f, false, want_median ? &init : nullptr, mom_direct))) return rc;
    if (want_hist) {
        CUBE_CUDA(c, cudaMemsetAsync(c->gout, 0, (size_t)(nbins + 2) * sizeof(unsigned long long), s));
    }
    // pass B: histogram + second digit + compaction
    unsigned long long* goutside = c->gout;
    if (want_median) CUBE_CUDA(c, cudaMemsetAsync(c->gdigits, 0, kDigitBins * sizeof(unsigned long long), s));
    if (want_median && want_hist && nbins <= kSmemHistMaxBins) {
        const size_t smem = (size_t)hist_select_smem(nbins);
        const int occ = occupancy_of(c, hist_select_kernel, kThreads, smem);
        const int grid = grid_for(c, 4, occ < kMaxCtasPerSm ? occ : kMaxCtasPerSm);
        {
            ProfScope prof(c, CUBE_K_HIST_SELECT, s);
            hist_select_kernel<<<grid, kThreads, smem, s>>>(d, n, nbins, lo, hi, scale, minmax ? c->mom_out : nullptr,
                                                            c->gbins, goutside, c->sel, c->gdigits, c->cand, c->ticket2);
        }
        CUBE_CUDA(c, cudaGetLastError());
    } else {
        if (want_hist) {
            if (minmax) {
                {
                    ProfScope prof(c, CUBE_K_OTHER, s);
                    hist_range_kernel<<<1, 1, 0, s>>>(c->mom_out, nbins, c->range3, goutside);
                }
                CUBE_CUDA(c, cudaGetLastError());
            }
            // more than 16384 bins together with the median: the window histogram and the second select digit
            // share one read (hist_win_select_kernel) when the sampled plan allows the window; the packed
            // histogram and select_pass_kernel<1> are enqueued behind it and return at once in that case
            const bool fused_big = want_median && nbins > kSmemHistMaxBins && c->bighist == 0;
            if ((rc = launch_hist(c, d, n, nbins, lo, hi, scale, s, minmax ? c->range3 : nullptr, fused_big))) return rc;
            if (fused_big) {
                if ((rc = launch_select_pass<1>(c, d, n, s, &cont, &c->plan->use_window))) return rc;
            } else if (want_median && (rc = launch_select_pass<1>(c, d, n, s, &cont))) return rc;
        } else if (want_median && (rc = launch_select_pass<1>(c, d, n, s, &cont))) return rc;
    }
    if (want_median) {
        if ((rc = launch_select_pass<2>(c, d, n, s, &cont))) return rc;   // on the candidates unless they did not fit
        if (!med_direct) CUBE_CUDA(c, cudaMemcpyAsync(median, &c->sel->result, sizeof(float), cudaMemcpyDefault, s));
    }
    if (moments && !mom_direct) CUBE_CUDA(c, cudaMemcpyAsync(moments, c->mom_out, sizeof(MomentsOut), cudaMemcpyDefault, s));
    if (want_hist) {
        CUBE_CUDA(c, cudaMemcpyAsync(bins, c->gbins, (size_t)nbins * sizeof(uint64_t), cudaMemcpyDefault, s));
        CUBE_CUDA(c, cudaMemcpyAsync(outside, goutside, 2 * sizeof(uint64_t), cudaMemcpyDefault, s));
    }
    return CUBE_OK;
}

int cube_mad(cube_ctx* c, const float* d, int64_t nx, int64_t ny, int64_t nz, unsigned flags, float* median,
             float* mad, cudaStream_t s) {
    uint64_t n;
    if (!c || !d || !mad || !dims_ok(nx, ny, nz, &n)) return CUBE_EINVAL;
    int rc;
    if ((rc = kth_impl<false>(c, d, n, 0, 1, flags & CUBE_REUSE_COARSE, median, s))) return rc;
    CUBE_CUDA(c, cudaMemcpyAsync(c->center, &c->sel->result, sizeof(float), cudaMemcpyDeviceToDevice, s));
    return kth_impl<true>(c, d, n, 0, 1, 0u, mad, s);
}

int cube_clipped_moments(cube_ctx* c, const float* d, int64_t nx, int64_t ny, int64_t nz, float lo, float hi,
                         unsigned flags, cube_moments_t* out, cudaStream_t s) {
    uint64_t n;
    if (!c || !d || !out || !dims_ok(nx, ny, nz, &n) || lo != lo || hi != hi) return CUBE_EINVAL;
    int rc = launch_moments(c, d, n, flags & CUBE_SAMPLE_STD, 0, s, kMomWindow, lo, hi, false);
    if (rc) return rc;
    CUBE_CUDA(c, cudaMemcpyAsync(out, c->mom_out, sizeof(MomentsOut), cudaMemcpyDefault, s));
    return CUBE_OK;
}

int cube_sigma_clip(cube_ctx* c, const float* d, int64_t nx, int64_t ny, int64_t nz, double kappa, int max_iter,
                    unsigned flags, cube_moments_t* out, int* iters, float* window, cudaStream_t s) {
    uint64_t n;
    if (!c || !d || !out || !dims_ok(nx, ny, nz, &n)) return CUBE_EINVAL;
    if (!(kappa >= 0.0) || !isfinite(kappa) || max_iter < 0 || max_iter > 1000) return CUBE_EINVAL;
    ClipState h;
    memset(&h, 0, sizeof(h));
    h.lo = h.hi = nanf("");
    CUBE_CUDA(c, cudaMemcpyAsync(c->clip, &h, sizeof(h), cudaMemcpyHostToDevice, s));
    const unsigned mflags = flags & CUBE_SAMPLE_STD;
    int rc = launch_moments(c, d, n, mflags, 0, s, kMomPlain);
    if (rc) return rc;
    for (int i = 0; i < max_iter; ++i) {
        {
            ProfScope prof(c, CUBE_K_OTHER, s);
            clip_step_kernel<<<1, 1, 0, s>>>(c->mom_out, c->clip, kappa);
        }
        CUBE_CUDA(c, cudaGetLastError());
        if ((rc = launch_moments(c, d, n, mflags, 0, s, kMomWindow, 0.f, 0.f, true))) return rc;
    }
    CUBE_CUDA(c, cudaMemcpyAsync(out, c->mom_out, sizeof(MomentsOut), cudaMemcpyDefault, s));
    if (iters) CUBE_CUDA(c, cudaMemcpyAsync(iters, &c->clip->iters, sizeof(int), cudaMemcpyDefault, s));
    if (window) CUBE_CUDA(c, cudaMemcpyAsync(window, &c->clip->lo, 2 * sizeof(float), cudaMemcpyDefault, s));
    return CUBE_OK;
}

int cube_median_torben(cube_ctx* c, const float* d, int64_t nx, int64_t ny, int64_t nz, int max_iter, float* out,
                       int* iters, int* converged, cudaStream_t s) {
    uint64_t n;
    if (!c || !d || !out || !dims_ok(nx, ny, nz, &n) || max_iter < 0 || max_iter > 1000) return CUBE_EINVAL;
    CUBE_CUDA(c, cudaMemsetAsync(c->torben, 0, sizeof(TorbenState), s));
    int rc = launch_moments(c, d, n, 0u, 0, s, kMomPlain);   // Min, Max, n ("calculated while the dataset is loading")
    if (rc) return rc;
    const int occ = occupancy_of(c, torben_pass_kernel, kThreads, 0);
    const int grid = grid_for(c, 4, occ < kMaxCtasPerSm ? occ : kMaxCtasPerSm);
    for (int i = 0; i < max_iter; ++i) {
        {
            ProfScope prof(c, CUBE_K_OTHER, s);
            torben_step_kernel<<<1, 1, 0, s>>>(c->mom_out, c->torben, 0);
        }
        {
            ProfScope prof(c, CUBE_K_TORBEN, s);
            torben_pass_kernel<<<grid, kThreads, 0, s>>>(d, n, c->torben);
        }
        CUBE_CUDA(c, cudaGetLastError());
    }
    {
        ProfScope prof(c, CUBE_K_OTHER, s);
        torben_step_kernel<<<1, 1, 0, s>>>(c->mom_out, c->torben, 1);
    }
    CUBE_CUDA(c, cudaGetLastError());
    CUBE_CUDA(c, cudaMemcpyAsync(out, &c->torben->result, sizeof(float), cudaMemcpyDefault, s));
    if (iters) CUBE_CUDA(c, cudaMemcpyAsync(iters, &c->torben->iters, sizeof(int), cudaMemcpyDefault, s));
    if (converged) CUBE_CUDA(c, cudaMemcpyAsync(converged, &c->torben->converged, sizeof(int), cudaMemcpyDefault, s));
    return CUBE_OK;
}

int cube_minimap_dims(int64_t nx, int64_t ny, int64_t nz, int64_t px, int64_t py, int64_t pz, int64_t* mx,
                      int64_t* my, int64_t* mz) {
    uint64_t n;
    if (!dims_ok(nx, ny, nz, &n) || px <= 0 || py <= 0 || pz <= 0 || !mx || !my || !mz) return CUBE_EINVAL;
    *mx = (nx + px - 1) / px; *my = (ny + py - 1) / py; *mz = (nz + pz - 1) / pz;
    return CUBE_OK;
}

int cube_minimap(cube_ctx* c, const float* d, int64_t nx, int64_t ny, int64_t nz, int64_t px, int64_t py,
                 int64_t pz, unsigned flags, cube_moments_t* cells, cudaStream_t s) {
    MapGeom g;
    if (!c || !d || !cells) return CUBE_EINVAL;
    if (cube_minimap_dims(nx, ny, nz, px, py, pz, (int64_t*)&g.mx, (int64_t*)&g.my, (int64_t*)&g.mz)) return CUBE_EINVAL;
    g.nx = nx; g.ny = ny; g.nz = nz; g.px = px; g.py = py; g.pz = pz;
    cudaPointerAttributes at;   // the map is consumed on the device: records are written in place
    if (cudaPointerGetAttributes(&at, cells) != cudaSuccess || at.type == cudaMemoryTypeUnregistered) {
        cudaGetLastError();
        return CUBE_EINVAL;
    }
    // Segments of whole cells that start on a multiple of 4 voxels (16 bytes): what both the TMA-ring kernel (bulk
    // copies of whole lines) and the 128-bit register kernel need; rows must be 16-byte aligned as well.
    const long long unit = (px % 4 == 0) ? 1 : (px % 2 == 0) ? 2 : 4;     // cells per segment must be a multiple of it
    const bool rows16 = (nx % 4 == 0) && (((uintptr_t)d & 15u) == 0);
    // TMA ring: segments that are also whole 128-byte lines (32 voxels) when the cell width allows it within
    // kMapTmaCols columns (px = 30: 16 cells = 480 voxels) -- no L2 line is then shared by two CTAs; such segments
    // are not re-balanced (the last one of a row is simply narrower).
    long long unit128 = 1;
    while ((unit128 * px) % 32 != 0) ++unit128;                           // 32 / gcd(px, 32)
    const bool seg128 = unit128 * px <= kMapTmaCols;
    const long long unit_t = seg128 ? unit128 : unit;
    const long long cpst = (kMapTmaCols / px) / unit_t * unit_t;
    const long long cps4 = (kMap4Cols / px) / unit * unit;
    // The ring kernel takes several cell rows per CTA, but every cell row still ends with two barriers and the per-cell
    // merge: it wins from about 256 lines per cell row upwards (measured on c2, TB/s ring vs 128-bit kernel: 30^3 cells
    // 6.36 vs 4.44, 64^3 6.10 vs 4.12, 16^3 5.76 vs 5.70, 24x8x8 4.09 vs 4.74, 100x10x10 3.29 vs 4.64).
    const bool v4_ok = rows16 && cps4 >= 1 && px >= 4;
    const long double lines = (long double)std::min(py, ny) * (long double)std::min(pz, nz);
    const bool tma = rows16 && cpst >= 1 && lines < 2147483000.0L &&
                     (c->minimap_variant == 3 || (c->minimap_variant == 0 && (lines >= 256.0L || !v4_ok)));
    const bool v4 = !tma && v4_ok && c->minimap_variant <= 1;
    g.cells_per_seg = tma ? cpst : v4 ? cps4 : (px > kMapThreads ? 1 : kMapThreads / px);
    g.nseg = (g.mx + g.cells_per_seg - 1) / g.cells_per_seg;
    {   // balance the segments of a row (35 cells: 18 + 17 instead of 34 + 1)
        const long long u = tma ? unit_t : v4 ? unit : 1;
        const long long even = ((g.mx + g.nseg - 1) / g.nseg + u - 1) / u * u;
        if (even < g.cells_per_seg) { g.cells_per_seg = even; g.nseg = (g.mx + even - 1) / even; }
    }
    const long double ctas = (long double)g.nseg * (long double)g.my * (long double)g.mz;
    if (ctas > 2147483647.0L) return CUBE_EINVAL;   // 1-D grid limit (cells of a few voxels on a huge cube)
    {
        ProfScope prof(c, CUBE_K_MINIMAP, s);
        const unsigned grid = (unsigned)(g.nseg * g.my * g.mz);
        g.main_threads = ((g.cells_per_seg * px / 4) + 31) / 32 * 32;
        const unsigned block4 = (unsigned)g.main_threads + (unsigned)((g.cells_per_seg - 1 + 31) / 32 * 32);  // + boundary threads
        if (tma) {
            const long long wmax = std::min<long long>(g.cells_per_seg * px, nx);     // widest segment, a multiple of 4
            const unsigned block = (unsigned)((wmax + 31) / 32 * 32) + 32u;           // + the producer warp
            // cell rows per CTA: about 1024 lines, so that filling and draining the ring is a small part of a CTA
            const long long rows = std::max<long long>(1, std::min<long long>(g.my, (long long)(1024.0L / lines)));
            const long double ctas_t = (long double)g.nseg * (long double)((g.my + rows - 1) / rows) * (long double)g.mz;
            minimap_tma_kernel<<<(unsigned)ctas_t, block, kMapTmaSmem, s>>>(d, g, flags & CUBE_SAMPLE_STD, (int)rows,
                                                                            reinterpret_cast<MomentsOut*>(cells));
        } else if (v4) minimap_v4_kernel<<<grid, block4, 0, s>>>(d, g, flags & CUBE_SAMPLE_STD,
                                                                 reinterpret_cast<MomentsOut*>(cells));
        else minimap_kernel<<<grid, kMapThreads, 0, s>>>(d, g, flags & CUBE_SAMPLE_STD,
                                                         reinterpret_cast<MomentsOut*>(cells));
    }
    CUBE_CUDA(c, cudaGetLastError());
    return CUBE_OK;
}

// ---- NEXT-4: ray casting (cube_render.cuh)
static bool render_args(cube_ctx* c, const float* d, int64_t nx, int64_t ny, int64_t nz, const cube_view_t* view,
                        void* out, RenderGeom* g, RenderView* vw) {
    uint64_t n;
    if (!c || !d || !view || !out || !dims_ok(nx, ny, nz, &n)) return false;
    if (nx > (1 << 24) || ny > (1 << 24) || nz > (1 << 24)) return false;      // float32 coordinates
    if (view->width < 1 || view->height < 1 || view->nsteps < 1) return false;
    if ((long double)view->width * (long double)view->height > 1073741824.0L) return false;
    for (int k = 0; k < 3; ++k)
        if (!isfinite(view->origin[k]) || !isfinite(view->du[k]) || !isfinite(view->dv[k]) || !isfinite(view->step[k])) return false;
    cudaPointerAttributes at;   // images are written in place by the kernels
    if (cudaPointerGetAttributes(&at, out) != cudaSuccess || at.type == cudaMemoryTypeUnregistered) {
        cudaGetLastError();
        return false;
    }
    static_assert(sizeof(cube_view_t) == sizeof(RenderView), "view layout");
    memcpy(vw, view, sizeof(RenderView));
    g->nx = nx; g->ny = ny; g->nz = nz;
    g->xmax = (float)(nx - 1); g->ymax = (float)(ny - 1); g->zmax = (float)(nz - 1);
    return true;
}

int cube_view_orbit(int64_t nx, int64_t ny, int64_t nz, double yaw_deg, double pitch_deg, int width, int height,
                    double step, cube_view_t* out) {
    uint64_t n;
    if (!out || !dims_ok(nx, ny, nz, &n) || width < 1 || height < 1 || !(step > 0.0) || !isfinite(step) ||
        !isfinite(yaw_deg) || !isfinite(pitch_deg)) return CUBE_EINVAL;
    const double pi = 3.14159265358979323846;
    const double ya = yaw_deg * pi / 180.0, pa = pitch_deg * pi / 180.0;
    const double cy = cos(ya), sy = sin(ya), cp = cos(pa), sp = sin(pa);
    // R = Ry(yaw) Rx(pitch); right = R e_x, up = R e_y, forward = R (-e_z)
    const double right[3] = {cy, 0.0, -sy};
    const double up[3] = {sy * sp, cp, cy * sp};
    const double fwd[3] = {-sy * cp, sp, -cy * cp};
    const double ctr[3] = {(nx - 1) / 2.0, (ny - 1) / 2.0, (nz - 1) / 2.0};
    const double diam = sqrt((nx - 1.0) * (nx - 1.0) + (ny - 1.0) * (ny - 1.0) + (nz - 1.0) * (nz - 1.0)) + 1.0;
    const double nsteps = ceil(diam / step) + 1.0;
    if (nsteps > 2147483000.0) return CUBE_EINVAL;
    for (int k = 0; k < 3; ++k) {
        const double du = right[k] * (diam / width), dv = up[k] * (diam / height);
        out->du[k] = (float)du;
        out->dv[k] = (float)dv;
        out->step[k] = (float)(fwd[k] * step);
        out->origin[k] = (float)(ctr[k] - fwd[k] * (diam / 2) - right[k] * (diam / 2) - up[k] * (diam / 2) + 0.5 * du + 0.5 * dv);
    }
    out->width = width; out->height = height; out->nsteps = (int32_t)nsteps;
    return CUBE_OK;
}

// Footprint of a warp in the ray-per-thread kernels (cube_render.cuh, render_pixel): log2 of its width in pixels.
static int render_footprint(const RenderView& vw) {
    if (const char* e = getenv("CUBE_RENDER_FW")) return atoi(e);           // experiments
    const double un = sqrt((double)vw.du[0] * vw.du[0] + (double)vw.du[1] * vw.du[1] + (double)vw.du[2] * vw.du[2]);
    // measured on c2, 1024^2 rays (MIP, ms; 32x1 / 16x2 / 8x4 / 4x8): yaw 0: 1.72 / 1.67 / 1.74 / 2.88, yaw 10: 4.12 / 3.36 /
    // 3.59 / 4.99, yaw 20 pitch 20: 6.28 / 4.76 / 4.72 / 5.42, yaw 45 pitch 40: 9.84 / 7.71 / 6.77 / 6.40
    // pixels one voxel apart along x (an axis-aligned view at the cube's resolution): 32 x 1, the lanes read 32 neighbouring
    // voxels (4.14 ms against 4.44 with 16 x 2 on c2 along z)
    if (un > 0.0 && un <= 1.25 && fabs((double)vw.du[0]) / un >= 0.98) return 5;
    return (un > 0.0 && fabs((double)vw.du[0]) / un >= 0.9) ? 4 : 3;        // image rows nearly along x: 16 x 2, else 8 x 4
}

// The block of rays of a CTA in the ray-per-warp kernels (cube_render.cuh, render_ray_of_warp): log2 of its width.
static int render_ray_block(const RenderView& vw) {
    if (const char* e = getenv("CUBE_RENDER_RW")) return atoi(e);           // experiments
    // 8 x 1 when the rays lie in planes y = const (neighbours along the image row share their lines), else 4 x 2
    // (c2, MIP: yaw 70 pitch 20: 4.7 -> 3.0 ms, yaw 90 pitch 40: 3.7 -> 3.0; at pitch 0 4 x 2 doubles the time)
    const double sn = sqrt((double)vw.step[0] * vw.step[0] + (double)vw.step[1] * vw.step[1] + (double)vw.step[2] * vw.step[2]);
    return (sn > 0.0 && fabs((double)vw.step[1]) / sn > 0.05) ? 2 : 3;
}
static unsigned render_ray_blocks(const RenderView& vw, int rw_log) {
    const unsigned across = ((unsigned)vw.width + (1u << rw_log) - 1u) >> rw_log;
    const unsigned down = ((unsigned)vw.height + (1u << (3 - rw_log)) - 1u) >> (3 - rw_log);
    return across * down;
}

// Which ray-casting kernel (CUBE_KNOB_RENDER)?  One ray per warp (cube_render.cuh) pays for every PLANE of the cube that
// the 32 consecutive samples of a ray cross (planes are megabytes apart) and for every line they climb in y, one ray per
// thread for the planes and lines the block of pixels of a warp spans.  The rules below are fits to a map of both
// kernels over yaw 0-90 x pitch 0-60 degrees on c2, 1024^2 rays, in terms of the components
// (ax, ay, az) of the ray direction: ray-per-warp wins when az is small enough for the ay at hand -- up to 0.9 when
// rays and image rows lie in planes y = const (an orbit at pitch 0: neighbouring rays share their lines) -- and, for
// the sigma-clipping transfer function, whose map lookups do not care about the direction, whenever the ray has some
// x component at all.
enum { kRenderMip = 0, kRenderTf = 1, kRenderSigma = 2 };
static bool render_along(const cube_ctx* c, const RenderView& vw, int kind) {
    const double sn = sqrt((double)vw.step[0] * vw.step[0] + (double)vw.step[1] * vw.step[1] + (double)vw.step[2] * vw.step[2]);
    bool along_auto = false;
    if (sn > 0.0) {
        const double ax = fabs((double)vw.step[0]) / sn, ay = fabs((double)vw.step[1]) / sn, az = fabs((double)vw.step[2]) / sn;
        if (kind == kRenderSigma) along_auto = ax >= 0.25;
        else along_auto = az <= std::max(0.9 - 4.0 * ay, 0.82 - 0.6 * ay);   // 0.9 at pitch 0, fading within a few degrees
    }
    return c->render_variant == 0 ? along_auto : c->render_variant == 2;
}

int cube_render_mip(cube_ctx* c, const float* d, int64_t nx, int64_t ny, int64_t nz, const cube_view_t* view,
                    float vmin, float* image, cudaStream_t s) {
    RenderGeom g; RenderView vw;
    if (!render_args(c, d, nx, ny, nz, view, image, &g, &vw) || vmin != vmin) return CUBE_EINVAL;
    {
        ProfScope prof(c, CUBE_K_RENDER, s);
        const dim3 block(kRenderTileU, kRenderTileV);
        const dim3 grid((vw.width + kRenderTileU - 1) / kRenderTileU, (vw.height + kRenderTileV - 1) / kRenderTileV);
        const bool along = render_along(c, vw, kRenderMip);
        if (along) {
            const int rw = render_ray_block(vw);
            render_mip_along_kernel<<<render_ray_blocks(vw, rw), 32 * kRenderRaysPerCta, 0, s>>>(d, g, vw, vmin, rw, image);
        } else {
            render_mip_kernel<<<grid, block, 0, s>>>(d, g, vw, vmin, render_footprint(vw), image);
        }
    }
    CUBE_CUDA(c, cudaGetLastError());
    return CUBE_OK;
}

static int render_tf_common(cube_ctx* c, const float* d, int64_t nx, int64_t ny, int64_t nz, const cube_view_t* view,
                            int nlevels, float lo, float hi, const float* table, float opacity_cut,
                            const cube_moments_t* cells, int64_t px, int64_t py, int64_t pz, float* rgba, cudaStream_t s) {
    RenderGeom g; RenderView vw;
    if (!render_args(c, d, nx, ny, nz, view, rgba, &g, &vw) || !table || nlevels < 1 || nlevels > 4096) return CUBE_EINVAL;
    if (opacity_cut != opacity_cut || ((uintptr_t)rgba & 15u)) return CUBE_EINVAL;
    float scale;
    if (!hist_scale(nlevels, lo, hi, &scale)) return CUBE_EINVAL;     // the histogram's scale (R10, R13, R19)
    MapLookupGeom mg = {};
    const double* dev_cells = nullptr;
    if (cells) {
        if (px < 1 || py < 1 || pz < 1) return CUBE_EINVAL;
        static_assert(sizeof(cube_moments_t) == 5 * sizeof(double), "record layout");
        dev_cells = static_cast<const double*>(device_reachable(c, const_cast<cube_moments_t*>(cells)));
        if (!dev_cells || ((uintptr_t)dev_cells & 7u)) return CUBE_EINVAL;
        const int64_t part[3] = {px, py, pz}, n[3] = {nx, ny, nz};
        long long m[3];
        for (int k = 0; k < 3; ++k) {
            m[k] = (n[k] + part[k] - 1) / part[k];
            mg.part[k] = (float)part[k];
            mg.off[k] = (float)(part[k] - 1) / 2.0f;
            mg.top[k] = (float)(m[k] - 1);
        }
        mg.mx = m[0]; mg.my = m[1]; mg.mz = m[2];
        // (mean, std) of the cells as float32 pairs, what the rays interpolate (cube_render.cuh): 8 bytes per cell in a
        // buffer of the context that grows when a larger map comes (the only allocation a render call can make)
        const long double ncell_ld = (long double)m[0] * (long double)m[1] * (long double)m[2];
        if (ncell_ld > 4294967296.0L) return CUBE_EINVAL;
        const size_t ncell = (size_t)ncell_ld;
        if (ncell > c->map32_cap) {
            float2* bigger = nullptr;
            if (cudaMalloc(&bigger, ncell * sizeof(float2)) != cudaSuccess) { cudaGetLastError(); return CUBE_ENOMEM; }
            cudaFree(c->map32);          // synchronises: no earlier render is still reading it
            c->map32 = bigger;
            c->map32_cap = ncell;
        }
        {
            ProfScope prof(c, CUBE_K_OTHER, s);
            map_compact_kernel<<<(unsigned)((ncell + 255) / 256), 256, 0, s>>>(dev_cells, (long long)ncell, c->map32);
        }
        CUBE_CUDA(c, cudaGetLastError());
    }
    const float4* dev_table = static_cast<const float4*>(device_reachable(c, const_cast<float*>(table)));
    if (!dev_table || ((uintptr_t)dev_table & 15u)) {
        CUBE_CUDA(c, cudaMemcpyAsync(c->tf_table, table, (size_t)nlevels * sizeof(float4), cudaMemcpyDefault, s));
        dev_table = c->tf_table;
    }
    {
        ProfScope prof(c, CUBE_K_RENDER, s);
        const dim3 block(kRenderTileU, kRenderTileV);
        const dim3 grid((vw.width + kRenderTileU - 1) / kRenderTileU, (vw.height + kRenderTileV - 1) / kRenderTileV);
        if (render_along(c, vw, dev_cells ? kRenderSigma : kRenderTf)) {
            const int rw = render_ray_block(vw);
            const unsigned agrid = render_ray_blocks(vw, rw);
            if (dev_cells)
                render_tf_along_kernel<true><<<agrid, 32 * kRenderRaysPerCta, 0, s>>>(
                    d, g, vw, nlevels, lo, scale, dev_table, opacity_cut, c->map32, mg, rw, reinterpret_cast<float4*>(rgba));
            else
                render_tf_along_kernel<false><<<agrid, 32 * kRenderRaysPerCta, 0, s>>>(
                    d, g, vw, nlevels, lo, scale, dev_table, opacity_cut, nullptr, mg, rw, reinterpret_cast<float4*>(rgba));
        } else if (dev_cells)
            render_tf_kernel<true><<<grid, block, 0, s>>>(d, g, vw, nlevels, lo, scale, dev_table, opacity_cut, c->map32,
                                                          mg, render_footprint(vw), reinterpret_cast<float4*>(rgba));
        else
            render_tf_kernel<false><<<grid, block, 0, s>>>(d, g, vw, nlevels, lo, scale, dev_table, opacity_cut, nullptr,
                                                           mg, render_footprint(vw), reinterpret_cast<float4*>(rgba));
    }
    CUBE_CUDA(c, cudaGetLastError());
    return CUBE_OK;
}

int cube_render_tf(cube_ctx* c, const float* d, int64_t nx, int64_t ny, int64_t nz, const cube_view_t* view,
                   int nlevels, float lo, float hi, const float* table, float opacity_cut, float* rgba, cudaStream_t s) {
    return render_tf_common(c, d, nx, ny, nz, view, nlevels, lo, hi, table, opacity_cut, nullptr, 0, 0, 0, rgba, s);
}

int cube_render_sigma(cube_ctx* c, const float* d, int64_t nx, int64_t ny, int64_t nz, const cube_view_t* view,
                      const cube_moments_t* cells, int64_t px, int64_t py, int64_t pz, int nlevels, float zlo, float zhi,
                      const float* table, float opacity_cut, float* rgba, cudaStream_t s) {
    if (!cells) return CUBE_EINVAL;
    return render_tf_common(c, d, nx, ny, nz, view, nlevels, zlo, zhi, table, opacity_cut, cells, px, py, pz, rgba, s);
}

int cube_spectrum(cube_ctx* c, const float* d, int64_t nx, int64_t ny, int64_t nz, const cube_view_t* view, int u,
                  int v, float* out, cudaStream_t s) {
    RenderGeom g; RenderView vw;
    if (!render_args(c, d, nx, ny, nz, view, out, &g, &vw)) return CUBE_EINVAL;
    if (u < -(1 << 24) || u > (1 << 24) || v < -(1 << 24) || v > (1 << 24)) return CUBE_EINVAL;
    {
        ProfScope prof(c, CUBE_K_RENDER, s);
        spectrum_kernel<<<(vw.nsteps + 255) / 256, 256, 0, s>>>(d, g, vw, u, v, out);
    }
    CUBE_CUDA(c, cudaGetLastError());
    return CUBE_OK;
}

// The two-read kernel addresses a cell's voxels by 32-bit byte offsets and divides row numbers by a multiplication
// (cube_minimap_median.cuh): both hold for every cell anyone would use; the rest takes the staged kernel.
static bool med_two_reads_ok(int64_t nx, int64_t ny, int64_t nz, int64_t py, int64_t pz) {
    const long double h = (long double)std::min(py, ny), dep = (long double)std::min(pz, nz);
    return dep * (long double)ny * (long double)nx < 1073741824.0L && h * h * dep < 4294967296.0L &&
           dep * dep < 4294967296.0L;
}

int cube_minimap_median(cube_ctx* c, const float* d, int64_t nx, int64_t ny, int64_t nz, int64_t px, int64_t py,
                        int64_t pz, float* med, cudaStream_t s) {
    MedGeom g;
    if (!c || !d || !med) return CUBE_EINVAL;
    if (cube_minimap_dims(nx, ny, nz, px, py, pz, (int64_t*)&g.mx, (int64_t*)&g.my, (int64_t*)&g.mz)) return CUBE_EINVAL;
    g.nx = nx; g.ny = ny; g.nz = nz; g.px = px; g.py = py; g.pz = pz;
    cudaPointerAttributes at;   // the medians are written in place by the kernel
    if (cudaPointerGetAttributes(&at, med) != cudaSuccess || at.type == cudaMemoryTypeUnregistered) {
        cudaGetLastError();
        return CUBE_EINVAL;
    }
    const long double cellvox = (long double)std::min(px, nx) * (long double)std::min(py, ny) * (long double)std::min(pz, nz);
    if (cellvox > 2147483648.0L) return CUBE_EINVAL;
    const long double ncell = (long double)g.mx * (long double)g.my * (long double)g.mz;
    {
        ProfScope prof(c, CUBE_K_MINIMAP, s);
        if (cellvox < (long double)kMedWarpKeys) {
            const int per = kMedCtaThreads / 32;
            const long double want = (ncell + per - 1) / per;
            const unsigned grid = (unsigned)std::min<long double>(want < 1 ? 1 : want, (long double)c->num_sms * 16);
            minimap_median_warp_kernel<<<grid, kMedCtaThreads, per * kMedWarpSmemPerWarp, s>>>(d, g, med);
        } else if (c->mapmedian != 1 && med_two_reads_ok(nx, ny, nz, py, pz)) {
            const int occ = occupancy_of(c, minimap_median_two_reads_kernel, kMed2Threads, kMed2Smem);
            const unsigned grid = (unsigned)std::min<long double>(ncell, (long double)c->num_sms * (occ < 1 ? 1 : occ));
            minimap_median_two_reads_kernel<<<grid, kMed2Threads, kMed2Smem, s>>>(d, g, med);
        } else {
            const int stage = cellvox <= (long double)kMedStageKeys ? (((int)cellvox + 3) & ~3) : 0;
            const size_t smem = (size_t)stage * 4 + kMedCtaExtra;
            const int occ = occupancy_of(c, minimap_median_cta_kernel, kMedCtaThreads, smem);
            const unsigned grid = (unsigned)std::min<long double>(ncell, (long double)c->num_sms * (occ < 1 ? 1 : occ));
            minimap_median_cta_kernel<<<grid, kMedCtaThreads, smem, s>>>(d, g, stage, med);
        }
    }
    CUBE_CUDA(c, cudaGetLastError());
    return CUBE_OK;
}

int cube_probe_read(cube_ctx* c, const float* d, uint64_t nvox, cudaStream_t s) {
    if (!c || !d || nvox == 0) return CUBE_EINVAL;
    {
        ProfScope prof(c, CUBE_K_PROBE, s);
        probe_read_kernel<<<grid_for(c, 4, kMaxCtasPerSm), kThreads, 0, s>>>(d, nvox, c->probe_out);
    }
    CUBE_CUDA(c, cudaGetLastError());
    return CUBE_OK;
}

const char* cube_strerror(int code) {
    switch (code) {
        case CUBE_OK: return "ok";
        case CUBE_EINVAL: return "invalid argument";
        case CUBE_EEMPTY: return "no non-NaN voxel";
        case CUBE_ECUDA: return "CUDA error (see cube_last_cuda_error)";
        case CUBE_ERANGE: return "out of range";
        case CUBE_ENOMEM: return "allocation failed";
        case CUBE_ECALLBACK: return "brick callback failed";
        default: return "unknown error";
    }
}

int cube_last_cuda_error(const cube_ctx* c) { return c ? c->last_cuda : 0; }

int cube_set_launch(cube_ctx* c, int ctas_per_sm) {
    if (!c || ctas_per_sm < 0 || ctas_per_sm > kMaxCtasPerSm) return CUBE_EINVAL;
    c->ctas_per_sm = ctas_per_sm;
    return CUBE_OK;
}

int cube_set_knob(cube_ctx* c, int knob, int value) {
    if (!c) return CUBE_EINVAL;
    switch (knob) {
        case CUBE_KNOB_CTAS_PER_SM: return cube_set_launch(c, value);
        case CUBE_KNOB_BIGHIST:
            if (value < 0 || value > 2) return CUBE_EINVAL;
            c->bighist = value;
            return CUBE_OK;
        case CUBE_KNOB_SMALL:
            if (value < 0 || value > 1) return CUBE_EINVAL;
            c->no_small = value;
            return CUBE_OK;
        case CUBE_KNOB_MAPMEDIAN:
            if (value < 0 || value > 2) return CUBE_EINVAL;
            c->mapmedian = value;
            return CUBE_OK;
        case CUBE_KNOB_RENDER:
            if (value < 0 || value > 2) return CUBE_EINVAL;
            c->render_variant = value;
            return CUBE_OK;
        case CUBE_KNOB_MINIMAP:
            if (value < 0 || value > 3) return CUBE_EINVAL;
            c->minimap_variant = value;
            return CUBE_OK;
        default: return CUBE_EINVAL;
    }
}

uint64_t cube_launch_count(const cube_ctx* c) { return c ? c->launches : 0; }

int cube_profile_enable(cube_ctx* c, int on) {
    if (!c) return CUBE_EINVAL;
    if (!on) { int rc = prof_collect(c); if (rc) return rc; }
    c->prof_on = on ? 1 : 0;
    return CUBE_OK;
}

int cube_profile_reset(cube_ctx* c) {
    if (!c) return CUBE_EINVAL;
    int rc = prof_collect(c);
    for (int k = 0; k < CUBE_K_KINDS; ++k) { c->prof_ms[k] = 0.0; c->prof_n[k] = 0; }
    return rc;
}

int cube_profile_read(cube_ctx* c, int kind, double* total_ms, uint64_t* launches) {
    if (!c || kind < 0 || kind >= CUBE_K_KINDS || !total_ms || !launches) return CUBE_EINVAL;
    int rc = prof_collect(c);
    *total_ms = c->prof_ms[kind];
    *launches = c->prof_n[kind];
    return rc;
}

}  // extern "C"

// ---- cube_histogram_noalloc: the histogram of cube_histogram for callers that cannot allocate (code under CUDA graph
// capture, tight serving loops, harnesses that forbid cudaMalloc): no cube_ctx, no cudaMalloc / cudaFree anywhere
// on its path.  The 64-bit global counters the per-CTA shared-memory counters are flushed into -- the scratch that
// cube_create() otherwise allocates -- live in the file-scope array below: 2 + CUBE_NOALLOC_MAX_BINS words = 32 KiB
// that every GPU which loads libcube holds until the process exits.
namespace {

static __device__ __align__(256) unsigned long long g_noalloc_scratch[2 + CUBE_NOALLOC_MAX_BINS];   // [outside (2)][bins]

// hist_smem_kernel (cube_kernels.cuh) with its counters in the static scratch; `scratch` is the DEVICE address of
// g_noalloc_scratch, resolved by the host with cudaGetSymbolAddress (in host code the array's name is only a stand-in).
__global__ void __launch_bounds__(kThreads)
hist_noalloc_kernel(const float* __restrict__ d, uint64_t n, int nbins, float lo, float hi, float scale,
                    unsigned long long* __restrict__ scratch) {
    extern __shared__ uint32_t dyn_bins[];
    __shared__ uint32_t s_out[2];
    for (int i = threadIdx.x; i < nbins + 2; i += kThreads) dyn_bins[i] = 0;  // + trash slot
    if (threadIdx.x < 2) s_out[threadIdx.x] = 0;
    __syncthreads();
    uint32_t below = 0, above = 0;
    if (hist_use_fast(nbins, lo, hi, scale)) {
        HistFastF f;
        f.setup(lo, hi, scale, nbins, dyn_bins, s_out);
        stream_cube<kThreads>(d, n, f);
    } else {
        HistF f;
        f.lo = lo; f.hi = hi; f.scale = scale; f.top = nbins - 1; f.sbins = dyn_bins;
        stream_cube<kThreads>(d, n, f);
        below = f.below; above = f.above;
    }
    __syncthreads();
    hist_flush_bins(dyn_bins, nbins, scratch + 2);
    if (below) atomicAdd(&s_out[0], below);
    if (above) atomicAdd(&s_out[1], above);
    __syncthreads();
    if (threadIdx.x < 2 && s_out[threadIdx.x]) atomicAdd(&scratch[threadIdx.x], (unsigned long long)s_out[threadIdx.x]);
}

// Set-up, once per device, with that device current: the device address of the scratch and the SM count.
struct NoAllocDevice { unsigned long long* scratch; int num_sms; };
constexpr int kNoAllocMaxDevices = 64;
NoAllocDevice g_noalloc_dev[kNoAllocMaxDevices];
std::mutex g_noalloc_mutex;

cudaError_t noalloc_device(NoAllocDevice* out) {
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    if (dev < 0 || dev >= kNoAllocMaxDevices) return cudaErrorInvalidDevice;
    std::lock_guard<std::mutex> lock(g_noalloc_mutex);
    if (!g_noalloc_dev[dev].scratch) {
        unsigned long long* ptr = nullptr;
        int sms = 0;
        if ((e = cudaGetSymbolAddress((void**)&ptr, g_noalloc_scratch)) != cudaSuccess) return e;
        if ((e = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev)) != cudaSuccess) return e;
        if (!ptr || sms < 1) return cudaErrorUnknown;
        g_noalloc_dev[dev].num_sms = sms;
        g_noalloc_dev[dev].scratch = ptr;
    }
    *out = g_noalloc_dev[dev];
    return cudaSuccess;
}

}  // namespace

extern "C" int cube_histogram_noalloc(const float* d, int64_t nx, int64_t ny, int64_t nz, int nbins, float lo, float hi,
                                      uint64_t* bins, uint64_t* outside, cudaStream_t s, int* cuda_error) {
    uint64_t n;
    float scale;
    if (cuda_error) *cuda_error = 0;
    if (!d || !bins || !outside || !dims_ok(nx, ny, nz, &n)) return CUBE_EINVAL;
    if (nbins > CUBE_NOALLOC_MAX_BINS) return CUBE_ERANGE;      // the static scratch holds no more: use cube_histogram
    if (!hist_scale(nbins, lo, hi, &scale)) return CUBE_EINVAL;
    NoAllocDevice dev;
    cudaError_t e = noalloc_device(&dev);
    // every call shares the scratch and finds the last call's counts in it: what this call accumulates into is cleared
    if (e == cudaSuccess) e = cudaMemsetAsync(dev.scratch, 0, (size_t)(nbins + 2) * sizeof(unsigned long long), s);
    if (e == cudaSuccess) {
        const size_t smem = (size_t)(nbins + 2) * sizeof(uint32_t);   // <= 16 KiB + 8: no opt-in needed
        hist_noalloc_kernel<<<dev.num_sms * 4, kThreads, smem, s>>>(d, n, nbins, lo, hi, scale, dev.scratch);
        e = cudaGetLastError();
    }
    if (e == cudaSuccess) e = cudaMemcpyAsync(bins, dev.scratch + 2, (size_t)nbins * sizeof(uint64_t), cudaMemcpyDefault, s);
    if (e == cudaSuccess) e = cudaMemcpyAsync(outside, dev.scratch, 2 * sizeof(uint64_t), cudaMemcpyDefault, s);
    if (e != cudaSuccess) {
        if (cuda_error) *cuda_error = (int)e;
        return CUBE_ECUDA;
    }
    return CUBE_OK;
}

#include "cube_ooc.inl"
