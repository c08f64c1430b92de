/* cube.h -- C ABI of libcube: global statistics of a float32 spectral cube on one B200.
 *
 * The operations are the "quantitative" tasks of arXiv:1211.4896 (cited as PAPER.md:<line> of
 * /root/reference/PAPER.md):
 *   - global mean / standard deviation (+ count of non-null voxels, min, max)   PAPER.md:263-275 (sec. 4.2),
 *     min/max "calculated while the dataset is loading"
 *   - global intensity histogram                                                PAPER.md:257-261 (sec. 4.1, Fig. 4)
 *   - exact global median / k-th value                                          PAPER.md:277-296 (sec. 4.3),
 *     Alg. 1; here reached by a 13/10/9-bit radix select on
 *     order-preserving keys instead of ~31 bisection passes
 *   - NULL (undefined) voxels are excluded from every statistic
 *     (NULL == IEEE NaN of any sign/payload, reading R6)
 *
 * Conventions
 *   - `d` is a DEVICE pointer to nx*ny*nz float32 voxels, x fastest, then y, then z. It is never
 *     written (the paper keeps the cube read-only) and stays owned by the caller.
 *     Any 4-byte alignment is accepted. All results are order independent, so only N = nx*ny*nz matters.
 *   - Every output pointer (`out`, `bins`, `outside`) may be a device pointer, pinned host memory or
 *     pageable host memory (detected by the driver through unified addressing). Results are produced
 *     on the device and copied with cudaMemcpyAsync on `stream`: for device/pinned destinations the
 *     call returns without synchronising the host; for pageable host memory the copy (and therefore
 *     the call) completes before returning.
 *   - All work is enqueued on `stream`; there is no hidden allocation after cube_create().
 *     A cube_ctx must not be used from two streams/threads at the same time.
 *   - Counts are 64-bit everywhere (N up to 2^37).
 *   - Return value: 0 (CUBE_OK) or a CUBE_E* code; never throws, exits or prints.
 *     Argument errors are detected before any work is enqueued.
 *   - There is NO CPU fallback: without a CUDA device cube_create() fails with CUBE_ECUDA.
 */
#ifndef CUBE_H_
#define CUBE_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#ifndef __DRIVER_TYPES_H__
typedef struct CUstream_st* cudaStream_t;
#endif

typedef struct cube_ctx cube_ctx; /* opaque; owns all device scratch (partials, bins, select state) */

enum {
    CUBE_OK = 0,
    CUBE_EINVAL = 1, /* null pointer, dim <= 0, nbins out of range, !(lo <= hi), non-finite lo/hi/scale */
    CUBE_EEMPTY = 2, /* reserved: not returned by the asynchronous calls (see cube_moments) */
    CUBE_ECUDA = 3,  /* a CUDA call failed; cube_last_cuda_error() gives the cudaError_t */
    CUBE_ERANGE = 4, /* a size beyond a fixed maximum (cube_histogram_noalloc: nbins > CUBE_NOALLOC_MAX_BINS) */
    CUBE_ENOMEM = 5, /* host or device allocation failed */
    CUBE_ECALLBACK = 6 /* the brick callback of cube_stats_stream returned non-zero */
};

/* flags */
enum {
    CUBE_SAMPLE_STD = 1u,  /* std = sqrt(M2/(n-1)) instead of the population sqrt(M2/n); n==1 -> NaN */
    CUBE_COARSE_HIST = 2u, /* cube_moments: also accumulate the first radix-select digit histogram
                              (8192 bins of key>>19) in the same pass and keep it in the context */
    CUBE_REUSE_COARSE = 4u,/* cube_kth_ex/cube_median_ex: skip the first select pass and use the digit
                              histogram left by the last cube_moments(CUBE_COARSE_HIST) or cube_stats(median)
                              call on the SAME data (the caller vouches for that) */
    CUBE_RANGE_MINMAX = 8u /* cube_stats: histogram over [data min, data max] (found by its first pass, never
                              leaves the device) instead of the lo/hi arguments */
};

#define CUBE_MAX_BINS 65536

typedef struct {
    uint64_t count;     /* voxels that are not NaN */
    uint64_t nan_count; /* NaN (blanked) voxels; count + nan_count == nx*ny*nz */
    float min, max;     /* extrema in IEEE total order (-0.0 < +0.0); NaN when count == 0 */
    double mean, std;   /* NaN when count == 0 */
} cube_moments_t;

/* Create a context on the CURRENT device. `scratch_bytes_hint` sizes the optional candidate buffer of
 * the select in bytes (0 = default, 256 MiB = 64 Mi keys); everything else is fixed size (< 4 MiB).
 * The buffer only saves a pass: when the median's first-digit bucket does not fit, the cube is read a third time. */
int cube_create(cube_ctx** out, size_t scratch_bytes_hint);
int cube_destroy(cube_ctx* ctx);

/* PAPER.md:263-275, 261. One streaming pass: count, nan_count, min, max, mean, std.
 * mean and std are accumulated in fp64 about per-thread pivots and merged with the pairwise
 * (n, mean, M2) update in a fixed tree (deterministic run to run); |rel. error| << 1e-9.
 * An all-NaN (or empty-of-values) cube gives count = 0 and NaN min/max/mean/std; the call still
 * returns CUBE_OK because the result is only known on the device. */
int cube_moments(cube_ctx* ctx, const float* d, int64_t nx, int64_t ny, int64_t nz, unsigned flags,
                 cube_moments_t* out, cudaStream_t stream);

/* PAPER.md:257-261. bins[b] = #{x : lo <= x <= hi, bin(x) == b}, 0 <= b < nbins, with
 *   bin(x) = min( floor( (x - lo) * ((float)nbins / (hi - lo)) ), nbins-1 )
 * every operation rounded to float32, no FMA contraction; hi == lo puts every in-range voxel in bin 0.
 * outside[0] = #{x < lo}, outside[1] = #{x > hi}; NaN voxels are counted nowhere, so
 * sum(bins) + outside[0] + outside[1] == count.  1 <= nbins <= CUBE_MAX_BINS. */
int cube_histogram(cube_ctx* ctx, const float* d, int64_t nx, int64_t ny, int64_t nz, int nbins, float lo,
                   float hi, uint64_t* bins /* [nbins] */, uint64_t* outside /* [2] */, cudaStream_t stream);

/* cube_histogram for callers that must not allocate (code under CUDA graph capture, tight serving loops, harnesses
 * that forbid cudaMalloc).  Same bins and outside counts as cube_histogram, bit for bit, but NO
 * cube_ctx and no cudaMalloc / cudaFree / allocating library call on its path: the 64-bit global counters the kernel
 * accumulates into are a file-scope `static __device__` array of the library, 2 + CUBE_NOALLOC_MAX_BINS words =
 * 32 KiB that every GPU which loads libcube holds until the process exits.  The work runs on the CURRENT device
 * (whose memory d must be); the first call on a device resolves the array's device address (cudaGetSymbolAddress,
 * checked) -- make that call outside a capture.  Enqueued on `stream`: a memset of the counters in use, one kernel,
 * two copies to `bins` [nbins] and `outside` [2] (device, pinned or pageable host memory; under capture: device or
 * pinned).  1 <= nbins <= CUBE_NOALLOC_MAX_BINS: more bins -> CUBE_ERANGE, nothing enqueued (use cube_histogram);
 * other argument errors -> CUBE_EINVAL as cube_histogram.  A failed CUDA call -> CUBE_ECUDA with the cudaError_t
 * in *cuda_error (may be NULL).  EVERY call on a device shares the one array, which keeps the last call's counts
 * until the next call clears them: calls that overlap on the GPU (two streams, or two threads on two streams) RACE
 * and give wrong counts -- keep them on one stream or order them with events. */
#define CUBE_NOALLOC_MAX_BINS 4096
int cube_histogram_noalloc(const float* d, int64_t nx, int64_t ny, int64_t nz, int nbins, float lo, float hi,
                           uint64_t* bins /* [nbins] */, uint64_t* outside /* [2] */, cudaStream_t stream,
                           int* cuda_error);

/* PAPER.md:277-296. *out = the element of rank k (0-based) of the non-NaN voxels sorted ascending in
 * IEEE total order. Exact. If k >= count (known only on the device) *out = NaN. */
int cube_kth(cube_ctx* ctx, const float* d, int64_t nx, int64_t ny, int64_t nz, uint64_t k, float* out,
             cudaStream_t stream);
int cube_kth_ex(cube_ctx* ctx, const float* d, int64_t nx, int64_t ny, int64_t nz, uint64_t k, unsigned flags,
                float* out, cudaStream_t stream);

/* Several ranks of the same cube (config 3 of BASELINE.json asks for the median and the values at n/100 and
 * 99n/100): out[i] = the element of rank k[i], i < nk, each exactly what cube_kth gives (NaN for k[i] >= count).
 * The first select digit is counted ONCE (read 1); then, per group of up to four ranks, ONE more read gathers the
 * keys of the voxels of all their first-digit buckets into the context's candidate buffer and the other two digits
 * are counted there: 1 + ceil(nk/4) reads instead of 2 nk.  If a group's buckets do not fit the candidate buffer
 * (cube_create's scratch_bytes_hint; decided on the device, no host synchronisation) each of its ranks costs one
 * more read.  `k` is a HOST array read before the call returns; `out` (nk floats) may be device, pinned or pageable
 * host memory.  The first-digit histogram stays in the context as after CUBE_COARSE_HIST; with CUBE_REUSE_COARSE in
 * `flags` the one already there is used (read 1 is skipped; the caller vouches that it belongs to this cube).
 * nk >= 1.  Like every selection here it replaces the ~31 passes of Alg. 1; the cube is
 * never written. */
int cube_kth_multi(cube_ctx* ctx, const float* d, int64_t nx, int64_t ny, int64_t nz, int nk, const uint64_t* k,
                   unsigned flags, float* out, cudaStream_t stream);

/* Lower median: k = (count-1)/2 with count = number of non-NaN voxels (what Alg. 1, PAPER.md:603-609,
 * returns). count == 0 -> NaN. */
int cube_median(cube_ctx* ctx, const float* d, int64_t nx, int64_t ny, int64_t nz, float* out,
                cudaStream_t stream);
int cube_median_ex(cube_ctx* ctx, const float* d, int64_t nx, int64_t ny, int64_t nz, unsigned flags,
                   float* out, cudaStream_t stream);

/* Everything at once, in TWO reads of the cube (SURVEY.md sec. 8(a) steps 1-8 fused):
 *   pass A  count/min/max/mean/std + first select digit;   pass B  histogram + second digit + compaction of
 *   the median's bucket;   then the last digit on the compacted candidates.
 * Results are those of cube_moments, cube_histogram and cube_median, bit for bit.  Any of `moments`,
 * (`bins`,`outside`) and `median` may be NULL to skip that output (bins and outside go together).
 * flags: CUBE_SAMPLE_STD; CUBE_RANGE_MINMAX = histogram over [min,max] (lo/hi ignored).  With
 * CUBE_RANGE_MINMAX, when there is no non-NaN voxel, an extremum is infinite, or max-min or nbins/(max-min)
 * overflows float32 (the cases cube_histogram rejects with CUBE_EINVAL), all bins are 0 and
 * outside[0] = outside[1] = UINT64_MAX.  More than 16384 bins: still two reads when the voxels concentrate in a
 * window of 32768 consecutive bins (decided on the device from a sample; the usual case for a noise-dominated cube),
 * else a third read (packed histogram and select as separate kernels).  The first-digit histogram stays in the
 * context for cube_kth_ex(..., CUBE_REUSE_COARSE).  A cube of at most 96 MiB (it stays in the L2 cache between the
 * two reads) with at most 4096 bins and the median takes ONE cooperative launch (CUBE_KNOB_SMALL). */
int cube_stats(cube_ctx* ctx, const float* d, int64_t nx, int64_t ny, int64_t nz, int nbins, float lo, float hi,
               unsigned flags, cube_moments_t* moments, uint64_t* bins /* [nbins] */, uint64_t* outside /* [2] */,
               float* median, cudaStream_t stream);

/* ---- Out-of-core / streamed cubes (north_star (4); the paper is in-core by design).
 * The cube is presented brick by brick (any split into contiguous runs of voxels); each brick is a device
 * buffer the caller has filled (e.g. by cudaMemcpyAsync from pinned host memory on a side stream).
 * With the median the bricks are read TWICE, like the cube in cube_stats (8 B per voxel): sweep 1 = moments + first
 * select digit (fused pass A), sweep 2 = histogram + second digit + candidate compaction (fused pass B), then the
 * last digit on the candidates; a third sweep only if the median's first-digit bucket did not fit the candidate
 * buffer.  Without the median: one sweep, moments + histogram.  cube_ooc_next_sweep() tells whether another sweep
 * is needed (*more); the call after sweep 2 synchronises `stream` once to read the "did it fit" decision. */
int cube_ooc_begin(cube_ctx* ctx, int nbins, float lo, float hi, int want_median, cudaStream_t stream);
/* flags: CUBE_RANGE_MINMAX = histogram over [data min, data max] (lo/hi ignored): the range is that of the running
 * record after sweep 1 (in a sharded run: after cube_shard_merge_records), never leaves the device, and the
 * histogram is accumulated in sweep 2 -- which then exists even without the median.  Unusable range: as cube_stats. */
int cube_ooc_begin_ex(cube_ctx* ctx, int nbins, float lo, float hi, int want_median, unsigned flags,
                      cudaStream_t stream);
int cube_ooc_brick(cube_ctx* ctx, const float* d_brick, uint64_t nvox, cudaStream_t stream);
int cube_ooc_next_sweep(cube_ctx* ctx, int* more, cudaStream_t stream);
int cube_ooc_result(cube_ctx* ctx, unsigned flags, cube_moments_t* moments, uint64_t* bins, uint64_t* outside,
                    float* median, cudaStream_t stream);

/* ---- NEXT-3: one cube sharded over several GPUs as contiguous z-slabs, one process
 * and one cube_ctx per GPU -- the paper's client/server decomposition whose merges are
 * "associative and commutative".  libcube itself does no communication: each rank
 * accumulates its slab with cube_ooc_begin() / cube_ooc_brick(), the caller combines the buffers below across ranks
 * with its own collectives on the same stream (paper_1211_4896_b200/shard.py: NCCL through torch.distributed), and
 * cube_shard_advance() then locates the bucket on the combined counts.  Per stage (three for an exact median, one
 * without):
 *     cube_ooc_brick(slab)                                   every rank, its own voxels (several bricks allowed)
 *     stage 0 only:  all-gather `record` (CUBE_SHARD_RECORD_BYTES per rank) -> cube_shard_merge_records()
 *     the stage that accumulates the histogram (stage 1 with the median or CUBE_RANGE_MINMAX, else stage 0):
 *                    all-reduce SUM `bins` (nbins x u64) and `outside` (2 x u64)
 *     every stage with the median:   all-reduce SUM `digits` (CUBE_SHARD_DIGITS x u64)
 *     cube_shard_advance(&more)
 * then cube_ooc_result() on any rank: every rank holds the same integers and, because the records are merged in
 * rank order on every rank, the same mean / std bits.  Three rounds of 64 KiB instead of the paper's ~31 rounds of
 * five scalars.  Every rank reads its slab twice (8 B per voxel).  Each rank counts the last digit
 * on its own compacted candidates ONCE, inside the cube_shard_advance() that ends stage 1; the bricks it presents in
 * stage 2 are read only when the candidates did not fit: decided on the device, no host synchronisation anywhere.
 * A rank without voxels (more ranks than z-planes) presents no brick and still takes part in every collective. */
#define CUBE_SHARD_RECORD_BYTES 40
#define CUBE_SHARD_DIGITS 8192
typedef struct {
    void* record;      /* device: this rank's running {count, mean, M2, min key, max key, voxel total} */
    uint64_t* bins;    /* device: histogram bins (the first nbins of CUBE_MAX_BINS) */
    uint64_t* outside; /* device: [2] */
    uint64_t* digits;  /* device: [CUBE_SHARD_DIGITS] digit counts of the current select pass */
} cube_shard_buffers_t;
int cube_shard_buffers(cube_ctx* ctx, cube_shard_buffers_t* out);
/* `gathered`: device pointer to world x CUBE_SHARD_RECORD_BYTES (rank order).  flags: CUBE_SAMPLE_STD. */
int cube_shard_merge_records(cube_ctx* ctx, const void* gathered, int world, unsigned flags, cudaStream_t stream);
int cube_shard_advance(cube_ctx* ctx, int* more, cudaStream_t stream);

/* Whole-cube convenience over HOST memory (pinned for full speed): streams the cube H2D through
 * double-buffered chunks overlapped with the kernels and returns moments, histogram and the exact lower
 * median in HOST memory. If the cube fits in the device workspace given at cube_host_workspace() it is kept
 * resident after the first sweep, so the host link is crossed once. Synchronises before returning. */
int cube_host_workspace(cube_ctx* ctx, size_t resident_bytes /* 0 = never keep resident */, size_t chunk_bytes);
int cube_stats_host(cube_ctx* ctx, const float* h_cube, int64_t nx, int64_t ny, int64_t nz, int nbins, float lo,
                    float hi, unsigned flags, cube_moments_t* moments, uint64_t* bins, uint64_t* outside,
                    float* median);

/* Cube PRODUCED brick by brick (BASELINE.json config 5: 256 GiB, larger than HBM and than host memory; north_star
 * (4)).  The cube is `nbricks` contiguous runs of voxels, `brick_vox` each (the last one total_vox - (nbricks-1) *
 * brick_vox).  For every brick that has to cross the host link the driver calls
 *     fill(user, brick, sweep, h_dst, nvox, fill_stream)
 * on the calling thread; it must put the brick's nvox float32 voxels into the PINNED HOST buffer h_dst, either
 * before returning or by work enqueued on fill_stream (e.g. a generator kernel plus a device-to-host copy); it
 * returns 0, or non-zero to abort (CUBE_ECALLBACK).  The same brick must get the same bytes in every sweep.
 * h_dst is one of `host_slots` staging buffers owned by the context; the driver blocks the calling thread
 * until the slot's previous host-to-device copy has completed, so at most host_slots bricks are in flight.
 * Pipeline per brick: fill (fill_stream) -> H2D (copy stream) into one of two device brick buffers -> kernels
 * (work stream), all three overlapped.  Sweep 1: moments + histogram + first select digit; sweep 2: second
 * digit + compaction; last digit on the candidates (3 sweeps only if the median's bucket does not fit the
 * candidate buffer).  The first resident_bytes / brick bytes bricks are kept in HBM after sweep 1 and are not
 * asked for again.  Results are those of cube_stats, bit for bit (mean/std to rounding: the merge order is
 * brick order).  Outputs are HOST pointers; synchronises before returning.
 * cube_stream_workspace() allocates (pinned host: host_slots * brick_bytes, 2 <= host_slots <= 8; device:
 * 2 * brick_bytes + resident_bytes); cube_stats_stream() calls it with (brick size, 3, 0) when it has not been. */
typedef int (*cube_fill_fn)(void* user, uint64_t brick, int sweep, float* h_dst, uint64_t nvox, cudaStream_t fill_stream);
int cube_stream_workspace(cube_ctx* ctx, size_t brick_bytes, int host_slots, size_t resident_bytes);
int cube_stats_stream(cube_ctx* ctx, uint64_t nbricks, uint64_t brick_vox, uint64_t total_vox, cube_fill_fn fill,
                      void* user, int nbins, float lo, float hi, unsigned flags, cube_moments_t* moments,
                      uint64_t* bins, uint64_t* outside, float* median);
/* After cube_stats_stream: bytes copied host-to-device and number of sweeps over the bricks. */
int cube_stream_info(const cube_ctx* ctx, uint64_t* h2d_bytes, int* sweeps);

/* ---- NEXT-1: robust noise estimates for source finding.
 *
 * cube_mad: *median = lower median m of the non-NaN voxels (may be NULL), *mad = lower median of
 *   y = |fl32(x - m)| over the non-NaN voxels (one float32 subtraction, sign cleared; R21) -- "easily
 *   modified to address the median absolute deviation".  Two exact selections with the same
 *   radix-select kernels, the second ranking y instead of x: four reads of the cube (three with
 *   CUBE_REUSE_COARSE after cube_moments(CUBE_COARSE_HIST) / cube_stats on the same data).  No non-NaN voxel -> NaN. */
int cube_mad(cube_ctx* ctx, const float* d, int64_t nx, int64_t ny, int64_t nz, unsigned flags, float* median,
             float* mad, cudaStream_t stream);

/* cube_clipped_moments: cube_moments over the voxels with lo <= x <= hi only (closed window, tested on x itself;
 *   NaN fails it).  out->count = voxels in the window, out->nan_count = nx*ny*nz - count = everything left out.
 *   lo > hi selects nothing (count 0, NaN statistics); NaN lo/hi -> CUBE_EINVAL. */
int cube_clipped_moments(cube_ctx* ctx, const float* d, int64_t nx, int64_t ny, int64_t nz, float lo, float hi,
                         unsigned flags, cube_moments_t* out, cudaStream_t stream);

/* cube_sigma_clip: iterated kappa-sigma clipping about the mean (the "Sigma-Clipping" threshold of PAPER.md:336
 *   chosen from mean and standard deviation; R22-R23).  m_0 = cube_moments; for i = 1..max_iter:
 *     lo = fl32(mean - kappa*std), hi = fl32(mean + kappa*std) from m_{i-1} (double product, double sum, one
 *     rounding to float32);  m_i = cube_clipped_moments over [lo, hi];
 *   stops after the first pass whose count equals the previous count, or when count == 0 or std is not finite.
 *   The whole loop stays on the device (no host synchronisation): max_iter + 1 launches over the cube are
 *   enqueued, and those after convergence return at once.  *out = the last statistics, *iters = clipped passes
 *   made (may be NULL), window[2] = the last window used, NaN if none (may be NULL).  All three may be device,
 *   pinned or pageable host memory.  CUBE_SAMPLE_STD applies to every std, including those that form the windows.
 *   0 <= kappa < inf, 0 <= max_iter <= 1000. */
int cube_sigma_clip(cube_ctx* ctx, const float* d, int64_t nx, int64_t ny, int64_t nz, double kappa, int max_iter,
                    unsigned flags, cube_moments_t* out, int* iters, float* window /* [2] */, cudaStream_t stream);

/* cube_median_torben: the paper's own median method, Alg. 1 (Torben's bisection, sec. 4.3), kept
 *   for comparison with the radix select and for the paper's early-stop approximation.  One pass over
 *   the cube per guess -- counts of voxels less / greater / equal, largest voxel below, smallest above -- and a
 *   1-thread kernel between passes in the role of the paper's server; at most max_iter passes
 *   (0..1000) are enqueued, those after the stop test has fired return at once; no host synchronisation.
 *   *out = the exact lower median when the stop test fired (*converged = 1; ~30 passes for float32 data), else the
 *   final selection of Alg. 1 applied to the counts of the last pass made (R26: within (max-min)/2^(p-1)
 *   of the median after p passes).  *iters = passes made.  Comparisons are numeric, so +0.0 and -0.0 are one
 *   value: a zero result carries no sign guarantee.  No non-NaN voxel, or max_iter == 0: NaN.  iters / converged
 *   may be NULL; all outputs device, pinned or pageable host memory. */
int cube_median_torben(cube_ctx* ctx, const float* d, int64_t nx, int64_t ny, int64_t nz, int max_iter, float* out,
                       int* iters, int* converged, cudaStream_t stream);

/* ---- NEXT-2: the statistical mini-map (Fig. 7): one cube_moments_t per partition of
 * px x py x pz voxels ("30x30x30 pixel"), cell (cx,cy,cz) covering x in [cx*px, min((cx+1)*px, nx)) and likewise
 * in y and z (ragged last cells are smaller; R25).  cells[(cz*my + cy)*mx + cx] with mx = ceil(nx/px),
 * my, mz from cube_minimap_dims().  `cells` must be memory the DEVICE can write (device or pinned host memory):
 * the map is consumed on the device (the second trilinear lookup of PAPER.md:354), so records are written in
 * place by the kernel.  One read of the cube.  flags: CUBE_SAMPLE_STD. */
int cube_minimap_dims(int64_t nx, int64_t ny, int64_t nz, int64_t px, int64_t py, int64_t pz, int64_t* mx,
                      int64_t* my, int64_t* mz);
int cube_minimap(cube_ctx* ctx, const float* d, int64_t nx, int64_t ny, int64_t nz, int64_t px, int64_t py,
                 int64_t pz, unsigned flags, cube_moments_t* cells, cudaStream_t stream);

/* ---- NEXT-4: volume ray casting and the 3-D spectrum tool as compute kernels writing into
 * headless buffers (the paper's renderer is CUDA as well; its viewer / window is left out).
 * Geometry (R27): data coordinates are voxel indices -- voxel (i,j,k) sits at (i,j,k) -- and the rays are
 * orthographic.  With every operation a float32 operation in the order written,
 *     first sample of pixel (u,v):  o = (origin + (float)u * du) + (float)v * dv
 *     sample i of that ray:         p = o + (float)i * step,   0 <= i < nsteps
 * a sample is inside iff 0 <= p_x <= nx-1, 0 <= p_y <= ny-1, 0 <= p_z <= nz-1, and its value is the trilinear
 * interpolation of the (up to) eight surrounding voxels, x then y then z, each step a + f * (b - a) (R28);
 * a neighbour of weight zero does not take part; a NULL (NaN) voxel among those that do makes the sample NULL.
 * Every dimension must be <= 2^24 (coordinates are float32).  The cube is never written. */
typedef struct {
    float origin[3], du[3], dv[3], step[3];
    int32_t width, height, nsteps;
} cube_view_t;

/* A camera orbiting the cube's centre (host-side convenience, no device work): viewing direction -z turned by
 * pitch about x, then by yaw about y (degrees); the image spans the bounding sphere of the cube, rays start on its
 * near side and take ceil(diameter / step) + 1 samples `step` voxels apart.  PAPER.md:400 ("2 degrees steps"). */
int cube_view_orbit(int64_t nx, int64_t ny, int64_t nz, double yaw_deg, double pitch_deg, int width, int height,
                    double step, cube_view_t* out);

/* Maximum intensity projection: image[v * width + u] = the largest sample of the ray of pixel
 * (u,v) among those inside the cube, not NULL and >= vmin (-INFINITY: no threshold; "the minimum data
 * value ... as a global thresholding technique"); NaN when there is none.  `image`: width * height floats the DEVICE
 * can write (device or pinned host memory).  `view` is a HOST pointer read before the call returns. */
int cube_render_mip(cube_ctx* ctx, const float* d, int64_t nx, int64_t ny, int64_t nz, const cube_view_t* view,
                    float vmin, float* image, cudaStream_t stream);

/* Generic transfer function with ordered front-to-back compositing (R30, R31).
 * table[L] = (r, g, b, opacity in [0,1]) for data level L < nlevels (1 <= nlevels <= 4096; host or device memory);
 * level of a sample s >= lo:  L = min(floor((s - lo) * ((float)nlevels / (hi - lo))), nlevels - 1) -- the histogram's
 * bin formula with everything above hi in the top level; samples below lo and NULL samples are skipped.  Per sample
 *     w = (1 - A) * a_L;   C = C + w * c_L;   A = A + w;   the ray stops once A >= opacity_cut (> 1: never).
 * rgba[(v * width + u) * 4 ...] = (C_r, C_g, C_b, A): opacity-weighted colour; device-writable memory, 16-byte aligned. */
int cube_render_tf(cube_ctx* ctx, const float* d, int64_t nx, int64_t ny, int64_t nz, const cube_view_t* view,
                   int nlevels, float lo, float hi, const float* table, float opacity_cut, float* rgba,
                   cudaStream_t stream);

/* Sigma-clipping transfer function (Fig. 7, Fig. 9; R34): cube_render_tf applied, sample
 * by sample, to   z = (s - mean(p)) / std(p)   where mean(p), std(p) are the LOCAL statistics at the sample point p,
 * trilinearly interpolated (the rule of the data lookup, float32) in the statistical mini-map `cells` that
 * cube_minimap(ctx, d, nx, ny, nz, px, py, pz, ...) wrote: cell (cx,cy,cz) sits at the centre of its nominal block,
 * data coordinate (cx*px + (px-1)/2, ...); map coordinate q = (p - (px-1)/2) / px clamped to [0, mx-1], likewise y, z.
 * "Two trilinear interpolation operations" per sample.  Levels partition [zlo, zhi] (zlo = the
 * clipping threshold in local sigmas, "2, 3, 4 and 7 sigma"); z < zlo, NULL samples and samples where
 * the interpolated std is not > 0 (or the map is NULL: an empty cell takes part) are skipped; compositing, table,
 * opacity_cut and rgba as cube_render_tf.  `cells`: memory the DEVICE can read (device or pinned host), mx*my*mz
 * records; read only.  Each call first rounds the cells' (mean, std) to float32 pairs in a buffer of the context
 * (8 bytes per cell; it is allocated -- the only allocation a render call can make -- when a map larger than any
 * before comes: CUBE_ENOMEM if that fails). */
int cube_render_sigma(cube_ctx* ctx, const float* d, int64_t nx, int64_t ny, int64_t nz, const cube_view_t* view,
                      const cube_moments_t* cells, int64_t px, int64_t py, int64_t pz, int nlevels, float zlo,
                      float zhi, const float* table, float opacity_cut, float* rgba, cudaStream_t stream);

/* 3-D spectrum tool (Fig. 6): out[i] = sample i of the ray of pixel (u,v) (any integers: the
 * pixel need not lie inside the image), NaN where the sample is outside the cube or NULL; nsteps floats,
 * device-writable memory. */
int cube_spectrum(cube_ctx* ctx, const float* d, int64_t nx, int64_t ny, int64_t nz, const cube_view_t* view,
                  int u, int v, float* out, cudaStream_t stream);

/* Per-cell lower median of the mini-map (NEXT-2, second half: SURVEY.md sec. 8(f) "mean/std (then median) per user
 * partition"): med[(cz*my + cy)*mx + cx] = the lower median (k = (count-1)/2 over the cell's non-NULL
 * voxels, as cube_median) of the cell cube_minimap defines; NaN for a cell without a non-NULL voxel.  Exact.  The
 * cube is read once (cells of up to 56000 voxels: their keys are kept in shared memory while four 8-bit digits are
 * fixed; larger cells are read once per digit).  A cell may hold at most 2^31 voxels.  `med`: mx*my*mz floats the
 * DEVICE can write (device or pinned host memory). */
int cube_minimap_median(cube_ctx* ctx, const float* d, int64_t nx, int64_t ny, int64_t nz, int64_t px, int64_t py,
                        int64_t pz, float* med, cudaStream_t stream);

const char* cube_strerror(int code);
int cube_last_cuda_error(const cube_ctx* ctx);

/* Launch-configuration knobs (0 keeps the default): threads per CTA, resident CTAs per SM. For tuning and
 * for the tests that check tiling invariance. */
int cube_set_launch(cube_ctx* ctx, int ctas_per_sm);
enum {
    CUBE_KNOB_CTAS_PER_SM = 0, /* same as cube_set_launch */
    CUBE_KNOB_BIGHIST = 1,     /* histograms with more than 16384 bins, one CTA of 1024 threads per SM:
                                  0 = automatic (default): 32-bit shared-memory counters for a window of 32768
                                      consecutive bins chosen by sampling + global REDs for the rest when at most
                                      1/32 of the sampled voxels fall outside the window, else 16-bit packed counters
                                      for all bins (the choice is made on the device),
                                  1 = clusters of two CTAs holding 32-bit counters in distributed shared memory,
                                  2 = always the 16-bit packed counters */
    CUBE_KNOB_SMALL = 3,       /* cube_stats with the median (histogram, if any, of at most 4096 bins), cube_median and
                                  cube_kth on a cube of at most 96 MiB: 0 = automatic (default): ONE cooperative launch
                                  (csrc/cube_small.cuh) when the device supports it, 1 = always the general three-launch
                                  path */
    CUBE_KNOB_MAPMEDIAN = 4,   /* cube_minimap_median on cells of at least 1024 voxels: 0 = automatic (default) = 2;
                                  1 = the cell's keys staged in shared memory, four 8-bit digits (cells of more than
                                      56000 voxels: re-read per digit); 2 = two reads of the cell, 11-bit first digit,
                                      the bucket's keys kept in shared memory (csrc/cube_minimap_median.cuh) */
    CUBE_KNOB_RENDER = 5,      /* cube_render_mip / _tf / _sigma: 0 = automatic (default): one ray per THREAD (a warp = 32
                                  neighbouring pixels of an image row) or one ray per WARP (lanes = consecutive samples),
                                  by the z component of the ray direction (csrc/cube.cu, render_along); 1 / 2 = always
                                  the former / the latter.  Same images bit for bit. */
    CUBE_KNOB_MINIMAP = 2      /* cube_minimap kernel: 0 = automatic (default): lines staged through a shared-memory
                                  ring by TMA bulk copies when the rows are 16-byte aligned, the cells at most 480
                                  voxels wide and a cell row has at least 256 lines (or the 128-bit kernel is not
                                  eligible), else as 1; 1 = 128-bit register kernel when eligible (rows 16-byte
                                  aligned, px >= 4), else the scalar one; 2 = always the scalar kernel; 3 = the TMA
                                  ring whenever it is eligible, whatever the number of lines */
};
int cube_set_knob(cube_ctx* ctx, int knob, int value);
/* Number of kernels launched through this context since creation (bench.py's gpu_launches). */
uint64_t cube_launch_count(const cube_ctx* ctx);

/* ---- Per-kernel timing (what bench.py's roofline reads).  When enabled, every kernel launched through the
 * context is bracketed by a cudaEvent pair on its own stream (about 2 us of stream time per launch, so keep
 * it off when timing whole steps).  cube_profile_read() synchronises the device, then returns the summed
 * duration and the number of launches of one kernel kind since the last cube_profile_reset(). */
enum {
    CUBE_K_MOMENTS = 0,        /* moments_kernel<plain> */
    CUBE_K_MOMENTS_COARSE = 1, /* moments_kernel<coarse>: moments + first select digit (pass A of cube_stats) */
    CUBE_K_HIST = 2,           /* histogram kernels */
    CUBE_K_SELECT_PASS0 = 3,   /* first digit over the cube */
    CUBE_K_SELECT_PASS1 = 4,   /* second digit + candidate compaction over the cube */
    CUBE_K_SELECT_PASS2 = 5,   /* last digit: on the candidate buffer (normal) or over the cube (fallback) */
    CUBE_K_SELECT_CAND = 6,    /* last digit on the candidates, brick-streamed path */
    CUBE_K_SELECT_SCAN = 7,    /* 1-CTA bucket location kernels */
    CUBE_K_HIST_SELECT = 8,    /* hist_select_kernel / hist_win_select_kernel (pass B of cube_stats) */
    CUBE_K_PROBE = 9,          /* cube_probe_read */
    CUBE_K_OTHER = 10,
    CUBE_K_MOMENTS_WINDOW = 11, /* moments_kernel<window>: cube_clipped_moments, cube_sigma_clip passes */
    CUBE_K_MINIMAP = 12,        /* minimap_kernel */
    CUBE_K_TORBEN = 13,         /* torben_pass_kernel (cube_median_torben) */
    CUBE_K_RENDER = 14,         /* render_mip_kernel / render_tf_kernel / spectrum_kernel */
    CUBE_K_STATS_SMALL = 15,    /* stats_small_kernel: cube_stats of an L2-resident cube in one cooperative launch (two reads) */
    CUBE_K_KINDS = 16
};
int cube_profile_enable(cube_ctx* ctx, int on);
/* Read-only STREAM probe: streams nvox float32 voxels through the same loop as the statistics kernels with one
 * FADD per voxel and discards the result.  Time it (CUBE_K_PROBE) to get the read ceiling of this GPU. */
int cube_probe_read(cube_ctx* ctx, const float* d, uint64_t nvox, cudaStream_t stream);
int cube_profile_reset(cube_ctx* ctx);
int cube_profile_read(cube_ctx* ctx, int kind, double* total_ms, uint64_t* launches);

#ifdef __cplusplus
}
#endif
#endif /* CUBE_H_ */
