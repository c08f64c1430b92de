// cube_oracle.cpp -- CPU ORACLE for the global-statistics path of arXiv:1211.4896.
//
// THIS IS TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only tests/, __graft_entry__.smoke()
// and bench.py's cpu_baseline / --impl reference legs may build, load or call it.
// It shares no code, header, table or helper with the CUDA path under
// paper_1211_4896_b200/ and neither side includes the other.
//
// Plain, single-threaded, obviously-correct C++.  Every result below has a plain
// definition; the oracle is that definition written out:
//
//   count / nan_count   PAPER.md:252, 265  "count of the non-null data values"; NULL == IEEE NaN
//   min / max           PAPER.md:261, 518  data minimum / maximum (total order: -0.0 < +0.0)
//   mean / std          PAPER.md:265, 273  from "summation and summation of squares and count";
//                       evaluated here as the exact-arithmetic value (long double, compensated,
//                       two-pass corrected) rounded to double -- NOT the paper's float32-per-slice
//                       partial sums, reading R17
//   histogram           PAPER.md:259-261   b = floor((x-lo) * (nbins/(hi-lo))) in float32,
//                       closed top bin, values outside [lo,hi] counted separately (R10-R13)
//   k-th / median       PAPER.md:281       "sort and select the middle element" is the definition
//                       the paper avoids for cost; here std::nth_element on a copy.  Lower
//                       median k=(n-1)/2 (R5), which is what Alg. 1 returns.
//   Torben (Alg. 1)     PAPER.md:570-610   restated step by step as a second, independent CPU
//                       algorithm for the median, with the garbled lines restored (R1-R4);
//                       Table 1 pins the restoration.
//   rank certificate    necessary-and-sufficient check of a claimed k-th value in one pass:
//                       #{x<m} <= k < #{x<m} + #{x==m}  (total order), independent of both
//                       selection algorithms.
//
//   MAD / clipped moments / sigma clip / mini-map   (PAPER.md:292, 336,
//                       344, 352-356): definitions stated at the functions near the end of this file.
//
// Parity pins (tests/test_oracle_*.py): closed forms (constant cube, ramp 0..N-1, two-value
// cube), exact rational sums computed with Python big integers, brute-force full sort on
// tiny cubes, power-of-two ramp histograms, Table 1 of the paper.  +-Inf voxels: mean = std = NaN by
// reading R8 (stated in oracle_moments, pinned in tests/test_oracle_pins.py).
//
//   ray casting: trilinear sample, maximum intensity
//                       projection, generic transfer function with front-to-back compositing, 3-D spectrum
//                       profile -- the march restated sample by sample at the end of this file
//                       (readings R27-R32, R34 of DESIGN.md; pins in tests/test_oracle_render_pins.py); the
//                       sigma-clipping transfer function with its second lookup in the mini-map.
//
// Build: g++ -O2 -std=c++17 -ffp-contract=off -fno-fast-math -fPIC -shared (oracle/build.py).

#include <algorithm>
#include <cmath>
#include <cstdint>
#include <cstring>
#include <limits>
#include <vector>

namespace {

inline bool is_nan(float x) { return x != x; }

// IEEE totalOrder restricted to non-NaN values: -0.0 < +0.0 (reading R7).
inline bool total_less(float a, float b) {
    if (a < b) return true;
    if (a == b) return std::signbit(a) && !std::signbit(b);
    return false;
}
inline bool total_equal(float a, float b) {
    return a == b && std::signbit(a) == std::signbit(b);
}

// Neumaier-compensated accumulator in long double.
struct Comp {
    long double s = 0.0L, c = 0.0L;
    inline void add(long double v) {
        long double t = s + v;
        if (fabsl(s) >= fabsl(v)) c += (s - t) + v; else c += (v - t) + s;
        s = t;
    }
    inline long double value() const { return s + c; }
};

}  // namespace

extern "C" {

struct oracle_moments_t {
    uint64_t count;      // non-NaN voxels
    uint64_t nan_count;  // NaN voxels
    float min, max;      // NaN if count == 0
    double mean, std;    // NaN if count == 0
};

// PAPER.md:265, 273.  sample_std != 0 -> divide M2 by (n-1) (n==1 -> NaN, reading R15).
int oracle_moments(const float* d, uint64_t N, int sample_std, oracle_moments_t* out) {
    uint64_t n = 0;
    float mn = 0.f, mx = 0.f;
    Comp sum;
    for (uint64_t i = 0; i < N; ++i) {
        float x = d[i];
        if (is_nan(x)) continue;
        if (n == 0) { mn = x; mx = x; }
        else {
            if (total_less(x, mn)) mn = x;
            if (total_less(mx, x)) mx = x;
        }
        ++n;
        sum.add((long double)x);
    }
    out->count = n;
    out->nan_count = N - n;
    if (n == 0) {
        out->min = out->max = std::numeric_limits<float>::quiet_NaN();
        out->mean = out->std = std::numeric_limits<double>::quiet_NaN();
        return 0;
    }
    // Reading R8: a set with an infinite member has no finite mean or deviation; both are reported as
    // NaN (count, min, max stay exact).  Stated here rather than left to what Inf does to a compensated sum.
    if (std::isinf(mn) || std::isinf(mx)) {
        out->min = mn;
        out->max = mx;
        out->mean = out->std = std::numeric_limits<double>::quiet_NaN();
        return 0;
    }
    long double mean = sum.value() / (long double)n;
    // second pass: corrected two-pass M2 = sum(delta^2) - (sum delta)^2 / n
    Comp sd, sd2;
    for (uint64_t i = 0; i < N; ++i) {
        float x = d[i];
        if (is_nan(x)) continue;
        long double delta = (long double)x - mean;
        sd.add(delta);
        sd2.add(delta * delta);
    }
    long double m2 = sd2.value() - sd.value() * sd.value() / (long double)n;
    if (m2 < 0.0L) m2 = 0.0L;
    out->min = mn;
    out->max = mx;
    out->mean = (double)(mean + sd.value() / (long double)n);
    long double denom = sample_std ? (long double)n - 1.0L : (long double)n;
    out->std = (denom > 0.0L) ? (double)sqrtl(m2 / denom)
                              : std::numeric_limits<double>::quiet_NaN();
    return 0;
}

// Float32 bin index of one in-range value (readings R10, R11, R13).  `scale` is
// (float)nbins / (hi - lo), both operations rounded to float32.  Exposed so tests can
// pin the formula on single values.
int oracle_bin_index(float x, int nbins, float lo, float hi) {
    if (hi == lo) return 0;
    float width = hi - lo;
    float scale = (float)nbins / width;
    float t = x - lo;
    float v = t * scale;
    if (!(v < (float)nbins)) return nbins - 1;  // closed top bin
    int b = (int)floorf(v);
    if (b > nbins - 1) b = nbins - 1;
    if (b < 0) b = 0;
    return b;
}

// PAPER.md:259-261.  bins[nbins], outside[2] = {#x<lo, #x>hi}; NaN counted nowhere.
// Returns 1 on invalid arguments (nbins<1, !(lo<=hi), non-finite lo/hi, width or scale; R19).
int oracle_histogram(const float* d, uint64_t N, int nbins, float lo, float hi,
                     uint64_t* bins, uint64_t* outside) {
    if (nbins < 1 || !(lo <= hi) || !std::isfinite(lo) || !std::isfinite(hi)) return 1;
    if (hi != lo && (!std::isfinite(hi - lo) || !std::isfinite((float)nbins / (hi - lo)))) return 1;
    for (int b = 0; b < nbins; ++b) bins[b] = 0;
    outside[0] = outside[1] = 0;
    for (uint64_t i = 0; i < N; ++i) {
        float x = d[i];
        if (is_nan(x)) continue;
        if (x < lo) { ++outside[0]; continue; }
        if (x > hi) { ++outside[1]; continue; }
        ++bins[oracle_bin_index(x, nbins, lo, hi)];
    }
    return 0;
}

// sort-and-select, k 0-based among the non-NaN values in total order.
// Returns 1 if k >= count (out = NaN).
int oracle_kth(const float* d, uint64_t N, uint64_t k, float* out) {
    std::vector<float> v;
    v.reserve(N);
    for (uint64_t i = 0; i < N; ++i) if (!is_nan(d[i])) v.push_back(d[i]);
    if (k >= v.size()) { *out = std::numeric_limits<float>::quiet_NaN(); return 1; }
    std::nth_element(v.begin(), v.begin() + (std::ptrdiff_t)k, v.end(), total_less);
    *out = v[k];
    return 0;
}

// Lower median: k = (n-1)/2 (reading R5).  Returns 1 if there is no non-NaN voxel.
int oracle_median(const float* d, uint64_t N, float* out) {
    std::vector<float> v;
    v.reserve(N);
    for (uint64_t i = 0; i < N; ++i) if (!is_nan(d[i])) v.push_back(d[i]);
    if (v.empty()) { *out = std::numeric_limits<float>::quiet_NaN(); return 1; }
    uint64_t k = (v.size() - 1) / 2;
    std::nth_element(v.begin(), v.begin() + (std::ptrdiff_t)k, v.end(), total_less);
    *out = v[k];
    return 0;
}

// One streaming pass: less = #{x < m}, equal = #{x == m} in total order over non-NaN x.
// m is the k-th value  <=>  equal >= 1 and less <= k < less + equal.
int oracle_rank_counts(const float* d, uint64_t N, float m, uint64_t* less, uint64_t* equal) {
    uint64_t l = 0, e = 0;
    for (uint64_t i = 0; i < N; ++i) {
        float x = d[i];
        if (is_nan(x)) continue;
        if (total_less(x, m)) ++l;
        else if (total_equal(x, m)) ++e;
    }
    *less = l; *equal = e;
    return 0;
}

// ---------------------------------------------------------------------------------
// Alg. 1, Torben's median method, restated in the paper's order.
// ---------------------------------------------------------------------------------

// PAPER.md:575 "Guess = (Min+Max)/" -- denominator lost in extraction; restored as /2
// evaluated in float32 (reading R1; every Guess printed in Table 1 equals this).
float oracle_torben_guess(float mn, float mx) { return (mn + mx) / 2.0f; }

// "if LessCount <= (data_length+1)/2 and GreaterCount <= (data_length+1)/2
// then" -- empty body restored as `break` (R2); integer division (R4).
int oracle_torben_stop(uint64_t less, uint64_t greater, uint64_t n) {
    uint64_t half = (n + 1) / 2;
    return (less <= half && greater <= half) ? 1 : 0;
}

// final selection.
float oracle_torben_pick(uint64_t less, uint64_t equal, uint64_t n,
                         float maxlt, float guess, float mingt) {
    uint64_t half = (n + 1) / 2;
    if (less >= half) return maxlt;
    if (less + equal >= half) return guess;
    return mingt;
}

// Full Alg. 1 over the non-NaN voxels.  trace (optional, may be NULL) receives up to
// max_trace rows of 6 doubles: guess, min, max, less, greater, equal.
// Returns the number of iterations, or -1 if there is no non-NaN voxel.
int oracle_torben_median(const float* d, uint64_t N, float* out, double* trace, int max_trace) {
    uint64_t n = 0;
    float Min = 0.f, Max = 0.f;
    for (uint64_t i = 0; i < N; ++i) {
        float x = d[i];
        if (is_nan(x)) continue;
        if (n == 0) { Min = Max = x; }
        else { if (x < Min) Min = x; if (x > Max) Max = x; }
        ++n;
    }
    if (n == 0) { *out = std::numeric_limits<float>::quiet_NaN(); return -1; }
    int iter = 0;
    float Guess, MaxLt, MinGt;
    uint64_t Less, Greater, Equal;
    for (;;) {
        Guess = oracle_torben_guess(Min, Max);
        Less = Greater = Equal = 0;
        MaxLt = Min;
        MinGt = Max;
        for (uint64_t i = 0; i < N; ++i) {          // i in [0, data_length)  (R3)
            float x = d[i];
            if (is_nan(x)) continue;                // NULL voxels excluded
            if (x < Guess) { ++Less; if (x > MaxLt) MaxLt = x; }
            else if (x > Guess) { ++Greater; if (x < MinGt) MinGt = x; }
            else ++Equal;
        }
        if (trace && iter < max_trace) {
            double* r = trace + 6 * iter;
            r[0] = Guess; r[1] = Min; r[2] = Max;
            r[3] = (double)Less; r[4] = (double)Greater; r[5] = (double)Equal;
        }
        ++iter;
        if (oracle_torben_stop(Less, Greater, n)) break;
        else if (Less > Greater) Max = MaxLt;
        else Min = MinGt;
    }
    *out = oracle_torben_pick(Less, Equal, n, MaxLt, Guess, MinGt);
    return iter;
}

// Alg. 1 stopped after at most max_iter passes over the data -- the paper's remark that "if a median approximation
// is accepted, the number of iterations could have been reduced to 20 with an error of order 1e-6" (
// "Torben-on-GPU as the paper-faithful comparison and early-stop approximate median").
// Same steps as oracle_torben_median; when the cap is reached before the stop test fires, the final
// selection is applied to the counts of the last pass made (reading R26).  *converged = 1 when
// the stop test fired (then the result is the exact lower median).  Returns the passes made; -1 and NaN when there
// is no non-NaN voxel; max_iter <= 0 makes no pass and returns NaN.
int oracle_torben_capped(const float* d, uint64_t N, int max_iter, float* out, int* converged) {
    uint64_t n = 0;
    float Min = 0.f, Max = 0.f;
    *converged = 0;
    *out = std::numeric_limits<float>::quiet_NaN();
    for (uint64_t i = 0; i < N; ++i) {
        float x = d[i];
        if (is_nan(x)) continue;
        if (n == 0) { Min = Max = x; }
        else { if (x < Min) Min = x; if (x > Max) Max = x; }
        ++n;
    }
    if (n == 0) return -1;
    if (max_iter <= 0) return 0;
    int iter = 0;
    float Guess, MaxLt, MinGt;
    uint64_t Less, Greater, Equal;
    for (;;) {
        Guess = oracle_torben_guess(Min, Max);
        Less = Greater = Equal = 0;
        MaxLt = Min;
        MinGt = Max;
        for (uint64_t i = 0; i < N; ++i) {
            float x = d[i];
            if (is_nan(x)) continue;
            if (x < Guess) { ++Less; if (x > MaxLt) MaxLt = x; }
            else if (x > Guess) { ++Greater; if (x < MinGt) MinGt = x; }
            else ++Equal;
        }
        ++iter;
        if (oracle_torben_stop(Less, Greater, n)) { *converged = 1; break; }
        if (iter >= max_iter) break;
        if (Less > Greater) Max = MaxLt;
        else Min = MinGt;
    }
    *out = oracle_torben_pick(Less, Equal, n, MaxLt, Guess, MinGt);
    return iter;
}

// ---------------------------------------------------------------------------------
// NEXT-1: median absolute deviation and sigma-clipped moments.
// The paper only names them: Torben's method "can be easily modified to address the median absolute
// deviation (MAD)"; "Thresholding (Sigma-Clipping) techniques where a data threshold is
// defined based on the estimated noise properties", the threshold being chosen from "the
// previously discussed statistical data computation ... (e.g mean and standard deviation)".
// Definitions taken (readings R21-R24):
//   MAD      med = lower median of the non-NaN voxels; y_i = |fl32(x_i - med)| (one float32 subtraction,
//            then the sign bit cleared); MAD = lower median of the non-NaN y_i (y is NaN only for
//            x = med = +-Inf, which is dropped like a NULL voxel).
//   clipped  moments (count, min, max, mean, std) of the voxels with lo <= x <= hi (closed window, the test
//            made on x itself; NaN fails it); nan_count = N - count = everything left out.
//   sigma clip (kappa, max_iter): m_0 = moments of all voxels; for i = 1..max_iter:
//            lo_i = fl32(mean - kappa*std), hi_i = fl32(mean + kappa*std) with mean, std of m_{i-1}
//            (product and sum rounded to double separately, then one rounding to float32);
//            m_i = clipped moments over [lo_i, hi_i]; stop after the first i with count_i == count_{i-1}
//            (that m_i is returned; it equals m_{i-1}), or when count_{i-1} == 0 or std_{i-1} is not finite.
//            Windows are always formed from the PREVIOUS iteration's statistics and applied to the
//            whole cube, so counts never increase.
// ---------------------------------------------------------------------------------

int oracle_clipped_moments(const float* d, uint64_t N, float lo, float hi, int sample_std,
                           oracle_moments_t* out) {
    std::vector<float> v;
    for (uint64_t i = 0; i < N; ++i) {
        float x = d[i];
        if (x >= lo && x <= hi) v.push_back(x);   // NaN fails both comparisons
    }
    oracle_moments(v.data(), v.size(), sample_std, out);
    out->nan_count = N - out->count;
    return 0;
}

// Returns the number of clipped passes made (0 .. max_iter).
int oracle_sigma_clip(const float* d, uint64_t N, double kappa, int max_iter, int sample_std,
                      oracle_moments_t* out, float* window /* [2]: last window used, NaN if none */) {
    oracle_moments_t m;
    oracle_moments(d, N, sample_std, &m);
    window[0] = window[1] = std::numeric_limits<float>::quiet_NaN();
    int iters = 0;
    while (iters < max_iter) {
        if (m.count == 0 || !std::isfinite(m.std) || !std::isfinite(m.mean)) break;
        volatile double w = kappa * m.std;             // rounded to double before the sum (no contraction)
        volatile double dl = m.mean - w, dh = m.mean + w;
        float lo = (float)dl, hi = (float)dh;
        oracle_moments_t m2;
        oracle_clipped_moments(d, N, lo, hi, sample_std, &m2);
        window[0] = lo; window[1] = hi;
        ++iters;
        bool same = (m2.count == m.count);
        m = m2;
        if (same) break;
    }
    *out = m;
    return iters;
}

// MAD.  Returns 1 when there is no non-NaN voxel (both outputs NaN).
int oracle_mad(const float* d, uint64_t N, float* median_out, float* mad_out) {
    float med;
    if (oracle_median(d, N, &med)) {
        *median_out = *mad_out = std::numeric_limits<float>::quiet_NaN();
        return 1;
    }
    std::vector<float> y;
    y.reserve(N);
    for (uint64_t i = 0; i < N; ++i) {
        float x = d[i];
        if (is_nan(x)) continue;
        volatile float t = x - med;                    // float32 subtraction
        y.push_back(fabsf(t));                         // NaN (Inf - Inf) is dropped by oracle_median below
    }
    *median_out = med;
    oracle_median(y.data(), y.size(), mad_out);
    return 0;
}

// ---------------------------------------------------------------------------------
// NEXT-2: the statistical mini-map (Fig. 7): "a scaled-down version
// of the data cube ... each data point represents the data statistics of a bigger region in the real
// dataset", partitions of px x py x pz voxels ("30x30x30 pixel").  Cell (cx,cy,cz) covers
// x in [cx*px, min((cx+1)*px, nx)) and likewise in y and z (ragged last cells are simply smaller; reading
// R25); its record is the moments of those voxels.  Map dims: mx = ceil(nx/px) etc., x fastest.
// ---------------------------------------------------------------------------------
int oracle_minimap(const float* d, int64_t nx, int64_t ny, int64_t nz, int64_t px, int64_t py, int64_t pz,
                   int sample_std, oracle_moments_t* cells) {
    if (nx <= 0 || ny <= 0 || nz <= 0 || px <= 0 || py <= 0 || pz <= 0) return 1;
    const int64_t mx = (nx + px - 1) / px, my = (ny + py - 1) / py, mz = (nz + pz - 1) / pz;
    std::vector<float> v;
    for (int64_t cz = 0; cz < mz; ++cz)
        for (int64_t cy = 0; cy < my; ++cy)
            for (int64_t cx = 0; cx < mx; ++cx) {
                v.clear();
                for (int64_t z = cz * pz; z < std::min((cz + 1) * pz, nz); ++z)
                    for (int64_t y = cy * py; y < std::min((cy + 1) * py, ny); ++y)
                        for (int64_t x = cx * px; x < std::min((cx + 1) * px, nx); ++x)
                            v.push_back(d[(z * ny + y) * nx + x]);
                oracle_moments(v.data(), v.size(), sample_std, &cells[(cz * my + cy) * mx + cx]);
            }
    return 0;
}


// Per-cell lower median of the mini-map (SURVEY.md sec. 8(f) NEXT-2 "mean/std (then median) per user partition";
// PAPER.md:352 "each data point represents the data statistics of a bigger region"): the lower median
// (k = (n-1)/2 over the cell's non-NaN voxels, reading R5) of every cell of oracle_minimap's partition; NaN for a cell
// without a non-NaN voxel.
int oracle_minimap_median(const float* d, int64_t nx, int64_t ny, int64_t nz, int64_t px, int64_t py, int64_t pz,
                          float* med) {
    if (nx <= 0 || ny <= 0 || nz <= 0 || px <= 0 || py <= 0 || pz <= 0) return 1;
    const int64_t mx = (nx + px - 1) / px, my = (ny + py - 1) / py, mz = (nz + pz - 1) / pz;
    std::vector<float> v;
    for (int64_t cz = 0; cz < mz; ++cz)
        for (int64_t cy = 0; cy < my; ++cy)
            for (int64_t cx = 0; cx < mx; ++cx) {
                v.clear();
                for (int64_t z = cz * pz; z < std::min((cz + 1) * pz, nz); ++z)
                    for (int64_t y = cy * py; y < std::min((cy + 1) * py, ny); ++y)
                        for (int64_t x = cx * px; x < std::min((cx + 1) * px, nx); ++x)
                            v.push_back(d[(z * ny + y) * nx + x]);
                oracle_median(v.data(), v.size(), &med[(cz * my + cy) * mx + cx]);
            }
    return 0;
}

// ---------------------------------------------------------------------------------
// NEXT-4: ray casting into a headless buffer -- the paper's volume rendering transfer
// functions and its 3-D spectrum tool (Fig. 6: "evaluating the sampled data
// points on an arbitrary ray with a constant sampling step ... in 3D with trilinear interpolation").  The paper
// gives no formulas beyond that; the readings (R27-R32) are restated at each function.  Everything is
// float32, one rounding per operation, no contraction (this file is built with -ffp-contract=off), in the order
// written, so that a kernel doing the same operations in the same order gives the same bits.
//
// Geometry (R27): data coordinates are voxel indices, voxel (i,j,k) sits at (i,j,k); orthographic rays.  A view is
//   origin[3], du[3], dv[3], step[3], width, height, nsteps:
//   first sample of pixel (u,v):  o_c = (origin_c + (float)u * du_c) + (float)v * dv_c        c = x, y, z
//   sample i of that ray:         p_c = o_c + (float)i * step_c,                              0 <= i < nsteps
// A sample is INSIDE iff 0 <= p_x <= nx-1, 0 <= p_y <= ny-1 and 0 <= p_z <= nz-1 (tested on the float32 p).
// ---------------------------------------------------------------------------------
struct oracle_view_t {
    float origin[3], du[3], dv[3], step[3];
    int32_t width, height, nsteps;
};

static inline void oracle_ray_origin(const oracle_view_t* vw, int u, int v, float o[3]) {
    for (int c = 0; c < 3; ++c) {
        volatile float a = (float)u * vw->du[c];
        volatile float b = vw->origin[c] + a;
        volatile float e = (float)v * vw->dv[c];
        o[c] = b + e;
    }
}
static inline void oracle_ray_point(const oracle_view_t* vw, const float o[3], int i, float p[3]) {
    for (int c = 0; c < 3; ++c) {
        volatile float a = (float)i * vw->step[c];
        p[c] = o[c] + a;
    }
}

// Trilinear sample (R28; "trilinear interpolation to interpolate the data values ... from the original
// data points"): x0 = floor(p_x), f_x = p_x - x0, x1 = x0 + 1 when f_x > 0 and x1 = x0 when f_x = 0 (a neighbour
// of weight zero does not take part: a sample at a voxel centre IS that voxel, whatever lies next to it, and
// p_x = nx - 1 needs no voxel beyond the cube); likewise y, z; interpolation along x, then y, then z, each step
// a + f * (b - a).  Returns 0 and leaves *out alone when the point is outside.
// A NULL (NaN) voxel among those that take part makes the sample NaN (IEEE propagation: the sample is NULL itself).
int oracle_trilinear(const float* d, int64_t nx, int64_t ny, int64_t nz, const float p[3], float* out) {
    if (!(p[0] >= 0.0f && p[0] <= (float)(nx - 1) && p[1] >= 0.0f && p[1] <= (float)(ny - 1) &&
          p[2] >= 0.0f && p[2] <= (float)(nz - 1))) return 0;
    const float flx = floorf(p[0]), fly = floorf(p[1]), flz = floorf(p[2]);
    const int64_t x0 = (int64_t)flx, y0 = (int64_t)fly, z0 = (int64_t)flz;
    const float fx = p[0] - flx, fy = p[1] - fly, fz = p[2] - flz;
    const int64_t x1 = x0 + (fx > 0.0f ? 1 : 0), y1 = y0 + (fy > 0.0f ? 1 : 0), z1 = z0 + (fz > 0.0f ? 1 : 0);
    auto at = [&](int64_t x, int64_t y, int64_t z) { return d[(z * ny + y) * nx + x]; };
    auto lerp = [](float a, float b, float f) {
        volatile float diff = b - a;
        volatile float prod = f * diff;
        return a + prod;
    };
    const float c00 = lerp(at(x0, y0, z0), at(x1, y0, z0), fx);
    const float c10 = lerp(at(x0, y1, z0), at(x1, y1, z0), fx);
    const float c01 = lerp(at(x0, y0, z1), at(x1, y0, z1), fx);
    const float c11 = lerp(at(x0, y1, z1), at(x1, y1, z1), fx);
    const float c0 = lerp(c00, c10, fy);
    const float c1 = lerp(c01, c11, fy);
    *out = lerp(c0, c1, fz);
    return 1;
}

// 3-D spectrum tool: the data profile along the line of sight of pixel (u,v): out[i] = the
// trilinear sample at sample i, NaN where the sample is outside the cube (or NULL).
int oracle_spectrum(const float* d, int64_t nx, int64_t ny, int64_t nz, const oracle_view_t* vw, int u, int v,
                    float* out) {
    float o[3], p[3];
    oracle_ray_origin(vw, u, v, o);
    for (int i = 0; i < vw->nsteps; ++i) {
        oracle_ray_point(vw, o, i, p);
        float s;
        out[i] = oracle_trilinear(d, nx, ny, nz, p, &s) ? s : std::numeric_limits<float>::quiet_NaN();
    }
    return 0;
}

// Maximum intensity projection ("only the value of the maximum voxel through each cast ray is
// shown for each pixel"; "the minimum data value" as a global threshold): image[v*width + u] = the largest sample of
// the ray among those that are inside, not NULL and >= vmin, taken in march order with  if (s > m) m = s  (R29);
// NaN when the ray has no such sample.
int oracle_render_mip(const float* d, int64_t nx, int64_t ny, int64_t nz, const oracle_view_t* vw, float vmin,
                      float* image) {
    for (int v = 0; v < vw->height; ++v)
        for (int u = 0; u < vw->width; ++u) {
            float o[3], p[3], m = 0.0f;
            bool have = false;
            oracle_ray_origin(vw, u, v, o);
            for (int i = 0; i < vw->nsteps; ++i) {
                oracle_ray_point(vw, o, i, p);
                float s;
                if (!oracle_trilinear(d, nx, ny, nz, p, &s)) continue;
                if (!(s >= vmin)) continue;                     // NULL samples fail the comparison
                if (!have || s > m) { m = s; have = true; }
            }
            image[(size_t)v * vw->width + u] = have ? m : std::numeric_limits<float>::quiet_NaN();
        }
    return 0;
}

// Generic transfer function ("The data values' range is partitioned into discrete levels.  Each
// data level is assigned a colour and opacity value ... from 0 to 1"), ordered front-to-back compositing (Levoy 1988,
// as the paper cites).  R30: level of a sample s with lo <= s (NULL and s < lo: skipped -- the global threshold of
// PAPER.md:170, 344):  L = min(floor((s - lo) * scale), nlevels - 1), scale = (float)nlevels / (hi - lo), every
// operation float32 -- the histogram's bin formula (R10, R11) with everything above hi in the top level (hi == lo:
// level 0).  R31: with table[L] = (r, g, b, a), accumulated colour C and opacity A start at 0 and per sample
//     w = (1 - A) * a;   C_c = C_c + w * c_c  (c = r, g, b);   A = A + w;   stop the ray when A >= opacity_cut.
// rgba[(v*width + u)*4 ..] = (C_r, C_g, C_b, A): opacity-weighted (premultiplied) colour.
int oracle_render_tf(const float* d, int64_t nx, int64_t ny, int64_t nz, const oracle_view_t* vw, int nlevels,
                     float lo, float hi, const float* table, float opacity_cut, float* rgba) {
    if (nlevels < 1 || !(lo <= hi)) return 1;
    volatile float width = hi - lo;
    volatile float scale_v = (hi == lo) ? 0.0f : (float)nlevels / width;
    const float scale = scale_v;
    for (int v = 0; v < vw->height; ++v)
        for (int u = 0; u < vw->width; ++u) {
            float o[3], p[3], C[3] = {0.0f, 0.0f, 0.0f}, A = 0.0f;
            oracle_ray_origin(vw, u, v, o);
            for (int i = 0; i < vw->nsteps; ++i) {
                oracle_ray_point(vw, o, i, p);
                float s;
                if (!oracle_trilinear(d, nx, ny, nz, p, &s)) continue;
                if (!(s >= lo)) continue;
                volatile float t = s - lo;
                volatile float q = t * scale;
                float fl = floorf(q);
                int L = (fl >= (float)(nlevels - 1)) ? nlevels - 1 : (int)fl;
                const float* e = table + 4 * (size_t)L;
                volatile float rem = 1.0f - A;
                volatile float w = rem * e[3];
                for (int c = 0; c < 3; ++c) {
                    volatile float wc = w * e[c];
                    C[c] = C[c] + wc;
                }
                A = A + w;
                if (A >= opacity_cut) break;
            }
            float* px = rgba + 4 * ((size_t)v * vw->width + u);
            px[0] = C[0]; px[1] = C[1]; px[2] = C[2]; px[3] = A;
        }
    return 0;
}


// Sigma-clipping transfer function (Fig. 7, Fig. 9): "For each sampled data point over the traced rays,
// two trilinear interpolation operations are required.  The first one is performed to get the actual data value at
// this point using the original data grid.  The second is performed to get the data properties at this point using
// the mini-map.  The point's data value is then scaled using its region's data properties to generate the look-up
// value used to calculate the colour and the opacity".  Reading R34 (the paper gives no formula):
//   * the mini-map is the array of cell records oracle_minimap produces; cell (cx, cy, cz) sits at the centre of its
//     nominal px x py x pz block: data coordinate  cx * px + (px - 1) / 2  along x, likewise y, z;
//   * map coordinate of a data point:  q_c = (p_c - (px_c - 1) / 2) / px_c  (float32: one subtraction, one IEEE
//     division), clamped to [0, m_c - 1]; local mean and std = trilinear interpolation (the rule of
//     oracle_trilinear: floor, a neighbour of weight zero does not take part, a + f * (b - a), x then y then z) of the
//     cells' mean and std, each rounded to float32 first; a cell without voxels (NaN record) makes them NaN;
//   * look-up value  z = (s - mean) / std  (float32, IEEE division); the sample is skipped unless std > 0 and z is
//     not NaN; levels over [zlo, zhi] and compositing exactly as in oracle_render_tf (R30, R31) with z in place of s:
//     zlo is the clipping threshold in units of the local sigma ("2 sigma, 3 sigma, 4 sigma and 7 sigma").
static inline float oracle_lerp(float a, float b, float f) {
    volatile float diff = b - a;
    volatile float prod = f * diff;
    return a + prod;
}

// mean and std of the mini-map at the data point p (see above).  Exposed for the pins.
int oracle_minimap_lookup(const oracle_moments_t* cells, int64_t nx, int64_t ny, int64_t nz, int64_t px, int64_t py,
                          int64_t pz, const float p[3], float* mean_out, float* std_out) {
    const int64_t n[3] = {nx, ny, nz}, part[3] = {px, py, pz};
    int64_t m[3], i0[3], i1[3];
    float f[3];
    for (int c = 0; c < 3; ++c) {
        m[c] = (n[c] + part[c] - 1) / part[c];
        volatile float off = (float)(part[c] - 1) / 2.0f;
        volatile float rel = p[c] - off;
        float q = rel / (float)part[c];
        if (!(q >= 0.0f)) q = 0.0f;                         // clamp (also a NaN coordinate)
        if (q > (float)(m[c] - 1)) q = (float)(m[c] - 1);
        const float fl = floorf(q);
        i0[c] = (int64_t)fl;
        f[c] = q - fl;
        i1[c] = i0[c] + (f[c] > 0.0f ? 1 : 0);
    }
    float out[2];
    for (int which = 0; which < 2; ++which) {
        auto at = [&](int64_t x, int64_t y, int64_t z) {
            const oracle_moments_t& r = cells[(z * m[1] + y) * m[0] + x];
            return (float)(which == 0 ? r.mean : r.std);
        };
        const float c00 = oracle_lerp(at(i0[0], i0[1], i0[2]), at(i1[0], i0[1], i0[2]), f[0]);
        const float c10 = oracle_lerp(at(i0[0], i1[1], i0[2]), at(i1[0], i1[1], i0[2]), f[0]);
        const float c01 = oracle_lerp(at(i0[0], i0[1], i1[2]), at(i1[0], i0[1], i1[2]), f[0]);
        const float c11 = oracle_lerp(at(i0[0], i1[1], i1[2]), at(i1[0], i1[1], i1[2]), f[0]);
        out[which] = oracle_lerp(oracle_lerp(c00, c10, f[1]), oracle_lerp(c01, c11, f[1]), f[2]);
    }
    *mean_out = out[0];
    *std_out = out[1];
    return 0;
}

int oracle_render_sigma(const float* d, int64_t nx, int64_t ny, int64_t nz, const oracle_view_t* vw,
                        const oracle_moments_t* cells, int64_t px, int64_t py, int64_t pz, int nlevels, float zlo,
                        float zhi, const float* table, float opacity_cut, float* rgba) {
    if (nlevels < 1 || !(zlo <= zhi) || px < 1 || py < 1 || pz < 1) return 1;
    volatile float width = zhi - zlo;
    volatile float scale_v = (zhi == zlo) ? 0.0f : (float)nlevels / width;
    const float scale = scale_v;
    for (int v = 0; v < vw->height; ++v)
        for (int u = 0; u < vw->width; ++u) {
            float o[3], p[3], C[3] = {0.0f, 0.0f, 0.0f}, A = 0.0f;
            oracle_ray_origin(vw, u, v, o);
            for (int i = 0; i < vw->nsteps; ++i) {
                oracle_ray_point(vw, o, i, p);
                float s, mean, sd;
                if (!oracle_trilinear(d, nx, ny, nz, p, &s)) continue;
                oracle_minimap_lookup(cells, nx, ny, nz, px, py, pz, p, &mean, &sd);
                if (!(sd > 0.0f)) continue;
                volatile float num = s - mean;
                const float z = num / sd;
                if (!(z >= zlo)) continue;                       // below the clipping threshold, or NULL
                volatile float t = z - zlo;
                volatile float q = t * scale;
                float fl = floorf(q);
                int L = (fl >= (float)(nlevels - 1)) ? nlevels - 1 : (int)fl;
                const float* e = table + 4 * (size_t)L;
                volatile float rem = 1.0f - A;
                volatile float w = rem * e[3];
                for (int c = 0; c < 3; ++c) {
                    volatile float wc = w * e[c];
                    C[c] = C[c] + wc;
                }
                A = A + w;
                if (A >= opacity_cut) break;
            }
            float* pxl = rgba + 4 * ((size_t)v * vw->width + u);
            pxl[0] = C[0]; pxl[1] = C[1]; pxl[2] = C[2]; pxl[3] = A;
        }
    return 0;
}

}  // extern "C"
