"""Pins for the CPU oracle (oracle/cube_oracle.cpp) against things OTHER than itself:
closed forms, exact rational arithmetic (Python big integers), brute-force sorts on tiny cubes,
invariants, and Table 1 of the paper (tests/golden/torben_table1.txt).

Chosen so that a plausible mistake in the oracle (dropped term, wrong sign/index, transposed
operand, open instead of closed top bin, upper instead of lower median, NaN counted) fails
at least one of them.  CPU only.
"""
import math
import os
from fractions import Fraction

import numpy as np
import pytest

import oracle

GOLD = os.path.join(os.path.dirname(__file__), "golden", "torben_table1.txt")
rng = np.random.default_rng(20121211)


# --------------------------------------------------------------------------- helpers
def total_key(v):
    """Sort key realising IEEE totalOrder on non-NaN floats without touching the bit pattern."""
    v = float(v)
    return (v, 0 if math.copysign(1.0, v) < 0 else 1)


def exact_mean_var(vals):
    fr = [Fraction(float(v)) for v in vals]          # float32 values are dyadic rationals
    n = len(fr)
    mean = sum(fr) / n
    var = sum((f - mean) ** 2 for f in fr) / n
    return mean, var


def frac_sqrt(fr, digits=40):
    """sqrt of a Fraction to ~digits significant digits, as float (via integer sqrt)."""
    if fr == 0:
        return 0.0
    scale = 10 ** (2 * digits)
    # bring the value to a comfortable magnitude first
    e = 0
    while fr < 1:
        fr *= 100
        e -= 1
    while fr >= 100:
        fr /= 100
        e += 1
    r = math.isqrt(int(fr * scale))
    return float(Fraction(r, 10 ** digits)) * (10.0 ** e)


# --------------------------------------------------------------------------- moments
@pytest.mark.parametrize("c", [0.1, 0.002, 1234.567, -3.0, 1e-40])
def test_moments_constant_cube(c):
    a = np.full(1 << 18, c, dtype=np.float32)
    m = oracle.moments(a)
    assert m["count"] == a.size and m["nan_count"] == 0
    assert m["min"] == np.float32(c) and m["max"] == np.float32(c)
    assert m["mean"] == float(np.float32(c))          # exactly
    assert m["std"] == 0.0                            # exactly


@pytest.mark.parametrize("logn", [10, 20, 24])
def test_moments_ramp_closed_form(logn):
    # x_i = i, i < 2^24 is exact in float32.  mean=(N-1)/2, population var=(N^2-1)/12
    # (north_star).  sample var = N(N+1)/12.
    N = 1 << logn
    a = np.arange(N, dtype=np.float32)
    m = oracle.moments(a)
    assert m["count"] == N
    assert m["min"] == 0.0 and m["max"] == np.float32(N - 1)
    assert m["mean"] == (N - 1) / 2.0
    assert m["std"] == pytest.approx(math.sqrt((N * N - 1) / 12.0), rel=2e-16)
    ms = oracle.moments(a, sample_std=True)
    assert ms["std"] == pytest.approx(math.sqrt(N * (N + 1) / 12.0), rel=2e-16)
    assert ms["mean"] == m["mean"]


def test_moments_ramp_reversed_and_shuffled_are_identical():
    N = 1 << 16
    a = np.arange(N, dtype=np.float32) * np.float32(0.37)
    m0 = oracle.moments(a)
    for b in (a[::-1].copy(), rng.permutation(a)):
        m = oracle.moments(b)
        assert m["mean"] == m0["mean"] and m["std"] == m0["std"]
        assert (m["min"], m["max"], m["count"]) == (m0["min"], m0["max"], m0["count"])


def test_moments_two_value_closed_form():
    # p copies of a, q copies of b: mean=(pa+qb)/n, var = pq (a-b)^2 / n^2
    a_, b_, p, q = np.float32(0.75), np.float32(-2.5), 1000, 3000
    a = np.concatenate([np.full(p, a_, np.float32), np.full(q, b_, np.float32)])
    m = oracle.moments(rng.permutation(a))
    n = p + q
    assert m["mean"] == (p * float(a_) + q * float(b_)) / n
    assert m["std"] == pytest.approx(math.sqrt(p * q) * abs(float(a_) - float(b_)) / n, rel=2e-16)


@pytest.mark.parametrize("seed", range(6))
def test_moments_exact_rational(seed):
    r = np.random.default_rng(seed)
    n = 700
    # wide dynamic range, mixed signs, heavy cancellation in the mean
    vals = (r.standard_normal(n) * 10.0 ** r.integers(-6, 6, n)).astype(np.float32)
    if seed % 2:
        vals += np.float32(1000.0)                    # large offset: Sum x^2 formulas lose digits here
    mean, var = exact_mean_var(vals)
    m = oracle.moments(vals)
    assert m["mean"] == pytest.approx(float(mean), rel=3e-16, abs=0.0)
    assert m["std"] == pytest.approx(frac_sqrt(var), rel=1e-15)
    ms = oracle.moments(vals, sample_std=True)
    assert ms["std"] == pytest.approx(frac_sqrt(var * n / (n - 1)), rel=1e-15)


def test_moments_nan_excluded_and_counted():
    a = np.arange(1000, dtype=np.float32)
    b = a.copy()
    b[::7] = np.float32("nan")
    b[3] = np.frombuffer(np.uint32(0xFFC00001).tobytes(), dtype=np.float32)[0]   # negative-sign NaN
    keep = b[~np.isnan(b)]
    m, mk = oracle.moments(b), oracle.moments(keep)
    assert m["count"] == keep.size and m["nan_count"] == b.size - keep.size
    for f in ("min", "max", "mean", "std"):
        assert m[f] == mk[f]
    mean, var = exact_mean_var(keep)
    assert m["mean"] == pytest.approx(float(mean), rel=3e-16)


def test_moments_empty_and_single():
    m = oracle.moments(np.full(10, np.nan, np.float32))
    assert m["count"] == 0 and m["nan_count"] == 10
    assert all(math.isnan(float(m[f])) for f in ("min", "max", "mean", "std"))
    m = oracle.moments(np.array([np.nan, 2.5, np.nan], np.float32))
    assert m["count"] == 1 and m["mean"] == 2.5 and m["std"] == 0.0
    assert math.isnan(oracle.moments(np.array([2.5], np.float32), sample_std=True)["std"])   # R15
    m = oracle.moments(np.zeros(0, np.float32))
    assert m["count"] == 0 and math.isnan(m["mean"])


def test_moments_signed_zero_total_order():
    a = np.array([0.0, -0.0, 0.0], np.float32)
    m = oracle.moments(a)
    assert math.copysign(1.0, float(m["min"])) == -1.0 and math.copysign(1.0, float(m["max"])) == 1.0
    assert m["mean"] == 0.0 and m["std"] == 0.0


def test_moments_subnormals_kept():
    a = np.array([1e-40, 3e-40, -2e-40], np.float32)
    mean, var = exact_mean_var(a)
    m = oracle.moments(a)
    assert m["mean"] == pytest.approx(float(mean), rel=1e-15) and m["mean"] != 0.0
    assert m["min"] == np.float32(-2e-40) and m["max"] == np.float32(3e-40)


# --------------------------------------------------------------------------- histogram
@pytest.mark.parametrize("logn,nbins", [(16, 256), (20, 1024), (20, 4096), (20, 65536), (12, 1)])
def test_histogram_pow2_ramp_is_uniform(logn, nbins):
    # x=i, lo=0, hi=N, nbins | N, all powers of two => every float op is exact (reading R10)
    N = 1 << logn
    a = rng.permutation(np.arange(N, dtype=np.float32))
    bins, outside = oracle.histogram(a, nbins, 0.0, float(N))
    assert (bins == N // nbins).all() and outside.tolist() == [0, 0]


def test_histogram_exact_arithmetic_on_dyadic_edges():
    # lo, width and every x are small dyadic rationals => (x-lo)*(nbins/(hi-lo)) is exact in
    # float32, so the float formula must equal the exact-arithmetic floor((x-lo)/w).
    nbins, lo, w = 37, Fraction(-3, 4), Fraction(1, 8)
    hi = lo + nbins * w
    xs = (rng.integers(-64, 400, 5000) / 64.0).astype(np.float32)       # multiples of 1/64
    bins, outside = oracle.histogram(xs, nbins, float(lo), float(hi))
    # nbins/(hi-lo) = 8 exactly
    exp = np.zeros(nbins, np.uint64)
    below = above = 0
    for x in xs:
        fx = Fraction(float(x))
        if fx < lo:
            below += 1
        elif fx > hi:
            above += 1
        else:
            exp[min(int((fx - lo) // w), nbins - 1)] += 1
    assert (bins == exp).all() and outside.tolist() == [below, above]


def test_histogram_closed_top_bin_and_outside():
    a = np.array([0.0, 1.0, 0.999999, -1e-9, 1.0000001, np.nan, 0.5], np.float32)
    bins, outside = oracle.histogram(a, 4, 0.0, 1.0)
    assert bins.tolist() == [1, 0, 1, 2] and outside.tolist() == [1, 1]     # x==hi lands in the top bin (R11)
    assert int(bins.sum() + outside.sum()) == 6                             # NaN counted nowhere (R12)


@pytest.mark.parametrize("nbins", [256, 1024, 4096, 65536])
def test_histogram_top_clamp_covers_all_in_range_values(nbins):
    # R11: for random (lo,hi) the raw index of x=hi or nextbelow(hi) can reach nbins; the
    # result must stay inside [0, nbins-1] and be monotone in x.
    for _ in range(300):
        lo = np.float32(rng.normal())
        hi = np.float32(lo + abs(rng.normal()) + 1e-3)
        xs = np.sort(np.concatenate([
            np.array([lo, hi, np.nextafter(hi, lo, dtype=np.float32), np.nextafter(lo, hi, dtype=np.float32)]),
            rng.uniform(lo, hi, 20).astype(np.float32)])).astype(np.float32)
        xs = xs[(xs >= lo) & (xs <= hi)]
        idx = [oracle.bin_index(x, nbins, lo, hi) for x in xs]
        assert idx[0] == 0 and 0 <= min(idx) and max(idx) <= nbins - 1
        assert idx[-1] == nbins - 1
        assert all(b1 <= b2 for b1, b2 in zip(idx, idx[1:]))


def test_histogram_bin_index_matches_exact_bin_within_one():
    # a transposed operand or wrong sign moves bins by far more than rounding can
    for _ in range(2000):
        lo = np.float32(rng.normal() * 3)
        hi = np.float32(lo + abs(rng.normal()) * 5 + 1e-2)
        nbins = int(rng.choice([7, 256, 1000, 4096]))
        x = np.float32(rng.uniform(lo, hi))
        if not (lo <= x <= hi):
            continue
        exact = (Fraction(float(x)) - Fraction(float(lo))) * nbins / (Fraction(float(hi)) - Fraction(float(lo)))
        b = oracle.bin_index(x, nbins, lo, hi)
        assert abs(b - min(int(exact), nbins - 1)) <= 1


def test_histogram_hi_equals_lo_and_invalid():
    a = np.array([2.0, 2.0, 1.0, 3.0, np.nan], np.float32)
    bins, outside = oracle.histogram(a, 8, 2.0, 2.0)                        # R13
    assert bins.tolist() == [2, 0, 0, 0, 0, 0, 0, 0] and outside.tolist() == [1, 1]
    for bad in ((0, 0.0, 1.0), (4, 1.0, 0.0), (4, float("nan"), 1.0), (4, 0.0, float("inf"))):
        with pytest.raises(ValueError):
            oracle.histogram(a, *bad)


def test_histogram_sum_invariant_and_permutation():
    a = (rng.standard_normal(50000) * 0.002).astype(np.float32)
    a[rng.integers(0, a.size, 500)] = np.nan
    n = int((~np.isnan(a)).sum())
    b0, o0 = oracle.histogram(a, 4096, -0.02, 0.5)
    assert int(b0.sum() + o0.sum()) == n
    b1, o1 = oracle.histogram(rng.permutation(a), 4096, -0.02, 0.5)
    assert (b0 == b1).all() and (o0 == o1).all()
    mm = oracle.moments(a)
    b2, o2 = oracle.histogram(a, 1024, mm["min"], mm["max"])                # over [min,max]: nothing outside
    assert o2.tolist() == [0, 0] and int(b2.sum()) == n and b2[0] >= 1 and b2[-1] >= 1


# --------------------------------------------------------------------------- k-th / median
def _tiny_cases():
    r = np.random.default_rng(7)
    cases = [np.array([5.0], np.float32), np.array([2.0, 1.0], np.float32),
             np.array([-0.0, 0.0, 0.0], np.float32), np.array([0.0, -0.0], np.float32),
             np.array([1e-40, -1e-40, 0.0, -0.0, 1e-45], np.float32),
             np.array([np.inf, -np.inf, 1.0, np.nan], np.float32)]
    for n in (3, 4, 7, 8, 33, 100, 257):
        cases.append(r.standard_normal(n).astype(np.float32))
        cases.append(r.integers(-3, 4, n).astype(np.float32))              # heavy ties
        c = r.standard_normal(n).astype(np.float32)
        c[r.integers(0, n, max(1, n // 5))] = np.nan
        cases.append(c)
    return cases


@pytest.mark.parametrize("a", _tiny_cases())
def test_kth_and_median_against_full_sort(a):
    s = sorted([v for v in a.tolist() if not math.isnan(v)], key=total_key)
    n = len(s)
    for k in range(n):
        got = float(oracle.kth(a, k))
        assert got == s[k] and math.copysign(1.0, got) == math.copysign(1.0, s[k])
        less, equal = oracle.rank_counts(a, got)
        assert equal >= 1 and less <= k < less + equal                      # rank certificate
    with pytest.raises(IndexError):
        oracle.kth(a, n)
    med = float(oracle.median(a))
    assert med == s[(n - 1) // 2]                                           # LOWER median (R5)
    if n % 2 == 0 and s[n // 2 - 1] != s[n // 2]:
        assert med != s[n // 2]


def test_kth_on_ramp_is_k():
    N = 1 << 16
    a = rng.permutation(np.arange(N, dtype=np.float32))
    for k in (0, 1, N // 100, (N - 1) // 2, 99 * N // 100, N - 1):
        assert oracle.kth(a, k) == np.float32(k)
    assert oracle.median(a) == np.float32((N - 1) // 2)


def test_median_nan_signs_do_not_leak_into_order():
    neg_nan = np.frombuffer(np.uint32(0xFFC00000).tobytes(), dtype=np.float32)[0]
    a = np.array([neg_nan, 3.0, np.nan, 1.0, 2.0, neg_nan], np.float32)     # R6
    assert oracle.median(a) == 2.0 and oracle.kth(a, 0) == 1.0 and oracle.kth(a, 2) == 3.0
    assert math.isnan(float(oracle.median(np.array([np.nan], np.float32))))


# --------------------------------------------------------------------------- Torben (Alg. 1) and Table 1
def _table1():
    rows, N, med = [], None, None
    for line in open(GOLD):
        if line.startswith("# N ="):
            parts = line.split()
            N, med = int(parts[3]), parts[6]
        if line.startswith("#") or not line.strip():
            continue
        t = line.split()
        rows.append((int(t[0]), t[1], float(t[2]), float(t[3]), int(t[4]), int(t[5]), int(t[6])))
    return rows, N, med


def test_table1_guess_is_float32_midpoint():
    # R1: "Guess = (Min+Max)/" restored as /2 in float32: every printed guess matches to all
    # 10 printed decimals (rows 2, 3 differ from the float64 midpoint in the 9th digit).
    rows, N, med = _table1()
    for it, guess, mn, mx, *_ in rows:
        g = oracle.torben_guess(np.float32(mn), np.float32(mx))
        assert "%.10f" % float(g) == "%.10f" % float(guess), (it, g, guess)
    g64 = (float(np.float32(rows[1][2])) + float(np.float32(rows[1][3]))) / 2.0
    assert "%.10f" % g64 != rows[1][1]


def test_table1_counts_stop_rule_and_pick():
    rows, N, med = _table1()
    assert N == 534397200
    for it, guess, mn, mx, less, greater, equal in rows:
        assert less + greater + equal == N                                   # R3: i in [0, N)
        assert oracle.torben_stop(less, greater, N) == (it == 31)            # R2/R4: stops at row 31 only
    it, guess, mn, mx, less, greater, equal = rows[-1]
    # final branch returns Guess, the quoted median
    got = oracle.torben_pick(less, equal, N, np.float32(mn), np.float32(guess), np.float32(mx))
    assert "%.10f" % float(got) == med
    # and that is the LOWER median: rank k=(N-1)/2 falls on the first of the 'equal' elements (R5)
    k = (N - 1) // 2
    assert less <= k < less + equal and less == k
    # interval updates follow "if Less > Greater then Max = MaxLess else Min = MinGreater"
    r1, r2, r3 = rows[0], rows[1], rows[2]
    assert r1[4] < r1[5] and r2[2] > r1[2] and r2[3] == r1[3]                # row1: Less<Greater -> Min moves
    assert r2[4] > r2[5] and r3[3] < r2[3] and r3[2] == r2[2]                # row2: Less>Greater -> Max moves


@pytest.mark.parametrize("seed", range(40))
def test_torben_equals_sort_definition(seed):
    r = np.random.default_rng(seed)
    n = int(r.integers(1, 400))
    kind = seed % 4
    if kind == 0:
        a = r.standard_normal(n).astype(np.float32)
    elif kind == 1:
        a = r.integers(-2, 3, n).astype(np.float32)                          # heavy ties
    elif kind == 2:
        a = (r.standard_normal(n) * 1e-41).astype(np.float32)                # subnormals
    else:
        a = r.standard_normal(n).astype(np.float32)
        a[r.integers(0, n, n // 4 + 1)] = np.nan
        if np.isnan(a).all():
            a[0] = 1.0
    med, iters, trace = oracle.torben_median(a)
    s = sorted(v for v in a.tolist() if not math.isnan(v))
    assert float(med) == s[(len(s) - 1) // 2]
    assert float(med) == float(oracle.median(a)) or float(med) == 0.0        # (+-0 may differ in sign only)
    assert iters >= 1 and (trace[:, 3] + trace[:, 4] + trace[:, 5] == len(s)).all()
    assert (np.diff(trace[:, 2] - trace[:, 1]) <= 0).all()                    # interval never grows


def test_torben_iteration_count_scales_like_log_n():
    # "estimated to be O(log N)"; 31 iterations for 5.3e8 voxels.
    a = (rng.standard_normal(200000) * 0.05).astype(np.float32)
    med, iters, _ = oracle.torben_median(a)
    assert med == oracle.median(a) and 10 <= iters <= 40


def test_moments_with_infinite_voxels_reading_r8():
    # DESIGN.md R8: count / min / max are exact, mean and std are NaN as soon as one voxel is infinite -- for either
    # sign, both signs, any position and any number of them; a cube without one is untouched by the rule
    base = np.array([1.0, -2.0, 0.5, 3.0, np.nan], dtype=np.float32)
    for extra in ([np.inf], [-np.inf], [np.inf, -np.inf], [np.inf] * 5, [-np.inf, -np.inf, 7.0]):
        for pos in (0, 3, 5):
            a = np.insert(base, pos, np.array(extra, dtype=np.float32))
            m = oracle.moments(a)
            assert m["count"] == a.size - 1 and m["nan_count"] == 1
            assert m["min"] == np.nanmin(a) and m["max"] == np.nanmax(a)
            assert np.isnan(m["mean"]) and np.isnan(m["std"])
            s = oracle.moments(a, sample_std=True)
            assert np.isnan(s["mean"]) and np.isnan(s["std"])
    m = oracle.moments(base)
    assert m["mean"] == 0.625 and abs(m["std"] - np.sqrt(np.mean((np.array([1.0, -2.0, 0.5, 3.0]) - 0.625) ** 2))) < 1e-15
    # the clipped moments see the rule only when the window holds an infinity
    a = np.array([1.0, 2.0, 3.0, np.inf], dtype=np.float32)
    assert oracle.clipped_moments(a, 0.0, 10.0)["mean"] == 2.0
    assert np.isnan(oracle.clipped_moments(a, 0.0, np.inf)["mean"])
