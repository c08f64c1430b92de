"""Pins for the NEXT-1 / NEXT-2 parts of the CPU oracle (MAD, clipped moments, sigma clipping, statistical
mini-map; readings R21-R25) against things other than the oracle:
closed forms on ramps, exact rational arithmetic, brute force with numpy sorts / block reshapes, invariants.
CPU only.
"""
import math
from fractions import Fraction

import numpy as np
import pytest

import oracle

rng = np.random.default_rng(4896)


def exact_mean_var(vals):
    fr = [Fraction(float(v)) for v in vals]
    n = len(fr)
    mean = sum(fr) / n
    return mean, sum((f - mean) ** 2 for f in fr) / n


def sqrt_fraction(fr):
    """Square root of a non-negative Fraction as the nearest double (integer square root on 2^200-scaled value)."""
    if fr == 0:
        return 0.0
    num = fr.numerator << 400
    r = math.isqrt(num // fr.denominator)
    return float(Fraction(r, 1 << 200))


# --------------------------------------------------------------------------------------- MAD
@pytest.mark.parametrize("m", [1, 2, 7, 50, 4095])
def test_mad_ramp_closed_form(m):
    # x = 0..2m: median m; deviations 0,1,1,2,2,...,m,m; the element of rank m is ceil(m/2)
    a = np.arange(2 * m + 1, dtype=np.float32)
    a = a[rng.permutation(a.size)]
    med, mad = oracle.mad(a)
    assert med == m and mad == (m + 1) // 2


@pytest.mark.parametrize("seed", range(12))
def test_mad_equals_sort_definition(seed):
    r = np.random.default_rng(seed)
    n = int(r.integers(1, 400))
    a = (r.standard_normal(n) * 10 ** r.uniform(-3, 3)).astype(np.float32)
    if seed % 3 == 0:
        a = np.round(a * 4) / 4          # heavy ties
    if seed % 4 == 1:
        a[r.integers(0, n, size=max(1, n // 10))] = np.nan
    v = np.sort(a[~np.isnan(a)])
    med, mad = oracle.mad(a)
    if v.size == 0:
        assert math.isnan(med) and math.isnan(mad)
        return
    m = v[(v.size - 1) // 2]
    y = np.sort(np.abs((v - m).astype(np.float32)))          # float32 subtraction, as the definition says
    assert med == m
    assert mad == y[(y.size - 1) // 2]


def test_mad_even_count_takes_lower_medians():
    a = np.array([1, 2, 4, 8], dtype=np.float32)              # lower median 2; deviations 1,0,2,6 -> sorted 0,1,2,6 -> 1
    assert oracle.mad(a) == (2.0, 1.0)
    assert oracle.mad(np.array([5.0], dtype=np.float32)) == (5.0, 0.0)


def test_mad_scale_and_nan_invariance():
    a = rng.standard_normal(1001).astype(np.float32)
    med, mad = oracle.mad(a)
    med2, mad2 = oracle.mad(np.concatenate([a * np.float32(4.0), np.full(17, np.nan, np.float32)]))
    assert med2 == med * 4 and mad2 == mad * 4               # scaling by a power of two is exact
    assert mad > 0
    # Gaussian: MAD ~ 0.6745 sigma (sanity, not a pin)
    assert 0.55 < mad < 0.8


def test_mad_constant_and_two_values():
    assert oracle.mad(np.full(100, 3.25, np.float32)) == (3.25, 0.0)
    a = np.array([1.0] * 60 + [9.0] * 40, dtype=np.float32)  # median 1; deviations: 60 zeros, 40 eights -> 0
    assert oracle.mad(a) == (1.0, 0.0)
    a = np.array([1.0] * 50 + [9.0] * 50, dtype=np.float32)  # lower median 1; rank 49 of (50 zeros, 50 eights) -> 0
    assert oracle.mad(a) == (1.0, 0.0)
    a = np.array([1.0] * 49 + [9.0] * 51, dtype=np.float32)  # median 9; 51 zeros
    assert oracle.mad(a) == (9.0, 0.0)


# --------------------------------------------------------------------------------------- clipped moments
def test_clipped_window_covering_everything_is_plain_moments():
    a = rng.standard_normal(5000).astype(np.float32)
    a[::97] = np.nan
    m = oracle.moments(a)
    c = oracle.clipped_moments(a, m["min"], m["max"])
    assert c == m


@pytest.mark.parametrize("lo,hi", [(10, 20), (0, 0), (100, 1023), (5.5, 9.5)])
def test_clipped_ramp_closed_form(lo, hi):
    N = 1024
    a = np.arange(N, dtype=np.float32)[rng.permutation(N)]
    c = oracle.clipped_moments(a, lo, hi)
    first, last = math.ceil(lo), math.floor(hi)              # closed window
    n = last - first + 1
    assert c["count"] == n and c["nan_count"] == N - n
    assert c["min"] == first and c["max"] == last
    assert c["mean"] == (first + last) / 2.0
    assert c["std"] == pytest.approx(math.sqrt((n * n - 1) / 12.0), rel=1e-15, abs=0)
    if n > 1:
        s = oracle.clipped_moments(a, lo, hi, sample_std=True)
        assert s["std"] == pytest.approx(math.sqrt(n * (n + 1) / 12.0), rel=1e-15)


def test_clipped_exact_rational_and_nan_and_empty():
    a = (rng.standard_normal(300) * 3).astype(np.float32)
    a[::13] = np.nan
    lo, hi = np.float32(-1.5), np.float32(2.25)
    sel = [v for v in a if lo <= v <= hi]
    c = oracle.clipped_moments(a, lo, hi)
    mean, var = exact_mean_var(sel)
    assert c["count"] == len(sel) and c["nan_count"] == a.size - len(sel)
    assert c["mean"] == pytest.approx(float(mean), rel=1e-15)
    assert c["std"] == pytest.approx(sqrt_fraction(var), rel=1e-15)
    assert c["min"] == min(sel) and c["max"] == max(sel)
    e = oracle.clipped_moments(a, 100.0, 200.0)
    assert e["count"] == 0 and e["nan_count"] == a.size and math.isnan(e["mean"]) and math.isnan(e["min"])
    # an inverted window selects nothing
    assert oracle.clipped_moments(a, 1.0, -1.0)["count"] == 0


# --------------------------------------------------------------------------------------- sigma clipping
def reference_sigma_clip(vals, kappa, max_iter):
    """Independent restatement with exact rational moments (integers / dyadic rationals in, doubles out)."""
    cur = [float(v) for v in vals if not math.isnan(v)]
    counts = [len(cur)]
    iters = 0
    allv = list(cur)
    while iters < max_iter and cur:
        mean, var = exact_mean_var(cur)
        mean, std = float(mean), sqrt_fraction(var)
        lo, hi = np.float32(mean - kappa * std), np.float32(mean + kappa * std)
        nxt = [v for v in allv if lo <= v <= hi]
        iters += 1
        same = len(nxt) == len(cur)
        cur = nxt
        counts.append(len(cur))
        if same:
            break
    return cur, iters, counts


@pytest.mark.parametrize("seed,kappa", [(0, 3.0), (1, 2.0), (2, 2.5), (3, 1.0), (4, 3.0)])
def test_sigma_clip_against_exact_restatement(seed, kappa):
    r = np.random.default_rng(100 + seed)
    a = np.round(r.standard_normal(400) * 16).astype(np.float32)       # integers: window edges never graze a value
    a[r.integers(0, 400, 12)] = np.float32(500 + 37 * seed)            # outliers
    a[r.integers(0, 400, 5)] = np.nan
    got, iters, win = oracle.sigma_clip(a, kappa, 20)
    cur, ref_iters, counts = reference_sigma_clip(a, kappa, 20)
    assert iters == ref_iters
    assert got["count"] == len(cur) and got["nan_count"] == a.size - len(cur)
    mean, var = exact_mean_var(cur)
    assert got["mean"] == pytest.approx(float(mean), rel=1e-14)
    assert got["std"] == pytest.approx(sqrt_fraction(var), rel=1e-14)
    assert got["min"] == min(cur) and got["max"] == max(cur)
    assert counts == sorted(counts, reverse=True)                      # counts never increase
    assert counts[0] > counts[-1]                                      # the outliers were clipped


def test_sigma_clip_limits_and_degenerate():
    a = rng.standard_normal(1000).astype(np.float32)
    m0, it0, w0 = oracle.sigma_clip(a, 3.0, 0)                         # no pass: plain moments
    assert it0 == 0 and m0 == oracle.moments(a) and math.isnan(w0[0])
    m1, it1, w1 = oracle.sigma_clip(a, 3.0, 1)
    p = oracle.moments(a)
    lo, hi = np.float32(p["mean"] - 3.0 * p["std"]), np.float32(p["mean"] + 3.0 * p["std"])
    assert it1 == 1 and (w1[0], w1[1]) == (lo, hi)
    assert m1 == oracle.clipped_moments(a, lo, hi)
    c, itc, _ = oracle.sigma_clip(np.full(64, 2.5, np.float32), 3.0, 10)  # constant: std 0, window [c,c], 1 pass
    assert itc == 1 and c["count"] == 64 and c["std"] == 0.0
    e, ite, _ = oracle.sigma_clip(np.full(8, np.nan, np.float32), 3.0, 10)
    assert ite == 0 and e["count"] == 0
    # a huge kappa keeps everything: converged after one pass with identical statistics
    k, itk, _ = oracle.sigma_clip(a, 1e6, 10)
    assert itk == 1 and k == p


def test_sigma_clip_gaussian_with_outliers_recovers_noise():
    a = rng.standard_normal(200000).astype(np.float32)
    a[:2000] = 50.0
    m, it, _ = oracle.sigma_clip(a, 3.0, 30)
    assert 2 <= it <= 30
    assert 0.95 < m["std"] < 1.0 and abs(m["mean"]) < 0.02
    assert oracle.moments(a)["std"] > 4.0


# --------------------------------------------------------------------------------------- mini-map
def test_minimap_even_partition_against_numpy_blocks():
    nx, ny, nz, px, py, pz = 12, 8, 6, 3, 4, 2
    a = rng.standard_normal(nx * ny * nz).astype(np.float32)
    mm = oracle.minimap(a, (nx, ny, nz), (px, py, pz))
    blk = a.astype(np.float64).reshape(nz // pz, pz, ny // py, py, nx // px, px)
    assert mm.shape == (3, 2, 4)
    assert (mm["count"] == px * py * pz).all() and (mm["nan_count"] == 0).all()
    np.testing.assert_allclose(mm["mean"], blk.mean(axis=(1, 3, 5)), rtol=1e-13, atol=1e-15)
    np.testing.assert_allclose(mm["std"], blk.std(axis=(1, 3, 5)), rtol=1e-13)
    assert (mm["min"] == blk.min(axis=(1, 3, 5)).astype(np.float32)).all()
    assert (mm["max"] == blk.max(axis=(1, 3, 5)).astype(np.float32)).all()


def test_minimap_ragged_cells_nan_and_index_order():
    nx, ny, nz, px, py, pz = 7, 5, 4, 3, 2, 3
    a = np.arange(nx * ny * nz, dtype=np.float32)
    a[3::11] = np.nan
    cube = a.reshape(nz, ny, nx)
    cube[0:3, 0:2, 0:3] = np.nan                                       # cell (0,0,0) fully blanked
    mm = oracle.minimap(cube.reshape(-1), (nx, ny, nz), (px, py, pz))
    assert mm.shape == (2, 3, 3)
    for cz in range(2):
        for cy in range(3):
            for cx in range(3):
                blk = cube[cz * pz:(cz + 1) * pz, cy * py:(cy + 1) * py, cx * px:(cx + 1) * px].reshape(-1)
                ok = blk[~np.isnan(blk)]
                c = mm[cz, cy, cx]
                assert c["count"] == ok.size and c["nan_count"] == blk.size - ok.size
                if ok.size == 0:
                    assert math.isnan(c["mean"]) and math.isnan(c["min"])
                    continue
                mean, var = exact_mean_var(ok)
                assert c["mean"] == pytest.approx(float(mean), rel=1e-15)
                assert c["std"] == pytest.approx(sqrt_fraction(var), rel=1e-14, abs=1e-300)
                assert c["min"] == ok.min() and c["max"] == ok.max()
    assert mm[0, 0, 0]["count"] == 0
    assert int(mm["count"].sum() + mm["nan_count"].sum()) == nx * ny * nz


def test_minimap_single_cell_is_global_moments_and_constant():
    a = rng.standard_normal(4 * 5 * 6).astype(np.float32)
    mm = oracle.minimap(a, (4, 5, 6), (10, 10, 10))
    g = oracle.moments(a)
    assert mm.shape == (1, 1, 1)
    for k in ("count", "nan_count", "min", "max", "mean", "std"):
        assert mm[0, 0, 0][k] == g[k]
    c = oracle.minimap(np.full(64, 1.5, np.float32), (4, 4, 4), (2, 2, 2))
    assert (c["std"] == 0).all() and (c["mean"] == 1.5).all() and (c["count"] == 8).all()
    s = oracle.minimap(np.arange(16, dtype=np.float32), (4, 2, 2), (2, 2, 2), sample_std=True)
    # cell (0,0,0): values 0,1,4,5,8,9,12,13
    vals = np.array([0, 1, 4, 5, 8, 9, 12, 13], dtype=np.float64)
    assert s[0, 0, 0]["std"] == pytest.approx(vals.std(ddof=1), rel=1e-15)


# --------------------------------------------------------------------------------------- capped Torben (Alg. 1)
def restated_torben(vals, max_iter):
    """Alg. 1 restated independently with numpy float32 scalars; stops after max_iter passes."""
    v = np.asarray([x for x in vals if not math.isnan(x)], dtype=np.float32)
    n = v.size
    mn, mx = v.min(), v.max()
    it = 0
    while True:
        guess = np.float32((mn + mx) / np.float32(2))
        less, greater = int((v < guess).sum()), int((v > guess).sum())
        equal = n - less - greater
        maxlt = v[v < guess].max() if less else mn
        mingt = v[v > guess].min() if greater else mx
        it += 1
        half = (n + 1) // 2
        conv = less <= half and greater <= half
        if conv or it >= max_iter:
            break
        if less > greater:
            mx = maxlt
        else:
            mn = mingt
    res = maxlt if less >= half else (guess if less + equal >= half else mingt)
    return np.float32(res), it, conv


@pytest.mark.parametrize("seed", range(10))
def test_torben_capped_against_restatement_and_sort(seed):
    r = np.random.default_rng(300 + seed)
    n = int(r.integers(2, 3000))
    a = (r.standard_normal(n) * 10 ** r.uniform(-3, 3) + r.uniform(-1, 1)).astype(np.float32)
    if seed % 3 == 0:
        a = np.round(a * 2) / 2
    a[r.integers(0, n, n // 20)] = np.nan
    if np.isnan(a).all():
        a[0] = 1.0
    full, it_full, conv_full = oracle.torben_capped(a, 10000)
    v = np.sort(a[~np.isnan(a)])
    assert conv_full and full == v[(v.size - 1) // 2]                   # uncapped: the exact lower median
    assert (full, it_full) == oracle.torben_median(a)[:2]
    for cap in (1, 2, 3, 5, 8, it_full - 1, it_full, it_full + 3):
        if cap < 1:
            continue
        got = oracle.torben_capped(a, cap)
        ref = restated_torben(a, cap)
        assert got[1] == ref[1] == min(cap, it_full) and got[2] == ref[2] and got[0] == ref[0], (cap, got, ref)
        assert v[0] <= got[0] <= v[-1]
    # the approximation tightens: after c passes the result is within (max-min) / 2^(c-1) of the median
    span = float(v[-1]) - float(v[0])
    for cap in (4, 8, 12):
        if cap < it_full:
            assert abs(float(oracle.torben_capped(a, cap)[0]) - float(full)) <= span / 2 ** (cap - 1) + 1e-30


def test_torben_capped_degenerate():
    assert oracle.torben_capped(np.full(5, np.nan, np.float32), 10)[1] == -1
    val, it, conv = oracle.torben_capped(np.full(9, 2.5, np.float32), 10)
    assert (val, it, conv) == (2.5, 1, True)
    val, it, conv = oracle.torben_capped(np.array([1, 2, 3], np.float32), 0)
    assert math.isnan(val) and it == 0 and not conv
