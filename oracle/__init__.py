"""CPU ORACLE loader -- TEST INFRASTRUCTURE, NOT THE PRODUCT.

Only ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s ``cpu_baseline`` /
``--impl reference`` legs may import this package.  It builds (g++) and loads
``oracle/cube_oracle.cpp`` through ctypes.  It shares nothing with, and never imports,
``paper_1211_4896_b200`` (the CUDA path); the CUDA path never imports this.

Every function is a thin marshalling wrapper over one ``extern "C"`` function of
cube_oracle.cpp; the passages each follows are cited there.
"""
import ctypes
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "cube_oracle.cpp")
_LIB = os.path.join(_HERE, "libcube_oracle.so")
_FLAGS = ["-O2", "-std=c++17", "-ffp-contract=off", "-fno-fast-math", "-fPIC", "-shared"]


# CUBE_ORACLE_SANITIZE=1: the same source built with AddressSanitizer + UndefinedBehaviorSanitizer into its own
# library; run the CPU pins under it with
#   CUBE_ORACLE_SANITIZE=1 LD_PRELOAD=$(gcc -print-file-name=libasan.so) ASAN_OPTIONS=detect_leaks=0 \
#       python -m pytest tests/test_oracle_pins.py tests/test_oracle_next_pins.py tests/test_oracle_render_pins.py -q
_SANITIZE = os.environ.get("CUBE_ORACLE_SANITIZE", "0") == "1"
if _SANITIZE:
    _LIB = os.path.join(_HERE, "libcube_oracle_san.so")
    _FLAGS = _FLAGS + ["-g", "-fsanitize=address,undefined", "-fno-sanitize-recover=undefined", "-fno-omit-frame-pointer"]


def build(force=False):
    """Compile cube_oracle.cpp -> libcube_oracle.so (no-op when up to date)."""
    if (not force and os.path.exists(_LIB)
            and os.path.getmtime(_LIB) >= os.path.getmtime(_SRC)):
        return _LIB
    tmp = _LIB + ".tmp.%d" % os.getpid()
    subprocess.check_call(["g++"] + _FLAGS + ["-o", tmp, _SRC])
    os.replace(tmp, _LIB)
    return _LIB


class Moments(ctypes.Structure):
    _fields_ = [("count", ctypes.c_uint64), ("nan_count", ctypes.c_uint64),
                ("min", ctypes.c_float), ("max", ctypes.c_float),
                ("mean", ctypes.c_double), ("std", ctypes.c_double)]


class View(ctypes.Structure):
    """oracle_view_t: origin, du, dv, step (data coordinates = voxel indices), width, height, nsteps."""
    _fields_ = [("origin", ctypes.c_float * 3), ("du", ctypes.c_float * 3), ("dv", ctypes.c_float * 3),
                ("step", ctypes.c_float * 3), ("width", ctypes.c_int32), ("height", ctypes.c_int32),
                ("nsteps", ctypes.c_int32)]


def _view(v):
    """dict(origin, du, dv, step, width, height, nsteps) (cubegen.view_*) -> View."""
    w = View()
    for name in ("origin", "du", "dv", "step"):
        a = np.asarray(v[name], dtype=np.float32)
        for c in range(3):
            getattr(w, name)[c] = float(a[c])
    w.width, w.height, w.nsteps = int(v["width"]), int(v["height"]), int(v["nsteps"])
    return w


_lib = None


def lib():
    global _lib
    if _lib is None:
        L = ctypes.CDLL(build())
        fp = ctypes.POINTER(ctypes.c_float)
        u64p = ctypes.POINTER(ctypes.c_uint64)
        L.oracle_moments.argtypes = [fp, ctypes.c_uint64, ctypes.c_int, ctypes.POINTER(Moments)]
        L.oracle_bin_index.argtypes = [ctypes.c_float, ctypes.c_int, ctypes.c_float, ctypes.c_float]
        L.oracle_bin_index.restype = ctypes.c_int
        L.oracle_histogram.argtypes = [fp, ctypes.c_uint64, ctypes.c_int, ctypes.c_float,
                                       ctypes.c_float, u64p, u64p]
        L.oracle_kth.argtypes = [fp, ctypes.c_uint64, ctypes.c_uint64, fp]
        L.oracle_median.argtypes = [fp, ctypes.c_uint64, fp]
        L.oracle_rank_counts.argtypes = [fp, ctypes.c_uint64, ctypes.c_float, u64p, u64p]
        L.oracle_torben_guess.argtypes = [ctypes.c_float, ctypes.c_float]
        L.oracle_torben_guess.restype = ctypes.c_float
        L.oracle_torben_stop.argtypes = [ctypes.c_uint64] * 3
        L.oracle_torben_pick.argtypes = [ctypes.c_uint64] * 3 + [ctypes.c_float] * 3
        L.oracle_torben_pick.restype = ctypes.c_float
        L.oracle_torben_median.argtypes = [fp, ctypes.c_uint64, fp,
                                           ctypes.POINTER(ctypes.c_double), ctypes.c_int]
        mp = ctypes.POINTER(Moments)
        L.oracle_clipped_moments.argtypes = [fp, ctypes.c_uint64, ctypes.c_float, ctypes.c_float, ctypes.c_int, mp]
        L.oracle_sigma_clip.argtypes = [fp, ctypes.c_uint64, ctypes.c_double, ctypes.c_int, ctypes.c_int, mp, fp]
        L.oracle_mad.argtypes = [fp, ctypes.c_uint64, fp, fp]
        L.oracle_minimap.argtypes = [fp] + [ctypes.c_int64] * 6 + [ctypes.c_int, mp]
        L.oracle_torben_capped.argtypes = [fp, ctypes.c_uint64, ctypes.c_int, fp, ctypes.POINTER(ctypes.c_int)]
        L.oracle_minimap_median.argtypes = [fp] + [ctypes.c_int64] * 6 + [fp]
        vwp = ctypes.POINTER(View)
        i64 = ctypes.c_int64
        L.oracle_trilinear.argtypes = [fp, i64, i64, i64, fp, fp]
        L.oracle_spectrum.argtypes = [fp, i64, i64, i64, vwp, ctypes.c_int, ctypes.c_int, fp]
        L.oracle_render_mip.argtypes = [fp, i64, i64, i64, vwp, ctypes.c_float, fp]
        L.oracle_minimap_lookup.argtypes = [mp] + [i64] * 6 + [fp, fp, fp]
        L.oracle_render_sigma.argtypes = [fp, i64, i64, i64, vwp, mp, i64, i64, i64, ctypes.c_int, ctypes.c_float,
                                          ctypes.c_float, fp, ctypes.c_float, fp]
        L.oracle_render_tf.argtypes = [fp, i64, i64, i64, vwp, ctypes.c_int, ctypes.c_float, ctypes.c_float, fp,
                                       ctypes.c_float, fp]
        _lib = L
    return _lib


def _arr(a):
    a = np.ascontiguousarray(a, dtype=np.float32).reshape(-1)
    return a, a.ctypes.data_as(ctypes.POINTER(ctypes.c_float))


def moments(a, sample_std=False):
    """-> dict(count, nan_count, min, max, mean, std).  PAPER.md:265, 273."""
    a, p = _arr(a)
    m = Moments()
    lib().oracle_moments(p, a.size, int(bool(sample_std)), ctypes.byref(m))
    return dict(count=m.count, nan_count=m.nan_count, min=np.float32(m.min),
                max=np.float32(m.max), mean=m.mean, std=m.std)


def bin_index(x, nbins, lo, hi):
    return lib().oracle_bin_index(float(np.float32(x)), int(nbins),
                                  float(np.float32(lo)), float(np.float32(hi)))


def histogram(a, nbins, lo, hi):
    """-> (bins[nbins] uint64, outside[2] uint64).  PAPER.md:259-261."""
    a, p = _arr(a)
    bins = np.zeros(nbins, dtype=np.uint64)
    outside = np.zeros(2, dtype=np.uint64)
    u64p = ctypes.POINTER(ctypes.c_uint64)
    rc = lib().oracle_histogram(p, a.size, int(nbins), float(np.float32(lo)), float(np.float32(hi)),
                                bins.ctypes.data_as(u64p), outside.ctypes.data_as(u64p))
    if rc != 0:
        raise ValueError("oracle_histogram: invalid arguments")
    return bins, outside


def kth(a, k):
    """k-th (0-based) smallest non-NaN value in total order.  PAPER.md:281."""
    a, p = _arr(a)
    out = ctypes.c_float()
    rc = lib().oracle_kth(p, a.size, int(k), ctypes.byref(out))
    if rc != 0:
        raise IndexError("k >= non-NaN count")
    return np.float32(out.value)


def median(a):
    """Lower median, k=(n-1)/2; NaN if there is no non-NaN voxel."""
    a, p = _arr(a)
    out = ctypes.c_float()
    lib().oracle_median(p, a.size, ctypes.byref(out))
    return np.float32(out.value)


def rank_counts(a, m):
    """-> (#{x<m}, #{x==m}) in total order over the non-NaN voxels."""
    a, p = _arr(a)
    less, equal = ctypes.c_uint64(), ctypes.c_uint64()
    lib().oracle_rank_counts(p, a.size, float(np.float32(m)), ctypes.byref(less), ctypes.byref(equal))
    return less.value, equal.value


def torben_guess(mn, mx):
    return np.float32(lib().oracle_torben_guess(float(np.float32(mn)), float(np.float32(mx))))


def torben_stop(less, greater, n):
    return bool(lib().oracle_torben_stop(int(less), int(greater), int(n)))


def torben_pick(less, equal, n, maxlt, guess, mingt):
    return np.float32(lib().oracle_torben_pick(int(less), int(equal), int(n), float(np.float32(maxlt)),
                                               float(np.float32(guess)), float(np.float32(mingt))))


def torben_median(a, max_trace=64):
    """Alg. 1.  -> (median, iterations, trace[iterations,6])."""
    a, p = _arr(a)
    out = ctypes.c_float()
    trace = np.zeros((max_trace, 6), dtype=np.float64)
    it = lib().oracle_torben_median(p, a.size, ctypes.byref(out),
                                    trace.ctypes.data_as(ctypes.POINTER(ctypes.c_double)), max_trace)
    return np.float32(out.value), it, trace[:max(0, min(it, max_trace))]


def _mdict(m):
    return dict(count=m.count, nan_count=m.nan_count, min=np.float32(m.min), max=np.float32(m.max),
                mean=m.mean, std=m.std)


def clipped_moments(a, lo, hi, sample_std=False):
    """Moments of the voxels with lo <= x <= hi (float32 window); nan_count = everything left out."""
    a, p = _arr(a)
    m = Moments()
    lib().oracle_clipped_moments(p, a.size, float(np.float32(lo)), float(np.float32(hi)), int(bool(sample_std)),
                                 ctypes.byref(m))
    return _mdict(m)


def sigma_clip(a, kappa, max_iter, sample_std=False):
    """Iterated kappa-sigma clipping about the mean.
    -> (moments dict of the last pass, clipped passes made, (lo, hi) of the last window)."""
    a, p = _arr(a)
    m = Moments()
    w = (ctypes.c_float * 2)()
    it = lib().oracle_sigma_clip(p, a.size, float(kappa), int(max_iter), int(bool(sample_std)), ctypes.byref(m), w)
    return _mdict(m), it, (np.float32(w[0]), np.float32(w[1]))


def mad(a):
    """-> (lower median, median absolute deviation |fl32(x - med)|).  PAPER.md:292."""
    a, p = _arr(a)
    med, out = ctypes.c_float(), ctypes.c_float()
    lib().oracle_mad(p, a.size, ctypes.byref(med), ctypes.byref(out))
    return np.float32(med.value), np.float32(out.value)


def minimap(a, dims, part, sample_std=False):
    """Statistical mini-map.  dims = (nx, ny, nz) with x fastest, part = (px, py, pz).
    -> structured array [mz, my, mx] with fields count, nan_count, min, max, mean, std."""
    a, p = _arr(a)
    nx, ny, nz = dims
    px, py, pz = part
    assert a.size == nx * ny * nz
    mx, my, mz = -(-nx // px), -(-ny // py), -(-nz // pz)
    cells = (Moments * (mx * my * mz))()
    rc = lib().oracle_minimap(p, nx, ny, nz, px, py, pz, int(bool(sample_std)), cells)
    if rc != 0:
        raise ValueError("oracle_minimap: invalid arguments")
    dt = np.dtype([("count", "<u8"), ("nan_count", "<u8"), ("min", "<f4"), ("max", "<f4"), ("mean", "<f8"),
                   ("std", "<f8")])
    return np.frombuffer(bytes(cells), dtype=dt).reshape(mz, my, mx).copy()


def torben_capped(a, max_iter):
    """Alg. 1 stopped after at most ``max_iter`` passes.  -> (value, passes made, converged)."""
    a, p = _arr(a)
    out, conv = ctypes.c_float(), ctypes.c_int()
    it = lib().oracle_torben_capped(p, a.size, int(max_iter), ctypes.byref(out), ctypes.byref(conv))
    return np.float32(out.value), it, bool(conv.value)


def minimap_median(a, dims, part):
    """Lower median of every mini-map cell (NaN for a cell without a non-NaN voxel) -> float32 [mz, my, mx]."""
    a, p = _arr(a)
    nx, ny, nz = dims
    px, py, pz = part
    assert a.size == nx * ny * nz
    mx, my, mz = -(-nx // px), -(-ny // py), -(-nz // pz)
    out = np.zeros(mx * my * mz, dtype=np.float32)
    rc = lib().oracle_minimap_median(p, nx, ny, nz, px, py, pz, out.ctypes.data_as(ctypes.POINTER(ctypes.c_float)))
    if rc != 0:
        raise ValueError("oracle_minimap_median: invalid arguments")
    return out.reshape(mz, my, mx)


# ---- NEXT-4: ray casting.  dims = (nx, ny, nz), x fastest; view = cubegen.view_* dict.
def trilinear(a, dims, point):
    """Trilinear sample at the data coordinates ``point`` (float32 x, y, z) -> float32, or None when outside."""
    a, p = _arr(a)
    nx, ny, nz = dims
    pt = (ctypes.c_float * 3)(*[float(np.float32(c)) for c in point])
    out = ctypes.c_float()
    ok = lib().oracle_trilinear(p, nx, ny, nz, pt, ctypes.byref(out))
    return np.float32(out.value) if ok else None


def spectrum(a, dims, view, u, v):
    """3-D spectrum tool: the nsteps trilinear samples of pixel (u, v)'s ray (NaN outside the cube)."""
    a, p = _arr(a)
    nx, ny, nz = dims
    w = _view(view)
    out = np.zeros(w.nsteps, dtype=np.float32)
    lib().oracle_spectrum(p, nx, ny, nz, ctypes.byref(w), int(u), int(v), out.ctypes.data_as(ctypes.POINTER(ctypes.c_float)))
    return out


def render_mip(a, dims, view, vmin=-np.inf):
    """Maximum intensity projection -> float32 [height, width] (NaN: no sample >= vmin on the ray)."""
    a, p = _arr(a)
    nx, ny, nz = dims
    w = _view(view)
    out = np.zeros(w.width * w.height, dtype=np.float32)
    lib().oracle_render_mip(p, nx, ny, nz, ctypes.byref(w), float(np.float32(vmin)),
                            out.ctypes.data_as(ctypes.POINTER(ctypes.c_float)))
    return out.reshape(w.height, w.width)


def render_tf(a, dims, view, table, lo, hi, opacity_cut=2.0):
    """Generic transfer function, front-to-back compositing.  table: [nlevels, 4] float32 (r, g, b, opacity).
    -> float32 [height, width, 4] (opacity-weighted r, g, b and the accumulated opacity)."""
    a, p = _arr(a)
    nx, ny, nz = dims
    w = _view(view)
    t = np.ascontiguousarray(table, dtype=np.float32).reshape(-1, 4)
    out = np.zeros(w.width * w.height * 4, dtype=np.float32)
    fp = ctypes.POINTER(ctypes.c_float)
    rc = lib().oracle_render_tf(p, nx, ny, nz, ctypes.byref(w), t.shape[0], float(np.float32(lo)), float(np.float32(hi)),
                                t.ctypes.data_as(fp), float(np.float32(opacity_cut)), out.ctypes.data_as(fp))
    if rc != 0:
        raise ValueError("oracle_render_tf: invalid arguments")
    return out.reshape(w.height, w.width, 4)


_MAP_DT = np.dtype([("count", "<u8"), ("nan_count", "<u8"), ("min", "<f4"), ("max", "<f4"), ("mean", "<f8"), ("std", "<f8")])


def _cells(cells):
    """mini-map records (structured array as returned by ``minimap``) -> ctypes array of Moments."""
    c = np.ascontiguousarray(cells, dtype=_MAP_DT).reshape(-1)
    return (Moments * c.size).from_buffer_copy(c.tobytes())


def minimap_lookup(cells, dims, part, point):
    """(mean, std) of the mini-map ``cells`` (structured array [mz, my, mx]) interpolated at the data point (R34)."""
    nx, ny, nz = dims
    px, py, pz = part
    pt = (ctypes.c_float * 3)(*[float(np.float32(c)) for c in point])
    m, s = ctypes.c_float(), ctypes.c_float()
    lib().oracle_minimap_lookup(_cells(cells), nx, ny, nz, px, py, pz, pt, ctypes.byref(m), ctypes.byref(s))
    return np.float32(m.value), np.float32(s.value)


def render_sigma(a, dims, view, cells, part, table, zlo, zhi, opacity_cut=2.0):
    """Sigma-clipping transfer function: levels of z = (sample - local mean) / local std over
    [zlo, zhi], local statistics interpolated in the mini-map.  -> float32 [height, width, 4]."""
    a, p = _arr(a)
    nx, ny, nz = dims
    px, py, pz = part
    w = _view(view)
    t = np.ascontiguousarray(table, dtype=np.float32).reshape(-1, 4)
    out = np.zeros(w.width * w.height * 4, dtype=np.float32)
    fp = ctypes.POINTER(ctypes.c_float)
    rc = lib().oracle_render_sigma(p, nx, ny, nz, ctypes.byref(w), _cells(cells), px, py, pz, t.shape[0],
                                   float(np.float32(zlo)), float(np.float32(zhi)), t.ctypes.data_as(fp),
                                   float(np.float32(opacity_cut)), out.ctypes.data_as(fp))
    if rc != 0:
        raise ValueError("oracle_render_sigma: invalid arguments")
    return out.reshape(w.height, w.width, 4)
