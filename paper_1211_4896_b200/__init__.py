"""paper_1211_4896_b200 -- thin Python binding of libcube (include/cube.h).

Argument marshalling only: every step of the statistics path runs in the CUDA
kernels of ``csrc/``.  PyTorch is used by callers for device memory and streams; this module itself
needs only ctypes.  There is NO CPU fallback: if ``libcube.so`` is missing or no CUDA device is
present, ``Context()`` raises.  This package never imports ``oracle``.

    ctx = Context()
    m = ctx.moments(ptr, nx, ny, nz)            # ptr: device pointer (int), e.g. tensor.data_ptr()
    bins, outside = ctx.histogram(ptr, nx, ny, nz, 4096, -0.02, 0.5)
    med = ctx.median(ptr, nx, ny, nz)
"""
import ctypes
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
# CUBE_LIBPATH: load another build of the same library instead (e.g. the bounds-checked one: build.py --checked)
_LIBPATH = os.environ.get("CUBE_LIBPATH") or os.path.join(_HERE, "libcube.so")

OK, EINVAL, EEMPTY, ECUDA, ERANGE, ENOMEM, ECALLBACK = 0, 1, 2, 3, 4, 5, 6
# int fill(void* user, uint64_t brick, int sweep, float* h_dst, uint64_t nvox, cudaStream_t fill_stream)
FILL_FN = ctypes.CFUNCTYPE(ctypes.c_int, ctypes.c_void_p, ctypes.c_uint64, ctypes.c_int, ctypes.c_void_p,
                           ctypes.c_uint64, ctypes.c_void_p)
SAMPLE_STD, COARSE_HIST, REUSE_COARSE, RANGE_MINMAX = 1, 2, 4, 8
MAX_BINS = 65536

# every symbol include/cube.h declares (checked by tests/test_abi.py)
SYMBOLS = ["cube_create", "cube_destroy", "cube_moments", "cube_histogram", "cube_kth", "cube_kth_ex", "cube_kth_multi",
           "cube_median", "cube_median_ex", "cube_stats", "cube_probe_read", "cube_ooc_begin", "cube_ooc_begin_ex", "cube_ooc_brick", "cube_ooc_next_sweep",
           "cube_ooc_result", "cube_host_workspace", "cube_stats_host", "cube_stream_workspace", "cube_stats_stream",
           "cube_stream_info", "cube_strerror",
           "cube_last_cuda_error", "cube_set_launch", "cube_set_knob", "cube_launch_count",
           "cube_profile_enable", "cube_profile_reset", "cube_profile_read",
           "cube_mad", "cube_clipped_moments", "cube_sigma_clip", "cube_minimap_dims", "cube_minimap",
           "cube_shard_buffers", "cube_shard_merge_records", "cube_shard_advance", "cube_median_torben",
           "cube_view_orbit", "cube_render_mip", "cube_render_tf", "cube_render_sigma", "cube_spectrum",
           "cube_minimap_median", "cube_histogram_noalloc"]
NOALLOC_MAX_BINS = 4096
SHARD_RECORD_BYTES, SHARD_DIGITS = 40, 8192
KNOB_CTAS_PER_SM, KNOB_BIGHIST, KNOB_MINIMAP, KNOB_SMALL, KNOB_MAPMEDIAN, KNOB_RENDER = 0, 1, 2, 3, 4, 5
KIND_NAMES = ["moments", "moments_coarse", "histogram", "select_pass0", "select_pass1", "select_pass2",
              "select_cand", "select_scan", "hist_select", "probe_read", "other", "moments_window", "minimap", "torben_pass",
              "render", "stats_small"]


class CubeError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__("libcube: %s (code %d)" % (msg, code))
        self.code = code


class MomentsT(ctypes.Structure):
    _fields_ = [("count", ctypes.c_uint64), ("nan_count", ctypes.c_uint64),
                ("min", ctypes.c_float), ("max", ctypes.c_float),
                ("mean", ctypes.c_double), ("std", ctypes.c_double)]

    def as_dict(self):
        return dict(count=int(self.count), nan_count=int(self.nan_count), min=np.float32(self.min),
                    max=np.float32(self.max), mean=float(self.mean), std=float(self.std))


class ShardBuffersT(ctypes.Structure):
    _fields_ = [("record", ctypes.c_void_p), ("bins", ctypes.c_void_p), ("outside", ctypes.c_void_p),
                ("digits", ctypes.c_void_p)]


class ViewT(ctypes.Structure):
    """cube_view_t (include/cube.h): orthographic rays in data coordinates."""
    _fields_ = [("origin", ctypes.c_float * 3), ("du", ctypes.c_float * 3), ("dv", ctypes.c_float * 3),
                ("step", ctypes.c_float * 3), ("width", ctypes.c_int32), ("height", ctypes.c_int32),
                ("nsteps", ctypes.c_int32)]

    @classmethod
    def from_dict(cls, v):
        """dict(origin, du, dv, step (3 floats each), width, height, nsteps) -> ViewT (marshalling only)."""
        if isinstance(v, cls):
            return v
        w = cls()
        for name in ("origin", "du", "dv", "step"):
            for c in range(3):
                getattr(w, name)[c] = float(v[name][c])
        w.width, w.height, w.nsteps = int(v["width"]), int(v["height"]), int(v["nsteps"])
        return w

    def as_dict(self):
        d = {k: np.array(list(getattr(self, k)), dtype=np.float32) for k in ("origin", "du", "dv", "step")}
        d.update(width=int(self.width), height=int(self.height), nsteps=int(self.nsteps))
        return d


# record layout of cube_moments_t as a numpy dtype (mini-map cells)
MINIMAP_DTYPE = np.dtype([("count", "<u8"), ("nan_count", "<u8"), ("min", "<f4"), ("max", "<f4"), ("mean", "<f8"),
                          ("std", "<f8")])

_lib = None


def load():
    """dlopen libcube.so (built by ``python -m paper_1211_4896_b200.build``).  Fails loudly."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(_LIBPATH):
        raise ImportError("libcube.so not built: run `python -m paper_1211_4896_b200.build` "
                          "(there is no CPU fallback)")
    L = ctypes.CDLL(_LIBPATH)
    vp, i64, u64, ci, cu, f32, sz = (ctypes.c_void_p, ctypes.c_int64, ctypes.c_uint64, ctypes.c_int,
                                     ctypes.c_uint, ctypes.c_float, ctypes.c_size_t)
    L.cube_create.argtypes = [ctypes.POINTER(vp), sz]
    L.cube_destroy.argtypes = [vp]
    L.cube_moments.argtypes = [vp, vp, i64, i64, i64, cu, vp, vp]
    L.cube_histogram.argtypes = [vp, vp, i64, i64, i64, ci, f32, f32, vp, vp, vp]
    L.cube_histogram_noalloc.argtypes = [vp, i64, i64, i64, ci, f32, f32, vp, vp, vp, ctypes.POINTER(ci)]
    L.cube_kth.argtypes = [vp, vp, i64, i64, i64, u64, vp, vp]
    L.cube_kth_ex.argtypes = [vp, vp, i64, i64, i64, u64, cu, vp, vp]
    L.cube_kth_multi.argtypes = [vp, vp, i64, i64, i64, ci, vp, cu, vp, vp]
    L.cube_median.argtypes = [vp, vp, i64, i64, i64, vp, vp]
    L.cube_median_ex.argtypes = [vp, vp, i64, i64, i64, cu, vp, vp]
    L.cube_stats.argtypes = [vp, vp, i64, i64, i64, ci, f32, f32, cu, vp, vp, vp, vp, vp]
    L.cube_probe_read.argtypes = [vp, vp, u64, vp]
    L.cube_ooc_begin.argtypes = [vp, ci, f32, f32, ci, vp]
    L.cube_ooc_begin_ex.argtypes = [vp, ci, f32, f32, ci, cu, vp]
    L.cube_ooc_brick.argtypes = [vp, vp, u64, vp]
    L.cube_ooc_next_sweep.argtypes = [vp, ctypes.POINTER(ci), vp]
    L.cube_ooc_result.argtypes = [vp, cu, vp, vp, vp, vp, vp]
    L.cube_host_workspace.argtypes = [vp, sz, sz]
    L.cube_stats_host.argtypes = [vp, vp, i64, i64, i64, ci, f32, f32, cu, vp, vp, vp, vp]
    L.cube_stream_workspace.argtypes = [vp, sz, ci, sz]
    L.cube_stats_stream.argtypes = [vp, u64, u64, u64, FILL_FN, vp, ci, f32, f32, cu, vp, vp, vp, vp]
    L.cube_stream_info.argtypes = [vp, ctypes.POINTER(u64), ctypes.POINTER(ci)]
    L.cube_strerror.argtypes = [ci]
    L.cube_strerror.restype = ctypes.c_char_p
    L.cube_last_cuda_error.argtypes = [vp]
    L.cube_set_launch.argtypes = [vp, ci]
    L.cube_set_knob.argtypes = [vp, ci, ci]
    L.cube_launch_count.argtypes = [vp]
    L.cube_launch_count.restype = u64
    L.cube_profile_enable.argtypes = [vp, ci]
    L.cube_profile_reset.argtypes = [vp]
    L.cube_profile_read.argtypes = [vp, ci, ctypes.POINTER(ctypes.c_double), ctypes.POINTER(u64)]
    f64 = ctypes.c_double
    L.cube_mad.argtypes = [vp, vp, i64, i64, i64, cu, vp, vp, vp]
    L.cube_clipped_moments.argtypes = [vp, vp, i64, i64, i64, f32, f32, cu, vp, vp]
    L.cube_sigma_clip.argtypes = [vp, vp, i64, i64, i64, f64, ci, cu, vp, vp, vp, vp]
    L.cube_minimap_dims.argtypes = [i64] * 6 + [ctypes.POINTER(i64)] * 3
    L.cube_minimap.argtypes = [vp, vp, i64, i64, i64, i64, i64, i64, cu, vp, vp]
    L.cube_minimap_median.argtypes = [vp, vp, i64, i64, i64, i64, i64, i64, vp, vp]
    L.cube_median_torben.argtypes = [vp, vp, i64, i64, i64, ci, vp, vp, vp, vp]
    vwp = ctypes.POINTER(ViewT)
    L.cube_view_orbit.argtypes = [i64, i64, i64, f64, f64, ci, ci, f64, vwp]
    L.cube_render_mip.argtypes = [vp, vp, i64, i64, i64, vwp, f32, vp, vp]
    L.cube_render_tf.argtypes = [vp, vp, i64, i64, i64, vwp, ci, f32, f32, vp, f32, vp, vp]
    L.cube_render_sigma.argtypes = [vp, vp, i64, i64, i64, vwp, vp, i64, i64, i64, ci, f32, f32, vp, f32, vp, vp]
    L.cube_spectrum.argtypes = [vp, vp, i64, i64, i64, vwp, ci, ci, vp, vp]
    L.cube_shard_buffers.argtypes = [vp, ctypes.POINTER(ShardBuffersT)]
    L.cube_shard_merge_records.argtypes = [vp, vp, ci, cu, vp]
    L.cube_shard_advance.argtypes = [vp, ctypes.POINTER(ci), vp]
    for name in SYMBOLS:
        getattr(L, name)
    _lib = L
    return L


def _ptr(p):
    """Device/host address as c_void_p.  Accepts int, ctypes pointers, numpy arrays, or anything with
    ``data_ptr()`` (torch tensors)."""
    if p is None:
        return ctypes.c_void_p(None)
    if hasattr(p, "data_ptr"):
        return ctypes.c_void_p(p.data_ptr())
    if isinstance(p, np.ndarray):
        return ctypes.c_void_p(p.ctypes.data)
    if isinstance(p, int):
        return ctypes.c_void_p(p)
    return ctypes.cast(p, ctypes.c_void_p)


def histogram_noalloc(d, nx, ny, nz, nbins, lo, hi, bins=None, outside=None, stream=0):
    """cube_histogram_noalloc: cube_histogram without a context and without any allocation on the device (the global
    counters are a static array of the library; nbins <= NOALLOC_MAX_BINS, else CubeError(ERANGE)).  Calls share that
    array: keep them on one stream.  ``bins`` / ``outside``: device or pinned buffers, else numpy arrays are returned."""
    L = load()
    err = ctypes.c_int(0)
    ret = None
    if bins is None:
        bins = np.zeros(max(int(nbins), 1), dtype=np.uint64)
        outside = np.zeros(2, dtype=np.uint64)
        ret = (bins, outside)
    rc = L.cube_histogram_noalloc(_ptr(d), nx, ny, nz, nbins, lo, hi, _ptr(bins), _ptr(outside), stream,
                                  ctypes.byref(err))
    if rc != OK:
        msg = L.cube_strerror(rc).decode()
        if rc == ECUDA:
            msg += " cudaError=%d" % err.value
        raise CubeError(rc, msg)
    return ret


class Context:
    """Owns one ``cube_ctx`` on the current CUDA device.  Methods with ``out=None`` return host values
    (and therefore synchronise, because results are copied to pageable host memory); pass device or
    pinned buffers (``out=`` / ``bins=``) for fully asynchronous use."""

    def __init__(self, scratch_bytes_hint=0):
        self._L = load()
        h = ctypes.c_void_p()
        rc = self._L.cube_create(ctypes.byref(h), scratch_bytes_hint)
        if rc != OK:
            raise CubeError(rc, "cube_create failed (%s) -- a CUDA device is required, there is no CPU "
                                "fallback" % self._L.cube_strerror(rc).decode())
        self._h = h

    def close(self):
        if getattr(self, "_h", None):
            self._L.cube_destroy(self._h)
            self._h = None

    __del__ = close

    def _check(self, rc):
        if rc != OK:
            msg = self._L.cube_strerror(rc).decode()
            if rc == ECUDA:
                msg += " cudaError=%d" % self._L.cube_last_cuda_error(self._h)
            raise CubeError(rc, msg)

    # --- in-core operations (d: device pointer) ---------------------------------------------------
    def moments(self, d, nx, ny, nz, flags=0, out=None, stream=0):
        if out is not None:
            self._check(self._L.cube_moments(self._h, _ptr(d), nx, ny, nz, flags, _ptr(out), stream))
            return None
        m = MomentsT()
        self._check(self._L.cube_moments(self._h, _ptr(d), nx, ny, nz, flags,
                                         ctypes.cast(ctypes.byref(m), ctypes.c_void_p), stream))
        return m.as_dict()

    def histogram(self, d, nx, ny, nz, nbins, lo, hi, bins=None, outside=None, stream=0):
        if bins is not None:
            self._check(self._L.cube_histogram(self._h, _ptr(d), nx, ny, nz, nbins, lo, hi,
                                               _ptr(bins), _ptr(outside), stream))
            return None
        b = np.zeros(max(int(nbins), 1), dtype=np.uint64)
        o = np.zeros(2, dtype=np.uint64)
        self._check(self._L.cube_histogram(self._h, _ptr(d), nx, ny, nz, nbins, lo, hi, _ptr(b), _ptr(o), stream))
        return b, o

    def kth(self, d, nx, ny, nz, k, flags=0, out=None, stream=0):
        if out is not None:
            self._check(self._L.cube_kth_ex(self._h, _ptr(d), nx, ny, nz, k, flags, _ptr(out), stream))
            return None
        r = ctypes.c_float()
        self._check(self._L.cube_kth_ex(self._h, _ptr(d), nx, ny, nz, k, flags,
                                        ctypes.cast(ctypes.byref(r), ctypes.c_void_p), stream))
        return np.float32(r.value)

    def kth_multi(self, d, nx, ny, nz, ks, flags=0, out=None, stream=0):
        """cube_kth_multi: the elements of ranks ``ks`` in 1 + ceil(len(ks)/4) reads of the cube (one less with
        REUSE_COARSE; one more per rank of a group whose buckets do not fit the candidate buffer).
        ``out``: device / pinned buffer of len(ks) floats, else the values come back as a float32 array."""
        karr = np.ascontiguousarray(ks, dtype=np.uint64)
        if out is not None:
            self._check(self._L.cube_kth_multi(self._h, _ptr(d), nx, ny, nz, karr.size, karr.ctypes.data, flags,
                                               _ptr(out), stream))
            return None
        r = np.full(karr.size, np.nan, dtype=np.float32)
        self._check(self._L.cube_kth_multi(self._h, _ptr(d), nx, ny, nz, karr.size, karr.ctypes.data, flags,
                                           r.ctypes.data, stream))
        return r

    def median(self, d, nx, ny, nz, flags=0, out=None, stream=0):
        if out is not None:
            self._check(self._L.cube_median_ex(self._h, _ptr(d), nx, ny, nz, flags, _ptr(out), stream))
            return None
        r = ctypes.c_float()
        self._check(self._L.cube_median_ex(self._h, _ptr(d), nx, ny, nz, flags,
                                           ctypes.cast(ctypes.byref(r), ctypes.c_void_p), stream))
        return np.float32(r.value)

    def stats(self, d, nx, ny, nz, nbins=0, lo=None, hi=None, flags=0, want_median=True,
              out=None, bins=None, outside=None, median=None, stream=0):
        """cube_stats: moments + histogram + exact lower median in two reads of the cube.
        lo=None -> histogram over [min,max] (CUBE_RANGE_MINMAX); nbins=0 -> no histogram.
        With no output buffers given returns (moments dict, bins, outside, median) on the host."""
        if nbins and lo is None:
            flags |= RANGE_MINMAX
            lo = hi = 0.0
        if out is not None or bins is not None or median is not None:
            self._check(self._L.cube_stats(self._h, _ptr(d), nx, ny, nz, nbins, lo or 0.0, hi or 0.0, flags,
                                           _ptr(out), _ptr(bins), _ptr(outside), _ptr(median), stream))
            return None
        m = MomentsT()
        b = np.zeros(max(int(nbins), 1), dtype=np.uint64)
        o = np.zeros(2, dtype=np.uint64)
        r = ctypes.c_float(float("nan"))
        self._check(self._L.cube_stats(self._h, _ptr(d), nx, ny, nz, nbins, lo or 0.0, hi or 0.0, flags,
                                       ctypes.cast(ctypes.byref(m), ctypes.c_void_p),
                                       _ptr(b) if nbins else None, _ptr(o) if nbins else None,
                                       ctypes.cast(ctypes.byref(r), ctypes.c_void_p) if want_median else None,
                                       stream))
        return m.as_dict(), (b if nbins else None), (o if nbins else None), (np.float32(r.value) if want_median else None)

    # --- NEXT-1 / NEXT-2 ------------------------------------------------------------
    def mad(self, d, nx, ny, nz, flags=0, median_out=None, mad_out=None, stream=0):
        """cube_mad -> (median, MAD) on the host, or None when device/pinned outputs are given."""
        if mad_out is not None:
            self._check(self._L.cube_mad(self._h, _ptr(d), nx, ny, nz, flags, _ptr(median_out), _ptr(mad_out), stream))
            return None
        m, r = ctypes.c_float(), ctypes.c_float()
        self._check(self._L.cube_mad(self._h, _ptr(d), nx, ny, nz, flags, ctypes.cast(ctypes.byref(m), ctypes.c_void_p),
                                     ctypes.cast(ctypes.byref(r), ctypes.c_void_p), stream))
        return np.float32(m.value), np.float32(r.value)

    def clipped_moments(self, d, nx, ny, nz, lo, hi, flags=0, out=None, stream=0):
        if out is not None:
            self._check(self._L.cube_clipped_moments(self._h, _ptr(d), nx, ny, nz, lo, hi, flags, _ptr(out), stream))
            return None
        m = MomentsT()
        self._check(self._L.cube_clipped_moments(self._h, _ptr(d), nx, ny, nz, lo, hi, flags,
                                                 ctypes.cast(ctypes.byref(m), ctypes.c_void_p), stream))
        return m.as_dict()

    def sigma_clip(self, d, nx, ny, nz, kappa, max_iter, flags=0, out=None, iters=None, window=None, stream=0):
        """cube_sigma_clip -> (moments dict, clipped passes made, (lo, hi) of the last window) on the host, or
        None when device/pinned outputs are given."""
        if out is not None:
            self._check(self._L.cube_sigma_clip(self._h, _ptr(d), nx, ny, nz, kappa, max_iter, flags, _ptr(out),
                                                _ptr(iters), _ptr(window), stream))
            return None
        m, it, w = MomentsT(), ctypes.c_int(), (ctypes.c_float * 2)()
        self._check(self._L.cube_sigma_clip(self._h, _ptr(d), nx, ny, nz, kappa, max_iter, flags,
                                            ctypes.cast(ctypes.byref(m), ctypes.c_void_p),
                                            ctypes.cast(ctypes.byref(it), ctypes.c_void_p),
                                            ctypes.cast(w, ctypes.c_void_p), stream))
        return m.as_dict(), int(it.value), (np.float32(w[0]), np.float32(w[1]))

    def median_torben(self, d, nx, ny, nz, max_iter=64, out=None, iters=None, converged=None, stream=0):
        """cube_median_torben (Alg. 1 of the paper) -> (value, passes made, converged) on the host, or None when
        device/pinned outputs are given."""
        if out is not None:
            self._check(self._L.cube_median_torben(self._h, _ptr(d), nx, ny, nz, max_iter, _ptr(out), _ptr(iters),
                                                   _ptr(converged), stream))
            return None
        r, it, cv = ctypes.c_float(), ctypes.c_int(), ctypes.c_int()
        self._check(self._L.cube_median_torben(self._h, _ptr(d), nx, ny, nz, max_iter,
                                               ctypes.cast(ctypes.byref(r), ctypes.c_void_p),
                                               ctypes.cast(ctypes.byref(it), ctypes.c_void_p),
                                               ctypes.cast(ctypes.byref(cv), ctypes.c_void_p), stream))
        return np.float32(r.value), int(it.value), bool(cv.value)

    def minimap_dims(self, nx, ny, nz, px, py, pz):
        mx, my, mz = ctypes.c_int64(), ctypes.c_int64(), ctypes.c_int64()
        self._check(self._L.cube_minimap_dims(nx, ny, nz, px, py, pz, ctypes.byref(mx), ctypes.byref(my),
                                              ctypes.byref(mz)))
        return int(mx.value), int(my.value), int(mz.value)

    def minimap(self, d, nx, ny, nz, px, py, pz, cells, flags=0, stream=0):
        """cube_minimap: ``cells`` = device (or pinned) buffer of mx*my*mz records of 40 bytes (MINIMAP_DTYPE)."""
        self._check(self._L.cube_minimap(self._h, _ptr(d), nx, ny, nz, px, py, pz, flags, _ptr(cells), stream))

    # --- NEXT-4: ray casting into headless buffers --------
    def view_orbit(self, nx, ny, nz, yaw_deg, pitch_deg, width, height, step=1.0):
        """cube_view_orbit -> ViewT (host-side geometry, no device work)."""
        w = ViewT()
        self._check(self._L.cube_view_orbit(nx, ny, nz, yaw_deg, pitch_deg, width, height, step, ctypes.byref(w)))
        return w

    def render_mip(self, d, nx, ny, nz, view, image, vmin=float("-inf"), stream=0):
        """cube_render_mip: ``image`` = device (or pinned) buffer of width * height floats."""
        w = ViewT.from_dict(view)
        self._check(self._L.cube_render_mip(self._h, _ptr(d), nx, ny, nz, ctypes.byref(w), vmin, _ptr(image), stream))

    def render_tf(self, d, nx, ny, nz, view, table, lo, hi, rgba, opacity_cut=2.0, stream=0):
        """cube_render_tf: ``table`` = [nlevels, 4] float32 (numpy array or device tensor); ``rgba`` = device (or
        pinned) buffer of width * height * 4 floats."""
        w = ViewT.from_dict(view)
        if isinstance(table, np.ndarray):
            table = np.ascontiguousarray(table, dtype=np.float32)
            nlevels = table.size // 4
        else:
            nlevels = table.numel() // 4
        self._check(self._L.cube_render_tf(self._h, _ptr(d), nx, ny, nz, ctypes.byref(w), nlevels, lo, hi, _ptr(table),
                                           opacity_cut, _ptr(rgba), stream))

    def render_sigma(self, d, nx, ny, nz, view, cells, px, py, pz, table, zlo, zhi, rgba, opacity_cut=2.0, stream=0):
        """cube_render_sigma: ``cells`` = the device (or pinned) buffer cube_minimap filled for partitions px, py, pz;
        levels of (sample - local mean) / local std over [zlo, zhi]; the rest as render_tf."""
        w = ViewT.from_dict(view)
        if isinstance(table, np.ndarray):
            table = np.ascontiguousarray(table, dtype=np.float32)
            nlevels = table.size // 4
        else:
            nlevels = table.numel() // 4
        self._check(self._L.cube_render_sigma(self._h, _ptr(d), nx, ny, nz, ctypes.byref(w), _ptr(cells), px, py, pz,
                                              nlevels, zlo, zhi, _ptr(table), opacity_cut, _ptr(rgba), stream))

    def spectrum(self, d, nx, ny, nz, view, u, v, out, stream=0):
        """cube_spectrum: ``out`` = device (or pinned) buffer of nsteps floats."""
        w = ViewT.from_dict(view)
        self._check(self._L.cube_spectrum(self._h, _ptr(d), nx, ny, nz, ctypes.byref(w), u, v, _ptr(out), stream))

    def minimap_median(self, d, nx, ny, nz, px, py, pz, med, stream=0):
        """cube_minimap_median: ``med`` = device (or pinned) buffer of mx*my*mz floats."""
        self._check(self._L.cube_minimap_median(self._h, _ptr(d), nx, ny, nz, px, py, pz, _ptr(med), stream))

    def probe_read(self, d, nvox, stream=0):
        self._check(self._L.cube_probe_read(self._h, _ptr(d), nvox, stream))

    # --- brick-streamed (out-of-core) ------------------------------------------------------------------
    def ooc_begin(self, nbins, lo, hi, want_median=True, stream=0, flags=0):
        self._check(self._L.cube_ooc_begin_ex(self._h, nbins, lo, hi, int(bool(want_median)), flags, stream))

    def ooc_brick(self, d_brick, nvox, stream=0):
        self._check(self._L.cube_ooc_brick(self._h, _ptr(d_brick), nvox, stream))

    def ooc_next_sweep(self, stream=0):
        more = ctypes.c_int()
        self._check(self._L.cube_ooc_next_sweep(self._h, ctypes.byref(more), stream))
        return bool(more.value)

    def ooc_result(self, nbins, flags=0, want_median=True, stream=0):
        m = MomentsT()
        b = np.zeros(max(int(nbins), 1), dtype=np.uint64)
        o = np.zeros(2, dtype=np.uint64)
        r = ctypes.c_float(float("nan"))
        self._check(self._L.cube_ooc_result(self._h, flags, ctypes.cast(ctypes.byref(m), ctypes.c_void_p),
                                            _ptr(b) if nbins else None, _ptr(o) if nbins else None,
                                            ctypes.cast(ctypes.byref(r), ctypes.c_void_p) if want_median else None,
                                            stream))
        return m.as_dict(), b, o, np.float32(r.value)

    # --- z-slab sharding over GPUs (NEXT-3; the collectives live in shard.py) ----------------------------
    def shard_buffers(self):
        """-> dict(record, bins, outside, digits) of device addresses (int)."""
        b = ShardBuffersT()
        self._check(self._L.cube_shard_buffers(self._h, ctypes.byref(b)))
        return dict(record=int(b.record), bins=int(b.bins), outside=int(b.outside), digits=int(b.digits))

    def shard_merge_records(self, gathered, world, flags=0, stream=0):
        self._check(self._L.cube_shard_merge_records(self._h, _ptr(gathered), world, flags, stream))

    def shard_advance(self, stream=0):
        more = ctypes.c_int()
        self._check(self._L.cube_shard_advance(self._h, ctypes.byref(more), stream))
        return bool(more.value)

    # --- whole cube in HOST memory ---------------------------------------------------------------------
    def host_workspace(self, resident_bytes=0, chunk_bytes=0):
        self._check(self._L.cube_host_workspace(self._h, resident_bytes, chunk_bytes))

    def stats_host(self, h_cube, nx, ny, nz, nbins, lo, hi, flags=0, want_median=True):
        m = MomentsT()
        b = np.zeros(max(int(nbins), 1), dtype=np.uint64)
        o = np.zeros(2, dtype=np.uint64)
        r = ctypes.c_float(float("nan"))
        self._check(self._L.cube_stats_host(self._h, _ptr(h_cube), nx, ny, nz, nbins, lo, hi, flags,
                                            ctypes.cast(ctypes.byref(m), ctypes.c_void_p), _ptr(b), _ptr(o),
                                            ctypes.cast(ctypes.byref(r), ctypes.c_void_p) if want_median else None))
        return m.as_dict(), b, o, np.float32(r.value)

    # --- cube produced brick by brick by a callback (config 5) -------------------------------------------
    def stream_workspace(self, brick_bytes, host_slots=3, resident_bytes=0):
        self._check(self._L.cube_stream_workspace(self._h, brick_bytes, host_slots, resident_bytes))

    def stats_stream(self, nbricks, brick_vox, total_vox, fill, nbins, lo, hi, flags=0, want_median=True):
        """``fill(brick, sweep, h_dst, nvox, fill_stream)``: put the brick's voxels into the pinned host buffer at
        address ``h_dst`` (now, or by work enqueued on the raw stream ``fill_stream``); return None/0, non-zero aborts.
        -> (moments dict, bins, outside, median, info dict(h2d_bytes, sweeps))."""
        err = []

        def _cb(user, brick, sweep, h_dst, nvox, fs):
            try:
                return int(fill(int(brick), int(sweep), int(h_dst), int(nvox), int(fs or 0)) or 0)
            except BaseException as e:      # never unwind through the C frames
                err.append(e)
                return 1
        cb = FILL_FN(_cb)
        m = MomentsT()
        b = np.zeros(max(int(nbins), 1), dtype=np.uint64)
        o = np.zeros(2, dtype=np.uint64)
        r = ctypes.c_float(float("nan"))
        rc = self._L.cube_stats_stream(self._h, nbricks, brick_vox, total_vox, cb, None, nbins, lo, hi, flags,
                                       ctypes.cast(ctypes.byref(m), ctypes.c_void_p),
                                       _ptr(b) if nbins else None, _ptr(o) if nbins else None,
                                       ctypes.cast(ctypes.byref(r), ctypes.c_void_p) if want_median else None)
        if err:
            raise err[0]
        self._check(rc)
        hb, sw = ctypes.c_uint64(), ctypes.c_int()
        self._check(self._L.cube_stream_info(self._h, ctypes.byref(hb), ctypes.byref(sw)))
        return m.as_dict(), b, o, np.float32(r.value), dict(h2d_bytes=int(hb.value), sweeps=int(sw.value))

    # --- knobs -----------------------------------------------------------------------------------------
    def set_launch(self, ctas_per_sm):
        self._check(self._L.cube_set_launch(self._h, ctas_per_sm))

    def set_knob(self, knob, value):
        self._check(self._L.cube_set_knob(self._h, knob, value))

    def profile(self, on):
        self._check(self._L.cube_profile_enable(self._h, int(bool(on))))

    def profile_reset(self):
        self._check(self._L.cube_profile_reset(self._h))

    def profile_read(self):
        """-> {kind name: (total_ms, launches)} since the last reset (synchronises the device)."""
        out = {}
        for k, name in enumerate(KIND_NAMES):
            ms, n = ctypes.c_double(), ctypes.c_uint64()
            self._check(self._L.cube_profile_read(self._h, k, ctypes.byref(ms), ctypes.byref(n)))
            out[name] = (ms.value, int(n.value))
        return out

    @property
    def launch_count(self):
        return int(self._L.cube_launch_count(self._h))
