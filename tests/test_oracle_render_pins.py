"""Pins for the ray-casting oracle (oracle_trilinear / _spectrum / _render_mip /
_render_tf and the per-cell mini-map median) against things that are NOT the oracle: closed forms, numpy brute force
along axis-aligned rays, analytically known projections, exact dyadic opacity sums.  CPU only."""
import math

import numpy as np
import pytest

import cubegen
import oracle


def ramp_cube(dims, coef, off):
    nx, ny, nz = dims
    z, y, x = np.meshgrid(np.arange(nz), np.arange(ny), np.arange(nx), indexing="ij")
    return (coef[0] * x + coef[1] * y + coef[2] * z + off).astype(np.float32)


def test_trilinear_reproduces_a_linear_ramp_exactly():
    # f = 2x + 4y + 8z + 1 with coordinates on a 1/8 grid: every difference, product and sum is a small dyadic
    # number, so the interpolation is exact and must equal f(p) -- a dropped term, a swapped axis or a wrong
    # neighbour changes the value
    dims = (9, 7, 5)
    a = ramp_cube(dims, (2.0, 4.0, 8.0), 1.0)
    r = np.random.default_rng(1)
    for _ in range(300):
        p = np.array([r.integers(0, 8 * (dims[c] - 1) + 1) / 8.0 for c in range(3)], dtype=np.float32)
        got = oracle.trilinear(a, dims, p)
        assert got is not None and float(got) == 2.0 * p[0] + 4.0 * p[1] + 8.0 * p[2] + 1.0
    # anisotropic check of the axis order: f = x only, y only, z only
    for c in range(3):
        coef = [0.0, 0.0, 0.0]
        coef[c] = 1.0
        b = ramp_cube(dims, coef, 0.0)
        p = np.array([1.25, 2.5, 3.75], dtype=np.float32)
        assert float(oracle.trilinear(b, dims, p)) == float(p[c])


def test_trilinear_domain_voxel_centres_and_null():
    dims = (4, 3, 2)
    r = np.random.default_rng(2)
    a = r.standard_normal(24).astype(np.float32)
    for z in range(2):
        for y in range(3):
            for x in range(4):                                   # at a voxel centre the sample IS the voxel (weights 0)
                assert float(oracle.trilinear(a, dims, (x, y, z))) == float(a[(z * 3 + y) * 4 + x])
    for p in ((-0.001, 0, 0), (3.001, 0, 0), (0, 2.5, 0), (0, 0, 1.0001), (0, -1, 0), (np.nan, 0, 0)):
        assert oracle.trilinear(a, dims, p) is None              # closed domain [0, n-1]^3
    assert oracle.trilinear(a, dims, (3.0, 2.0, 1.0)) is not None
    # midpoint of a cell = mean of its 8 corners (exact here: small integers)
    b = np.arange(8, dtype=np.float32)
    assert float(oracle.trilinear(b, (2, 2, 2), (0.5, 0.5, 0.5))) == 3.5
    # a NULL voxel among the eight makes the sample NULL; far from it nothing changes
    c = a.copy()
    c[0] = np.nan
    assert math.isnan(float(oracle.trilinear(c, dims, (0.5, 0.5, 0.5))))
    assert float(oracle.trilinear(c, dims, (2.5, 1.5, 0.5))) == float(oracle.trilinear(a, dims, (2.5, 1.5, 0.5)))
    # one voxel thick along an axis: the clamped neighbour is the voxel itself
    d1 = np.array([5.0, 7.0], dtype=np.float32)
    assert float(oracle.trilinear(d1, (2, 1, 1), (0.5, 0.0, 0.0))) == 6.0


@pytest.mark.parametrize("axis", [0, 1, 2])
def test_axis_aligned_mip_and_spectrum_are_numpy_slices(axis):
    dims = (13, 11, 9)
    r = np.random.default_rng(10 + axis)
    a = r.standard_normal(dims[0] * dims[1] * dims[2]).astype(np.float32)
    a[r.integers(0, a.size, 40)] = np.nan
    vol = a.reshape(dims[2], dims[1], dims[0])                   # [z, y, x]
    view = cubegen.view_axis(dims, axis)
    img = oracle.render_mip(a, dims, view)
    np_axis = 2 - axis
    with np.errstate(all="ignore"):
        ref = np.nanmax(vol, axis=np_axis) if not np.isnan(vol).all(axis=np_axis).any() else None
    assert ref is not None
    # image[v, u]: u runs over the first remaining axis (x, y, z order), v over the second
    other = [c for c in (0, 1, 2) if c != axis]
    ref_t = ref if (2 - other[1]) < (2 - other[0]) else ref.T
    assert img.shape == (dims[other[1]], dims[other[0]])
    assert np.array_equal(img, ref_t.astype(np.float32))
    # the profile of one pixel is the voxel column
    u, v = 3, 2
    idx = [0, 0, 0]
    idx[other[0]], idx[other[1]] = u, v
    sl = [slice(None)] * 3
    sl[2 - other[0]], sl[2 - other[1]] = u, v
    col = vol[tuple(sl)]
    prof = oracle.spectrum(a, dims, view, u, v)
    assert prof.shape == (dims[axis],) and np.array_equal(prof, col, equal_nan=True)
    # threshold: samples below vmin do not count; a pixel with none is NaN
    thr = oracle.render_mip(a, dims, view, vmin=1.0)
    assert np.array_equal(np.isnan(thr), ~(ref_t >= 1.0)) and np.array_equal(thr[~np.isnan(thr)], ref_t[ref_t >= 1.0])


def test_half_step_profile_of_a_ramp_and_outside_samples():
    dims = (8, 4, 4)
    a = ramp_cube(dims, (1.0, 0.0, 0.0), 0.0)
    view = cubegen.view_axis(dims, 0, step=0.5)
    prof = oracle.spectrum(a, dims, view, 1, 2)
    assert np.array_equal(prof, np.arange(15, dtype=np.float32) * 0.5)
    # a ray that starts before the cube and runs past it: NaN outside, the ramp inside
    view = dict(view, origin=np.array([-2.0, 0, 0], dtype=np.float32), nsteps=30)
    prof = oracle.spectrum(a, dims, view, 1, 2)
    xs = -2.0 + 0.5 * np.arange(30)
    inside = (xs >= 0) & (xs <= 7)
    assert np.array_equal(np.isnan(prof), ~inside) and np.array_equal(prof[inside], xs[inside].astype(np.float32))


def test_rotated_mip_of_a_single_bright_voxel_lands_on_its_projection():
    dims = (21, 17, 13)
    a = np.zeros(dims[0] * dims[1] * dims[2], dtype=np.float32)
    pos = np.array([14, 5, 9])
    a[(pos[2] * dims[1] + pos[1]) * dims[0] + pos[0]] = 100.0
    for yaw, pitch in ((0, 0), (30, 0), (0, 40), (57, -23), (180, 10), (270, 80)):
        view = cubegen.view_orbit(dims, yaw, pitch, 96, 96, step=0.25)
        img = oracle.render_mip(a, dims, view)
        v, u = np.unravel_index(np.nanargmax(img), img.shape)
        # analytic projection: solve origin + u du + v dv + t step = pos for (u, v, t) (du, dv, step are orthogonal)
        du, dv, st, o = (view[k].astype(np.float64) for k in ("du", "dv", "step", "origin"))
        rel = pos - o
        ue, ve = rel @ du / (du @ du), rel @ dv / (dv @ dv)
        assert abs(u - ue) <= 1.0 and abs(v - ve) <= 1.0, (yaw, pitch, u, v, ue, ve)
        assert 0 < np.nanmax(img) <= 100.0
        # far from the projection the ray sees only zeros (or misses the cube: NaN)
        far = (np.hypot(*(np.indices(img.shape) - np.array([ve, ue])[:, None, None])) > 8)
        assert np.all((img[far] == 0) | np.isnan(img[far]))
    # the rays of a view are parallel and the image plane is orthogonal to them
    view = cubegen.view_orbit(dims, 33, 21, 64, 48)
    assert abs(float(view["du"] @ view["step"])) < 1e-5 and abs(float(view["dv"] @ view["step"])) < 1e-5


def test_transfer_function_closed_forms():
    dims = (4, 4, 12)
    a = np.full(4 * 4 * 12, 0.5, dtype=np.float32)
    view = cubegen.view_axis(dims, 2)                             # 12 samples per ray, all equal to 0.5
    one = np.array([[0.25, 0.5, 1.0, 0.5]], dtype=np.float32)    # one level, opacity 1/2
    img = oracle.render_tf(a, dims, view, one, 0.0, 1.0)
    acc = 1.0 - 2.0 ** -12                                        # A_n = 1 - (1 - a)^n, exact in float32
    assert np.all(img[..., 3] == np.float32(acc))
    assert np.all(img[..., 0] == np.float32(0.25 * acc)) and np.all(img[..., 2] == np.float32(acc))
    # early termination: stop as soon as A >= cut -- after 3 samples A = 7/8
    img = oracle.render_tf(a, dims, view, one, 0.0, 1.0, opacity_cut=0.8)
    assert np.all(img[..., 3] == np.float32(0.875)) and np.all(img[..., 1] == np.float32(0.5 * 0.875))
    # an opaque front level hides everything behind it; level lookup = the histogram's bin formula (4 levels on [0,1])
    vol = a.reshape(12, 4, 4).copy()
    vol[0] = 0.1       # level 0
    vol[1] = 0.3       # level 1
    vol[2:] = 0.9      # level 3
    table = np.array([[1, 0, 0, 0.0], [0, 1, 0, 1.0], [0, 0, 1, 1.0], [1, 1, 1, 1.0]], dtype=np.float32)
    img = oracle.render_tf(vol.reshape(-1), dims, view, table, 0.0, 1.0)
    assert np.all(img == np.array([0, 1, 0, 1], dtype=np.float32))       # transparent level 0, then opaque green
    # seen from the other side (rays along -z): the white top level comes first
    back = dict(view, origin=np.array([0, 0, 11], dtype=np.float32), step=np.array([0, 0, -1], dtype=np.float32))
    img = oracle.render_tf(vol.reshape(-1), dims, back, table, 0.0, 1.0)
    assert np.all(img == np.array([1, 1, 1, 1], dtype=np.float32))
    # below lo and NULL samples are skipped, above hi saturates in the top level, x == hi is in the top level
    vol2 = np.full((12, 4, 4), -5.0, dtype=np.float32)
    vol2[3] = np.nan
    vol2[5] = 7.0
    vol2[6] = 1.0
    half = np.array([[1, 0, 0, 0.5], [0, 1, 0, 0.5], [0, 0, 1, 0.5], [0.5, 0.5, 0.5, 0.5]], dtype=np.float32)
    img = oracle.render_tf(vol2.reshape(-1), dims, view, half, 0.0, 1.0)
    assert np.all(img[..., 3] == np.float32(0.75)) and np.all(img[..., 0] == np.float32(0.5 * 0.75))
    # order matters: front-to-back weights 1/2, 1/4 for two different levels
    vol3 = np.full((12, 4, 4), -1.0, dtype=np.float32)
    vol3[2] = 0.1
    vol3[7] = 0.6
    img = oracle.render_tf(vol3.reshape(-1), dims, view, half, 0.0, 1.0)
    assert np.all(img[..., 0] == 0.5) and np.all(img[..., 2] == 0.25) and np.all(img[..., 3] == 0.75)
    with pytest.raises(ValueError):
        oracle.render_tf(a, dims, view, one, 1.0, 0.0)


def test_minimap_median_is_the_block_sort():
    r = np.random.default_rng(4)
    nx, ny, nz = 23, 10, 9
    a = np.round(r.standard_normal(nx * ny * nz) * 3).astype(np.float32)
    a[r.integers(0, a.size, 300)] = np.nan
    a[:5 * 4] = np.nan
    vol = a.reshape(nz, ny, nx)
    for part in ((5, 4, 3), (23, 10, 9), (1, 1, 1), (30, 30, 30), (8, 3, 2)):
        px, py, pz = part
        got = oracle.minimap_median(a, (nx, ny, nz), part)
        mx, my, mz = -(-nx // px), -(-ny // py), -(-nz // pz)
        assert got.shape == (mz, my, mx)
        for cz in range(mz):
            for cy in range(my):
                for cx in range(mx):
                    blk = vol[cz * pz:(cz + 1) * pz, cy * py:(cy + 1) * py, cx * px:(cx + 1) * px].reshape(-1)
                    ok = np.sort(blk[~np.isnan(blk)])
                    if ok.size == 0:
                        assert math.isnan(got[cz, cy, cx])
                    else:
                        assert float(got[cz, cy, cx]) == float(ok[(ok.size - 1) // 2])


def map_cells(shape, mean, std):
    """a mini-map (structured array [mz, my, mx]) with the given mean / std arrays"""
    dt = np.dtype([("count", "<u8"), ("nan_count", "<u8"), ("min", "<f4"), ("max", "<f4"), ("mean", "<f8"),
                   ("std", "<f8")])
    c = np.zeros(shape, dtype=dt)
    c["count"] = 1
    c["mean"] = mean
    c["std"] = std
    return c


def test_minimap_lookup_centres_linear_maps_and_clamping():
    # cells of 4 x 2 x 8 voxels on a 20 x 6 x 16 cube -> a 5 x 3 x 2 map; cell (cx, cy, cz) sits at data coordinate
    # (4 cx + 1.5, 2 cy + 0.5, 8 cz + 3.5)
    dims, part = (20, 6, 16), (4, 2, 8)
    mz, my, mx = 2, 3, 5
    cz, cy, cx = np.meshgrid(np.arange(mz), np.arange(my), np.arange(mx), indexing="ij")
    mean = 2.0 * cx + 8.0 * cy + 32.0 * cz + 1.0          # linear in the map index: trilinear reproduces it exactly
    std = 0.5 * cx + 0.25 * cy + 4.0 * cz + 1.0
    cells = map_cells((mz, my, mx), mean, std)
    # at the cell centres: the cell's own values
    for (z, y, x) in [(0, 0, 0), (1, 2, 4), (0, 1, 3), (1, 0, 2)]:
        p = (4 * x + 1.5, 2 * y + 0.5, 8 * z + 3.5)
        m, s = oracle.minimap_lookup(cells, dims, part, p)
        assert float(m) == mean[z, y, x] and float(s) == std[z, y, x]
    # between centres, on a dyadic grid: the linear function of q = (p - (part - 1) / 2) / part
    r = np.random.default_rng(3)
    for _ in range(200):
        q = np.array([r.integers(0, 8 * (mx - 1) + 1) / 8.0, r.integers(0, 8 * (my - 1) + 1) / 8.0,
                      r.integers(0, 8 * (mz - 1) + 1) / 8.0])
        p = q * np.array(part) + (np.array(part) - 1) / 2.0
        m, s = oracle.minimap_lookup(cells, dims, part, p)
        assert float(m) == 2.0 * q[0] + 8.0 * q[1] + 32.0 * q[2] + 1.0
        assert float(s) == 0.5 * q[0] + 0.25 * q[1] + 4.0 * q[2] + 1.0
    # outside the centres' hull the map is clamped: the cube's corner voxels see the corner cells
    m, s = oracle.minimap_lookup(cells, dims, part, (0.0, 0.0, 0.0))
    assert float(m) == mean[0, 0, 0] and float(s) == std[0, 0, 0]
    m, s = oracle.minimap_lookup(cells, dims, part, (19.0, 5.0, 15.0))
    assert float(m) == mean[1, 2, 4] and float(s) == std[1, 2, 4]
    m, s = oracle.minimap_lookup(cells, dims, part, (19.0, 0.0, 3.5))
    assert float(m) == mean[0, 0, 4]
    # an empty cell (NaN record) poisons what touches it, and only that: weight-zero neighbours do not take part
    mean2 = mean.copy()
    mean2[0, 1, 2] = np.nan
    cells2 = map_cells((mz, my, mx), mean2, std)
    m, _ = oracle.minimap_lookup(cells2, dims, part, (4 * 2 + 1.5 - 1.0, 2 * 1 + 0.5, 3.5))    # between cx = 1 and 2
    assert math.isnan(float(m))
    m, _ = oracle.minimap_lookup(cells2, dims, part, (4 * 1 + 1.5, 2 * 1 + 0.5, 3.5))          # exactly on cell cx = 1
    assert float(m) == mean[0, 1, 1]
    # a ragged map (21 voxels in cells of 4 -> 6 cells): the last centre is nominal, x = 21.5, beyond the cube
    cells3 = map_cells((1, 1, 6), np.arange(6.0).reshape(1, 1, 6), np.ones((1, 1, 6)))
    m, _ = oracle.minimap_lookup(cells3, (21, 1, 1), (4, 1, 1), (20.0, 0.0, 0.0))
    assert float(m) == (20.0 - 1.5) / 4.0


def test_sigma_clipping_transfer_function_closed_forms():
    dims, part = (4, 4, 12), (2, 2, 4)
    view = cubegen.view_axis(dims, 2)
    a = np.full(4 * 4 * 12, 3.0, dtype=np.float32)
    one = np.array([[0.25, 0.5, 1.0, 0.5]], dtype=np.float32)
    # uniform map, mean 1, std 0.5: every sample has z = (3 - 1) / 0.5 = 4 -> inside [3, 5]: A = 1 - 2^-12
    cells = map_cells((3, 2, 2), 1.0, 0.5)
    img = oracle.render_sigma(a, dims, view, cells, part, one, 3.0, 5.0)
    acc = 1.0 - 2.0 ** -12
    assert np.all(img[..., 3] == np.float32(acc)) and np.all(img[..., 0] == np.float32(0.25 * acc))
    # threshold above z: everything is clipped
    img = oracle.render_sigma(a, dims, view, cells, part, one, 4.5, 5.0)
    assert np.all(img == 0)
    # std = 0 or NaN cells: the samples are skipped
    for bad in (0.0, np.nan):
        img = oracle.render_sigma(a, dims, view, map_cells((3, 2, 2), 1.0, bad), part, one, 3.0, 5.0)
        assert np.all(img == 0)
    # the LOCAL statistics decide: mean grows along z (cells at z = 1.5, 5.5, 9.5 with mean 0, 2, 4 -> mean(z) =
    # (z - 1.5) / 2 clamped to [0, 4]), std 1, data 3: z-score = 3 - mean(z); threshold 1.5 -> the samples with
    # mean(z) <= 1.5, i.e. z <= 4.5: slices 0 .. 4 pass, five samples: A = 1 - 2^-5
    mean = np.zeros((3, 2, 2))
    mean[1] = 2.0
    mean[2] = 4.0
    img = oracle.render_sigma(a, dims, view, map_cells((3, 2, 2), mean, 1.0), part, one, 1.5, 10.0)
    assert np.all(img[..., 3] == np.float32(1.0 - 2.0 ** -5))
    # level lookup on z: 4 levels over [0, 4]; data 3, std 1, uniform mean m -> level floor(3 - m)
    table = np.array([[1, 0, 0, 1.0], [0, 1, 0, 1.0], [0, 0, 1, 1.0], [1, 1, 1, 1.0]], dtype=np.float32)
    for m, colour in [(2.5, (1, 0, 0, 1)), (1.5, (0, 1, 0, 1)), (0.5, (0, 0, 1, 1)), (-0.5, (1, 1, 1, 1)),
                      (-7.0, (1, 1, 1, 1))]:
        img = oracle.render_sigma(a, dims, view, map_cells((3, 2, 2), m, 1.0), part, table, 0.0, 4.0)
        assert np.all(img == np.array(colour, dtype=np.float32)), m
    # with mean 0 and std 1 everywhere it is oracle.render_tf on the data values (same bins, same compositing)
    r = np.random.default_rng(9)
    b = r.standard_normal(4 * 4 * 12).astype(np.float32)
    half = np.array([[1, 0, 0, 0.5], [0, 1, 0, 0.25], [0, 0, 1, 0.5], [0.5, 0.5, 0.5, 0.125]], dtype=np.float32)
    rot = cubegen.view_orbit(dims, 30.0, 20.0, 24, 24, 0.5)
    for v in (view, rot):
        assert np.array_equal(oracle.render_sigma(b, dims, v, map_cells((3, 2, 2), 0.0, 1.0), part, half, -1.0, 2.0),
                              oracle.render_tf(b, dims, v, half, -1.0, 2.0))
    with pytest.raises(ValueError):
        oracle.render_sigma(a, dims, view, cells, part, one, 1.0, 0.0)
