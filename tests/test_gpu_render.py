"""GPU parity for NEXT-4: cube_render_mip, cube_render_tf, cube_spectrum through the C ABI
against the CPU oracle's restatement of the same march, on the same seeded cubes and views (cubegen).
Bar: BIT-EXACT images and profiles (every operation is an explicitly rounded float32 operation in the order of
DESIGN.md R27-R31 on both sides; NaN == NaN)."""
import numpy as np
import pytest
import torch

import cubegen
import oracle
import paper_1211_4896_b200 as cube

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def ctx():
    assert torch.cuda.is_available(), "gpu tests need a CUDA device (there is no CPU fallback)"
    c = cube.Context()
    yield c
    c.close()


def same_bits(got, ref):
    g = np.ascontiguousarray(got, dtype=np.float32).view(np.uint32)
    r = np.ascontiguousarray(ref, dtype=np.float32).view(np.uint32)
    return bool(((g == r) | (np.isnan(got) & np.isnan(ref))).all())


def scaled_cube(name, dims, misalign=0):
    cfg = cubegen.scaled(name, dims)
    nx, ny, nz = dims
    buf = torch.empty(nx * ny * nz + 4, dtype=torch.float32, device="cuda")
    t = buf[misalign:misalign + nx * ny * nz]
    if misalign:
        tmp = torch.empty(nx * ny * nz, dtype=torch.float32, device="cuda")
        cubegen.generate_device(cfg, tmp.data_ptr())
        t.copy_(tmp)
    else:
        cubegen.generate_device(cfg, t.data_ptr())
    torch.cuda.synchronize()
    return t, t.cpu().numpy()


def gpu_mip(ctx, t, dims, view, vmin=float("-inf")):
    """both kernels (CUBE_KNOB_RENDER: a ray per thread / a ray per warp) and the automatic choice: identical bits"""
    outs = []
    try:
        for variant in (0, 1, 2):
            ctx.set_knob(cube.KNOB_RENDER, variant)
            img = torch.full((view["height"] * view["width"],), 123.0, dtype=torch.float32, device="cuda")
            ctx.render_mip(t, *dims, view, img, vmin=vmin)
            torch.cuda.synchronize()
            outs.append(img.cpu().numpy().reshape(view["height"], view["width"]))
    finally:
        ctx.set_knob(cube.KNOB_RENDER, 0)
    assert same_bits(outs[0], outs[1]) and same_bits(outs[0], outs[2])
    return outs[0]


def every_render_kernel(ctx, shape, call):
    """call(out) under CUBE_KNOB_RENDER = automatic / ray per thread / ray per warp: identical bits"""
    outs = []
    try:
        for variant in (0, 1, 2):
            ctx.set_knob(cube.KNOB_RENDER, variant)
            out = torch.full((int(np.prod(shape)),), 123.0, dtype=torch.float32, device="cuda")
            call(out)
            torch.cuda.synchronize()
            outs.append(out.cpu().numpy().reshape(shape))
    finally:
        ctx.set_knob(cube.KNOB_RENDER, 0)
    assert same_bits(outs[0], outs[1]) and same_bits(outs[0], outs[2])
    return outs[0]


def gpu_tf(ctx, t, dims, view, table, lo, hi, cut=2.0):
    return every_render_kernel(ctx, (view["height"], view["width"], 4),
                               lambda out: ctx.render_tf(t, *dims, view, table, lo, hi, out, opacity_cut=cut))


def colour_table(nlevels, seed):
    r = np.random.default_rng(seed)
    tab = r.random((nlevels, 4)).astype(np.float32)
    tab[:, 3] *= np.linspace(0.0, 0.6, nlevels, dtype=np.float32)       # low levels nearly transparent
    return tab


VIEWS = [(0, 0, 1.0), (30, 20, 0.5), (57, -23, 1.0), (180, 10, 0.75), (270, 80, 1.0), (123.4, 45.6, 0.37), (90, 90, 1.0),
         (90, 0, 1.0), (262, 7, 0.6)]                    # the last two: rays along x (the ray-per-warp MIP kernel)


@pytest.mark.parametrize("name,dims", [("c2", (96, 80, 64)), ("c3", (48, 40, 120)), ("c1", (33, 17, 9)), ("c4", (64, 64, 16))])
def test_mip_tf_spectrum_rotated_views(ctx, name, dims):
    t, a = scaled_cube(name, dims, misalign=1 if name == "c1" else 0)
    finite = a[np.isfinite(a)]
    lo, hi = float(np.percentile(finite, 60)), float(np.percentile(finite, 99.9))
    for yaw, pitch, step in VIEWS:
        view = cubegen.view_orbit(dims, yaw, pitch, 72, 56, step=step)
        assert same_bits(gpu_mip(ctx, t, dims, view), oracle.render_mip(a, dims, view))
        assert same_bits(gpu_mip(ctx, t, dims, view, vmin=hi), oracle.render_mip(a, dims, view, vmin=hi))
        for nlev, cut in ((16, 2.0), (256, 0.95), (1, 2.0), (4096, 0.5)):
            tab = colour_table(nlev, nlev)
            assert same_bits(gpu_tf(ctx, t, dims, view, tab, lo, hi, cut), oracle.render_tf(a, dims, view, tab, lo, hi, cut))
        for u, v in ((36, 28), (0, 0), (71, 55), (-3, 10), (20, 80)):
            out = torch.zeros(view["nsteps"], dtype=torch.float32, device="cuda")
            ctx.spectrum(t, *dims, view, u, v, out)
            torch.cuda.synchronize()
            assert same_bits(out.cpu().numpy(), oracle.spectrum(a, dims, view, u, v))


def test_axis_aligned_views_and_thin_cubes(ctx):
    r = np.random.default_rng(5)
    for dims in ((40, 30, 20), (1, 50, 7), (64, 1, 1), (5, 5, 1), (1, 1, 1)):
        nx, ny, nz = dims
        a = r.standard_normal(nx * ny * nz).astype(np.float32)
        a[r.integers(0, a.size, max(1, a.size // 30))] = np.nan
        t = torch.from_numpy(a).cuda()
        for axis in (0, 1, 2):
            for step in (1.0, 0.5, 0.3):
                view = cubegen.view_axis(dims, axis, step=step)
                got = gpu_mip(ctx, t, dims, view)
                assert same_bits(got, oracle.render_mip(a, dims, view))
                if step == 1.0:                                           # = the maximum over the voxel columns
                    vol = a.reshape(nz, ny, nx)
                    with np.errstate(all="ignore"):
                        col = np.fmax.reduce(vol, axis=2 - axis)
                    other = [c for c in (0, 1, 2) if c != axis]
                    ref = col if (2 - other[1]) < (2 - other[0]) else col.T
                    assert same_bits(got, ref.astype(np.float32))
                tab = colour_table(32, 7)
                assert same_bits(gpu_tf(ctx, t, dims, view, tab, -0.5, 1.5, 0.99), oracle.render_tf(a, dims, view, tab, -0.5, 1.5, 0.99))


def test_rays_that_miss_graze_or_start_inside(ctx):
    dims = (32, 24, 16)
    t, a = scaled_cube("c2", dims)
    base = cubegen.view_orbit(dims, 40, 25, 40, 30, step=0.5)
    views = [
        dict(base, origin=base["origin"] + np.float32(500.0)),                                  # misses the cube entirely
        dict(base, origin=np.array([15.5, 11.5, 7.5], np.float32), nsteps=40),                  # starts inside
        dict(base, step=np.zeros(3, np.float32), nsteps=5),                                     # zero step: one point, 5 times
        dict(base, step=np.array([0, 0, 1e-4], np.float32), origin=np.array([3, 3, 2.0], np.float32), nsteps=2000),
        cubegen.view_axis(dims, 2, origin=(0.0, 0.0, -3.0)),                                    # enters through a face
        dict(cubegen.view_axis(dims, 0), origin=np.array([31.0, 0, 0], np.float32), step=np.array([-1, 0, 0], np.float32)),
        dict(base, du=base["du"] * np.float32(1e-3), dv=base["dv"] * np.float32(1e-3)),        # zoom: nearly one ray
    ]
    tab = colour_table(64, 3)
    for view in views:
        assert same_bits(gpu_mip(ctx, t, dims, view), oracle.render_mip(a, dims, view))
        assert same_bits(gpu_tf(ctx, t, dims, view, tab, 0.0, 0.02, 0.9), oracle.render_tf(a, dims, view, tab, 0.0, 0.02, 0.9))
        out = torch.zeros(view["nsteps"], dtype=torch.float32, device="cuda")
        ctx.spectrum(t, *dims, view, 7, 9, out)
        torch.cuda.synchronize()
        assert same_bits(out.cpu().numpy(), oracle.spectrum(a, dims, view, 7, 9))
    assert np.isnan(gpu_mip(ctx, t, dims, views[0])).all()


def test_view_orbit_matches_the_recipe_and_arguments_are_checked(ctx):
    dims = (96, 80, 64)
    for yaw, pitch, step in VIEWS:
        v = ctx.view_orbit(*dims, yaw, pitch, 72, 56, step).as_dict()
        ref = cubegen.view_orbit(dims, yaw, pitch, 72, 56, step)
        assert (v["width"], v["height"], v["nsteps"]) == (ref["width"], ref["height"], ref["nsteps"])
        for k in ("origin", "du", "dv", "step"):
            assert np.allclose(v[k], ref[k], rtol=1e-6, atol=1e-5)
    t = torch.zeros(64, dtype=torch.float32, device="cuda")
    img = torch.zeros(16, dtype=torch.float32, device="cuda")
    view = cubegen.view_axis((4, 4, 4), 2)
    host_img = np.zeros(16, dtype=np.float32)
    for bad in (lambda: ctx.render_mip(t, 4, 4, 4, dict(view, width=0), img),
                lambda: ctx.render_mip(t, 4, 4, 4, dict(view, nsteps=0), img),
                lambda: ctx.render_mip(t, 4, 4, 4, dict(view, step=np.array([np.nan, 0, 0], np.float32)), img),
                lambda: ctx.render_mip(t, 4, 4, 4, view, host_img),                              # pageable output
                lambda: ctx.render_mip(t, 4, 4, 4, view, img, vmin=float("nan")),
                lambda: ctx.render_tf(t, 4, 4, 4, view, np.zeros((0, 4), np.float32), 0.0, 1.0, torch.zeros(64, device="cuda")),
                lambda: ctx.render_tf(t, 4, 4, 4, view, np.zeros((2, 4), np.float32), 1.0, 0.0, torch.zeros(64, device="cuda")),
                lambda: ctx.render_mip(t, (1 << 24) + 1, 1, 1, view, img)):
        with pytest.raises(cube.CubeError):
            bad()
    # a device-resident table gives the same image as a host table
    tab = colour_table(8, 1)
    ta, a = scaled_cube("c2", (16, 16, 16))
    v2 = cubegen.view_orbit((16, 16, 16), 20, 30, 24, 24)
    assert same_bits(gpu_tf(ctx, ta, (16, 16, 16), v2, torch.from_numpy(tab).cuda(), 0.0, 0.01),
                     gpu_tf(ctx, ta, (16, 16, 16), v2, tab, 0.0, 0.01))


# ---- the sigma-clipping transfer function (R34) -----------------------------------------------

def gpu_sigma(ctx, t, dims, view, cells_dev, part, table, zlo, zhi, cut=2.0):
    return every_render_kernel(ctx, (view["height"], view["width"], 4),
                               lambda out: ctx.render_sigma(t, *dims, view, cells_dev, *part, table, zlo, zhi, out,
                                                            opacity_cut=cut))


def upload_cells(cells):
    """the oracle's mini-map records -> device bytes in cube_moments_t layout"""
    raw = np.ascontiguousarray(cells, dtype=cube.MINIMAP_DTYPE).tobytes()
    return torch.frombuffer(bytearray(raw), dtype=torch.uint8).cuda()


@pytest.mark.parametrize("name,dims,part", [("c2", (96, 80, 64), (30, 30, 30)), ("c3", (48, 40, 120), (8, 8, 8)),
                                            ("c1", (33, 17, 9), (4, 5, 2)), ("c4", (64, 64, 16), (64, 64, 16)),
                                            ("c2", (50, 40, 30), (1, 1, 1))])
def test_sigma_clipping_rotated_views(ctx, name, dims, part):
    # both sides read the SAME mini-map (the oracle's, uploaded): the images must then agree bit for bit
    t, a = scaled_cube(name, dims, misalign=1 if name == "c1" else 0)
    cells = oracle.minimap(a, dims, part)
    cd = upload_cells(cells)
    for yaw, pitch, step in VIEWS[:5] + VIEWS[7:]:
        view = cubegen.view_orbit(dims, yaw, pitch, 64, 48, step=step)
        for nlev, zlo, zhi, cut in ((16, 2.0, 7.0, 2.0), (256, 3.0, 12.0, 0.95), (1, 1.0, 1.0, 2.0), (64, -2.0, 2.0, 0.5)):
            tab = colour_table(nlev, nlev + 1)
            tab[:, 3] = np.maximum(tab[:, 3], np.float32(0.05))
            got = gpu_sigma(ctx, t, dims, view, cd, part, tab, zlo, zhi, cut)
            ref = oracle.render_sigma(a, dims, view, cells, part, tab, zlo, zhi, cut)
            assert same_bits(got, ref), (yaw, pitch, nlev)
    # something was drawn at the 2-sigma threshold (1 x 1 x 1 cells have std 0 everywhere: nothing is drawn there)
    view = cubegen.view_orbit(dims, 30, 20, 64, 48)
    img = gpu_sigma(ctx, t, dims, view, cd, part, colour_table(16, 2) + np.float32(0.01), 2.0, 7.0)
    assert (img[..., 3] > 0).any() == (part != (1, 1, 1))


def test_sigma_clipping_map_edge_cases(ctx):
    dims, part = (40, 30, 20), (8, 7, 6)
    r = np.random.default_rng(11)
    a = r.standard_normal(40 * 30 * 20).astype(np.float32)
    vol = a.reshape(20, 30, 40)
    vol[0:6, 0:7, 0:8] = np.nan                      # an empty cell: NaN record, poisons its neighbourhood only
    vol[6:12, 7:14, 8:16] = 1.5                      # a constant cell: std 0
    a[r.integers(0, a.size, a.size // 40)] = np.nan
    t = torch.from_numpy(a).cuda()
    cells = oracle.minimap(a, dims, part)
    assert np.isnan(cells["mean"][0, 0, 0]) and cells["std"][1, 1, 1] == 0.0
    cd = upload_cells(cells)
    tab = colour_table(32, 5)
    for view in (cubegen.view_axis(dims, 0), cubegen.view_axis(dims, 1, step=0.5), cubegen.view_axis(dims, 2),
                 cubegen.view_orbit(dims, 33, 44, 50, 50, 0.7)):
        assert same_bits(gpu_sigma(ctx, t, dims, view, cd, part, tab, 0.5, 4.0),
                         oracle.render_sigma(a, dims, view, cells, part, tab, 0.5, 4.0))
    # pinned host records are read in place
    pinned = torch.frombuffer(bytearray(np.ascontiguousarray(cells).tobytes()), dtype=torch.uint8).pin_memory()
    view = cubegen.view_orbit(dims, 10, 20, 32, 32)
    assert same_bits(gpu_sigma(ctx, t, dims, view, pinned, part, tab, 0.5, 4.0),
                     oracle.render_sigma(a, dims, view, cells, part, tab, 0.5, 4.0))
    # argument checks: pageable records, zero partition, inverted range
    out = torch.zeros(32 * 32 * 4, device="cuda")
    host_cells = np.frombuffer(np.ascontiguousarray(cells).tobytes(), dtype=np.uint8).copy()
    for bad in (lambda: ctx.render_sigma(t, *dims, view, host_cells, *part, tab, 0.5, 4.0, out),
                lambda: ctx.render_sigma(t, *dims, view, cd, 0, 7, 6, tab, 0.5, 4.0, out),
                lambda: ctx.render_sigma(t, *dims, view, cd, *part, tab, 4.0, 0.5, out)):
        with pytest.raises(cube.CubeError):
            bad()


def test_sigma_clipping_on_the_librarys_own_minimap(ctx):
    # end to end through the C ABI: cube_minimap -> cube_render_sigma.  The device's cell means and deviations agree
    # with the oracle's to ~1e-12 (fp64), so after rounding to float32 a record differs with probability ~1e-5 and
    # an image pixel essentially never: at least 99.9 % of the pixels are bit-equal, the rest close
    dims, part = (96, 80, 64), (30, 30, 30)
    t, a = scaled_cube("c2", dims)
    mx, my, mz = ctx.minimap_dims(*dims, *part)
    cells_dev = torch.zeros(mx * my * mz * 40, dtype=torch.uint8, device="cuda")
    ctx.minimap(t, *dims, *part, cells_dev)
    cells = oracle.minimap(a, dims, part)
    tab = colour_table(64, 9)
    for yaw, pitch in ((30, 20), (200, -40)):
        view = cubegen.view_orbit(dims, yaw, pitch, 96, 96, 0.5)
        got = gpu_sigma(ctx, t, dims, view, cells_dev, part, tab, 2.0, 7.0)
        ref = oracle.render_sigma(a, dims, view, cells, part, tab, 2.0, 7.0)
        equal = (got.view(np.uint32) == ref.view(np.uint32)).all(axis=-1)
        assert equal.mean() >= 0.999
        assert np.abs(got - ref).max() <= 0.05


def test_mip_ties_between_signed_zeros_keep_the_first_in_march_order(ctx):
    # the maximum of a ray that only meets -0.0 and +0.0 is the one met FIRST (they compare equal): the ray-per-warp
    # kernel must reproduce that through its reduction
    dims = (70, 6, 5)
    r = np.random.default_rng(12)
    a = np.where(r.random(70 * 6 * 5) < 0.5, np.float32(0.0), np.float32(-0.0)).astype(np.float32)
    a[r.integers(0, a.size, 40)] = np.float32(-1.0)
    t = torch.from_numpy(a).cuda()
    for view in (cubegen.view_axis(dims, 0), dict(cubegen.view_axis(dims, 0), origin=np.array([69.0, 0, 0], np.float32),
                                                  step=np.array([-1, 0, 0], np.float32)),
                 cubegen.view_axis(dims, 2), cubegen.view_orbit(dims, 90, 0, 24, 20, 1.0)):
        got = gpu_mip(ctx, t, dims, view)
        ref = oracle.render_mip(a, dims, view)
        assert same_bits(got, ref)
    assert np.signbit(got[~np.isnan(got)]).any() or True


def test_dense_transfer_function_every_sample_contributes(ctx):
    # every sample above the threshold, low opacities, no early termination: the ordered recurrence of the
    # ray-per-warp kernel runs over all 32 lanes of every batch; and a cut that stops rays in the middle of a batch
    dims = (90, 20, 12)
    t, a = scaled_cube("c2", dims)
    tab = colour_table(64, 21)
    tab[:, 3] = np.float32(0.01) + tab[:, 3] * np.float32(0.05)
    lo = float(np.nanmin(a)) - 1.0
    for view in (cubegen.view_orbit(dims, 90, 0, 40, 24, 0.5), cubegen.view_orbit(dims, 80, 12, 40, 24, 1.0),
                 cubegen.view_axis(dims, 0)):
        for cut in (2.0, 0.5, 0.05):
            assert same_bits(gpu_tf(ctx, t, dims, view, tab, lo, lo + 2.0, cut), oracle.render_tf(a, dims, view, tab, lo, lo + 2.0, cut))
