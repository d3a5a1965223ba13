"""Parity: the CUDA path (through the C ABI) against the CPU oracle, element by element, on the same seeded
inputs.  Bit-exact for min/max and counts, MIP <= 1e-6 scale-relative, EA <= 1e-4 absolute per channel
(north_star); because both sides run the same canonical float32 op sequence the tests also assert bit identity.

Every test takes the backend fixture `be` (tests/backends.py): `gpu` = libvr.so on a B200 (marked gpu), `simt` =
the same .cu sources executed thread by thread on the host (runs without a GPU, reduced case matrix)."""
import numpy as np
import pytest

import oracle as O
import paper_1111_6661_b200 as vr
import workload as W
from backends import BACKENDS, be, render, statistics, summary  # noqa: F401  (be is a fixture)
from parity import FRAGILE_FRAC_OPAQUE, check_ea, check_mip


def assert_summary_equal(g, o):
    assert g["vmin"] == o.vmin and g["vmax"] == o.vmax, (g["vmin"], o.vmin, g["vmax"], o.vmax)
    assert int(g["n_nonfinite"]) == o.n_nonfinite and int(g["n_below"]) == o.n_below and int(g["n_above"]) == o.n_above
    assert np.array_equal(g["counts"], o.counts)


# ------------------------------------------------------------------ A1 / A2
@pytest.mark.parametrize("dims", [(128, 128, 128), (37, 29, 41), (130, 67, 3), (2, 2, 2)])
def test_minmax_hist_bit_exact(be, dims):
    nx, ny, nz = dims
    if not be.full and nx * ny * nz > 200000:
        nx, ny, nz = 96, 50, 40                                      # several CTAs, loop + tail, at emulation speed
    v = W.make_cube(W.Recipe(nx, ny, nz, seed=21, n_sources=4 if nx > 8 else 0))
    with vr.Volume(be.dev(v), (nx, ny, nz)) as vol:
        assert_summary_equal(summary(be, vol), O.minmax_hist(v))
        assert_summary_equal(summary(be, vol, 64, (-1.0, 1.5)), O.minmax_hist(v, 64, (-1.0, 1.5)))
        assert_summary_equal(summary(be, vol, 1000), O.minmax_hist(v, 1000))
        assert_summary_equal(summary(be, vol, 4096, (0.0, 0.0)), O.minmax_hist(v, 4096, (0.0, 0.0)))


def test_minmax_hist_nonfinite_and_constant(be):
    v = W.make_cube(W.Recipe(40, 33, 27, seed=5)).copy()
    v[0, 0, 0], v[5, 6, 7], v[26, 32, 39], v[13, 1, 2] = np.nan, np.inf, -np.inf, np.nan
    with vr.Volume(be.dev(v), (40, 33, 27)) as vol:
        g, o = summary(be, vol), O.minmax_hist(v)
        assert_summary_equal(g, o)
        assert int(g["counts"].sum() + g["n_below"] + g["n_above"] + g["n_nonfinite"]) == v.size
    c = np.full((9, 10, 11), 3.5, dtype=np.float32)
    with vr.Volume(be.dev(c), (11, 10, 9)) as vol:
        assert_summary_equal(summary(be, vol), O.minmax_hist(c))
    k = (np.arange(8 * 16 * 32) % 256).astype(np.float32).reshape(8, 16, 32)
    with vr.Volume(be.dev(k), (32, 16, 8)) as vol:
        g = summary(be, vol)
        assert np.all(g["counts"] == k.size // 256)


def test_histogram_ranges_that_overflow_the_bin_arithmetic(be):
    """S41: caller ranges whose bin arithmetic overflows (scale_h = 0 with an infinite v - lo, or scale_h = inf): NaN goes
    to bin 0 and +inf to the last bin on both sides (the float-to-int conversion of the GPU, made explicit in the oracle)."""
    v = np.array([-3.0e38, 3.0e38, 0.0, 1.0, -1.0, 2.5, 1e-40, 7.0], dtype=np.float32).reshape(2, 2, 2)
    w = np.array([0.0, 1e-40, 5e-41, 0.0, 1e-40, -1.0, 1.0, 1e-40], dtype=np.float32).reshape(2, 2, 2)
    for a, rng in ((v, (-3.4e38, 3.4e38)), (w, (0.0, 1e-40)), (v, (-3.0e38, 3.0e38))):
        with vr.Volume(be.dev(a), (2, 2, 2)) as vol:
            assert_summary_equal(summary(be, vol, 16, rng), O.minmax_hist(a, 16, rng))


# ------------------------------------------------------------------ §8(f) #1: mean, standard deviation, median
def assert_statistics_equal(g, o, v):
    """Counts and the median (a data value) bit-exact; the float64 moments within 1e-13 of the data scale: both
    sides sum in compensated float64, in different orders (S35-S36)."""
    assert int(g["n_finite"]) == o.n_finite and int(g["n_nonfinite"]) == o.n_nonfinite
    if o.n_finite == 0:
        assert np.isnan(g["mean"]) and np.isnan(g["stddev"]) and np.isnan(g["median"])
        return
    assert np.float32(g["median"]).tobytes() == np.float32(o.median).tobytes(), (g["median"], o.median)
    f = v[np.isfinite(v)].astype(np.float64)
    scale = np.abs(f).mean()
    assert abs(float(g["mean"]) - o.mean) <= 1e-13 * scale, (g["mean"], o.mean)
    assert abs(float(g["stddev"]) - o.stddev) <= 1e-13 * max(o.stddev, scale), (g["stddev"], o.stddev)


@pytest.mark.parametrize("dims", [(128, 128, 128), (37, 29, 41), (130, 67, 3), (2, 2, 2)])
def test_statistics_match_oracle(be, dims):
    nx, ny, nz = dims
    if not be.full and nx * ny * nz > 200000:
        nx, ny, nz = 96, 50, 40
    v = W.make_cube(W.Recipe(nx, ny, nz, seed=23, n_sources=4 if nx > 8 else 0)).copy()
    if v.size > 100:
        v.reshape(-1)[[3, 50, 97]] = np.nan, np.inf, -np.inf
    with vr.Volume(be.dev(v), (nx, ny, nz)) as vol:
        g = statistics(be, vol)
        assert_statistics_equal(g, O.statistics(v), v)
        g2 = statistics(be, vol, device=False)                       # pinned host output, and run-to-run determinism
        assert g.tobytes() == g2.tobytes()


def test_statistics_special_cubes(be):
    """Constant cube (the key interval is a single key after pass 0), a two-valued cube with even n (LOWER median),
    signed zeros (totalOrder: -0 before +0), integers 0..255 (closed forms), no finite voxel at all."""
    cases = []
    cases.append(np.full((5, 6, 7), -3.25, dtype=np.float32))
    two = np.array([1.0] * 30 + [5.0] * 30, dtype=np.float32).reshape(3, 4, 5)
    cases.append(two)
    two2 = two.copy(); two2[0, 0, 0] = 5.0
    cases.append(two2)
    z = np.array([0.0, -0.0, -0.0, 0.0, 1.0, -1.0, -0.0, 2.0], dtype=np.float32).reshape(2, 2, 2)
    cases.append(z)
    z2 = z.copy(); z2[0, 0, 1] = 0.0
    cases.append(z2)
    k = np.repeat(np.arange(256), 32).astype(np.float32)
    np.random.default_rng(4).shuffle(k)
    cases.append(k.reshape(8, 32, 32))
    cases.append(np.full((3, 4, 5), np.nan, dtype=np.float32))
    wide = np.array([-3.0e38, 3.0e38, 1e-45, -1e-45, 0.5, 7.0, -2.0, 1.0], dtype=np.float32).reshape(2, 2, 2)   # the whole key space
    cases.append(wide)
    for c in cases:
        nz, ny, nx = c.shape
        with vr.Volume(be.dev(c), (nx, ny, nz)) as vol:
            g = statistics(be, vol)
        o = O.statistics(c)
        assert_statistics_equal(g, o, c)
        if np.isfinite(c).all():
            assert np.float32(g["median"]).tobytes() == np.sort(c.reshape(-1))[(c.size - 1) // 2].tobytes() or \
                float(g["median"]) == 0.0                             # np.sort does not order the signed zeros
    with vr.Volume(be.dev(cases[5]), (32, 32, 8)) as vol:
        g = statistics(be, vol)
    assert g["mean"] == 127.5 and g["median"] == 127.0 and abs(g["stddev"] - np.sqrt((256 ** 2 - 1) / 12)) < 1e-12


@pytest.mark.parametrize("where", ["device", "host_ooc"])
def test_statistics_bricked_halo_and_streamed(be, where):
    """Halo voxels are not counted; out of core all five passes ride the brick streamer."""
    n, B = (45, 38, 52), 16
    v = W.make_cube(W.Recipe(*n, seed=36, n_sources=4)).copy()
    v[7, 8, 9] = np.nan
    t = W.retile_halo(v, B)
    kw = dict(resident_bytes=7 * (B + 1) ** 3 * 4, n_copy_streams=3) if where == "host_ooc" else {}
    data = be.dev(t) if where == "device" else be.pinned(t)
    with vr.Volume(data, n, brick=B, layout=vr.VR_BRICKED_HALO1, **kw) as vol:
        g = statistics(be, vol)
        assert_statistics_equal(g, O.statistics(v), v)
        if where == "host_ooc":
            assert vol.stats()["h2d_bytes"] > 4 * t.size              # the non-resident bricks were streamed five times


# ------------------------------------------------------------------ cfg1: A3, A6-A9
def test_cfg1(be):
    """cfg1 at full size (128^3, 256x256 ortho view along z, step 0.5, 1.68e7 samples per mode) on both backends."""
    cfg = W.get_config(1)
    v = W.make_cube(cfg.recipe)
    cam = cfg.camera()
    o_sum = O.minmax_hist(v)
    tf = W.tf_haze(cfg.dims, cfg.step)
    with vr.Volume(be.dev(v), cfg.dims) as vol:
        g = summary(be, vol)
        assert_summary_equal(g, o_sum)
        vol.set_transfer_function(tf, float(g["vmin"]), float(g["vmax"]))
        mip = render(be, vol, cam, vr.VR_MIP)
        ea = render(be, vol, cam, vr.VR_EA)
        ea2 = render(be, vol, cam, vr.VR_EA)
        st = vol.stats()
        vol.set_option(vr.VR_OPT_RENDER_PATH, vr.VR_PATH_RAY_MAJOR)
        mip_r = render(be, vol, cam, vr.VR_MIP)
        ea_r = render(be, vol, cam, vr.VR_EA)
        st_r = vol.stats()
    R = float(max(abs(o_sum.vmin), abs(o_sum.vmax)))
    om = O.render(v, cam, O.MIP)
    oe = O.render(v, cam, O.EA, tf, o_sum.vmin, o_sum.vmax)
    sm = check_mip(mip, om.image, R)
    se = check_ea(ea, oe.image)
    assert sm["bit_exact"] == 1.0 and se["bit_exact"] == 1.0        # same canonical op sequence
    assert np.array_equal(ea, ea2)                                   # run-to-run determinism
    assert st["path"] == 7 and st["kernel_launches"] == 1           # auto = lane-mapped rows; a view along z needs no z-fastest copy
    assert st["zfast_copy"] == 0
    assert st_r["path"] == 1 and st_r["kernel_launches"] == 1
    assert check_mip(mip_r, om.image, R)["bit_exact"] == 1.0 and check_ea(ea_r, oe.image)["bit_exact"] == 1.0


def _views(n):
    c = np.array(n) / 2
    yield "persp", W.perspective_camera(c + np.array([1.9, 0.8, 1.5]) * max(n), c, (0, 1, 0), 40.0, 97, 61, step=0.5)
    yield "ortho", W.ortho_lookat_camera(c + np.array([-1.7, 0.6, 1.1]) * max(n), c, (0, 1, 0), 1.6 * max(n), 80, 50, step=0.7)
    yield "inside", W.perspective_camera((16.3, 7.25, 32.45), (30, 40, 10), (0, 0, 1), 70.0, 64, 48, step=0.5)
    yield "axis", W.ortho_axis_camera(n, 0, -1, step=1.0)


# (path option, z-fastest copy allowed, lane lag): path 0 = lane-mapped rows (the default), 1 = ray-major tiles
_VARIANTS = [(0, 1, 1), (0, 0, 1), (0, 1, 0), (0, 1, 4), (1, 1, 1)]


def _set_variant(vol, variant):
    path, zcopy, lag = variant
    vol.set_option(vr.VR_OPT_RENDER_PATH, path)
    vol.set_option(vr.VR_OPT_ZFAST_COPY, zcopy)
    vol.set_option(vr.VR_OPT_LANE_LAG, lag)
    return 7 if path == 0 else 1


@pytest.mark.parametrize("variant", _VARIANTS)
@pytest.mark.parametrize("ert", [0.0, 0.99])
def test_single_march_views(be, ert, variant):
    n = (61, 47, 83)
    v = W.make_cube(W.Recipe(*n, seed=31, n_sources=5))
    s = O.minmax_hist(v)
    R = float(max(abs(s.vmin), abs(s.vmax)))
    tf = W.tf_opaque(n, 0.5) if ert else W.tf_haze(n, 0.5)
    with vr.Volume(be.dev(v), n) as vol:
        path_id = _set_variant(vol, variant)
        vol.set_transfer_function(tf, s.vmin, s.vmax)
        for name, cam in _views(n):
            cam = cam.with_(ert_alpha=ert)
            om = O.render(v, cam, O.MIP)
            sm = check_mip(render(be, vol, cam, vr.VR_MIP), om.image, R)
            assert vol.stats()["path"] == path_id
            oe = O.render(v, cam, O.EA, tf, s.vmin, s.vmax)
            se = check_ea(render(be, vol, cam, vr.VR_EA), oe.image, oe.fragile, oe.K > 0,
                          max_fragile_frac=FRAGILE_FRAC_OPAQUE if ert else 0.005)
            assert sm["bit_exact"] == 1.0 and se["bit_exact"] == 1.0, (name, sm, se)   # same canonical op sequence
            if ert:
                assert (oe.K_ert < oe.K).sum() > 20, name          # ERT really fires in this workload


def _axis_views(n, full=True):
    """Views that travel along +-x, +-y, +-z (all three principal-axis classes, both directions), oblique
    ones that mix the two pixel classes across the image, a wide-angle one from inside, image sizes that are
    not multiples of the 32x8 tile, and cameras rolled by 90 degrees (lanes along image j)."""
    c = np.array(n, dtype=np.float64) / 2
    m = float(max(n))
    size = (150, 105) if full else (75, 52)
    for k, e in enumerate([(1.6, 0.25, 0.3), (-1.5, -0.2, 0.35), (0.3, 1.7, 0.2), (0.25, -1.6, -0.3),
                           (0.3, 0.2, 1.8), (-0.2, 0.35, -1.7), (1.2, 1.1, 1.3), (-1.0, 1.2, -1.1)]):
        up = (0, 0, 1) if abs(e[1]) > 1 else (0, 1, 0)
        yield f"persp{k}", W.perspective_camera(c + np.array(e) * m, c, up, 42.0, *size, step=0.5)
    yield "rolled_z", W.perspective_camera(c + np.array([0.3, 0.2, 1.8]) * m, c, (1, 0.2, 0), 42.0, size[1], size[0], step=0.5)
    yield "rolled_x", W.perspective_camera(c + np.array([1.7, -0.3, 0.4]) * m, c, (0, 0.3, 1), 42.0, size[1], size[0], step=0.5)
    yield "ortho_x", W.ortho_lookat_camera(c + np.array([1.7, 0.4, -0.5]) * m, c, (0, 1, 0), 1.5 * m, 90, 70, step=0.75)
    yield "ortho_z", W.ortho_lookat_camera(c + np.array([-0.3, 0.5, 1.9]) * m, c, (0, 1, 0), 1.5 * m, 100, 60, step=0.6)
    yield "inside", W.perspective_camera(c + np.array([0.11, -0.07, 0.2]) * m, c + np.array([0.5, 0.4, -0.3]) * m,
                                         (0, 1, 0), 75.0, size[0] + 26, size[1] + 23, step=0.5)
    if full:
        yield "axis_z", W.ortho_axis_camera(n, 2, +1, step=0.5, width=2 * n[0], height=2 * n[1])
    yield "axis_x", W.ortho_axis_camera(n, 0, -1, step=1.0)


@pytest.mark.parametrize("variant", [(0, 1, 1), (0, 0, 2)])
@pytest.mark.parametrize("n", [(132, 72, 100), (64, 200, 40), (61, 47, 83)])
def test_lane_mapped_views(be, n, variant):
    """The default path over views travelling along +-x, +-y, +-z, with and without the z-fastest copy: EA with
    and without ERT and MIP, bit-identical to the oracle's single march (same canonical op sequence)."""
    if not be.full:
        n = tuple(max(24, d // 2) for d in n)
    v = W.make_cube(W.Recipe(*n, seed=91, n_sources=14))
    s = O.minmax_hist(v)
    R = float(max(abs(s.vmin), abs(s.vmax)))
    tf = W.tf_opaque(n, 0.5)
    with vr.Volume(be.dev(v), n) as vol:
        _set_variant(vol, variant)
        vol.set_transfer_function(tf, s.vmin, s.vmax)
        for name, cam in _axis_views(n, be.full):
            for ert in (0.0, 0.99):
                cam2 = cam.with_(ert_alpha=ert)
                oe = O.render(v, cam2, O.EA, tf, s.vmin, s.vmax)
                se = check_ea(render(be, vol, cam2, vr.VR_EA), oe.image, oe.fragile, oe.K > 0,
                              max_fragile_frac=FRAGILE_FRAC_OPAQUE)
                assert vol.stats()["path"] == 7, name
                assert se["bit_exact"] == 1.0, (name, ert, se)
            om = O.render(v, cam, O.MIP)
            assert check_mip(render(be, vol, cam, vr.VR_MIP), om.image, R)["bit_exact"] == 1.0, name
        assert vol.stats()["zfast_copy"] == variant[1]            # the x-travelling views made the copy (when allowed)


# ------------------------------------------------------------------ §8(f) #2: exact empty-space skipping
@pytest.mark.parametrize("n", [(132, 72, 100), (61, 47, 83)])
def test_empty_space_skipping_is_exact(be, n):
    """TF_SOURCES makes the noise floor transparent (opacity exactly 0 on a table interval): most macrocells are
    empty, the kernel skips their samples, and the image is STILL bit-identical to the oracle, which skips nothing
    (C.5: compositing a sample of opacity 0 changes nothing).  Cells next to sources, cells with NaN / Inf voxels
    and the clamped outer half voxel are the cases a wrong cell range would get wrong."""
    if not be.full:
        n = tuple(max(24, d // 2) for d in n)
    v = W.make_cube(W.Recipe(*n, seed=93, n_sources=10 if be.full else 2)).copy()
    v[n[2] // 2, n[1] // 2, n[0] // 3] = np.nan
    v[3, 4, 5] = np.inf
    s = O.minmax_hist(v)
    tf = W.tf_sources(n, 0.5, alpha_scale=8.0)
    views = [(k, c) for k, c in _axis_views(n, be.full) if k in ("persp0", "persp2", "persp5", "persp6", "ortho_x", "inside", "axis_x")]
    with vr.Volume(be.dev(v), n) as vol:
        vol.set_transfer_function(tf, s.vmin, s.vmax)
        for name, cam in views:
            for ert in (0.0, 0.99):
                cam2 = cam.with_(ert_alpha=ert)
                oe = O.render(v, cam2, O.EA, tf, s.vmin, s.vmax)
                g = render(be, vol, cam2, vr.VR_EA)
                assert np.array_equal(g, oe.image, equal_nan=True), (name, ert)
                st = vol.stats()
                assert st["path"] == 7 and st["skip_variant"] == 1
        st = vol.stats()
        assert st["macro_cells"] == np.prod([(d - 2) // 8 + 1 for d in n])
        assert st["empty_cells"] >= st["macro_cells"] // 4          # the skipping really happened
        # a transfer function without an empty interval: the plain variant, same handle
        tf2 = W.tf_opaque(n, 0.5).copy(); tf2[:, 3] = np.maximum(tf2[:, 3], 1e-3)
        vol.set_transfer_function(tf2, s.vmin, s.vmax)
        name, cam = views[0]
        oe = O.render(v, cam, O.EA, tf2, s.vmin, s.vmax)
        assert np.array_equal(render(be, vol, cam, vr.VR_EA), oe.image, equal_nan=True)
        assert vol.stats()["skip_variant"] == 0
        # TF_HAZE has an empty interval but no cell of a noise cube falls into it: either the skipping variant is
        # launched and decides on the device not to skip (the count has not reached the host yet), or the host already
        # knows and launches the plain variant (always so in the emulation, whose runtime is synchronous)
        tf3 = W.tf_haze(n, 0.5)
        vol.set_transfer_function(tf3, s.vmin, s.vmax)
        oe = O.render(v, cam, O.EA, tf3, s.vmin, s.vmax)
        assert np.array_equal(render(be, vol, cam, vr.VR_EA), oe.image, equal_nan=True)
        be.sync()
        assert vol.stats()["empty_cells"] < max(1, vol.stats()["macro_cells"] // 64)
        assert np.array_equal(render(be, vol, cam, vr.VR_EA), oe.image, equal_nan=True)
        assert vol.stats()["skip_variant"] == 0                      # by now the host knows: plain variant
        vol.set_option(vr.VR_OPT_EMPTY_SKIP, 0)
        vol.set_transfer_function(tf, s.vmin, s.vmax)
        oe = O.render(v, cam, O.EA, tf, s.vmin, s.vmax)
        assert np.array_equal(render(be, vol, cam, vr.VR_EA), oe.image, equal_nan=True)
        assert vol.stats()["skip_variant"] == 0


def test_empty_space_leaps_over_whole_blocks(be):
    """A cube that is empty (under the transfer function) except for one corner: blocks of 8x8x8 cells are empty as
    a whole and rays leap 64 base indices at a time; rays that graze the blob, enter through the clamped outer half
    voxel or end inside an empty block exercise the verification of every leap."""
    n = (150, 80, 90) if be.full else (136, 72, 72)
    nx, ny, nz = n
    rng = np.random.default_rng(17)
    v = (-1.0 + 0.05 * rng.standard_normal((nz, ny, nx))).astype(np.float32)
    z, y, x = np.mgrid[0:nz, 0:ny, 0:nx]
    v += (12.0 * np.exp(-((x - 20.0) ** 2 + (y - 15.0) ** 2 + (z - 18.0) ** 2) / (2 * 6.0 ** 2))).astype(np.float32)
    v[nz - 1, ny - 1, nx - 1] = 9.0                                  # one bright voxel in the far corner
    s = O.minmax_hist(v)
    tf = W.tf_sources(n, 0.5, alpha_scale=6.0)
    c = np.array(n, dtype=np.float64) / 2
    m = float(max(n))
    size = (64, 40) if be.full else (40, 26)
    cams = [W.perspective_camera(c + np.array(e) * m, c, (0, 1, 0), 40.0, *size, step=st)
            for e, st in (((1.7, 0.3, 0.2), 0.5), ((-0.4, 0.5, 1.6), 1.0), ((-1.2, -0.9, -1.1), 0.25))]
    cams.append(W.ortho_axis_camera(n, 0, +1, step=1.0, width=size[0], height=size[1]))
    if be.name == "simt":
        import simt_lib
        simt_lib.lib().simt_reset_counters()
    with vr.Volume(be.dev(v), n) as vol:
        vol.set_transfer_function(tf, s.vmin, s.vmax)
        for cam in cams:
            for ert in (0.0, 0.99):
                cam2 = cam.with_(ert_alpha=ert)
                oe = O.render(v, cam2, O.EA, tf, s.vmin, s.vmax)
                assert np.array_equal(render(be, vol, cam2, vr.VR_EA), oe.image), ert
                assert oe.image[..., 3].max() > 0.05                 # the blob is visible: not everything was skipped
        st = vol.stats()
        assert st["skip_variant"] == 1 and st["empty_cells"] > 0.8 * st["macro_cells"]
    if be.name == "simt":                                           # the emulation counts what the kernel did
        cnt = [simt_lib.lib().simt_counter(i) for i in range(4)]
        assert cnt[0] > 1000 and cnt[1] > 1000, cnt                  # leaps over single cells AND over whole blocks
        assert cnt[2] < 0.2 * (cnt[0] + cnt[1]), cnt                 # the estimate is rarely rejected by the verification


def test_zfast_copy_skipped_when_memory_is_short(be):
    """Without room for a second copy of the volume the x-travelling views render from the x-fastest array."""
    if be.name != "simt":
        pytest.skip("needs control over the free device memory (emulated runtime only)")
    import simt_lib
    n = (40, 36, 44)
    v = W.make_cube(W.Recipe(*n, seed=12, n_sources=2))
    cam = W.orbit_camera(n, 2, 8, 60, 40, step=0.5)                 # travels mostly along x
    d = be.dev(v)
    simt_lib.lib().simt_set_device_capacity(simt_lib.lib().simt_device_bytes_in_use() + v.nbytes // 2 + (1 << 16))
    try:
        with vr.Volume(d, n) as vol:
            g = render(be, vol, cam, vr.VR_MIP)
            assert vol.stats()["zfast_copy"] == 0 and vol.stats()["path"] == 7
    finally:
        simt_lib.lib().simt_set_device_capacity(4 << 30)
    assert np.array_equal(g, O.render(v, cam, O.MIP).image)


@pytest.mark.parametrize("how", ["lanes", "tiles", "sort_last", "chain"])
def test_64_bit_offsets_at_small_size(be, how):
    """VR_OPT_FORCE_WIDE: the 64-bit voxel-offset arithmetic that volumes of more than 2^32 voxels (cfg4) run, at a
    size the oracle and the host emulation finish in seconds; z- and x-travelling views (both volume copies)."""
    n, B = (52, 40, 61), 16
    v = W.make_cube(W.Recipe(*n, seed=77, n_sources=4))
    s = O.minmax_hist(v)
    R = float(max(abs(s.vmin), abs(s.vmax)))
    tf = W.tf_opaque(n, 0.5)
    views = [c for k, c in _axis_views(n, False) if k in ("persp0", "persp4", "persp6", "ortho_x")]
    data = be.dev(W.retile_halo(v, B)) if how == "chain" else be.dev(v)
    with vr.Volume(data, n, brick=B, layout=vr.VR_BRICKED_HALO1 if how == "chain" else vr.VR_LINEAR) as vol:
        vol.set_option(vr.VR_OPT_FORCE_WIDE, 1)
        if how == "tiles":
            vol.set_option(vr.VR_OPT_RENDER_PATH, vr.VR_PATH_RAY_MAJOR)
        vol.set_transfer_function(tf, s.vmin, s.vmax)
        for cam in views:
            sl = how == "sort_last"
            cam2 = cam.with_(ert_alpha=0.0 if sl else 0.99, flags=W.cameras.VR_SORT_LAST if sl else 0)
            oe = O.render(v, cam2, O.EA, tf, s.vmin, s.vmax, brick=B if sl else 0)
            assert np.array_equal(render(be, vol, cam2, vr.VR_EA), oe.image)
            om = O.render(v, cam2, O.MIP, brick=B if sl else 0)
            assert np.array_equal(render(be, vol, cam2, vr.VR_MIP), om.image)


@pytest.mark.parametrize("n", [(2, 5, 9), (64, 2, 33), (7, 40, 2), (2, 2, 2)])
def test_degenerate_dimensions(be, n):
    """An axis of length 2 (one cell: i0 is always 0 and the whole axis is 'outer half voxel'), every render path;
    bricks larger than the cube and bricks of edge 2."""
    v = W.make_cube(W.Recipe(*n, seed=101, n_sources=0))
    s = O.minmax_hist(v)
    tf = W.bake_tf(W.TF_HAZE_POINTS, 0.5, alpha_scale=20.0)
    c = np.array(n, dtype=np.float64) / 2
    m = float(max(n))
    cams = [W.perspective_camera(c + np.array(e) * m * 1.5, c, (0, 1, 0), 50.0, 45, 37, step=0.3)
            for e in ((1.2, 0.5, 0.8), (-0.3, 0.2, 1.5), (0.2, 1.6, 0.1))]
    cams.append(W.ortho_axis_camera(n, 1, +1, step=0.5))
    for path in (0, 1):
        with vr.Volume(be.dev(v), n, brick=2) as vol:
            vol.set_option(vr.VR_OPT_RENDER_PATH, path)
            vol.set_transfer_function(tf, s.vmin, s.vmax)
            for k, up in enumerate(cams):
                for ert in (0.0, 0.9):
                    oe = O.render(v, up.with_(ert_alpha=ert), O.EA, tf, s.vmin, s.vmax)
                    assert np.array_equal(render(be, vol, up.with_(ert_alpha=ert), vr.VR_EA), oe.image), (n, path, k, ert)
                om = O.render(v, up, O.MIP)
                assert np.array_equal(render(be, vol, up, vr.VR_MIP), om.image), (n, path, k)
                if up.is_perspective or up.is_orthographic:
                    sl = up.with_(flags=W.cameras.VR_SORT_LAST)
                    ob = O.render(v, sl, O.EA, tf, s.vmin, s.vmax, brick=2)
                    assert np.array_equal(render(be, vol, sl, vr.VR_EA), ob.image), (n, path, k, "sort-last")
    with vr.Volume(be.dev(v), n, brick=1000) as vol:               # one brick larger than the cube
        vol.set_transfer_function(tf, s.vmin, s.vmax)
        sl = cams[0].with_(flags=W.cameras.VR_SORT_LAST)
        assert np.array_equal(render(be, vol, sl, vr.VR_EA), O.render(v, sl, O.EA, tf, s.vmin, s.vmax, brick=1000).image)


def test_rays_along_brick_planes_and_opaque_first_sample(be):
    """Orthographic rays with d_a = 0 whose origin lies exactly on an ownership plane o_a = B b + 1/2 (every sample
    sits on the boundary between two bricks: C.7 gives it to exactly one); alpha = 1 everywhere with ERT (K = 1:
    the ray stops after its first sample, P7)."""
    n, B = (32, 24, 40), 8
    v = W.make_cube(W.Recipe(*n, seed=55, n_sources=2))
    s = O.minmax_hist(v)
    cam = W.ortho_axis_camera(n, 2, +1, step=0.5, width=8, height=6)   # pixel centres at x = 2, 6, .. ; y = 2, 6, ..
    vec = cam.vectors()
    o0 = vec[0].copy(); o0[0] += 8.5 - 2.0; o0[1] += 8.5 - 2.0            # first pixel centre on the planes x = y = 8.5
    cam = cam.with_(o0=o0, ou=np.array([8.0, 0, 0], np.float32), ov=np.array([0, 8.0, 0], np.float32), width=3, height=2)
    tf = W.tf_haze(n, 0.5)
    one = np.ones((256, 4), dtype=np.float32)
    with vr.Volume(be.dev(v), n, brick=B) as vol:
        vol.set_transfer_function(tf, s.vmin, s.vmax)
        for flags in (0, W.cameras.VR_SORT_LAST):
            c2 = cam.with_(flags=flags)
            o = O.render(v, c2, O.EA, tf, s.vmin, s.vmax, brick=B if flags else 0)
            assert o.n_order_mismatch == 0 and o.n_noncontig == 0
            assert np.array_equal(render(be, vol, c2, vr.VR_EA), o.image), flags
            om = O.render(v, c2, O.MIP, brick=B if flags else 0)
            assert np.array_equal(render(be, vol, c2, vr.VR_MIP), om.image), flags
        vol.set_transfer_function(one, s.vmin, s.vmax)
        view = W.orbit_camera(n, 1, 8, 40, 30, step=0.5, ert_alpha=0.5)
        o = O.render(v, view, O.EA, one, s.vmin, s.vmax)
        assert (o.K_ert[o.K > 0] == 1).all()
        g = render(be, vol, view, vr.VR_EA)
        assert np.array_equal(g, o.image) and (g[o.K > 0] == 1.0).all()


@pytest.mark.parametrize("n,wide", [((64, 44, 60), 0), ((64, 44, 60), 1), ((36, 40, 61), 0)])
def test_16_byte_row_loads(be, n, wide):
    """VR_OPT_ROW_LOADS = 1: one aligned 16-byte load per row (+ a scalar load where x ends its quad) instead of two
    scalar loads — the same eight voxels, so bit-identical images; the memory-fast dimension must be a multiple of 4
    (nz = 61: the z-fastest launches keep scalar loads, the x-fastest ones use quads); with and without 64-bit offsets."""
    v = W.make_cube(W.Recipe(*n, seed=88, n_sources=6))
    s = O.minmax_hist(v)
    R = float(max(abs(s.vmin), abs(s.vmax)))
    tf = W.tf_opaque(n, 0.5)
    with vr.Volume(be.dev(v), n) as vol:
        vol.set_option(vr.VR_OPT_ROW_LOADS, 1)
        vol.set_option(vr.VR_OPT_FORCE_WIDE, wide)
        vol.set_transfer_function(tf, s.vmin, s.vmax)
        for name, cam in _axis_views(n, False):
            for ert in (0.0, 0.99):
                cam2 = cam.with_(ert_alpha=ert)
                oe = O.render(v, cam2, O.EA, tf, s.vmin, s.vmax)
                assert np.array_equal(render(be, vol, cam2, vr.VR_EA), oe.image), (name, ert)
            om = O.render(v, cam, O.MIP)
            assert np.array_equal(render(be, vol, cam, vr.VR_MIP), om.image), name
        assert vol.stats()["path"] == 7


@pytest.mark.parametrize("path", [0, 1])
def test_progressive_passes(be, path):
    """VR_SUBSAMPLE: a pass renders one sub-lattice of the pixels in place; every rendered pixel is bit-identical to the
    oracle's pixel (its `mask` is the same lattice), every other pixel of the buffer is untouched, and after all
    stride^2 phases the buffer IS the full render.  Views with both pixel classes, an image that is not a multiple of
    the stride, a phase without any pixel."""
    n = (52, 40, 61)
    v = W.make_cube(W.Recipe(*n, seed=71, n_sources=4))
    s = O.minmax_hist(v)
    tf = W.tf_opaque(n, 0.5)
    cams = [c.with_(ert_alpha=0.99) for k, c in _axis_views(n, False) if k in ("persp0", "persp6", "ortho_z")]
    with vr.Volume(be.dev(v), n) as vol:
        vol.set_option(vr.VR_OPT_RENDER_PATH, path)
        vol.set_transfer_function(tf, s.vmin, s.vmax)
        for cam in cams:
            H, Wd = cam.height, cam.width
            full = O.render(v, cam, O.EA, tf, s.vmin, s.vmax).image
            for stride in (4, 3):
                buf = be.empty((H, Wd, 4), fill=7.0)
                seen = np.zeros((H, Wd), dtype=bool)
                for py in range(stride):
                    for px in range(stride):
                        vol.render(cam.with_(flags=vr.VR_SUBSAMPLE(stride, px, py)), vr.VR_EA, out=buf, stream=be.stream)
                        seen[py::stride, px::stride] = True
                        g = be.numpy(buf)
                        assert np.array_equal(g[seen], full[seen]) and (g[~seen] == 7.0).all(), (stride, px, py)
                        if (px, py) == (0, 0):                   # the oracle with the same lattice as its mask
                            mask = seen.astype(np.uint8)
                            o = O.render(v, cam, O.EA, tf, s.vmin, s.vmax, mask=mask).image
                            assert np.array_equal(g[seen], o[seen])
                assert np.array_equal(be.numpy(buf), full)
            mbuf = be.empty((H, Wd), fill=-3.0)
            vol.render(cam.with_(flags=vr.VR_SUBSAMPLE(5, 2, 1)), vr.VR_MIP, out=mbuf, stream=be.stream)
            gm, om = be.numpy(mbuf), O.render(v, cam, O.MIP).image
            assert np.array_equal(gm[1::5, 2::5], om[1::5, 2::5]) and (np.delete(np.delete(gm, np.s_[1::5], 0), np.s_[2::5], 1) == -3.0).all()
        tiny = cams[0].with_(width=3, height=2)
        tb = be.empty((2, 3, 4), fill=7.0)
        vol.render(tiny.with_(flags=vr.VR_SUBSAMPLE(4, 3, 3)), vr.VR_EA, out=tb, stream=be.stream)     # no pixel has j % 4 == 3
        assert (be.numpy(tb) == 7.0).all()
        with pytest.raises(vr.VrError) as e:
            vol.render(cams[0].with_(flags=vr.VR_SUBSAMPLE(2, 2, 0)), vr.VR_EA, out=tb, stream=be.stream)
        assert e.value.status == vr.VR_ERR_INVALID_ARG
    with vr.Volume(be.dev(v), n, brick=16) as vol:
        vol.set_transfer_function(tf, s.vmin, s.vmax)
        with pytest.raises(vr.VrError) as e:
            vol.render(cams[0].with_(ert_alpha=0.0, flags=vr.VR_SUBSAMPLE(2, 0, 0) | vr.VR_SORT_LAST), vr.VR_EA,
                       out=be.empty((cams[0].height, cams[0].width, 4)), stream=be.stream)
        assert e.value.status == vr.VR_ERR_UNSUPPORTED


def test_row_loads_default_follows_the_view(be):
    """VR_OPT_ROW_LOADS = 2 (default): 16-byte row loads for the launches whose rays can enter through the face
    perpendicular to the memory-fast axis (oblique views of the orbit: both lateral faces visible), scalar loads for
    the others; volumes whose fast dimension is not a multiple of 4 never use them.  Results are the same either way
    (test_16_byte_row_loads); this pins the rule the traffic model (profiles/r2_lane_traffic_model.md) is quoted for."""
    n = (64, 64, 128)
    v = W.make_cube(W.Recipe(*n, seed=3))
    want = {0: 0, 2: 2, 8: 0, 10: 2, 14: 2}                       # orbit of 16 views: view -> launches with quads (axis / oblique)
    with vr.Volume(be.dev(v), n) as vol:
        for view, quads in want.items():
            cam = W.orbit_camera(n, view, 16, 64, 48, step=1.0)
            render(be, vol, cam, vr.VR_MIP)
            st = vol.stats()
            assert st["quad_launches"] == quads, (view, st["quad_launches"], st["kernel_launches"])
        vol.set_option(vr.VR_OPT_ROW_LOADS, 0)
        render(be, vol, W.orbit_camera(n, 2, 16, 64, 48, step=1.0), vr.VR_MIP)
        assert vol.stats()["quad_launches"] == 0
    n2 = (62, 64, 126)
    with vr.Volume(be.dev(W.make_cube(W.Recipe(*n2, seed=3))), n2) as vol:
        render(be, vol, W.orbit_camera(n2, 2, 16, 64, 48, step=1.0), vr.VR_MIP)
        assert vol.stats()["quad_launches"] == 0


def test_mixed_camera_renders(be):
    """A camera whose origins AND directions vary per pixel (neither perspective nor orthographic)."""
    n = (32, 32, 32)
    v = W.make_cube(W.Recipe(*n, seed=3))
    cam = W.perspective_camera((80.0, 20.0, 16.0), (16, 16, 16), (0, 1, 0), 30.0, 40, 30)
    cam = cam.with_(ou=np.array([0.01, 0, 0], dtype=np.float32))
    with vr.Volume(be.dev(v), n) as vol:
        g = render(be, vol, cam, vr.VR_MIP)
        assert vol.stats()["path"] == 7
    assert np.array_equal(g, O.render(v, cam, O.MIP).image)


def test_set_option_rejects_bad_values(be):
    v = W.make_cube(W.Recipe(16, 16, 16, seed=1))
    with vr.Volume(be.dev(v), (16, 16, 16)) as vol:
        for opt, val in ((vr.VR_OPT_RENDER_PATH, 5), (vr.VR_OPT_ZFAST_COPY, 2), (vr.VR_OPT_LANE_LAG, -1),
                         (vr.VR_OPT_EMPTY_SKIP, 2), (vr.VR_OPT_FORCE_WIDE, -1), (vr.VR_OPT_ROW_LOADS, 3), (77, 0)):
            with pytest.raises(vr.VrError) as e:
                vol.set_option(opt, val)
            assert e.value.status == vr.VR_ERR_INVALID_ARG


def test_all_miss_camera(be):
    n = (20, 24, 28)
    v = W.make_cube(W.Recipe(*n, seed=2))
    cam = W.perspective_camera((100.0, 100.0, 100.0), (200, 200, 200), (0, 1, 0), 20.0, 33, 17)
    with vr.Volume(be.dev(v), n) as vol:
        vol.set_transfer_function(W.tf_haze(n, 0.5), -5.0, 5.0)
        assert np.isneginf(render(be, vol, cam, vr.VR_MIP)).all()
        assert (render(be, vol, cam, vr.VR_EA) == 0).all()


# ------------------------------------------------------------------ bricks: A0, A4, A10
@pytest.mark.parametrize("B,how", [(7, "lanes"), (16, "lanes"), (32, "lanes"), (100, "lanes"), (16, "quads"), (16, "tiles"), (16, "halo")])
def test_sort_last_equals_oracle_bricked(be, B, how):
    """Fragments from the lane-mapped march that flushes at every change of owner brick (`lanes`, the default for
    linear volumes), from one CTA per (brick, pixel tile) on a linear volume (`tiles`) and on a resident brick-major
    volume with halo (`halo`): all bit-identical to the oracle's bricked render (same partials, same fold order)."""
    n = (60, 47, 84) if how == "quads" else (61, 47, 83)            # quads need nx and nz to be multiples of 4
    v = W.make_cube(W.Recipe(*n, seed=33, n_sources=5))
    s = O.minmax_hist(v)
    R = float(max(abs(s.vmin), abs(s.vmax)))
    tf = W.bake_tf(W.TF_HAZE_POINTS, 0.5, alpha_scale=6.0)
    data = be.dev(W.retile_halo(v, B)) if how == "halo" else be.dev(v)
    if be.name == "simt":
        import simt_lib
        simt_lib.lib().simt_reset_counters()
    with vr.Volume(data, n, brick=B, layout=vr.VR_BRICKED_HALO1 if how == "halo" else vr.VR_LINEAR) as vol:
        if how == "tiles":
            vol.set_option(vr.VR_OPT_RENDER_PATH, vr.VR_PATH_RAY_MAJOR)
        if how == "quads":
            vol.set_option(vr.VR_OPT_ROW_LOADS, 1)
        vol.set_transfer_function(tf, s.vmin, s.vmax)
        for name, cam in _views(n):
            cam = cam.with_(flags=W.cameras.VR_SORT_LAST)
            om = O.render(v, cam, O.MIP, brick=B)
            assert om.n_noncontig == 0 and om.n_order_mismatch == 0
            sm = check_mip(render(be, vol, cam, vr.VR_MIP), om.image, R)
            assert sm["bit_exact"] == 1.0, name
            oe = O.render(v, cam, O.EA, tf, s.vmin, s.vmax, brick=B)
            se = check_ea(render(be, vol, cam, vr.VR_EA), oe.image)
            assert se["bit_exact"] == 1.0, (name, se)                # same partials, same fold order
            st = vol.stats()
            assert st["path"] == 2 and st["fragments"] > 0
    if be.name == "simt":                # no fragment fell outside its brick's rectangle, no owner brick was missing from the plan
        assert simt_lib.lib().simt_counter(4) == 0 and simt_lib.lib().simt_counter(5) == 0


def test_sort_last_rejections(be):
    n = (16, 16, 16)
    v = W.make_cube(W.Recipe(*n, seed=1))
    cam = W.ortho_axis_camera(n, 2, +1).with_(flags=W.cameras.VR_SORT_LAST)
    out = be.empty((16, 16))
    out4 = be.empty((16, 16, 4))
    with vr.Volume(be.dev(v), n, brick=0) as vol:
        with pytest.raises(vr.VrError) as e:
            vol.render(cam, vr.VR_MIP, out=out, stream=be.stream)
        assert e.value.status == vr.VR_ERR_UNSUPPORTED
    with vr.Volume(be.dev(v), n, brick=8) as vol:
        with pytest.raises(vr.VrError) as e:
            vol.render(cam, vr.VR_EA, out=out4, stream=be.stream)
        assert e.value.status == vr.VR_ERR_NOT_READY
        vol.set_transfer_function(W.tf_haze(n, 0.5), -1.0, 1.0)
        with pytest.raises(vr.VrError) as e:
            vol.render(cam.with_(ert_alpha=0.99), vr.VR_EA, out=out4, stream=be.stream)
        assert e.value.status == vr.VR_ERR_UNSUPPORTED


# ------------------------------------------------------------------ bricked-halo layout, chain, out-of-core: A5
@pytest.mark.parametrize("where", ["device", "host_resident", "host_ooc"])
def test_bricked_halo_chain_and_streaming(be, where):
    n = (61, 47, 83)
    B = 16
    v = W.make_cube(W.Recipe(*n, seed=35, n_sources=5))
    t = W.retile_halo(v, B)
    s = O.minmax_hist(v)
    R = float(max(abs(s.vmin), abs(s.vmax)))
    tf = W.tf_opaque(n, 0.5)
    brick_bytes = (B + 1) ** 3 * 4
    kw = {}
    data = be.dev(t) if where == "device" else be.pinned(t)
    if where == "host_ooc":
        kw = dict(resident_bytes=11 * brick_bytes, n_copy_streams=4)     # 11 of 72 bricks fit
    with vr.Volume(data, n, brick=B, layout=vr.VR_BRICKED_HALO1, **kw) as vol:
        assert_summary_equal(summary(be, vol), s)
        assert_summary_equal(summary(be, vol, 100, (-0.5, 2.0)), O.minmax_hist(v, 100, (-0.5, 2.0)))
        vol.set_transfer_function(tf, s.vmin, s.vmax)
        for name, cam in _views(n):
            for ert in (0.0, 0.99):
                cam2 = cam.with_(ert_alpha=ert)
                om = O.render(v, cam2, O.MIP)
                sm = check_mip(render(be, vol, cam2, vr.VR_MIP), om.image, R)
                assert sm["bit_exact"] == 1.0, name
                oe = O.render(v, cam2, O.EA, tf, s.vmin, s.vmax)
                se = check_ea(render(be, vol, cam2, vr.VR_EA), oe.image, oe.fragile, oe.K > 0,
                              max_fragile_frac=FRAGILE_FRAC_OPAQUE)
                assert se["bit_exact"] == 1.0, (name, ert, se)           # chained state == single march
        st = vol.stats()
        assert st["path"] == 3
        if where == "host_ooc":
            assert st["h2d_bytes"] > 0 and st["resident_bytes"] == 11 * brick_bytes


@pytest.mark.parametrize("where", ["device", "host_ooc"])
def test_empty_bricks_are_dropped_before_upload(be, where):
    """A brick-major cube that is transparent under TF_SOURCES except around one blob: after the first summary pass
    has gathered the value range of every brick slot, an EA render drops the empty bricks — out of core they are not
    even uploaded — and the image is still bit-identical to the oracle (S38).  MIP never drops a brick."""
    n, B = (60, 44, 52), 12
    nx, ny, nz = n
    rng = np.random.default_rng(23)
    v = (-1.0 + 0.05 * rng.standard_normal((nz, ny, nx))).astype(np.float32)
    z, y, x = np.mgrid[0:nz, 0:ny, 0:nx]
    v += (12.0 * np.exp(-((x - 40.0) ** 2 + (y - 30.0) ** 2 + (z - 12.0) ** 2) / (2 * 4.0 ** 2))).astype(np.float32)
    v[0, 0, 0] = np.nan                                             # a brick with a non-finite voxel is never dropped
    t = W.retile_halo(v, B)
    s = O.minmax_hist(v)
    tf = W.tf_sources(n, 0.5, alpha_scale=6.0)
    brick_bytes = (B + 1) ** 3 * 4
    kw = dict(resident_bytes=10 * brick_bytes, n_copy_streams=3) if where == "host_ooc" else {}
    data = be.dev(t) if where == "device" else be.pinned(t)
    cams = [c for _, c in _views(n)]
    with vr.Volume(data, n, brick=B, layout=vr.VR_BRICKED_HALO1, **kw) as vol:
        vol.set_transfer_function(tf, s.vmin, s.vmax)
        g0 = render(be, vol, cams[0], vr.VR_EA)                      # before any summary pass: nothing is known, nothing dropped
        st0 = vol.stats()
        assert st0["bricks_empty"] == 0
        assert_summary_equal(summary(be, vol), s)                    # gathers the brick ranges
        be.sync()
        for cam in cams:
            for ert in (0.0, 0.99):
                cam2 = cam.with_(ert_alpha=ert)
                oe = O.render(v, cam2, O.EA, tf, s.vmin, s.vmax)
                g = render(be, vol, cam2, vr.VR_EA)
                assert np.array_equal(g, oe.image, equal_nan=True)
                st = vol.stats()
                assert st["bricks_empty"] > 0.5 * st["n_bricks"] and st["bricks_drawn"] + st["bricks_empty"] + st["bricks_culled"] == st["n_bricks"]
            om = O.render(v, cam, O.MIP)
            assert np.array_equal(render(be, vol, cam, vr.VR_MIP), om.image) and vol.stats()["bricks_empty"] == 0
        assert np.array_equal(g0, O.render(v, cams[0], O.EA, tf, s.vmin, s.vmax).image, equal_nan=True)
        if where == "host_ooc":
            render(be, vol, cams[0], vr.VR_EA)
            assert vol.stats()["h2d_bytes"] < 0.5 * st0["h2d_bytes"]  # most of the streamed bricks were not uploaded
        # sort-last on the resident brick-major volume drops them too
        if where == "device":
            sl = cams[0].with_(flags=W.cameras.VR_SORT_LAST)
            ob = O.render(v, sl, O.EA, tf, s.vmin, s.vmax, brick=B)
            assert np.array_equal(render(be, vol, sl, vr.VR_EA), ob.image, equal_nan=True) and vol.stats()["bricks_empty"] > 0
        vol.set_option(vr.VR_OPT_EMPTY_SKIP, 0)
        render(be, vol, cams[0], vr.VR_EA)
        assert vol.stats()["bricks_empty"] == 0


def test_host_linear_mirror_and_host_outputs(be):
    n = (40, 36, 52)
    v = W.make_cube(W.Recipe(*n, seed=37, n_sources=3))
    s = O.minmax_hist(v)
    tf = W.tf_haze(n, 0.5)
    cam = W.orbit_camera(n, 1, 8, 96, 64, step=0.5, ert_alpha=0.99)
    with vr.Volume(be.pinned(v), n, brick=16) as vol:
        assert_summary_equal(summary(be, vol, device=False), s)
        assert vol.stats()["h2d_bytes"] == v.nbytes
        vol.set_transfer_function(tf, s.vmin, s.vmax)
        out = be.empty((64, 96, 4), device=False)
        g = render(be, vol, cam, vr.VR_EA, out=out)
        oe = O.render(v, cam, O.EA, tf, s.vmin, s.vmax)
        check_ea(g, oe.image, oe.fragile, oe.K > 0)
        assert vol.stats()["d2h_bytes"] == g.size * 4
        assert vol.stats()["h2d_bytes"] <= 257 * 16                      # the transfer function only; the cube is not re-uploaded


def test_pageable_host_memory_is_rejected(be):
    v = W.make_cube(W.Recipe(16, 16, 16, seed=1))

    class Pageable:                          # a plain numpy buffer: neither device nor page-locked memory
        is_cuda = False

        def data_ptr(self):
            return v.ctypes.data

    if (v.ctypes.data & 15) != 0:
        pytest.skip("unaligned numpy buffer")
    with pytest.raises(vr.VrError) as e:
        vr.Volume(Pageable(), (16, 16, 16))
    assert e.value.status == vr.VR_ERR_INVALID_ARG


def test_two_handles_two_streams_and_pitch(be):
    n = (32, 32, 32)
    a = W.make_cube(W.Recipe(*n, seed=41))
    b = W.make_cube(W.Recipe(*n, seed=42))
    cam = W.orbit_camera(n, 0, 4, 70, 50, step=0.5)
    if be.name == "gpu":
        import torch
        s1, s2 = torch.cuda.Stream(), torch.cuda.Stream()
    else:
        s1 = s2 = 0
    with vr.Volume(be.dev(a), n) as va, vr.Volume(be.dev(b), n) as vb:
        big = be.empty((50, 96), fill=0.0)
        be.sync()
        if be.name == "gpu":
            view = big[:, :70]
        else:                                # a 70-wide window of the 96-wide buffer: same pointer, pitch 96
            class View:
                is_cuda = True
                shape = (50, 70)
                data_ptr = big.data_ptr
                stride = big.stride
            view = View()
        va.render(cam, vr.VR_MIP, out=view, stream=s1)
        ib = be.empty((50, 70))
        vb.render(cam, vr.VR_MIP, out=ib, stream=s2)
        be.sync()
        g = be.numpy(big)
        assert np.array_equal(g[:, :70], O.render(a, cam, O.MIP).image)
        assert np.array_equal(be.numpy(ib), O.render(b, cam, O.MIP).image)
        assert (g[:, 70:] == 0).all()


# ------------------------------------------------------------------ full-size configs, bench launch configuration
def _host_cube(cfg):
    """The config's cube in host memory, filled in z-slabs by the shared generator (as bench.py does)."""
    nx, ny, nz = cfg.dims
    out = np.empty((nz, ny, nx), dtype=np.float32)
    gen = W.CubeGenerator(cfg.recipe)
    slab = max(1, (1 << 28) // (nx * ny))
    for z0 in range(0, nz, slab):
        z1 = min(nz, z0 + slab)
        gen.fill(out[z0:z1], z0, z1)
    return out


def _lattice(cfg, stride=8):
    m = np.zeros((cfg.height, cfg.width), dtype=np.uint8)
    m[stride // 2::stride, stride // 2::stride] = 1
    return m


def _check_statistics_by_definition(g, v):
    """At sizes the oracle's sort cannot finish in seconds: the properties that DEFINE the results.  The median m is
    a voxel value with #(v < m) <= rank < #(v <= m), rank = (n-1)//2; the mean against float64 slab sums; the standard
    deviation against float64 slab sums of squared deviations (cubes up to 16 GiB: the conversion passes take minutes
    beyond that, and the larger cube adds nothing the 8 GiB one — more than 2^31 voxels — does not cover)."""
    n = v.size
    assert int(g["n_finite"]) == n and int(g["n_nonfinite"]) == 0
    m = np.float32(g["median"])
    below = le = 0
    s1 = 0.0
    slabs = np.array_split(np.arange(v.shape[0]), max(1, v.nbytes >> 28))
    for idx in slabs:
        blk = v[idx[0]:idx[-1] + 1]
        below += int(np.count_nonzero(blk < m)); le += int(np.count_nonzero(blk <= m))
        s1 += float(blk.sum(dtype=np.float64))
    assert below <= (n - 1) // 2 < le, (below, le, n)
    mean = s1 / n
    assert abs(float(g["mean"]) - mean) <= 1e-11
    if v.nbytes > (16 << 30):
        return
    s2 = 0.0
    for idx in slabs:
        d = v[idx[0]:idx[-1] + 1].astype(np.float64) - mean
        s2 += float(np.dot(d.reshape(-1), d.reshape(-1)))
    assert abs(float(g["stddev"]) - np.sqrt(s2 / n)) <= 1e-11


def _full_size_case(number, views, summary_exact=True, stride=8):
    """vr_minmax_histogram on the whole cube (bit-exact) and vr_render of `views` at the config's own image
    size, step, ERT and flags — the launches bench.py times — compared with the oracle on a lattice of every
    8th pixel in x and y (C.11), which the oracle computes ray by ray."""
    import torch
    b = BACKENDS["gpu"]
    cfg = W.get_config(number)
    v = _host_cube(cfg)
    d = torch.from_numpy(v).cuda()
    tf = W.tf_haze(cfg.dims, cfg.step)
    mask = _lattice(cfg, stride)
    sel = mask.astype(bool)
    with vr.Volume(d, cfg.dims, brick=cfg.brick) as vol:
        g = summary(b, vol)
        if summary_exact:
            assert_summary_equal(g, O.minmax_hist(v))
        vmin, vmax = float(g["vmin"]), float(g["vmax"])
        R = max(abs(vmin), abs(vmax))
        _check_statistics_by_definition(statistics(b, vol), v)
        vol.set_transfer_function(tf, vmin, vmax)
        for view in views:
            cam = cfg.camera(view)
            for mode in cfg.modes:
                if mode == "mip":
                    o = O.render(v, cam, O.MIP, brick=cfg.brick if cfg.sort_last else 0, mask=mask)
                    gi = render(b, vol, cam, vr.VR_MIP)
                    s = check_mip(gi[sel], o.image[sel], R)
                else:
                    o = O.render(v, cam, O.EA, tf, vmin, vmax, brick=cfg.brick if cfg.sort_last else 0, mask=mask)
                    gi = render(b, vol, cam, vr.VR_EA)
                    s = check_ea(gi[sel], o.image[sel], o.fragile[sel], (o.K > 0)[sel])
                assert s["bit_exact"] == 1.0, (number, view, mode, s)      # same canonical op sequence
                assert o.n_nominal > 1000
    del d
    torch.cuda.empty_cache()


@pytest.mark.gpu
def test_cfg2_full_size_sampled():
    """cfg2 (512x512x1024, 1024^2, step 0.5, EA + ERT 0.99): a z-travelling, a mixed and an x-travelling orbit view."""
    _full_size_case(2, views=(0, 2, 3))


@pytest.mark.gpu
def test_cfg3_full_size_sampled():
    """cfg3 (1024x1024x2048, 8 GiB; summary pass; 1920x1080 MIP + EA, 128^3 bricks, sort-last compositing)."""
    import torch
    if torch.cuda.get_device_properties(0).total_memory < 24 << 30:
        pytest.skip("needs 24 GB of device memory")
    _full_size_case(3, views=(1,))


@pytest.mark.gpu
def test_cfg4_full_size_sampled():
    """cfg4 (2048x2048x4096, 64 GiB resident + the 64 GiB z-fastest copy; 3840x2160, step 1, EA + ERT): a z-travelling
    and an x-travelling orbit view on the every-16th-pixel lattice (3e4 rays, ~6e7 oracle samples per view)."""
    import torch
    if torch.cuda.get_device_properties(0).total_memory < 150 << 30:
        pytest.skip("needs 150 GB of device memory")
    try:
        with open("/proc/meminfo") as f:
            avail = next(int(ln.split()[1]) * 1024 for ln in f if ln.startswith("MemAvailable:"))
    except Exception:
        avail = 0
    if avail < 80 << 30:
        pytest.skip("needs 80 GB of host memory for the cube the oracle reads")
    _full_size_case(4, views=(5, 12), summary_exact=True, stride=16)


@pytest.mark.gpu
def test_cfg5_scaled_out_of_core():
    """cfg5 at 1/8 linear scale: 512x512x384 brick-major (+1 halo) in pinned host memory as 32^3 bricks — the SAME
    16x16x12 = 3072-brick grid as cfg5 —, 25 % of the cube resident, 4 copy streams, 8 orbit views 480x270, step 0.5,
    EA + ERT 0.99, plus the streamed min/max + histogram and statistics.  Renders on the every-4th-pixel lattice and the
    summary are bit-identical to the oracle reading the same brick-major bytes."""
    import torch
    from dataclasses import replace
    b = BACKENDS["gpu"]
    cfg = W.get_config(5)
    n, B = (512, 512, 384), 32
    rec = replace(cfg.recipe, nx=n[0], ny=n[1], nz=n[2], n_sources=40)
    n_el = W.bricked_halo_elems(n, B)
    host = torch.empty(n_el, dtype=torch.float32, pin_memory=True)
    W.fill_bricked_halo_ptr(rec, B, host.data_ptr())
    hn = host.numpy().reshape(-1, B + 1, B + 1, B + 1)
    o_sum = O.minmax_hist(hn, layout=O.BRICKED_HALO1, layout_brick=B, dims=n)
    tf = W.tf_haze(n, 0.5)
    Wd, H = 480, 270
    mask = np.zeros((H, Wd), dtype=np.uint8)
    mask[2::4, 2::4] = 1
    sel = mask.astype(bool)
    with vr.Volume(host, n, brick=B, layout=vr.VR_BRICKED_HALO1, resident_bytes=n_el * 4 // 4, n_copy_streams=4) as vol:
        assert_summary_equal(summary(b, vol, device=False), o_sum)
        h2d_summary = vol.stats()["h2d_bytes"]
        assert h2d_summary >= n_el * 4                                # pass 1 streams everything, pass 2 the non-resident rest
        g = statistics(b, vol)
        assert int(g["n_finite"]) == n[0] * n[1] * n[2]
        vol.set_transfer_function(tf, float(o_sum.vmin), float(o_sum.vmax))
        for view in range(8):
            cam = W.orbit_camera(n, view, 8, Wd, H, step=0.5, ert_alpha=0.99)
            o = O.render(hn, cam, O.EA, tf, o_sum.vmin, o_sum.vmax, mask=mask, layout=O.BRICKED_HALO1, layout_brick=B, dims=n)
            gi = render(b, vol, cam, vr.VR_EA)
            st = vol.stats()
            assert st["path"] == 3 and st["h2d_bytes"] >= 0.7 * n_el * 4 and st["bricks_drawn"] + st["bricks_culled"] == 3072
            s = check_ea(gi[sel], o.image[sel], o.fragile[sel], (o.K > 0)[sel])
            assert s["bit_exact"] == 1.0, (view, s)
    del host


# ------------------------------------------------------------------ §8(f) #4: the 8-bit frame a thin client displays
def test_encode_rgba8_matches_oracle(be):
    """vr_encode_rgba8 of rendered EA and MIP images (device and pinned-host outputs, a padded output pitch), byte for
    byte against the oracle's C.14; plus a synthetic image with ties, out-of-range values and NaN."""
    n = (40, 36, 52)
    v = W.make_cube(W.Recipe(*n, seed=61, n_sources=3))
    s = O.minmax_hist(v)
    tf = W.tf_opaque(n, 0.5)
    cam = W.orbit_camera(n, 1, 8, 90, 61, step=0.5, ert_alpha=0.99)
    bg = (0.1, 0.25, 0.8)
    with vr.Volume(be.dev(v), n) as vol:
        vol.set_transfer_function(tf, s.vmin, s.vmax)
        ea_buf = be.empty((61, 90, 4)); vol.render(cam, vr.VR_EA, out=ea_buf, stream=be.stream)
        mip_buf = be.empty((61, 90)); vol.render(cam, vr.VR_MIP, out=mip_buf, stream=be.stream)
        ea, mip = be.numpy(ea_buf), be.numpy(mip_buf)
        for device in (True, False):
            out = be.empty((61, 90, 4), np.uint8, device=device)
            vol.encode_rgba8(ea_buf, vr.VR_EA, out, background=bg, stream=be.stream)
            assert np.array_equal(be.numpy(out), O.encode_rgba8(ea, O.EA, background=bg))
            vol.encode_rgba8(mip_buf, vr.VR_MIP, out, vmin=float(s.vmin), vmax=float(s.vmax), stream=be.stream)
            assert np.array_equal(be.numpy(out), O.encode_rgba8(mip, O.MIP, vmin=s.vmin, vmax=s.vmax))
        syn = np.random.default_rng(5).random((33, 47, 4)).astype(np.float32) * 1.4 - 0.2
        syn[0, 0] = (np.nan, np.inf, -np.inf, 0.5); syn[1, :, :3] = 0.5; syn[1, :, 3] = 1.0; syn[2] = 0.0
        sb = be.dev(syn)
        out = be.empty((33, 47, 4), np.uint8)
        vol.encode_rgba8(sb, vr.VR_EA, out, background=(0.5, 0.5, 0.5), stream=be.stream)
        g = be.numpy(out)
        assert np.array_equal(g, O.encode_rgba8(syn, O.EA, background=(0.5, 0.5, 0.5)))
        assert (g[1, :, :3] == 128).all() and (g[2, :, :3] == 128).all() and (g[..., 3] == 255).all()
        with pytest.raises(vr.VrError) as e:
            vol.encode_rgba8(sb, vr.VR_EA, out, background=(0.5, 2.0, 0.5), stream=be.stream)
        assert e.value.status == vr.VR_ERR_INVALID_ARG


# ------------------------------------------------------------------ S24: non-finite voxels in a rendered cube
def test_nonfinite_voxels_render_like_the_oracle(be):
    """FITS blanks: NaN and +-Inf voxels.  A NaN sample classifies as table entry 0 and is ignored by MIP (C.4, C.6,
    S24; pinned for the oracle by P15); every render path must reproduce the oracle bit for bit, NaN for NaN."""
    n = (40, 33, 27)
    v = W.make_cube(W.Recipe(*n, seed=5, n_sources=2)).copy()
    v[0, 0, 0], v[5, 6, 7], v[20, 30, 35], v[13, 1, 2], v[14, 16, 20] = np.nan, np.inf, -np.inf, np.nan, np.nan
    s = O.minmax_hist(v)
    tf = W.tf_opaque(n, 0.5)
    c = np.array(n) / 2
    cams = [W.perspective_camera(c + np.array([0.4, 0.5, 1.7]) * 40, c, (0, 1, 0), 40.0, 70, 50, step=0.5),
            W.perspective_camera(c + np.array([1.8, 0.3, -0.4]) * 40, c, (0, 1, 0), 40.0, 70, 50, step=0.5, ert_alpha=0.99),
            W.ortho_axis_camera(n, 2, +1, step=1.0)]
    for path, brick, flags in ((0, 0, 0), (1, 0, 0), (0, 16, W.cameras.VR_SORT_LAST)):
        with vr.Volume(be.dev(v), n, brick=brick) as vol:
            vol.set_option(vr.VR_OPT_RENDER_PATH, path)
            vol.set_transfer_function(tf, s.vmin, s.vmax)
            for cam in cams:
                if flags and cam.ert_alpha:
                    continue
                cam = cam.with_(flags=flags)
                om = O.render(v, cam, O.MIP, brick=brick if flags else 0)
                oe = O.render(v, cam, O.EA, tf, s.vmin, s.vmax, brick=brick if flags else 0)
                gm = render(be, vol, cam, vr.VR_MIP)
                ge = render(be, vol, cam, vr.VR_EA)
                assert np.array_equal(gm, om.image, equal_nan=True) and np.array_equal(ge, oe.image, equal_nan=True)
                assert not np.isnan(om.image).any()          # MIP never returns NaN (fmaxf drops it)
