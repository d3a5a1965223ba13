"""GPU parity: the CUDA path (through the C ABI) against the CPU oracle, element by element,
on the same seeded inputs.  Bit-exact for min/max and counts, MIP <= 1e-6 scale-relative,
EA <= 1e-4 absolute per channel (north_star)."""
import numpy as np
import pytest
import torch

import oracle as O
import paper_1111_6661_b200 as vr
import workload as W
from parity import check_ea, check_mip

pytestmark = pytest.mark.gpu


def dev(a):
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def pinned(a):
    t = torch.from_numpy(np.ascontiguousarray(a)).pin_memory()
    return t


def gpu_summary(vol, nbins=256, range_=None):
    buf = vol.minmax_histogram(nbins, range_)
    return vr.Volume.read_summary(buf, nbins)


def assert_summary_equal(g, o):
    assert g["vmin"] == o.vmin and g["vmax"] == o.vmax, (g["vmin"], o.vmin, g["vmax"], o.vmax)
    assert int(g["n_nonfinite"]) == o.n_nonfinite and int(g["n_below"]) == o.n_below and int(g["n_above"]) == o.n_above
    assert np.array_equal(g["counts"], o.counts)


# ------------------------------------------------------------------ A1 / A2
@pytest.mark.parametrize("dims", [(128, 128, 128), (37, 29, 41), (130, 67, 3), (2, 2, 2)])
def test_minmax_hist_bit_exact(dims):
    nx, ny, nz = dims
    v = W.make_cube(W.Recipe(nx, ny, nz, seed=21, n_sources=4 if nx > 8 else 0))
    # the flat kernel needs a 16-byte aligned base: torch allocations are
    with vr.Volume(dev(v), dims) as vol:
        assert_summary_equal(gpu_summary(vol), O.minmax_hist(v))
        assert_summary_equal(gpu_summary(vol, 64, (-1.0, 1.5)), O.minmax_hist(v, 64, (-1.0, 1.5)))
        assert_summary_equal(gpu_summary(vol, 1000), O.minmax_hist(v, 1000))
        assert_summary_equal(gpu_summary(vol, 4096, (0.0, 0.0)), O.minmax_hist(v, 4096, (0.0, 0.0)))


def test_minmax_hist_nonfinite_and_constant():
    v = W.make_cube(W.Recipe(40, 33, 27, seed=5)).copy()
    v[0, 0, 0], v[5, 6, 7], v[26, 32, 39], v[13, 1, 2] = np.nan, np.inf, -np.inf, np.nan
    with vr.Volume(dev(v), (40, 33, 27)) as vol:
        g, o = gpu_summary(vol), O.minmax_hist(v)
        assert_summary_equal(g, o)
        assert int(g["counts"].sum() + g["n_below"] + g["n_above"] + g["n_nonfinite"]) == v.size
    c = np.full((9, 10, 11), 3.5, dtype=np.float32)
    with vr.Volume(dev(c), (11, 10, 9)) as vol:
        assert_summary_equal(gpu_summary(vol), O.minmax_hist(c))
    k = (np.arange(8 * 16 * 32) % 256).astype(np.float32).reshape(8, 16, 32)
    with vr.Volume(dev(k), (32, 16, 8)) as vol:
        g = gpu_summary(vol)
        assert np.all(g["counts"] == k.size // 256)


# ------------------------------------------------------------------ cfg1 (full size): A3, A6-A9
def test_cfg1_full():
    cfg = W.get_config(1)
    v = W.make_cube(cfg.recipe)
    cam = cfg.camera()
    o_sum = O.minmax_hist(v)
    tf = W.tf_haze(cfg.dims, cfg.step)
    with vr.Volume(dev(v), cfg.dims) as vol:
        g = gpu_summary(vol)
        assert_summary_equal(g, o_sum)
        vol.set_transfer_function(tf, float(g["vmin"]), float(g["vmax"]))
        mip = vol.render(cam, vr.VR_MIP).cpu().numpy()
        ea = vol.render(cam, vr.VR_EA).cpu().numpy()
        ea2 = vol.render(cam, vr.VR_EA).cpu().numpy()
        st = vol.stats()
        vol.set_option(vr.VR_OPT_RENDER_PATH, vr.VR_PATH_RAY_MAJOR)
        mip_r = vol.render(cam, vr.VR_MIP).cpu().numpy()
        ea_r = vol.render(cam, vr.VR_EA).cpu().numpy()
        st_r = vol.stats()
    R = float(max(abs(o_sum.vmin), abs(o_sum.vmax)))
    om = O.render(v, cam, O.MIP)
    oe = O.render(v, cam, O.EA, tf, o_sum.vmin, o_sum.vmax)
    sm = check_mip(mip, om.image, R)
    se = check_ea(ea, oe.image)
    assert sm["bit_exact"] == 1.0 and se["bit_exact"] == 1.0        # same canonical op sequence
    assert np.array_equal(ea, ea2)                                   # run-to-run determinism
    assert st["path"] == 6 and st["kernel_launches"] == 1           # auto = sheared-plane beams for a pure ortho camera
    assert st["beam_overflow"] == 0
    assert st_r["path"] == 1 and st_r["kernel_launches"] == 1
    assert check_mip(mip_r, om.image, R)["bit_exact"] == 1.0 and check_ea(ea_r, oe.image)["bit_exact"] == 1.0


def _views(n):
    c = np.array(n) / 2
    yield "persp", W.perspective_camera(c + np.array([1.9, 0.8, 1.5]) * max(n), c, (0, 1, 0), 40.0, 97, 61, step=0.5)
    yield "ortho", W.ortho_lookat_camera(c + np.array([-1.7, 0.6, 1.1]) * max(n), c, (0, 1, 0), 1.6 * max(n), 80, 50, step=0.7)
    yield "inside", W.perspective_camera((16.3, 7.25, 32.45), (30, 40, 10), (0, 0, 1), 70.0, 64, 48, step=0.5)
    yield "axis", W.ortho_axis_camera(n, 0, -1, step=1.0)


# path 1 = ray-major through global memory; path 2 = tile-wave with each staging-tile shape; path 3 = beam-slab
# (nx = 61 is not a multiple of 4, so the beam path runs its plain-load fallback here; the TMA loader is
# covered by test_beam_views); path 4 = sheared-plane beams (the default)
_PATH_ID = {0: 6, 1: 1, 2: 4, 3: 5, 4: 6}


@pytest.mark.parametrize("path,tile", [(0, 0), (1, 0), (2, 1), (2, 2), (2, 3), (2, 4), (3, 0), (4, 0)])
@pytest.mark.parametrize("ert", [0.0, 0.99])
def test_single_march_views(ert, path, tile):
    n = (61, 47, 83)
    v = W.make_cube(W.Recipe(*n, seed=31, n_sources=5))
    s = O.minmax_hist(v)
    R = float(max(abs(s.vmin), abs(s.vmax)))
    tf = W.tf_opaque(n, 0.5) if ert else W.tf_haze(n, 0.5)
    with vr.Volume(dev(v), n) as vol:
        vol.set_option(vr.VR_OPT_RENDER_PATH, path)
        vol.set_option(vr.VR_OPT_TILE_SHAPE, tile)
        vol.set_transfer_function(tf, s.vmin, s.vmax)
        for name, cam in _views(n):
            cam = cam.with_(ert_alpha=ert)
            om = O.render(v, cam, O.MIP)
            sm = check_mip(vol.render(cam, vr.VR_MIP).cpu().numpy(), om.image, R)
            assert vol.stats()["path"] == _PATH_ID[path]
            oe = O.render(v, cam, O.EA, tf, s.vmin, s.vmax)
            se = check_ea(vol.render(cam, vr.VR_EA).cpu().numpy(), oe.image, oe.fragile, oe.K > 0, max_fragile_frac=0.05)
            assert sm["bit_exact"] == 1.0 and se["bit_exact"] == 1.0, (name, sm, se)   # same canonical op sequence
            if ert:
                assert (oe.K_ert < oe.K).sum() > 20, name          # ERT really fires in this workload


@pytest.mark.parametrize("tile", [1, 2, 4])
def test_tile_wave_many_tiles_ragged(tile):
    """Several tiles per axis with a ragged last tile (n-1 not a multiple of the tile edge), eye outside on a
    diagonal and eye inside the volume, ERT on an opaque TF: the wave order must reproduce the k order."""
    n = (131, 70, 98)
    v = W.make_cube(W.Recipe(*n, seed=77, n_sources=12))
    s = O.minmax_hist(v)
    R = float(max(abs(s.vmin), abs(s.vmax)))
    tf = W.tf_opaque(n, 0.5)
    c = np.array(n) / 2
    cams = [W.perspective_camera(c + np.array([1.1, 0.9, -1.3]) * max(n), c, (0, 1, 0), 35.0, 160, 120, step=0.5),
            W.perspective_camera((65.5, 33.2, 40.7), (0, 10, 98), (0, 1, 0), 80.0, 128, 96, step=0.5),
            W.ortho_lookat_camera(c + np.array([0.7, -1.2, 0.4]) * max(n), c, (0, 0, 1), 1.3 * max(n), 120, 90, step=0.75)]
    with vr.Volume(dev(v), n) as vol:
        vol.set_option(vr.VR_OPT_RENDER_PATH, vr.VR_PATH_TILE_WAVE)
        vol.set_option(vr.VR_OPT_TILE_SHAPE, tile)
        vol.set_transfer_function(tf, s.vmin, s.vmax)
        for cam in cams:
            for ert in (0.0, 0.99):
                cam2 = cam.with_(ert_alpha=ert)
                oe = O.render(v, cam2, O.EA, tf, s.vmin, s.vmax)
                se = check_ea(vol.render(cam2, vr.VR_EA).cpu().numpy(), oe.image, oe.fragile, oe.K > 0, max_fragile_frac=0.05)
                assert se["bit_exact"] == 1.0 and vol.stats()["path"] == 4, se
            om = O.render(v, cam, O.MIP)
            assert check_mip(vol.render(cam, vr.VR_MIP).cpu().numpy(), om.image, R)["bit_exact"] == 1.0


def _axis_views(n):
    """Views whose beams travel along +-x, +-y, +-z (all three principal-axis classes, both directions), oblique
    ones that mix classes across the image, a wide-angle one from inside, and image sizes that are not
    multiples of the 16x16 beam."""
    c = np.array(n, dtype=np.float64) / 2
    m = float(max(n))
    for k, e in enumerate([(1.6, 0.25, 0.3), (-1.5, -0.2, 0.35), (0.3, 1.7, 0.2), (0.25, -1.6, -0.3),
                           (0.3, 0.2, 1.8), (-0.2, 0.35, -1.7), (1.2, 1.1, 1.3), (-1.0, 1.2, -1.1)]):
        up = (0, 0, 1) if abs(e[1]) > 1 else (0, 1, 0)
        yield f"persp{k}", W.perspective_camera(c + np.array(e) * m, c, up, 42.0, 150, 105, step=0.5)
    yield "ortho_x", W.ortho_lookat_camera(c + np.array([1.7, 0.4, -0.5]) * m, c, (0, 1, 0), 1.5 * m, 90, 70, step=0.75)
    yield "ortho_z", W.ortho_lookat_camera(c + np.array([-0.3, 0.5, 1.9]) * m, c, (0, 1, 0), 1.5 * m, 100, 60, step=0.6)
    yield "inside", W.perspective_camera(c + np.array([0.11, -0.07, 0.2]) * m, c + np.array([0.5, 0.4, -0.3]) * m,
                                         (0, 1, 0), 75.0, 176, 128, step=0.5)
    yield "axis_z", W.ortho_axis_camera(n, 2, +1, step=0.5, width=2 * n[0], height=2 * n[1])
    yield "axis_x", W.ortho_axis_camera(n, 0, -1, step=1.0)


@pytest.mark.parametrize("path", [3, 4])
@pytest.mark.parametrize("n", [(132, 72, 100), (64, 200, 40), (61, 47, 83)])
def test_beam_views(n, path):
    """Both beam paths (3: TMA slab boxes when nx % 4 == 0, else its plain loader; 4: sheared planes by
    cp.async) over views travelling along +-x, +-y, +-z: EA with and without ERT and MIP, bit-identical to the
    oracle's single march (same canonical op sequence), no slab-box overflow."""
    v = W.make_cube(W.Recipe(*n, seed=91, n_sources=14))
    s = O.minmax_hist(v)
    R = float(max(abs(s.vmin), abs(s.vmax)))
    tf = W.tf_opaque(n, 0.5)
    with vr.Volume(dev(v), n) as vol:
        vol.set_option(vr.VR_OPT_RENDER_PATH, path)
        vol.set_transfer_function(tf, s.vmin, s.vmax)
        for name, cam in _axis_views(n):
            for ert in (0.0, 0.99):
                cam2 = cam.with_(ert_alpha=ert)
                oe = O.render(v, cam2, O.EA, tf, s.vmin, s.vmax)
                se = check_ea(vol.render(cam2, vr.VR_EA).cpu().numpy(), oe.image, oe.fragile, oe.K > 0, max_fragile_frac=0.05)
                st = vol.stats()
                assert st["path"] == _PATH_ID[path] and st["beam_overflow"] == 0, (name, st)
                assert se["bit_exact"] == 1.0, (name, ert, se)
            om = O.render(v, cam, O.MIP)
            assert check_mip(vol.render(cam, vr.VR_MIP).cpu().numpy(), om.image, R)["bit_exact"] == 1.0, name


def test_beam_slab_falls_back_for_mixed_camera():
    """A camera whose origins AND directions vary per pixel is outside the beam path: auto must use ray-major."""
    n = (32, 32, 32)
    v = W.make_cube(W.Recipe(*n, seed=3))
    cam = W.perspective_camera((80.0, 20.0, 16.0), (16, 16, 16), (0, 1, 0), 30.0, 40, 30)
    cam = cam.with_(ou=np.array([0.01, 0, 0], dtype=np.float32))
    with vr.Volume(dev(v), n) as vol:
        g = vol.render(cam, vr.VR_MIP).cpu().numpy()
        assert vol.stats()["path"] == 1
    assert np.array_equal(g, O.render(v, cam, O.MIP).image)


def test_set_option_rejects_bad_values():
    v = W.make_cube(W.Recipe(16, 16, 16, seed=1))
    with vr.Volume(dev(v), (16, 16, 16)) as vol:
        for opt, val in ((vr.VR_OPT_RENDER_PATH, 5), (vr.VR_OPT_TILE_SHAPE, 9), (77, 0)):
            with pytest.raises(vr.VrError) as e:
                vol.set_option(opt, val)
            assert e.value.status == vr.VR_ERR_INVALID_ARG


def test_all_miss_camera_and_eye_inside():
    n = (20, 24, 28)
    v = W.make_cube(W.Recipe(*n, seed=2))
    cam = W.perspective_camera((100.0, 100.0, 100.0), (200, 200, 200), (0, 1, 0), 20.0, 33, 17)
    with vr.Volume(dev(v), n) as vol:
        vol.set_transfer_function(W.tf_haze(n, 0.5), -5.0, 5.0)
        assert torch.isneginf(vol.render(cam, vr.VR_MIP)).all()
        assert (vol.render(cam, vr.VR_EA) == 0).all()


# ------------------------------------------------------------------ bricks: A0, A4, A10
@pytest.mark.parametrize("B", [7, 16, 32, 100])
def test_sort_last_equals_oracle_bricked(B):
    n = (61, 47, 83)
    v = W.make_cube(W.Recipe(*n, seed=33, n_sources=5))
    s = O.minmax_hist(v)
    R = float(max(abs(s.vmin), abs(s.vmax)))
    tf = W.bake_tf(W.TF_HAZE_POINTS, 0.5, alpha_scale=6.0)
    with vr.Volume(dev(v), n, brick=B) as vol:
        vol.set_transfer_function(tf, s.vmin, s.vmax)
        for name, cam in _views(n):
            cam = cam.with_(flags=W.cameras.VR_SORT_LAST)
            om = O.render(v, cam, O.MIP, brick=B)
            assert om.n_noncontig == 0 and om.n_order_mismatch == 0
            sm = check_mip(vol.render(cam, vr.VR_MIP).cpu().numpy(), om.image, R)
            assert sm["bit_exact"] == 1.0, name
            oe = O.render(v, cam, O.EA, tf, s.vmin, s.vmax, brick=B)
            se = check_ea(vol.render(cam, vr.VR_EA).cpu().numpy(), oe.image)
            assert se["bit_exact"] == 1.0, (name, se)                # same partials, same fold order
            st = vol.stats()
            assert st["path"] == 2 and st["fragments"] > 0


def test_sort_last_rejections():
    n = (16, 16, 16)
    v = W.make_cube(W.Recipe(*n, seed=1))
    cam = W.ortho_axis_camera(n, 2, +1).with_(flags=W.cameras.VR_SORT_LAST)
    with vr.Volume(dev(v), n, brick=0) as vol:
        with pytest.raises(vr.VrError) as e:
            vol.render(cam, vr.VR_MIP)
        assert e.value.status == vr.VR_ERR_UNSUPPORTED
    with vr.Volume(dev(v), n, brick=8) as vol:
        with pytest.raises(vr.VrError) as e:
            vol.render(cam, vr.VR_EA)
        assert e.value.status == vr.VR_ERR_NOT_READY
        vol.set_transfer_function(W.tf_haze(n, 0.5), -1.0, 1.0)
        with pytest.raises(vr.VrError) as e:
            vol.render(cam.with_(ert_alpha=0.99), vr.VR_EA)
        assert e.value.status == vr.VR_ERR_UNSUPPORTED


# ------------------------------------------------------------------ bricked-halo layout, chain, out-of-core: A5
@pytest.mark.parametrize("where", ["device", "host_resident", "host_ooc"])
def test_bricked_halo_chain_and_streaming(where):
    n = (61, 47, 83)
    B = 16
    v = W.make_cube(W.Recipe(*n, seed=35, n_sources=5))
    t = W.retile_halo(v, B)
    s = O.minmax_hist(v)
    R = float(max(abs(s.vmin), abs(s.vmax)))
    tf = W.tf_opaque(n, 0.5)
    brick_bytes = (B + 1) ** 3 * 4
    kw = {}
    data = dev(t) if where == "device" else pinned(t)
    if where == "host_ooc":
        kw = dict(resident_bytes=11 * brick_bytes, n_copy_streams=4)     # 11 of 72 bricks fit
    with vr.Volume(data, n, brick=B, layout=vr.VR_BRICKED_HALO1, **kw) as vol:
        assert_summary_equal(gpu_summary(vol), s)
        assert_summary_equal(gpu_summary(vol, 100, (-0.5, 2.0)), O.minmax_hist(v, 100, (-0.5, 2.0)))
        vol.set_transfer_function(tf, s.vmin, s.vmax)
        for name, cam in _views(n):
            for ert in (0.0, 0.99):
                cam2 = cam.with_(ert_alpha=ert)
                om = O.render(v, cam2, O.MIP)
                sm = check_mip(vol.render(cam2, vr.VR_MIP).cpu().numpy(), om.image, R)
                assert sm["bit_exact"] == 1.0, name
                oe = O.render(v, cam2, O.EA, tf, s.vmin, s.vmax)
                se = check_ea(vol.render(cam2, vr.VR_EA).cpu().numpy(), oe.image, oe.fragile, oe.K > 0, max_fragile_frac=0.05)
                assert se["bit_exact"] == 1.0, (name, ert, se)           # chained state == single march
        st = vol.stats()
        assert st["path"] == 3
        if where == "host_ooc":
            assert st["h2d_bytes"] > 0 and st["resident_bytes"] == 11 * brick_bytes


def test_host_linear_mirror_and_host_outputs():
    n = (40, 36, 52)
    v = W.make_cube(W.Recipe(*n, seed=37, n_sources=3))
    s = O.minmax_hist(v)
    tf = W.tf_haze(n, 0.5)
    cam = W.orbit_camera(n, 1, 8, 96, 64, step=0.5, ert_alpha=0.99)
    with vr.Volume(pinned(v), n, brick=16) as vol:
        hbuf = torch.empty(32 + 8 * 256, dtype=torch.uint8).pin_memory()
        vol.minmax_histogram(256, None, out=hbuf)
        torch.cuda.synchronize()
        assert_summary_equal(vr.Volume.read_summary(hbuf), s)
        assert vol.stats()["h2d_bytes"] == v.nbytes
        vol.set_transfer_function(tf, s.vmin, s.vmax)
        out = torch.empty((64, 96, 4), dtype=torch.float32).pin_memory()
        vol.render(cam, vr.VR_EA, out=out)
        torch.cuda.synchronize()
        oe = O.render(v, cam, O.EA, tf, s.vmin, s.vmax)
        check_ea(out.numpy(), oe.image, oe.fragile, oe.K > 0, max_fragile_frac=0.05)
        assert vol.stats()["d2h_bytes"] == out.numel() * 4
        assert vol.stats()["h2d_bytes"] < 4096                           # per-frame tables only; the cube is not re-uploaded


def test_pageable_host_memory_is_rejected():
    v = W.make_cube(W.Recipe(16, 16, 16, seed=1))
    t = torch.from_numpy(v)                  # pageable
    if (t.data_ptr() & 15) != 0:
        pytest.skip("unaligned numpy buffer")
    with pytest.raises(vr.VrError) as e:
        vr.Volume(t, (16, 16, 16))
    assert e.value.status == vr.VR_ERR_INVALID_ARG


def test_two_handles_two_streams_and_pitch():
    n = (32, 32, 32)
    a = W.make_cube(W.Recipe(*n, seed=41))
    b = W.make_cube(W.Recipe(*n, seed=42))
    cam = W.orbit_camera(n, 0, 4, 70, 50, step=0.5)
    s1, s2 = torch.cuda.Stream(), torch.cuda.Stream()
    with vr.Volume(dev(a), n) as va, vr.Volume(dev(b), n) as vb:
        big = torch.zeros((50, 96), dtype=torch.float32, device="cuda")
        torch.cuda.synchronize()
        with torch.cuda.stream(s1):
            ia = va.render(cam, vr.VR_MIP, out=big[:, :70], stream=s1)
        with torch.cuda.stream(s2):
            ib = vb.render(cam, vr.VR_MIP, stream=s2)
        torch.cuda.synchronize()
        assert np.array_equal(ia.cpu().numpy(), O.render(a, cam, O.MIP).image)
        assert np.array_equal(ib.cpu().numpy(), O.render(b, cam, O.MIP).image)
        assert (big[:, 70:] == 0).all()


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


def _full_size_case(number, views, summary_exact=True):
    """vr_minmax_histogram on the whole cube (bit-exact) and vr_render of `views` at the config's own image
    size, step, ERT and flags — the launches bench.py times — compared with the oracle on a lattice of every
    8th pixel in x and y (C.11), which the oracle computes ray by ray."""
    cfg = W.get_config(number)
    v = _host_cube(cfg)
    d = torch.from_numpy(v).cuda()
    tf = W.tf_haze(cfg.dims, cfg.step)
    mask = _lattice(cfg)
    sel = mask.astype(bool)
    with vr.Volume(d, cfg.dims, brick=cfg.brick) as vol:
        g = gpu_summary(vol)
        if summary_exact:
            assert_summary_equal(g, O.minmax_hist(v))
        vmin, vmax = float(g["vmin"]), float(g["vmax"])
        R = max(abs(vmin), abs(vmax))
        vol.set_transfer_function(tf, vmin, vmax)
        for view in views:
            cam = cfg.camera(view)
            for mode in cfg.modes:
                if mode == "mip":
                    o = O.render(v, cam, O.MIP, brick=cfg.brick if cfg.sort_last else 0, mask=mask)
                    gi = vol.render(cam, vr.VR_MIP).cpu().numpy()
                    s = check_mip(gi[sel], o.image[sel], R)
                else:
                    o = O.render(v, cam, O.EA, tf, vmin, vmax, brick=cfg.brick if cfg.sort_last else 0, mask=mask)
                    gi = vol.render(cam, vr.VR_EA).cpu().numpy()
                    s = check_ea(gi[sel], o.image[sel], o.fragile[sel], (o.K > 0)[sel])
                st = vol.stats()
                assert st["beam_overflow"] == 0
                assert s["bit_exact"] == 1.0, (number, view, mode, s)      # same canonical op sequence
                assert o.n_nominal > 1000
    del d
    torch.cuda.empty_cache()


def test_cfg2_full_size_sampled():
    """cfg2 (512x512x1024, 1024^2, step 0.5, EA + ERT 0.99): a z-class, a mixed and an x-class orbit view."""
    _full_size_case(2, views=(0, 2, 3))


def test_cfg3_full_size_sampled():
    """cfg3 (1024x1024x2048, 8 GiB; summary pass; 1920x1080 MIP + EA, 128^3 bricks, sort-last compositing)."""
    if torch.cuda.get_device_properties(0).total_memory < 24 << 30:
        pytest.skip("needs 24 GB of device memory")
    _full_size_case(3, views=(1,))


@pytest.mark.skipif(not __import__("os").environ.get("VR_TEST_BIG"), reason="64 GiB cube: set VR_TEST_BIG=1 (takes minutes)")
def test_cfg4_full_size_sampled():
    """cfg4 (2048x2048x4096, 64 GiB resident; 3840x2160, step 1, EA + ERT): one orbit view on the pixel lattice."""
    _full_size_case(4, views=(5,), summary_exact=True)


def test_sparse_direct_option_same_results():
    """VR_OPT_SPARSE_DIRECT (experimental): sparse views (several voxels per pixel) of classes 1 and 2 read through
    L1 instead of staging planes — same canonical arithmetic, so bit-identical images."""
    n = (96, 80, 112)
    v = W.make_cube(W.Recipe(*n, seed=57, n_sources=6))
    s = O.minmax_hist(v)
    tf = W.tf_opaque(n, 1.0)
    c = np.array(n, dtype=np.float64) / 2
    cams = [W.perspective_camera(c + np.array(e) * 140.0, c, up, 50.0, 40, 28, step=1.0, ert_alpha=0.99)
            for e, up in (((0.2, 0.3, 1.7), (0, 1, 0)), ((0.3, 1.6, 0.2), (0, 0, 1)), ((1.7, 0.2, 0.3), (0, 1, 0)))]
    with vr.Volume(dev(v), n) as vol:
        vol.set_option(vr.VR_OPT_SPARSE_DIRECT, 1)
        vol.set_transfer_function(tf, s.vmin, s.vmax)
        for cam in cams:
            oe = O.render(v, cam, O.EA, tf, s.vmin, s.vmax)
            se = check_ea(vol.render(cam, vr.VR_EA).cpu().numpy(), oe.image, oe.fragile, oe.K > 0, max_fragile_frac=0.05)
            assert se["bit_exact"] == 1.0 and vol.stats()["path"] == 6 and vol.stats()["beam_overflow"] == 0
            om = O.render(v, cam, O.MIP)
            assert np.array_equal(vol.render(cam, vr.VR_MIP).cpu().numpy(), om.image)
