"""Seeded random parity: random volume sizes (odd, tiny, long), random perspective / orthographic / mixed cameras
(eyes outside, inside and on faces of the volume, rolled, wide and narrow fields of view, non-square images that are
not multiples of the warp tile), random steps, both modes, ERT on and off, every implementation choice the library
offers (render path, z-fastest copy, lag, empty-space skipping, 16-byte row loads, 64-bit offsets, sort-last with
random brick edges) — each image bit-identical to the oracle.  Runs in the host emulation (no GPU); the same cases run
on the GPU under -m gpu."""
import numpy as np
import pytest

import oracle as O
import paper_1111_6661_b200 as vr
import workload as W
from backends import be, render  # noqa: F401  (be is a fixture)


def _random_case(rng, k):
    n = tuple(int(x) for x in rng.integers(2, 40, size=3))
    if k % 5 == 0:
        n = (int(rng.integers(2, 6)), int(rng.integers(30, 70)), int(rng.integers(2, 30)))
    if k % 7 == 0:
        n = tuple(4 * int(x) for x in rng.integers(2, 12, size=3))          # 16-byte row loads apply on both copies
    c = np.array(n, dtype=np.float64) / 2
    m = float(max(n))
    W_, H_ = int(rng.integers(1, 70)), int(rng.integers(1, 50))
    step = float(rng.choice([0.25, 0.5, 0.7, 1.0, 1.6]))
    kind = k % 4
    direction = rng.normal(size=3)
    direction /= np.linalg.norm(direction)
    up = rng.normal(size=3)
    if kind == 0:       # perspective from outside
        cam = W.perspective_camera(c + direction * m * rng.uniform(1.2, 3.0), c + rng.normal(size=3) * 0.1 * m, up,
                                   float(rng.uniform(15, 80)), W_, H_, step=step)
    elif kind == 1:     # orthographic, oblique
        cam = W.ortho_lookat_camera(c + direction * m * 2.0, c, up, float(rng.uniform(0.8, 2.5)) * m, W_, H_, step=step)
    elif kind == 2:     # eye inside the volume (or exactly on a face)
        eye = rng.uniform(0, 1, size=3) * np.array(n)
        if k % 8 == 2:
            eye[int(rng.integers(0, 3))] = 0.0
        cam = W.perspective_camera(eye, eye + direction, up, float(rng.uniform(40, 100)), W_, H_, step=step)
    else:               # mixed: origins and directions both vary per pixel
        cam = W.perspective_camera(c + direction * m * 2.0, c, up, 35.0, W_, H_, step=step)
        cam = cam.with_(ou=(rng.normal(size=3) * 0.05).astype(np.float32), ov=(rng.normal(size=3) * 0.05).astype(np.float32))
    return n, cam


@pytest.mark.parametrize("seed", range(6))
def test_random_cameras_and_options(be, seed):
    rng = np.random.default_rng(1000 + seed)
    if be.name == "simt":
        import simt_lib
        simt_lib.lib().simt_reset_counters()
    for k in range(8 if be.full else 5):
        n, cam = _random_case(rng, seed * 8 + k)
        v = W.make_cube(W.Recipe(*n, seed=500 + seed * 8 + k, n_sources=int(rng.integers(0, 4))))
        if rng.random() < 0.3:
            v = v.copy(); v.reshape(-1)[int(rng.integers(0, v.size))] = np.nan
        s = O.minmax_hist(v)
        tf = [W.tf_opaque(n, cam.step), W.tf_haze(n, cam.step), W.tf_sources(n, cam.step, alpha_scale=10.0)][int(rng.integers(0, 3))]
        ert = float(rng.choice([0.0, 0.9, 0.99]))
        opts = dict(path=int(rng.random() < 0.15), zcopy=int(rng.random() < 0.8), lag=int(rng.choice([0, 1, 1, 3])),
                    skip=int(rng.random() < 0.8), quad=int(rng.random() < 0.5), wide=int(rng.random() < 0.3))
        B = int(rng.choice([0, 3, 8, 16, 50]))
        with vr.Volume(be.dev(v), n, brick=B) as vol:
            vol.set_option(vr.VR_OPT_RENDER_PATH, opts["path"]); vol.set_option(vr.VR_OPT_ZFAST_COPY, opts["zcopy"])
            vol.set_option(vr.VR_OPT_LANE_LAG, opts["lag"]); vol.set_option(vr.VR_OPT_EMPTY_SKIP, opts["skip"])
            vol.set_option(vr.VR_OPT_ROW_LOADS, opts["quad"]); vol.set_option(vr.VR_OPT_FORCE_WIDE, opts["wide"])
            vol.set_transfer_function(tf, s.vmin, s.vmax)
            tag = (seed, k, n, opts, B, ert, cam.width, cam.height, cam.step)
            c2 = cam.with_(ert_alpha=ert)
            oe = O.render(v, c2, O.EA, tf, s.vmin, s.vmax)
            assert np.array_equal(render(be, vol, c2, vr.VR_EA), oe.image, equal_nan=True), ("EA",) + tag
            om = O.render(v, cam, O.MIP)
            assert np.array_equal(render(be, vol, cam, vr.VR_MIP), om.image), ("MIP",) + tag
            if B and (cam.is_perspective or cam.is_orthographic):
                sl = cam.with_(flags=W.cameras.VR_SORT_LAST)
                ob = O.render(v, sl, O.EA, tf, s.vmin, s.vmax, brick=B)
                assert ob.n_order_mismatch == 0 and ob.n_noncontig == 0, ("order",) + tag
                assert np.array_equal(render(be, vol, sl, vr.VR_EA), ob.image, equal_nan=True), ("sort-last EA",) + tag
                obm = O.render(v, sl, O.MIP, brick=B)
                assert np.array_equal(render(be, vol, sl, vr.VR_MIP), obm.image), ("sort-last MIP",) + tag
    if be.name == "simt":                # sort-last: every fragment inside its rectangle, every owner brick in the plan
        assert simt_lib.lib().simt_counter(4) == 0 and simt_lib.lib().simt_counter(5) == 0


@pytest.mark.parametrize("seed", range(4))
def test_random_summaries_and_statistics(be, seed):
    """Random sizes, bin counts, caller ranges, layouts (linear, brick-major with halo on the device, out of core with a
    random pool size and stream count), planted non-finite voxels: counts, min / max and the median bit-exact, the
    float64 moments within 1e-13 of the data scale."""
    from backends import statistics, summary
    from test_parity import assert_statistics_equal, assert_summary_equal
    rng = np.random.default_rng(2000 + seed)
    for k in range(5):
        n = tuple(int(x) for x in rng.integers(2, 48, size=3))
        v = W.make_cube(W.Recipe(*n, seed=700 + seed * 8 + k, n_sources=int(rng.integers(0, 3)))).copy()
        for _ in range(int(rng.integers(0, 4))):
            v.reshape(-1)[int(rng.integers(0, v.size))] = rng.choice([np.nan, np.inf, -np.inf])
        nbins = int(rng.choice([1, 7, 256, 1000, 4096]))
        rng_arg = None if rng.random() < 0.5 else tuple(sorted(float(x) for x in rng.normal(size=2) * 2))
        layout = int(rng.integers(0, 3))
        B = int(rng.choice([4, 9, 16]))
        kw = {}
        if layout == 0:
            data, lay = be.dev(v), vr.VR_LINEAR
        else:
            t = W.retile_halo(v, B)
            lay = vr.VR_BRICKED_HALO1
            if layout == 1:
                data = be.dev(t)
            else:
                data = be.pinned(t)
                n_bricks = int(np.prod([(d + B - 1) // B for d in n]))
                if n_bricks > 2:
                    kw = dict(resident_bytes=int(rng.integers(2, n_bricks)) * (B + 1) ** 3 * 4, n_copy_streams=int(rng.integers(1, 5)))
        with vr.Volume(data, n, brick=B if layout else 0, layout=lay, **kw) as vol:
            o = O.minmax_hist(v, nbins, rng_arg)
            assert_summary_equal(summary(be, vol, nbins, rng_arg), o)
            assert_statistics_equal(statistics(be, vol), O.statistics(v), v)


@pytest.mark.parametrize("seed", range(4))
def test_random_chain_renders(be, seed):
    """Brick-major volumes (resident and out of core, random brick edge, pool size and stream count) rendered brick by
    brick with the ray state carried in the image, with and without the brick ranges of a prior summary pass (empty
    bricks dropped), random pure perspective / orthographic cameras: bit-identical to the oracle's single march."""
    from backends import summary
    rng = np.random.default_rng(3000 + seed)
    for k in range(4):
        n, cam = _random_case(rng, 4 * (seed * 4 + k) + int(rng.integers(0, 3)))     # kinds 0, 1, 2: never mixed
        if not (cam.is_perspective or cam.is_orthographic):
            continue
        B = int(rng.choice([3, 8, 16]))
        v = W.make_cube(W.Recipe(*n, seed=900 + seed * 4 + k, n_sources=int(rng.integers(0, 3))))
        s = O.minmax_hist(v)
        tf = [W.tf_opaque(n, cam.step), W.tf_sources(n, cam.step, alpha_scale=10.0)][int(rng.integers(0, 2))]
        t = W.retile_halo(v, B)
        n_bricks = int(np.prod([(d + B - 1) // B for d in n]))
        kw = {}
        if rng.random() < 0.6 and n_bricks > 2:
            data = be.pinned(t)
            kw = dict(resident_bytes=int(rng.integers(2, n_bricks)) * (B + 1) ** 3 * 4, n_copy_streams=int(rng.integers(1, 5)))
        else:
            data = be.dev(t)
        ert = float(rng.choice([0.0, 0.99]))
        with vr.Volume(data, n, brick=B, layout=vr.VR_BRICKED_HALO1, **kw) as vol:
            vol.set_transfer_function(tf, s.vmin, s.vmax)
            if rng.random() < 0.6:
                summary(be, vol)                                     # gathers the brick ranges: empty bricks get dropped
            c2 = cam.with_(ert_alpha=ert)
            oe = O.render(v, c2, O.EA, tf, s.vmin, s.vmax)
            assert np.array_equal(render(be, vol, c2, vr.VR_EA), oe.image, equal_nan=True), (seed, k, n, B, kw, ert)
            assert vol.stats()["path"] == 3
            om = O.render(v, cam, O.MIP)
            assert np.array_equal(render(be, vol, cam, vr.VR_MIP), om.image), (seed, k, n, B, kw)
