"""Pins P1-P14: the oracle against closed forms, invariants, library
routines and brute force — never against itself and never against the CUDA path.

The paper prints no worked example (PAPER.md has no equations or numeric fixtures), so every
pin is a mathematical one; each is chosen so that a plausible mistake (dropped term, wrong
sign or index, transposed axis, off-by-half lattice) fails at least one of them.
"""
import math

import numpy as np
import pytest

import oracle as O
import workload as W

RNG = np.random.default_rng(20241104)


def noise_cube(nx, ny, nz, seed=11):
    return W.make_cube(W.Recipe(nx, ny, nz, seed=seed))


KS = 255.0 / 256.0


def ramp_alpha_tf(amax=0.5):
    """Entries i/256-based so every entry is exact in float32 and the table lerp IS the line:
    rgb(u) = (KS*u, 1-KS*u, 0.25), alpha(u) = amax*KS*u   (amax a power of two)."""
    w = np.arange(256, dtype=np.float64) / 256.0
    t = np.stack([w, 1 - w, np.full_like(w, 0.25), amax * w], axis=1)
    assert np.array_equal(t.astype(np.float32).astype(np.float64), t)
    return t.astype(np.float32)


def const_tf(rgba):
    return np.tile(np.asarray(rgba, dtype=np.float32), (256, 1))


# --------------------------------------------------------------------------- P1 / P10
@pytest.mark.parametrize("axis", [0, 1, 2])
@pytest.mark.parametrize("sign", [+1, -1])
def test_p1_axis_aligned_ortho_mip_is_column_max(axis, sign):
    v = noise_cube(13, 9, 17)                       # shape (nz, ny, nx)
    cam = W.ortho_axis_camera((13, 9, 17), axis, sign, step=1.0)
    r = O.render(v, cam, O.MIP)
    want = v.max(axis={0: 2, 1: 1, 2: 0}[axis])     # image[j, i]: i <-> u axis, j <-> v axis
    assert r.image.shape == want.shape
    assert np.array_equal(r.image, want)            # bit-exact, incl. the last voxel (i0=n-2, f=1)
    assert np.all(r.K == (13, 9, 17)[axis])
    r64 = O.render(v, cam, O.MIP, precision=O.F64)
    assert np.array_equal(r64.image, want)


def test_p1_argmax_location_distinguishes_axes():
    v = np.zeros((6, 5, 4), dtype=np.float32)       # nz=6, ny=5, nx=4
    v[4, 1, 2] = 7.0                                # z=4, y=1, x=2
    img = O.render(v, W.ortho_axis_camera((4, 5, 6), 2, +1, step=1.0), O.MIP).image
    assert img.shape == (5, 4) and img[1, 2] == 7.0 and (img > 0).sum() == 1
    img = O.render(v, W.ortho_axis_camera((4, 5, 6), 0, +1, step=1.0), O.MIP).image
    assert img.shape == (6, 5) and img[4, 1] == 7.0 and (img > 0).sum() == 1


# --------------------------------------------------------------------------- P2
@pytest.mark.parametrize("step", [1.0, 0.5, 0.25])
@pytest.mark.parametrize("prec,tol", [(O.F32, 1e-5), (O.F64, 1e-12)])
def test_p2_constant_cube_axis_aligned(step, prec, tol):
    n = (16, 12, 20)
    v = np.full((20, 12, 16), 0.6, dtype=np.float32)
    tf = ramp_alpha_tf(0.5)
    vmin, vmax = 0.0, 1.0
    u = float(np.float32(0.6))                      # the stored voxel value
    a, rgb = 0.5 * KS * u, np.array([KS * u, 1 - KS * u, 0.25])
    for axis in range(3):
        cam = W.ortho_axis_camera(n, axis, +1, step=step)
        r = O.render(v, cam, O.EA, tf, vmin, vmax, precision=prec)
        K = int(round(n[axis] / step))
        assert np.all(r.K == K)
        A = 1 - (1 - a) ** K
        assert np.max(np.abs(r.image64[..., 3] - A)) <= tol
        assert np.max(np.abs(r.image64[..., :3] - rgb * A)) <= 2 * tol


def test_p2_constant_cube_oblique_rays_chord_count():
    n = (24, 20, 28)
    v = np.full((28, 20, 24), 0.3, dtype=np.float32)
    a = 1.0 / 64.0                                  # dyadic: exact in the float32 table
    tf = const_tf([0.25, 0.5, 0.875, a])
    cam = W.perspective_camera((60.0, 45.0, -40.0), (12, 10, 14), (0, 1, 0), 30.0, 40, 30, step=0.5)
    r = O.render(v, cam, O.EA, tf, 0.0, 1.0, precision=O.F64)
    vec = cam.vectors().astype(np.float64)
    i, j = np.meshgrid(np.arange(40) + 0.5, np.arange(30) + 0.5)
    g = vec[3] + i[..., None] * vec[4] + j[..., None] * vec[5]
    d = g / np.linalg.norm(g, axis=-1, keepdims=True)
    o = vec[0]
    with np.errstate(divide="ignore", invalid="ignore"):
        t0 = (0 - o) / d
        t1 = (np.array(n) - o) / d
    te = np.maximum(np.minimum(t0, t1).max(-1), 0.0)
    tx = np.maximum(t0, t1).min(-1)
    hit = tx > te
    L = np.where(hit, tx - te, 0.0)
    Kcf = np.where(hit, np.ceil(L / 0.5 - 0.5), 0)
    assert hit.sum() > 200
    assert np.all(np.abs(r.K - Kcf) <= 1)
    assert (r.K == Kcf).mean() > 0.98
    A = 1 - (1 - a) ** r.K
    assert np.max(np.abs(r.image64[..., 3] - A)) < 1e-12
    assert np.max(np.abs(r.image64[..., 0] - 0.25 * A)) < 1e-12
    assert np.all(r.image64[~hit] == 0)
    r32 = O.render(v, cam, O.EA, tf, 0.0, 1.0)
    assert np.max(np.abs(r32.image - r.image64)) < 1e-5


# --------------------------------------------------------------------------- P3
def _cams_for_bricks(n):
    c = np.array(n) / 2
    yield W.perspective_camera(c + np.array([90.0, 40.0, 70.0]), c, (0, 1, 0), 40.0, 48, 36, step=0.5)
    yield W.ortho_lookat_camera(c + np.array([-80.0, 30.0, 55.0]), c, (0, 1, 0), 90.0, 40, 30, step=0.7)
    # adversarial: eye inside the volume, within half a voxel of a brick plane
    yield W.perspective_camera((16.3, 7.25, 32.45), (30, 40, 10), (0, 0, 1), 70.0, 40, 30, step=0.5)
    yield W.perspective_camera((15.6, 14.01, 16.49), (0, 50, 70), (0, 1, 0), 80.0, 40, 30, step=0.35)


@pytest.mark.parametrize("B", [2, 7, 16, 72, 100])
def test_p3_bricked_equals_unbricked(B):
    n = (40, 56, 72)
    v = noise_cube(*n, seed=3)
    tf = W.bake_tf(W.TF_HAZE_POINTS, 0.5, alpha_scale=4.0)
    s = O.minmax_hist(v)
    for cam in _cams_for_bricks(n):
        m0 = O.render(v, cam, O.MIP)
        m1 = O.render(v, cam, O.MIP, brick=B)
        assert m1.n_noncontig == 0 and m1.n_order_mismatch == 0
        assert np.array_equal(m0.image, m1.image)                          # MIP bit-exact
        e0 = O.render(v, cam, O.EA, tf, s.vmin, s.vmax)
        e1 = O.render(v, cam, O.EA, tf, s.vmin, s.vmax, brick=B)
        assert e1.n_noncontig == 0 and e1.n_order_mismatch == 0
        assert np.max(np.abs(e0.image - e1.image)) <= 1e-5
        d0 = O.render(v, cam, O.EA, tf, s.vmin, s.vmax, precision=O.F64)
        d1 = O.render(v, cam, O.EA, tf, s.vmin, s.vmax, brick=B, precision=O.F64)
        assert d1.n_noncontig == 0 and d1.n_order_mismatch == 0
        assert np.max(np.abs(d0.image64 - d1.image64)) <= 1e-12
        assert np.array_equal(m0.K, m1.K)


def test_p3_wrong_order_would_be_detected():
    """The fold is order-sensitive: reversing the view must change EA (sanity of the pin)."""
    n = (40, 56, 72)
    v = noise_cube(*n, seed=3)
    tf = W.bake_tf(W.TF_HAZE_POINTS, 0.5, alpha_scale=30.0)
    s = O.minmax_hist(v)
    a = O.render(v, W.ortho_axis_camera(n, 2, +1, step=0.5), O.EA, tf, s.vmin, s.vmax, brick=16)
    b = O.render(v, W.ortho_axis_camera(n, 2, -1, step=0.5), O.EA, tf, s.vmin, s.vmax, brick=16)
    assert np.max(np.abs(a.image[..., :3] - b.image[..., :3])) > 1e-3
    assert np.max(np.abs(a.image[..., 3] - b.image[..., 3])) < 1e-5     # opacity is order-free


def test_bricked_halo_layout_equals_linear():
    n = (21, 18, 13)
    v = noise_cube(*n, seed=5)
    t = W.retile_halo(v, 8)
    cam = W.perspective_camera((50.0, 30.0, 40.0), (10, 9, 6), (0, 1, 0), 35.0, 32, 24, step=0.5)
    a = O.render(v, cam, O.MIP)
    b = O.render(t, cam, O.MIP, layout=O.BRICKED_HALO1, layout_brick=8, dims=n)
    assert np.array_equal(a.image, b.image)
    sa, sb = O.minmax_hist(v), O.minmax_hist(t, layout=O.BRICKED_HALO1, layout_brick=8, dims=n)   # P14
    assert sa.vmin == sb.vmin and sa.vmax == sb.vmax and np.array_equal(sa.counts, sb.counts)
    assert sb.counts.sum() == v.size                                        # halo not double counted


# --------------------------------------------------------------------------- P4
def test_p4_minmax_hist_closed_forms():
    # integers 0..255 uniformly: each of 256 bins holds exactly N/256; v == max lands in the last bin
    v = (np.arange(8 * 16 * 32) % 256).astype(np.float32).reshape(8, 16, 32)
    RNG.shuffle(v.reshape(-1))
    s = O.minmax_hist(v)
    assert s.vmin == 0 and s.vmax == 255 and np.all(s.counts == v.size // 256)
    assert s.n_below == s.n_above == s.n_nonfinite == 0
    # constant cube -> everything in bin 0 (hi == lo)
    s = O.minmax_hist(np.full((4, 5, 6), 3.5, dtype=np.float32))
    assert s.vmin == s.vmax == np.float32(3.5) and s.counts[0] == 120 and s.counts[1:].sum() == 0
    # planted NaN / +-Inf are skipped by min/max and counted
    v = noise_cube(10, 11, 12).copy()
    v[0, 0, 0], v[3, 4, 5], v[9, 9, 9], v[5, 5, 5] = np.nan, np.inf, -np.inf, np.nan
    s = O.minmax_hist(v)
    fin = v[np.isfinite(v)]
    assert s.n_nonfinite == 4 and s.vmin == fin.min() and s.vmax == fin.max()
    assert s.counts.sum() + s.n_below + s.n_above + s.n_nonfinite == v.size
    assert s.counts[-1] >= 1 and s.counts[0] >= 1
    # caller range narrower than the data
    s = O.minmax_hist(v, 16, (-1.0, 1.0))
    assert s.n_below == (fin < -1).sum() and s.n_above == (fin > 1).sum()
    assert s.counts.sum() == ((fin >= -1) & (fin <= 1)).sum()


def test_p4_histogram_matches_numpy_library_routine():
    # values at bin centres: no edge ambiguity, must equal np.histogram exactly
    nb, lo, hi = 64, -2.0, 6.0
    k = RNG.integers(0, nb, size=5000)
    v = (lo + (k + 0.5) * (hi - lo) / nb).astype(np.float32).reshape(10, 20, 25)
    s = O.minmax_hist(v, nb, (lo, hi))
    want, _ = np.histogram(v.astype(np.float64), bins=nb, range=(lo, hi))
    assert np.array_equal(s.counts, want.astype(np.uint64))
    # random data over [min,max]: float32 edge rounding may move a voxel to the adjacent bin only
    v = noise_cube(40, 30, 20, seed=8)
    s = O.minmax_hist(v)
    want, _ = np.histogram(v.astype(np.float64), bins=256, range=(float(s.vmin), float(s.vmax)))
    diff = s.counts.astype(np.int64) - want
    assert diff.sum() == 0 and np.abs(diff).sum() <= 8
    assert np.abs(np.cumsum(diff)).max() <= 2


# --------------------------------------------------------------------------- P5 / P7
def _affine_setup():
    n = (20, 16, 24)
    al, be, ga, de = 0.031, -0.017, 0.023, 0.4
    z, y, x = np.meshgrid(np.arange(24), np.arange(16), np.arange(20), indexing="ij")
    v = (al * x + be * y + ga * z + de).astype(np.float32)
    cam = W.perspective_camera((55.0, 38.0, -30.0), (10, 8, 12), (0, 1, 0), 32.0, 36, 28, step=0.5)
    return n, (al, be, ga, de), v, cam


def _closed_form_samples(n, coef, cam, K):
    """Double-precision sample positions (C.1-C.2) and the affine value at each (clamp-to-edge)."""
    al, be, ga, de = coef
    vec = cam.vectors().astype(np.float64)
    out = {}
    for j in range(cam.height):
        for i in range(cam.width):
            if K[j, i] == 0:
                continue
            g = vec[3] + (i + 0.5) * vec[4] + (j + 0.5) * vec[5]
            d = g / np.linalg.norm(g)
            o = vec[0] + (i + 0.5) * vec[1] + (j + 0.5) * vec[2]
            with np.errstate(divide="ignore"):
                t0, t1 = (0 - o) / d, (np.array(n) - o) / d
            te = max(0.0, np.minimum(t0, t1).max())
            tx = np.maximum(t0, t1).min()
            t = te + (np.arange(K[j, i]) + 0.5) * cam.step
            if not (t[-1] < tx - 1e-6 and te + (K[j, i] + 0.5) * cam.step > tx + 1e-6):
                continue                                    # K ambiguous at the exit face: skip
            p = o + t[:, None] * d - 0.5
            p = np.clip(p, 0, np.array(n) - 1.0)
            out[(j, i)] = al * p[:, 0] + be * p[:, 1] + ga * p[:, 2] + de
    return out


def test_p5_affine_cube_mip_and_ea_closed_sum():
    n, coef, v, cam = _affine_setup()
    tf = ramp_alpha_tf(0.125)
    vmin, vmax = 0.0, 2.0
    m32, m64 = O.render(v, cam, O.MIP), O.render(v, cam, O.MIP, precision=O.F64)
    e32 = O.render(v, cam, O.EA, tf, vmin, vmax)
    e64 = O.render(v, cam, O.EA, tf, vmin, vmax, precision=O.F64)
    S = _closed_form_samples(n, coef, cam, m64.K)
    assert len(S) > 150
    for (j, i), s in S.items():
        mx = s.max()
        assert abs(m64.image64[j, i] - mx) < 5e-7        # float32 voxels of an affine field: ~6e-8 each
        assert abs(m32.image[j, i] - mx) < 2e-5
        u = np.clip((s - vmin) / (vmax - vmin), 0, 1)
        a = 0.125 * KS * u
        Tk = np.concatenate([[1.0], np.cumprod(1 - a)])[:-1]
        w = Tk * a
        want = np.array([(w * KS * u).sum(), (w * (1 - KS * u)).sum(), (w * 0.25).sum(), 1 - np.prod(1 - a)])
        assert np.max(np.abs(e64.image64[j, i] - want)) < 2e-6
        assert np.max(np.abs(e32.image[j, i] - want)) < 2e-5


def test_p7_alpha_zero_and_alpha_one():
    n, coef, v, cam = _affine_setup()
    r = O.render(v, cam, O.EA, const_tf([0.3, 0.6, 0.9, 0.0]), 0.0, 2.0)
    assert np.all(r.image == 0)
    w = np.arange(256, dtype=np.float64) / 256.0
    tf = np.stack([w, 1 - w, 0.5 * w, np.ones_like(w)], axis=1).astype(np.float32)
    r = O.render(v, cam.with_(ert_alpha=0.99), O.EA, tf, 0.0, 2.0, precision=O.F64)
    S = _closed_form_samples(n, coef, cam, r.K)
    hit = r.K > 0
    assert np.all(r.K_ert[hit] == 1) and np.all(r.image64[hit][:, 3] == 1.0)
    for (j, i), s in S.items():
        u0 = KS * s[0] / 2.0
        assert np.max(np.abs(r.image64[j, i, :3] - [u0, 1 - u0, 0.5 * u0])) < 1e-6
    r0 = O.render(v, cam, O.EA, tf, 0.0, 2.0, precision=O.F64)               # ERT off: same image, all K
    assert np.array_equal(r0.image64, r.image64) and np.array_equal(r0.K_ert, r0.K)


# --------------------------------------------------------------------------- P6
def test_p6_impulse_tent_footprint():
    n = (9, 8, 7)
    v = np.zeros((7, 8, 9), dtype=np.float32)
    x0, y0, z0, amp = 4, 3, 2, 8.0
    v[z0, y0, x0] = amp
    W_, H_ = 9 * 4, 8 * 4
    cam = W.ortho_axis_camera(n, 2, +1, step=0.25, width=W_, height=H_)
    r = O.render(v, cam, O.MIP)
    xs = (np.arange(W_) + 0.5) * 9 / W_
    ys = (np.arange(H_) + 0.5) * 8 / H_
    wx = np.maximum(0, 1 - np.abs(xs - (x0 + 0.5)))
    wy = np.maximum(0, 1 - np.abs(ys - (y0 + 0.5)))
    want = amp * wy[:, None] * wx[None, :] * 0.875          # nearest sample is 1/8 voxel from the centre plane
    assert np.max(np.abs(r.image - want)) < 1e-6
    # boundary voxel: clamp-to-edge extends the value constantly through the outer half voxel
    v[:] = 0
    v[3, 0, 0] = amp
    r = O.render(v, W.ortho_axis_camera(n, 2, +1, step=0.25, width=W_, height=H_), O.MIP)
    wx = np.where(xs <= 0.5, 1.0, np.maximum(0, 1 - np.abs(xs - 0.5)))
    wy = np.where(ys <= 0.5, 1.0, np.maximum(0, 1 - np.abs(ys - 0.5)))
    assert np.max(np.abs(r.image - amp * wy[:, None] * wx[None, :] * 0.875)) < 1e-6


# --------------------------------------------------------------------------- P8
@pytest.mark.parametrize("step", [1.0, 0.5, 0.25])
def test_p8_sample_counts(step):
    n = (10, 12, 14)
    v = noise_cube(*n)
    for axis in range(3):
        cam = W.ortho_axis_camera(n, axis, -1, step=step)
        r = O.render(v, cam, O.MIP)
        assert r.n_nominal == cam.width * cam.height * int(n[axis] / step)
        assert r.n_ert == r.n_nominal


def test_misses_and_degenerate_rays():
    n = (10, 12, 14)
    v = noise_cube(*n)
    cam = W.perspective_camera((100.0, 100.0, 100.0), (200, 200, 200), (0, 1, 0), 20.0, 16, 12)   # looks away
    r = O.render(v, cam, O.MIP)
    assert np.all(np.isneginf(r.image)) and r.n_nominal == 0
    r = O.render(v, cam, O.EA, const_tf([1, 1, 1, 0.5]), 0.0, 1.0)
    assert np.all(r.image == 0)
    # d_a == 0 with the origin outside that slab: miss (S6), inside: hit
    cam = W.ortho_axis_camera(n, 2, +1, step=1.0, width=20, height=12)
    cam = cam.with_(ou=np.array([1.0, 0, 0], dtype=np.float32), o0=np.array([-5.0, 0, -1], dtype=np.float32))
    r = O.render(v, cam, O.MIP)
    assert np.all(np.isneginf(r.image[:, :5])) and np.all(np.isfinite(r.image[:, 5:15])) and np.all(np.isneginf(r.image[:, 15:]))


# --------------------------------------------------------------------------- P9
def test_p9_mirror_symmetry():
    n = (24, 18, 20)
    v = noise_cube(*n, seed=2)
    tf = W.bake_tf(W.TF_HAZE_POINTS, 0.5, alpha_scale=8.0)
    s = O.minmax_hist(v)
    cam = W.perspective_camera((70.0, 41.0, -33.0), (12, 9, 10), (0, 1, 0), 30.0, 40, 30, step=0.5)
    vec = cam.vectors().copy()
    mir = vec.copy()
    mir[:, 0] *= -1
    mir[0, 0] = 24.0 - vec[0, 0]
    camm = cam.with_(o0=mir[0], ou=mir[1], ov=mir[2], d0=mir[3], du=mir[4], dv=mir[5])
    vm = np.ascontiguousarray(v[:, :, ::-1])
    for mode, kw in ((O.MIP, {}), (O.EA, dict(tf=tf, vmin=s.vmin, vmax=s.vmax))):
        a = O.render(v, cam, mode, precision=O.F64, **kw)
        b = O.render(vm, camm, mode, precision=O.F64, **kw)
        assert np.array_equal(a.K, b.K)
        fin = np.isfinite(a.image64)
        assert np.array_equal(fin, np.isfinite(b.image64))
        assert np.max(np.abs(a.image64[fin] - b.image64[fin])) < 1e-9
        a = O.render(v, cam, mode, **kw)
        b = O.render(vm, camm, mode, **kw)
        fin = np.isfinite(a.image)
        assert np.max(np.abs(a.image[fin] - b.image[fin])) < 2e-4


# --------------------------------------------------------------------------- P11
def test_p11_ert_bound_and_fragility():
    n = (40, 40, 48)
    v = W.make_cube(W.Recipe(*n, seed=4, n_sources=6))
    s = O.minmax_hist(v)
    tf = W.bake_tf(W.TF_HAZE_POINTS, 0.5, alpha_scale=40.0)
    cam = W.perspective_camera((110.0, 60.0, 95.0), (20, 20, 24), (0, 1, 0), 30.0, 64, 48, step=0.5)
    full = O.render(v, cam, O.EA, tf, s.vmin, s.vmax)
    ert = O.render(v, cam.with_(ert_alpha=0.99), O.EA, tf, s.vmin, s.vmax)
    assert ert.n_ert < full.n_ert and ert.n_nominal == full.n_nominal
    assert (ert.K_ert < ert.K).sum() > 50                       # ERT actually fires
    assert np.all(ert.image <= full.image + 1e-6)
    assert np.max(full.image - ert.image) <= (1 - 0.99) + 1e-4
    stopped = ert.K_ert < ert.K
    assert np.all(ert.image[stopped][:, 3] >= 0.99 - 1e-6)
    assert ert.fragile.mean() < 0.005
    # bricked request with ERT on renders by the single march (C.7 / S15)
    eb = O.render(v, cam.with_(ert_alpha=0.99), O.EA, tf, s.vmin, s.vmax, brick=16)
    assert np.array_equal(eb.image, ert.image)


# --------------------------------------------------------------------------- P12 / P13
def test_p12_f32_canonical_close_to_f64_truth():
    n = (96, 96, 96)
    v = noise_cube(*n, seed=6)
    cam = W.orbit_camera(n, 1, 8, 96, 96, step=0.5)
    a = O.render(v, cam, O.MIP)
    b = O.render(v, cam, O.MIP, precision=O.F64)
    hit = np.isfinite(b.image64)
    assert np.array_equal(hit, np.isfinite(a.image))
    R = float(np.abs(v).max())
    rel = np.abs(a.image[hit] - b.image64[hit]) / np.maximum(np.abs(b.image64[hit]), R)
    assert np.median(rel) < 1e-5 and rel.max() < 1e-3


def test_p13_step_halving_converges_on_smooth_cube():
    n = (48, 48, 48)
    v = W.make_cube(W.Recipe(*n, seed=10, n_sources=5, noise_amp=0.0))
    cam0 = W.perspective_camera((130.0, 70.0, 110.0), (24, 24, 24), (0, 1, 0), 28.0, 40, 40)
    imgs = []
    for step in (1.0, 0.5, 0.25, 0.125):
        tf = W.bake_tf(W.TF_HAZE_POINTS, step, alpha_scale=3.0)
        imgs.append(O.render(v, cam0.with_(step=step), O.EA, tf, 0.0, float(v.max()), precision=O.F64).image64)
    e = [np.abs(imgs[k] - imgs[k + 1]).max() for k in range(3)]
    assert e[0] > e[1] > e[2] and e[2] < 0.35 * e[0]


def test_oracle_matches_its_committed_golden():
    """Regression guard: the oracle's bits on one tiny seeded case (tests/golden/oracle_tiny.txt, written by
    tests/golden/make_oracle_golden.py from the oracle alone).  Not a pin against the paper — it prints no numbers."""
    import importlib.util
    import os
    here = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden")
    spec = importlib.util.spec_from_file_location("make_oracle_golden", os.path.join(here, "make_oracle_golden.py"))
    mod = importlib.util.module_from_spec(spec)
    spec.loader.exec_module(mod)
    with open(os.path.join(here, "oracle_tiny.txt")) as f:
        stored = f.read().splitlines()
    assert list(mod.lines()) == stored


# --------------------------------------------------------------------------- P15: S24, non-finite voxels in a render
def _nonfinite_cube():
    v = noise_cube(11, 9, 13, seed=77).copy()       # (nz, ny, nx) = (13, 9, 11)
    v[4, 3, 5] = np.nan
    v[9, 7, 2] = np.inf
    v[1, 1, 8] = -np.inf
    return v


def _polluted(v):
    """Voxel-centre samples whose 8 corners (C.3: i0 = min(i, n-2), corners i0, i0+1) are not all finite.  The
    exact-ends lerp L(a,b,f) = fma(f, b, fma(-f, a, a)) multiplies BOTH ends by a weight, so a NaN or infinite
    corner makes the sample NaN even at weight 0 (0 * inf = NaN) — also when the infinite corner is the sampled
    voxel itself (-0 * inf).  (No non-finite voxel of these cubes lies on a high face, where f = 1.)"""
    nz, ny, nx = v.shape
    bad = np.zeros(v.shape, dtype=bool)
    for z in range(nz):
        for y in range(ny):
            for x in range(nx):
                x0, y0, z0 = min(x, nx - 2), min(y, ny - 2), min(z, nz - 2)
                bad[z, y, x] = not np.all(np.isfinite(v[z0:z0 + 2, y0:y0 + 2, x0:x0 + 2]))
    return bad


def test_p15_nonfinite_voxels_mip_ignores_nan_samples():
    """S24: a NaN sample is ignored by MIP (fmaxf keeps the other operand).  Axis view at voxel centres, so every
    sample is one voxel unless a non-finite corner turns it into NaN: expected = brute-force column max over the
    unpolluted voxels."""
    v = _nonfinite_cube()
    bad = _polluted(v)
    r = O.render(v, W.ortho_axis_camera((11, 9, 13), 2, +1, step=1.0), O.MIP)
    want = np.where(bad, -np.inf, v).max(axis=0)
    assert np.array_equal(r.image, want)
    assert bad.sum() >= 24 and np.isfinite(r.image).all()          # 3 voxels x >= 8 base cells; every column keeps clean samples
    assert not np.isnan(r.image).any()


def test_p15_nonfinite_voxels_ea_classifies_nan_as_entry_zero():
    """S24 / C.4: u = sat(fma(s, scale, bias)) maps a NaN sample to table entry 0 (+inf to entry 255, -inf to 0).
    With a table whose alpha is 1 only at entry 0 (and 0 elsewhere, exact), a ray is opaque after its first
    NaN / -inf / below-range sample and transparent before it: A = 1 exactly where the column holds such a sample."""
    v = np.abs(_nonfinite_cube()) + 1.0            # finite voxels in [1, ~6]; nan stays nan, inf stays +inf
    v[1, 1, 8] = -np.inf
    tf = np.zeros((256, 4), dtype=np.float32)
    tf[0] = (0.25, 0.5, 0.75, 1.0)
    vmin, vmax = 0.0, 8.0                           # finite samples land on u >= 1/8 -> entries >= 31: alpha exactly 0
    r = O.render(v, W.ortho_axis_camera((11, 9, 13), 2, +1, step=1.0), O.EA, tf, vmin, vmax)
    bad = _polluted(v)
    want_a = bad.any(axis=0).astype(np.float32)
    assert np.array_equal(r.image[..., 3], want_a)
    assert np.array_equal(r.image[..., 0], 0.25 * want_a) and np.array_equal(r.image[..., 2], 0.75 * want_a)


# --------------------------------------------------------------------------- P16: mean / standard deviation / median
def test_p16_statistics_closed_forms():
    """C.13 (S35-S37).  Integers 0..255, each 32 times: mean 127.5, population variance (256^2-1)/12, lower median
    127 (rank (8192-1)//2 = 4095 -> value 4095 // 32).  Constant cube: std 0, median c.  Two-point cube."""
    k = np.repeat(np.arange(256), 32).astype(np.float32)
    RNG.shuffle(k)
    s = O.statistics(k.reshape(8, 32, 32))
    assert s.n_finite == 8192 and s.n_nonfinite == 0
    assert s.mean == 127.5 and abs(s.stddev - math.sqrt((256 ** 2 - 1) / 12)) < 1e-12 and s.median == 127.0
    c = np.full((5, 6, 7), -3.25, dtype=np.float32)
    s = O.statistics(c)
    assert s.mean == -3.25 and s.stddev == 0.0 and s.median == np.float32(-3.25)
    two = np.array([1.0] * 30 + [5.0] * 30, dtype=np.float32).reshape(3, 4, 5)     # even n: LOWER median
    s = O.statistics(two)
    assert s.mean == 3.0 and s.stddev == 2.0 and s.median == 1.0
    two[0, 0, 0] = 5.0                                                              # 29 ones, 31 fives
    assert O.statistics(two).median == 5.0


def test_p16_statistics_match_numpy_and_sorting():
    """Against library routines on a noise+sources cube with planted non-finite voxels: float64 mean / std of numpy
    (pairwise summation) within 1e-13 relative; the median is EXACTLY the element of rank (n-1)//2 of np.sort."""
    v = W.make_cube(W.Recipe(37, 29, 41, seed=8, n_sources=3)).copy()
    v[3, 4, 5], v[7, 7, 7], v[20, 1, 30] = np.nan, np.inf, -np.inf
    s = O.statistics(v)
    f = v[np.isfinite(v)].astype(np.float64)
    assert s.n_finite == f.size and s.n_nonfinite == 3
    assert abs(s.mean - f.mean()) <= 1e-13 * np.abs(f).mean()
    assert abs(s.stddev - f.std()) <= 1e-13 * f.std()
    assert s.median == np.sort(v[np.isfinite(v)])[(f.size - 1) // 2]
    # n even and odd, and the signed-zero order (-0 sorts before +0)
    z = np.array([0.0, -0.0, -0.0, 0.0, 1.0, -1.0, -0.0, 2.0], dtype=np.float32).reshape(2, 2, 2)   # sorted: -1 -0 -0 -0 +0 +0 1 2
    m = O.statistics(z).median
    assert m == 0.0 and np.signbit(m)                # rank 3 is the last -0
    z[0, 0, 1] = 0.0                                 # sorted: -1 -0 -0 +0 +0 +0 1 2 -> rank 3 is +0
    m = O.statistics(z).median
    assert m == 0.0 and not np.signbit(m)


def test_p16_statistics_bricked_halo_layout_equals_linear():
    v = W.make_cube(W.Recipe(21, 18, 26, seed=9, n_sources=2))
    t = W.retile_halo(v, 8)
    a, b = O.statistics(v), O.statistics(t, layout=O.BRICKED_HALO1, layout_brick=8, dims=(21, 18, 26))
    assert a.n_finite == b.n_finite and a.median == b.median
    assert abs(a.mean - b.mean) < 1e-14 and abs(a.stddev - b.stddev) < 1e-14      # same values, another voxel order


# --------------------------------------------------------------------------- P17: 8-bit frame for delivery (C.14, S40)
def test_p17_encode_closed_forms():
    """Opaque pixels of colour k/255 give byte k for every k; transparent pixels give the background; the tie 127.5 goes
    to the even byte 128; values outside [0,1] clamp; NaN gives 0; the alpha byte is 255.  MIP: grey ramp, miss = 0."""
    k = np.arange(256, dtype=np.float64)
    img = np.zeros((1, 256, 4), dtype=np.float32)
    img[0, :, 0] = (k / 255).astype(np.float32); img[0, :, 1] = ((255 - k) / 255).astype(np.float32); img[0, :, 3] = 1.0
    out = O.encode_rgba8(img, O.EA, background=(0.3, 0.6, 0.9))
    assert np.array_equal(out[0, :, 0], np.arange(256)) and np.array_equal(out[0, :, 1], 255 - np.arange(256))
    assert (out[0, :, 2] == 0).all() and (out[..., 3] == 255).all()
    clear = np.zeros((2, 3, 4), dtype=np.float32)
    out = O.encode_rgba8(clear, O.EA, background=(0.5, 0.2, 1.0))
    assert (out[..., 0] == 128).all() and (out[..., 1] == 51).all() and (out[..., 2] == 255).all()     # 127.5 -> 128 (even)
    half = np.zeros((1, 1, 4), dtype=np.float32); half[0, 0] = (0.25, 2.0, -1.0, 0.5)       # C + (1 - A) bg
    out = O.encode_rgba8(half, O.EA, background=(0.5, 0.5, 0.5))
    assert tuple(out[0, 0]) == (128, 255, 0, 255)                                           # 0.5 -> 127.5 -> 128; clamps
    bad = np.zeros((1, 1, 4), dtype=np.float32); bad[0, 0] = (np.nan, np.inf, -np.inf, 0.0)
    assert tuple(O.encode_rgba8(bad, O.EA)[0, 0]) == (0, 255, 0, 255)
    m = np.array([[-np.inf, 2.0, 3.0, 4.0, 10.0, np.nan]], dtype=np.float32)
    out = O.encode_rgba8(m, O.MIP, vmin=2.0, vmax=4.0)
    assert out[0, :, 0].tolist() == [0, 0, 128, 255, 255, 0] and np.array_equal(out[..., 0], out[..., 1]) and (out[..., 3] == 255).all()


def test_p17_encode_against_float64():
    """A random EA image against the formula evaluated in float64: equal bytes wherever the float64 value is not
    within 1e-4 of a rounding tie, never more than one byte apart elsewhere."""
    img = RNG.random((37, 53, 4)).astype(np.float32)
    img[..., :3] *= img[..., 3:4]                                                         # premultiplied
    bg = np.array([0.1, 0.7, 0.35], dtype=np.float32)
    out = O.encode_rgba8(img, O.EA, background=bg).astype(np.int64)
    x = np.clip(img[..., :3].astype(np.float64) + (1.0 - img[..., 3:4].astype(np.float64)) * bg.astype(np.float64), 0, 1) * 255
    want = np.rint(x).astype(np.int64)
    near_tie = np.abs(x - np.floor(x) - 0.5) < 1e-4
    assert np.array_equal(out[..., :3][~near_tie], want[~near_tie]) and np.abs(out[..., :3] - want).max() <= 1
    assert near_tie.mean() < 0.01


def test_p4_histogram_ranges_that_overflow_the_bin_arithmetic():
    """S41.  A caller range of the whole float32 span: hi - lo = inf, scale_h = 0, every t is 0 or inf * 0 = NaN -> bin 0.
    A range narrower than nbins / FLT_MAX: scale_h = inf, v == lo gives NaN -> bin 0, v > lo gives inf -> last bin."""
    v = np.array([-3.0e38, 3.0e38, 0.0, 1.0, -1.0, 2.5, 1e-40, 7.0], dtype=np.float32).reshape(2, 2, 2)
    s = O.minmax_hist(v, 16, (-3.4e38, 3.4e38))
    assert s.counts[0] == 8 and s.counts[1:].sum() == 0 and s.n_below == s.n_above == 0
    w = np.array([0.0, 1e-40, 5e-41, 0.0, 1e-40, -1.0, 1.0, 1e-40], dtype=np.float32).reshape(2, 2, 2)
    s = O.minmax_hist(w, 16, (0.0, 1e-40))
    assert s.counts[0] == 2 and s.counts[15] == 4 and s.n_below == 1 and s.n_above == 1 and s.counts.sum() == 6
