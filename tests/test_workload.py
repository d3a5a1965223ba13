"""The seeded input generators: determinism, statistics, on-demand == bulk."""
import math

import numpy as np
import pytest

import workload as W
from workload import cubes


def test_det_functions_match_libm():
    rng = np.random.default_rng(0)
    for x in rng.uniform(1e-9, 1.0, 2000):
        assert abs(cubes.det_log(x) - math.log(x)) <= 4e-16 * max(1.0, abs(math.log(x)))
    for a in rng.uniform(0.0, 60.0, 2000):
        assert abs(cubes.det_exp_neg(a) - math.exp(-a)) <= 4e-16 * math.exp(-a)
    for u in rng.uniform(0.0, 1.0, 2000):
        s, c = cubes.det_sincos2pi(u)
        assert abs(s - math.sin(2 * math.pi * u)) < 2e-15 and abs(c - math.cos(2 * math.pi * u)) < 2e-15


def test_noise_moments_and_determinism():
    r = W.Recipe(96, 80, 64, seed=1234)
    a = W.make_cube(r)
    b = W.make_cube(r)
    assert np.array_equal(a, b) and W.checksum(a) == W.checksum(b)
    n = a.size
    assert abs(a.mean()) < 5 / math.sqrt(n)
    assert abs(a.var() - 1.0) < 5 * math.sqrt(2.0 / n)
    assert abs((a.astype(np.float64) ** 4).mean() - 3.0) < 0.05
    c = W.make_cube(W.Recipe(96, 80, 64, seed=1235))
    assert abs(np.corrcoef(a.ravel(), c.ravel())[0, 1]) < 0.01
    # neighbours uncorrelated (i.i.d.)
    assert abs(np.corrcoef(a[:, :, :-1].ravel(), a[:, :, 1:].ravel())[0, 1]) < 0.01


def test_on_demand_equals_bulk_and_slabs():
    r = W.Recipe(37, 29, 41, seed=7, n_sources=6, ramp_max=2.0, sigma_mod=0.5)
    g = W.CubeGenerator(r)
    full = W.make_cube(r)
    rng = np.random.default_rng(1)
    for _ in range(300):
        x, y, z = int(rng.integers(37)), int(rng.integers(29)), int(rng.integers(41))
        assert g.voxel(x, y, z) == full[z, y, x]
    slab = np.empty((7, 29, 37), dtype=np.float32)
    g.fill(slab, 10, 17)
    assert np.array_equal(slab, full[10:17])


def test_sources_ramp_and_sigma_profile():
    r0 = W.Recipe(64, 64, 64, seed=5, n_sources=0, noise_amp=0.0, ramp_max=2.0)
    v = W.make_cube(r0)
    assert np.allclose(v[3, 4, :], 2.0 * np.arange(64) / 63.0, atol=1e-6)
    r1 = W.Recipe(64, 64, 64, seed=5, n_sources=3, noise_amp=0.0)
    g = W.CubeGenerator(r1)
    v = W.make_cube(r1)
    src = g.sources()
    assert np.all((src[:, 0] >= 5) & (src[:, 0] <= 20))
    sxy = src[:, 6] / 5.0
    sz = src[:, 7] / 5.0
    assert np.all((sxy >= 2) & (sxy <= 6)) and np.all((sz >= 4) & (sz <= 12))
    # brute-force evaluation of the sum of truncated Gaussians at a few voxels
    rng = np.random.default_rng(2)
    for _ in range(200):
        s = src[int(rng.integers(len(src)))]
        x = int(np.clip(s[3] + rng.integers(-6, 7), 0, 63)); y = int(np.clip(s[4] + rng.integers(-6, 7), 0, 63))
        z = int(np.clip(s[5] + rng.integers(-10, 11), 0, 63))
        want = 0.0
        for A, hxy, hz, cx, cy, cz, rxy, rz in src:
            dx, dy, dz = x - cx, y - cy, z - cz
            if abs(dx) <= rxy and abs(dy) <= rxy and abs(dz) <= rz:
                want += A * math.exp(-(dx * dx + dy * dy) * hxy - dz * dz * hz)
        assert abs(v[z, y, x] - want) <= 1e-6 * max(1.0, want)
    r2 = W.Recipe(32, 32, 256, seed=9, sigma_mod=0.5)
    n = W.make_cube(r2)
    sd = n.reshape(256, -1).std(axis=1)
    want = 1 + 0.5 * np.sin(2 * np.pi * np.arange(256) / 256)
    assert np.max(np.abs(sd / want - 1)) < 0.12


def test_retile_halo_roundtrip():
    r = W.Recipe(21, 18, 13, seed=3)
    v = W.make_cube(r)
    B = 8
    t = W.retile_halo(v, B)
    nbx, nby, nbz = 3, 3, 2
    assert t.shape == (nbx * nby * nbz, B + 1, B + 1, B + 1)
    for b in range(t.shape[0]):
        bx, by, bz = b % nbx, (b // nbx) % nby, b // (nbx * nby)
        zi = np.minimum(bz * B + np.arange(B + 1), 12); yi = np.minimum(by * B + np.arange(B + 1), 17)
        xi = np.minimum(bx * B + np.arange(B + 1), 20)
        assert np.array_equal(t[b], v[np.ix_(zi, yi, xi)])


def test_configs_shapes():
    for i, dims in {1: (128, 128, 128), 2: (512, 512, 1024), 3: (1024, 1024, 2048), 4: (2048, 2048, 4096),
                    5: (4096, 4096, 3072)}.items():
        assert W.CONFIGS[i].dims == dims
    c = W.CONFIGS[1].camera()
    assert c.is_orthographic and c.width == 256 and np.allclose(c.vectors()[1], [0.5, 0, 0])
    c2 = W.CONFIGS[2].camera(3)
    assert c2.is_perspective and c2.ert_alpha == pytest.approx(0.99)
    assert abs(c2.meta["R"] - 1639) < 1.0
    tf = W.tf_haze((512, 512, 1024), 0.5)
    assert tf.shape == (256, 4) and tf.min() >= 0 and tf.max() <= 1 and tf[0, 3] == 0


def test_fill_bricked_halo_layerwise_equals_retile():
    """The layer-by-layer generator of the brick-major layout (used for cubes that do not fit host memory twice)
    writes the same bytes as retiling the whole linear cube."""
    r = W.Recipe(21, 18, 23, seed=99, n_sources=2)
    for B in (4, 7, 16, 32):
        ref = W.retile_halo(W.make_cube(r), B)
        out = np.empty(W.bricked_halo_elems((r.nx, r.ny, r.nz), B), dtype=np.float32)
        W.fill_bricked_halo_ptr(r, B, out.ctypes.data)
        assert np.array_equal(out.reshape(ref.shape).view(np.uint32), ref.view(np.uint32))
