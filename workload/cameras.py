"""Camera construction (input generation; SURVEY.md §8(c) C.1 harness part, §8(d) D.2).

The six camera vectors are derived in double from (eye, look-at, up, fov / extent,
W, H), rounded to float32 ONCE, and the same 18 floats are handed to the oracle and
to the library:   origin(i,j) = o0 + (i+.5) ou + (j+.5) ov
                  dir(i,j)    = normalize(d0 + (i+.5) du + (j+.5) dv)
Row j = 0 is the v-minimum row (no flip).
"""
from __future__ import annotations

from dataclasses import dataclass, field, replace

import numpy as np

VR_SORT_LAST = 1  # camera flag: force per-brick partial images + sort-last compositor


def _f3(v):
    return np.asarray(v, dtype=np.float64).astype(np.float32)


@dataclass(frozen=True)
class Camera:
    width: int
    height: int
    o0: np.ndarray
    ou: np.ndarray
    ov: np.ndarray
    d0: np.ndarray
    du: np.ndarray
    dv: np.ndarray
    step: float = 0.5
    ert_alpha: float = 0.0
    flags: int = 0
    meta: dict = field(default_factory=dict, compare=False)

    def vectors(self) -> np.ndarray:
        """(6,3) float32: o0, ou, ov, d0, du, dv."""
        return np.stack([_f3(self.o0), _f3(self.ou), _f3(self.ov), _f3(self.d0), _f3(self.du), _f3(self.dv)])

    def with_(self, **kw) -> "Camera":
        return replace(self, **kw)

    @property
    def is_perspective(self) -> bool:
        v = self.vectors()
        return not v[1].any() and not v[2].any()

    @property
    def is_orthographic(self) -> bool:
        v = self.vectors()
        return not v[4].any() and not v[5].any()


def ortho_axis_camera(dims, axis: int, sign: int = +1, step: float = 1.0, width=None, height=None,
                      standoff: float = 1.0, **kw) -> Camera:
    """Axis-aligned orthographic view; u,v = the two transverse axes in cyclic order.

    With default W,H = transverse dims and standoff 1, rays pass through voxel centres and
    all t are exactly representable (pin P1).  dims = (nx, ny, nz)."""
    n = np.asarray(dims, dtype=np.float64)
    ua, va = [(1, 2), (0, 2), (0, 1)][axis]
    W = int(n[ua]) if width is None else width
    H = int(n[va]) if height is None else height
    o0 = np.zeros(3); ou = np.zeros(3); ov = np.zeros(3); d0 = np.zeros(3)
    ou[ua] = n[ua] / W
    ov[va] = n[va] / H
    d0[axis] = float(sign)
    o0[axis] = -standoff if sign > 0 else n[axis] + standoff
    z = np.zeros(3)
    return Camera(W, H, _f3(o0), _f3(ou), _f3(ov), _f3(d0), _f3(z), _f3(z), step=step,
                  meta={"kind": "ortho_axis", "axis": axis, "sign": sign}, **kw)


def _basis(eye, look_at, up):
    eye = np.asarray(eye, dtype=np.float64); look_at = np.asarray(look_at, dtype=np.float64)
    f = look_at - eye
    f /= np.linalg.norm(f)
    r = np.cross(f, np.asarray(up, dtype=np.float64))
    r /= np.linalg.norm(r)
    u = np.cross(r, f)
    return eye, f, r, u


def perspective_camera(eye, look_at, up, fov_y_deg: float, width: int, height: int, step: float = 0.5,
                       **kw) -> Camera:
    eye, f, r, u = _basis(eye, look_at, up)
    th = np.tan(np.deg2rad(fov_y_deg) / 2.0)
    asp = width / height
    d0 = f - th * asp * r - th * u
    du = (2.0 * th * asp / width) * r
    dv = (2.0 * th / height) * u
    z = np.zeros(3)
    return Camera(width, height, _f3(eye), _f3(z), _f3(z), _f3(d0), _f3(du), _f3(dv), step=step,
                  meta={"kind": "perspective", "eye": eye.tolist(), "fov_y": fov_y_deg}, **kw)


def ortho_lookat_camera(eye, look_at, up, extent_y: float, width: int, height: int, step: float = 0.5,
                        **kw) -> Camera:
    """General (oblique) orthographic camera: image plane through ``eye``, height ``extent_y`` voxels."""
    eye, f, r, u = _basis(eye, look_at, up)
    asp = width / height
    o0 = eye - 0.5 * extent_y * asp * r - 0.5 * extent_y * u
    ou = (extent_y * asp / width) * r
    ov = (extent_y / height) * u
    z = np.zeros(3)
    return Camera(width, height, _f3(o0), _f3(ou), _f3(ov), _f3(f), _f3(z), _f3(z), step=step,
                  meta={"kind": "ortho_lookat"}, **kw)


def orbit_camera(dims, view: int, n_views: int, width: int, height: int, step: float = 0.5,
                 fov_y_deg: float = 45.0, elevation_deg: float = 20.0, **kw) -> Camera:
    """circular orbit, bounding sphere fills the vertical FOV."""
    n = np.asarray(dims, dtype=np.float64)
    c = n / 2.0
    r_b = 0.5 * np.linalg.norm(n)
    R = r_b / np.sin(np.deg2rad(fov_y_deg) / 2.0)
    th = 2.0 * np.pi * (view + 0.25) / n_views
    el = np.deg2rad(elevation_deg)
    eye = c + R * np.array([np.cos(el) * np.sin(th), np.sin(el), np.cos(el) * np.cos(th)])
    cam = perspective_camera(eye, c, (0.0, 1.0, 0.0), fov_y_deg, width, height, step=step, **kw)
    cam.meta.update({"kind": "orbit", "view": view, "n_views": n_views, "R": R})
    return cam


def nominal_samples(cam: Camera, dims) -> int:
    """Size of one view as a workload: how many sample positions its rays hold inside the box
    [0,nx]x[0,ny]x[0,nz] at spacing ``cam.step`` (mid-point lattice from the volume entry), counted
    analytically in float64 from the camera geometry.  A descriptor of the input (like a token
    count), used by bench.py to turn frame times into samples/s; it may differ from the renderer's
    own float32 count by at most one sample per ray."""
    v = cam.vectors().astype(np.float64)
    W, H = cam.width, cam.height
    px = (np.arange(W, dtype=np.float64) + 0.5)[None, :, None]
    py = (np.arange(H, dtype=np.float64) + 0.5)[:, None, None]
    o = v[0] + px * v[1] + py * v[2]
    g = v[3] + px * v[4] + py * v[5]
    d = g / np.linalg.norm(g, axis=-1, keepdims=True)
    n = np.asarray(dims, dtype=np.float64)
    with np.errstate(divide="ignore", invalid="ignore"):
        ta, tb = (0.0 - o) / d, (n - o) / d
    lo, hi = np.minimum(ta, tb), np.maximum(ta, tb)
    par = d == 0.0
    inside = (o >= 0.0) & (o <= n)
    lo = np.where(par, np.where(inside, -np.inf, np.inf), lo)
    hi = np.where(par, np.where(inside, np.inf, -np.inf), hi)
    t_enter = np.maximum(lo.max(axis=-1), 0.0)
    t_exit = hi.min(axis=-1)
    chord = np.where(t_exit > t_enter, t_exit - t_enter, 0.0)
    return int(np.maximum(np.ceil(chord / float(cam.step) - 0.5), 0.0).sum())
