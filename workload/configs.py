"""The five BASELINE.json configs as data (SURVEY.md §8(a) sizes, §8(d) D.1/D.2).

``scale`` < 1 shrinks every dimension (and the source count with the volume) for tests
that need the *shape* of a config at a size the oracle finishes in seconds.
"""
from __future__ import annotations

from dataclasses import dataclass

from .cameras import Camera, orbit_camera, ortho_axis_camera, VR_SORT_LAST
from .cubes import Recipe

_SEED = 0x1111666100000000


@dataclass(frozen=True)
class WorkloadConfig:
    name: str
    number: int
    recipe: Recipe
    brick: int               # 0 = one brick = whole cube
    width: int
    height: int
    n_views: int             # 1 => the single orthographic view of cfg1
    step: float
    ert_alpha: float
    modes: tuple             # subset of ("ea", "mip")
    sort_last: bool
    out_of_core: bool = False
    n_copy_streams: int = 0
    summary: bool = False    # config also runs the min/max + histogram pass

    @property
    def dims(self):
        return (self.recipe.nx, self.recipe.ny, self.recipe.nz)

    def camera(self, view: int = 0) -> Camera:
        flags = VR_SORT_LAST if self.sort_last else 0
        if self.number == 1:
            return ortho_axis_camera(self.dims, axis=2, sign=+1, step=self.step, width=self.width,
                                     height=self.height, ert_alpha=self.ert_alpha, flags=flags)
        return orbit_camera(self.dims, view, self.n_views, self.width, self.height, step=self.step,
                            ert_alpha=self.ert_alpha, flags=flags)


def _mk(number, dims, n_src, brick, wh, views, step, ert, modes, sort_last, ramp=0.0, smod=0.0,
        ooc=False, streams=0, summary=False, scale=1.0):
    nx, ny, nz = (max(8, int(round(d * scale))) for d in dims)
    n_src = max(1, int(round(n_src * scale ** 3))) if scale != 1.0 else n_src
    w, h = (max(16, int(round(v * scale))) for v in wh) if scale != 1.0 else wh
    b = max(4, int(round(brick * scale))) if (brick and scale != 1.0) else brick
    rec = Recipe(nx, ny, nz, _SEED + number, n_sources=n_src, ramp_max=ramp, sigma_mod=smod)
    return WorkloadConfig(f"cfg{number}" + ("" if scale == 1.0 else f"@{scale:g}"), number, rec, b, w, h,
                          views, step, ert, modes, sort_last, ooc, streams, summary)


def get_config(number: int, scale: float = 1.0) -> WorkloadConfig:
    if number == 1:   # 128^3, one ortho view along z, 256x256, step 0.5, MIP + EA, + summary pass
        return _mk(1, (128, 128, 128), 8, 0, (256, 256), 1, 0.5, 0.0, ("mip", "ea"), False, summary=True, scale=scale)
    if number == 2:   # 512x512x1024 (1 GiB), 128^3 bricks, 16 orbit views, 1024^2, EA + ERT 0.99
        return _mk(2, (512, 512, 1024), 200, 128, (1024, 1024), 16, 0.5, 0.99, ("ea",), False, scale=scale)
    if number == 3:   # 1024x1024x2048 (8 GiB), ramp, summary, 1920x1080, 32 views, MIP + EA, sort-last
        return _mk(3, (1024, 1024, 2048), 1000, 128, (1920, 1080), 32, 0.5, 0.0, ("mip", "ea"), True,
                   ramp=2.0, summary=True, scale=scale)
    if number == 4:   # 2048x2048x4096 (64 GiB), sigma(z), 3840x2160, 64 views, step 1, EA + ERT
        return _mk(4, (2048, 2048, 4096), 5000, 128, (3840, 2160), 64, 1.0, 0.99, ("ea",), False,
                   smod=0.5, scale=scale)
    if number == 5:   # out-of-core 4096x4096x3072 (192 GiB) pinned host, 256^3 bricks, 4 streams, 8 views
        return _mk(5, (4096, 4096, 3072), 20000, 256, (1920, 1080), 8, 0.5, 0.99, ("ea",), False,
                   smod=0.5, ooc=True, streams=4, summary=True, scale=scale)
    raise ValueError(f"no config {number}")


CONFIGS = {i: get_config(i) for i in range(1, 6)}
