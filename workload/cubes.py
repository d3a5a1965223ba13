"""ctypes front-end of ``vrgen.c`` (seeded noise + sources cubes)."""
from __future__ import annotations

import ctypes as C
import os
import subprocess
from dataclasses import dataclass

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "vrgen.c")
_LIB = os.path.join(_HERE, "libvrgen.so")
_lib = None


def build(force: bool = False) -> str:
    """Compile vrgen.c -> libvrgen.so (in-tree) if missing or stale."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        cmd = ["gcc", "-O2", "-fopenmp", "-mfma", "-ffp-contract=off", "-fvisibility=hidden",
               "-shared", "-fPIC", "-o", _LIB, _SRC, "-lm"]
        subprocess.run(cmd, check=True)
    return _LIB


class _RecipeC(C.Structure):
    _fields_ = [("struct_size", C.c_uint32), ("nx", C.c_uint32), ("ny", C.c_uint32), ("nz", C.c_uint32),
                ("seed", C.c_uint64), ("n_sources", C.c_uint32), ("ramp_max", C.c_float),
                ("sigma_mod", C.c_float), ("noise_amp", C.c_float)]


def _load():
    global _lib
    if _lib is None:
        lib = C.CDLL(build())
        lib.vrgen_create.restype = C.c_void_p
        lib.vrgen_create.argtypes = [C.POINTER(_RecipeC)]
        lib.vrgen_destroy.argtypes = [C.c_void_p]
        lib.vrgen_voxel.restype = C.c_float
        lib.vrgen_voxel.argtypes = [C.c_void_p, C.c_uint32, C.c_uint32, C.c_uint32]
        lib.vrgen_fill.restype = C.c_int
        lib.vrgen_fill.argtypes = [C.c_void_p, C.c_uint32, C.c_uint32, C.c_void_p]
        lib.vrgen_sources.restype = C.c_int
        lib.vrgen_sources.argtypes = [C.c_void_p, C.c_void_p]
        lib.vrgen_checksum.restype = C.c_uint64
        lib.vrgen_checksum.argtypes = [C.c_void_p, C.c_uint64]
        lib.vrgen_retile_halo.restype = C.c_int
        lib.vrgen_retile_halo.argtypes = [C.c_void_p, C.c_uint32, C.c_uint32, C.c_uint32, C.c_uint32, C.c_void_p]
        lib.vrgen_retile_halo_layer.restype = C.c_int
        lib.vrgen_retile_halo_layer.argtypes = [C.c_void_p, C.c_uint32, C.c_uint32, C.c_uint32, C.c_uint32, C.c_void_p]
        lib.vrgen_det_log.restype = C.c_double
        lib.vrgen_det_log.argtypes = [C.c_double]
        lib.vrgen_det_exp_neg.restype = C.c_double
        lib.vrgen_det_exp_neg.argtypes = [C.c_double]
        lib.vrgen_det_sincos2pi.argtypes = [C.c_double, C.POINTER(C.c_double), C.POINTER(C.c_double)]
        _lib = lib
    return _lib


@dataclass(frozen=True)
class Recipe:
    nx: int
    ny: int
    nz: int
    seed: int
    n_sources: int = 0
    ramp_max: float = 0.0     # cfg3: 2.0 (sky-continuum gradient along x)
    sigma_mod: float = 0.0    # cfg4/5: 0.5 (noise sigma varies per spectral channel)
    noise_amp: float = 1.0    # 0 => smooth (sources/ramp only) cubes for convergence tests

    @property
    def shape(self):
        return (self.nz, self.ny, self.nx)

    @property
    def n_voxels(self):
        return self.nx * self.ny * self.nz


class CubeGenerator:
    """Handle on one recipe: bulk fill and on-demand single voxels (same bits)."""

    def __init__(self, recipe: Recipe):
        self.recipe = recipe
        lib = _load()
        rc = _RecipeC(C.sizeof(_RecipeC), recipe.nx, recipe.ny, recipe.nz, recipe.seed & (2**64 - 1),
                      recipe.n_sources, recipe.ramp_max, recipe.sigma_mod, recipe.noise_amp)
        self._h = lib.vrgen_create(C.byref(rc))
        if not self._h:
            raise ValueError("vrgen_create failed")

    def __del__(self):
        if getattr(self, "_h", None) and _lib is not None:
            _lib.vrgen_destroy(self._h)
            self._h = None

    def voxel(self, ix: int, iy: int, iz: int) -> np.float32:
        return np.float32(_lib.vrgen_voxel(self._h, ix, iy, iz))

    def fill(self, out: np.ndarray, z0: int = 0, z1: int | None = None) -> np.ndarray:
        """Fill ``out`` (float32, C-contiguous, shape (z1-z0, ny, nx)) with slices z0..z1."""
        r = self.recipe
        z1 = r.nz if z1 is None else z1
        assert out.dtype == np.float32 and out.flags["C_CONTIGUOUS"]
        assert out.size == (z1 - z0) * r.ny * r.nx
        if _lib.vrgen_fill(self._h, z0, z1, out.ctypes.data) != 0:
            raise ValueError("vrgen_fill failed")
        return out

    def fill_ptr(self, ptr: int, z0: int, z1: int) -> None:
        """Fill raw host memory (e.g. a pinned torch tensor's data_ptr())."""
        if _lib.vrgen_fill(self._h, z0, z1, C.c_void_p(ptr)) != 0:
            raise ValueError("vrgen_fill failed")

    def sources(self) -> np.ndarray:
        """(n_sources, 8): A, 1/(2 sxy^2), 1/(2 sz^2), cx, cy, cz, 5 sxy, 5 sz."""
        out = np.zeros((max(self.recipe.n_sources, 1), 8), dtype=np.float64)
        _lib.vrgen_sources(self._h, out.ctypes.data)
        return out[: self.recipe.n_sources]


def make_cube(recipe: Recipe) -> np.ndarray:
    """float32 array of shape (nz, ny, nx), x fastest."""
    out = np.empty(recipe.shape, dtype=np.float32)
    CubeGenerator(recipe).fill(out)
    return out


def checksum(a: np.ndarray) -> int:
    """64-bit wrap-around sum of the float32 bit patterns (identity of a cube's bytes)."""
    a = np.ascontiguousarray(a, dtype=np.float32)
    return int(_load().vrgen_checksum(a.ctypes.data, a.size))


def retile_halo(lin: np.ndarray, brick: int) -> np.ndarray:
    """Linear (nz,ny,nx) -> brick-major with +1 high-side halo: (n_bricks, B+1, B+1, B+1)."""
    nz, ny, nx = lin.shape
    nb = -(-nx // brick) * -(-ny // brick) * -(-nz // brick)
    out = np.empty((nb, brick + 1, brick + 1, brick + 1), dtype=np.float32)
    lin = np.ascontiguousarray(lin, dtype=np.float32)
    if _load().vrgen_retile_halo(lin.ctypes.data, nx, ny, nz, brick, out.ctypes.data) != 0:
        raise ValueError("vrgen_retile_halo failed")
    return out


def bricked_halo_elems(dims, brick: int) -> int:
    """Number of float32 elements of the brick-major (B+1)^3 layout of a cube of ``dims`` = (nx, ny, nz)."""
    nx, ny, nz = dims
    return -(-nx // brick) * -(-ny // brick) * -(-nz // brick) * (brick + 1) ** 3


def fill_bricked_halo_ptr(recipe: Recipe, brick: int, ptr: int) -> None:
    """Generate the recipe's cube straight into brick-major-with-halo layout at raw host address ``ptr``
    (e.g. a pinned torch tensor), one brick layer at a time: the linear cube is never held as a whole."""
    lib = _load()
    gen = CubeGenerator(recipe)
    nx, ny, nz = recipe.nx, recipe.ny, recipe.nz
    E3 = (brick + 1) ** 3
    per_layer = -(-nx // brick) * -(-ny // brick)
    for bz in range(-(-nz // brick)):
        z0, z1 = bz * brick, min(bz * brick + brick + 1, nz)
        slab = np.empty((z1 - z0, ny, nx), dtype=np.float32)
        gen.fill(slab, z0, z1)
        dst = ptr + 4 * bz * per_layer * E3
        if lib.vrgen_retile_halo_layer(slab.ctypes.data, nx, ny, z1 - z0, brick, C.c_void_p(dst)) != 0:
            raise ValueError("vrgen_retile_halo_layer failed")
        del slab


def det_log(x: float) -> float:
    return _load().vrgen_det_log(x)


def det_exp_neg(a: float) -> float:
    return _load().vrgen_det_exp_neg(a)


def det_sincos2pi(u: float):
    s, c = C.c_double(), C.c_double()
    _load().vrgen_det_sincos2pi(u, C.byref(s), C.byref(c))
    return s.value, c.value
