"""ctypes front-end of vr_oracle.c (argument marshalling only)."""
from __future__ import annotations

import ctypes as C
import os
import subprocess
from dataclasses import dataclass

import numpy as np

EA, MIP = 0, 1
F32, F64 = 0, 1
LINEAR, BRICKED_HALO1 = 0, 1

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "vr_oracle.c")
_LIB = os.path.join(_HERE, "libvroracle.so")
_lib = None


def build(force: bool = False) -> str:
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        subprocess.run(["gcc", "-O2", "-fopenmp", "-mfma", "-ffp-contract=off", "-fvisibility=hidden",
                        "-shared", "-fPIC", "-o", _LIB, _SRC, "-lm"], check=True)
    return _LIB


class _Cam(C.Structure):
    _fields_ = [("struct_size", C.c_uint32), ("width", C.c_uint32), ("height", C.c_uint32),
                ("o0", C.c_float * 3), ("ou", C.c_float * 3), ("ov", C.c_float * 3),
                ("d0", C.c_float * 3), ("du", C.c_float * 3), ("dv", C.c_float * 3),
                ("step", C.c_float), ("ert_alpha", C.c_float)]


class _Args(C.Structure):
    _fields_ = [("struct_size", C.c_uint32), ("nx", C.c_uint32), ("ny", C.c_uint32), ("nz", C.c_uint32),
                ("layout", C.c_uint32), ("layout_brick", C.c_uint32),
                ("vol", C.c_void_p), ("tf", C.c_void_p), ("vmin", C.c_float), ("vmax", C.c_float),
                ("mode", C.c_int32), ("precision", C.c_int32), ("brick", C.c_uint32),
                ("mask", C.c_void_p), ("image", C.c_void_p), ("image64", C.c_void_p),
                ("K", C.c_void_p), ("K_ert", C.c_void_p), ("fragile", C.c_void_p),
                ("n_nominal", C.c_uint64), ("n_ert", C.c_uint64),
                ("n_noncontig", C.c_uint64), ("n_order_mismatch", C.c_uint64)]


class _Head(C.Structure):
    _fields_ = [("vmin", C.c_float), ("vmax", C.c_float), ("n_nonfinite", C.c_uint64),
                ("n_below", C.c_uint64), ("n_above", C.c_uint64)]


class _Stats(C.Structure):
    _fields_ = [("n_finite", C.c_uint64), ("n_nonfinite", C.c_uint64), ("mean", C.c_double), ("stddev", C.c_double),
                ("median", C.c_float), ("pad", C.c_float)]


def _load():
    global _lib
    if _lib is None:
        lib = C.CDLL(build())
        lib.oracle_render.restype = C.c_int
        lib.oracle_render.argtypes = [C.POINTER(_Cam), C.POINTER(_Args)]
        lib.oracle_minmax_hist.restype = C.c_int
        lib.oracle_minmax_hist.argtypes = [C.c_void_p, C.c_uint32, C.c_uint32, C.c_uint32, C.c_uint32, C.c_uint32,
                                           C.c_uint32, C.c_void_p, C.POINTER(_Head), C.c_void_p]
        lib.oracle_statistics.restype = C.c_int
        lib.oracle_statistics.argtypes = [C.c_void_p, C.c_uint32, C.c_uint32, C.c_uint32, C.c_uint32, C.c_uint32,
                                          C.POINTER(_Stats)]
        lib.oracle_num_threads.restype = C.c_int
        _lib = lib
    return _lib


def num_threads() -> int:
    return int(_load().oracle_num_threads())


@dataclass
class RenderResult:
    image: np.ndarray            # (H,W,4) EA or (H,W) MIP, float32
    image64: np.ndarray          # same shape, float64 (f64-truth unrounded; f32 results widened)
    K: np.ndarray                # (H,W) int32 nominal sample counts
    K_ert: np.ndarray            # (H,W) int32
    fragile: np.ndarray          # (H,W) bool
    n_nominal: int
    n_ert: int
    n_noncontig: int
    n_order_mismatch: int


def _cam_struct(cam) -> _Cam:
    v = cam.vectors()
    c = _Cam()
    c.struct_size = C.sizeof(_Cam)
    c.width, c.height = cam.width, cam.height
    for name, row in zip(("o0", "ou", "ov", "d0", "du", "dv"), v):
        setattr(c, name, (C.c_float * 3)(*[float(x) for x in row]))
    c.step = float(cam.step)
    c.ert_alpha = float(cam.ert_alpha)
    return c


def render(vol: np.ndarray, cam, mode: int, tf: np.ndarray | None = None, vmin: float = 0.0, vmax: float = 1.0,
           brick: int = 0, precision: int = F32, mask: np.ndarray | None = None,
           layout: int = LINEAR, layout_brick: int = 0, dims=None) -> RenderResult:
    """vol: float32 (nz,ny,nx) [LINEAR] or (n_bricks,B+1,B+1,B+1) [BRICKED_HALO1 with dims=(nx,ny,nz)]."""
    lib = _load()
    assert vol.dtype == np.float32 and vol.flags["C_CONTIGUOUS"]
    if layout == LINEAR:
        nz, ny, nx = vol.shape
    else:
        nx, ny, nz = dims
    W, H = cam.width, cam.height
    ch = 4 if mode == EA else 1
    image = np.zeros((H, W, ch), dtype=np.float32)
    image64 = np.zeros((H, W, ch), dtype=np.float64)
    if mode == MIP:
        image[:] = -np.inf
        image64[:] = -np.inf
    K = np.zeros((H, W), dtype=np.int32)
    Ke = np.zeros((H, W), dtype=np.int32)
    frag = np.zeros((H, W), dtype=np.uint8)
    a = _Args()
    a.struct_size = C.sizeof(_Args)
    a.nx, a.ny, a.nz = nx, ny, nz
    a.layout, a.layout_brick = layout, layout_brick
    a.vol = vol.ctypes.data
    if tf is not None:
        tf = np.ascontiguousarray(tf, dtype=np.float32)
        assert tf.shape == (256, 4)
        a.tf = tf.ctypes.data
    a.vmin, a.vmax = float(vmin), float(vmax)
    a.mode, a.precision, a.brick = mode, precision, brick
    if mask is not None:
        mask = np.ascontiguousarray(mask, dtype=np.uint8)
        assert mask.shape == (H, W)
        a.mask = mask.ctypes.data
    a.image, a.image64 = image.ctypes.data, image64.ctypes.data
    a.K, a.K_ert, a.fragile = K.ctypes.data, Ke.ctypes.data, frag.ctypes.data
    c = _cam_struct(cam)
    rc = lib.oracle_render(C.byref(c), C.byref(a))
    if rc != 0:
        raise ValueError(f"oracle_render failed: {rc}")
    if mode == MIP:
        image, image64 = image[..., 0], image64[..., 0]
    return RenderResult(image, image64, K, Ke, frag.astype(bool), int(a.n_nominal), int(a.n_ert),
                        int(a.n_noncontig), int(a.n_order_mismatch))


@dataclass
class Summary:
    vmin: np.float32
    vmax: np.float32
    n_nonfinite: int
    n_below: int
    n_above: int
    counts: np.ndarray           # (nbins,) uint64


def minmax_hist(vol: np.ndarray, nbins: int = 256, range_=None, layout: int = LINEAR, layout_brick: int = 0,
                dims=None) -> Summary:
    lib = _load()
    assert vol.dtype == np.float32 and vol.flags["C_CONTIGUOUS"]
    if layout == LINEAR:
        nz, ny, nx = vol.shape
    else:
        nx, ny, nz = dims
    head = _Head()
    counts = np.zeros(nbins, dtype=np.uint64)
    rng = None
    if range_ is not None:
        rng = np.asarray(range_, dtype=np.float32)
    rc = lib.oracle_minmax_hist(vol.ctypes.data, nx, ny, nz, layout, layout_brick, nbins,
                                rng.ctypes.data if rng is not None else None, C.byref(head), counts.ctypes.data)
    if rc != 0:
        raise ValueError(f"oracle_minmax_hist failed: {rc}")
    return Summary(np.float32(head.vmin), np.float32(head.vmax), int(head.n_nonfinite), int(head.n_below),
                   int(head.n_above), counts)


@dataclass
class Statistics:
    n_finite: int
    n_nonfinite: int
    mean: float                  # double
    stddev: float                # double, population
    median: np.float32           # lower median, a data value


def statistics(vol: np.ndarray, layout: int = LINEAR, layout_brick: int = 0, dims=None) -> Statistics:
    lib = _load()
    assert vol.dtype == np.float32 and vol.flags["C_CONTIGUOUS"]
    if layout == LINEAR:
        nz, ny, nx = vol.shape
    else:
        nx, ny, nz = dims
    st = _Stats()
    rc = lib.oracle_statistics(vol.ctypes.data, nx, ny, nz, layout, layout_brick, C.byref(st))
    if rc != 0:
        raise ValueError(f"oracle_statistics failed: {rc}")
    return Statistics(int(st.n_finite), int(st.n_nonfinite), float(st.mean), float(st.stddev), np.float32(st.median))


def encode_rgba8(image: np.ndarray, mode: int, background=(0.0, 0.0, 0.0), vmin: float = 0.0, vmax: float = 1.0) -> np.ndarray:
    """C.14 (S40): 8-bit RGBA frame of an EA image (H,W,4) composited over an opaque background, or of a MIP image
    (H,W) as a grey ramp over [vmin, vmax]."""
    lib = _load()
    img = np.ascontiguousarray(image, dtype=np.float32)
    H, W = img.shape[:2]
    assert img.shape == ((H, W, 4) if mode == EA else (H, W))
    bg = np.asarray(background, dtype=np.float32)
    out = np.empty((H, W, 4), dtype=np.uint8)
    lib.oracle_encode_rgba8.restype = C.c_int
    lib.oracle_encode_rgba8.argtypes = [C.c_void_p, C.c_uint32, C.c_uint32, C.c_uint64, C.c_int, C.c_void_p, C.c_float,
                                        C.c_float, C.c_void_p]
    rc = lib.oracle_encode_rgba8(img.ctypes.data, W, H, W * (4 if mode == EA else 1), mode, bg.ctypes.data,
                                 float(vmin), float(vmax), out.ctypes.data)
    if rc != 0:
        raise ValueError(f"oracle_encode_rgba8 failed: {rc}")
    return out
