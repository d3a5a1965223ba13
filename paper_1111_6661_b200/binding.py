"""Thin ctypes binding of libvr.so (include/vr.h) — argument marshalling only.

Every step of the path runs in the CUDA kernels of csrc/; this module converts tensors to raw
pointers and structs, nothing else.  There is NO CPU fallback: if the shared library is missing
or no CUDA device is present, calls raise.  torch is used for device memory and streams only.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

from . import _build

VR_OK, VR_ERR_INVALID_ARG, VR_ERR_UNSUPPORTED, VR_ERR_OUT_OF_MEMORY, VR_ERR_CUDA, VR_ERR_NOT_READY = range(6)
VR_LINEAR, VR_BRICKED_HALO1 = 0, 1
VR_DEVICE, VR_HOST_PINNED = 0, 1
VR_EA, VR_MIP = 0, 1
VR_SORT_LAST = 1


def VR_SUBSAMPLE(stride: int, phase_x: int = 0, phase_y: int = 0) -> int:
    """vr_camera.flags of a progressive pass (include/vr.h)."""
    return (int(stride) << 8) | (int(phase_x) << 16) | (int(phase_y) << 24)

VR_OPT_RENDER_PATH, VR_OPT_ZFAST_COPY, VR_OPT_LANE_LAG, VR_OPT_EMPTY_SKIP, VR_OPT_FORCE_WIDE, VR_OPT_ROW_LOADS, VR_OPT_TILE_SHEAR = 1, 2, 3, 4, 5, 6, 7
VR_PATH_AUTO, VR_PATH_RAY_MAJOR = 0, 1

_STATUS = {0: "VR_OK", 1: "VR_ERR_INVALID_ARG", 2: "VR_ERR_UNSUPPORTED", 3: "VR_ERR_OUT_OF_MEMORY",
           4: "VR_ERR_CUDA", 5: "VR_ERR_NOT_READY"}


class VrError(RuntimeError):
    def __init__(self, status: int, message: str):
        super().__init__(f"{_STATUS.get(status, status)}: {message}")
        self.status = status


class vr_volume_desc(C.Structure):
    _fields_ = [("struct_size", C.c_uint32), ("nx", C.c_uint32), ("ny", C.c_uint32), ("nz", C.c_uint32),
                ("brick", C.c_uint32), ("layout", C.c_uint32), ("location", C.c_uint32),
                ("n_copy_streams", C.c_uint32), ("data", C.c_void_p), ("resident_bytes", C.c_uint64)]


class vr_camera(C.Structure):
    _fields_ = [("struct_size", C.c_uint32), ("width", C.c_uint32), ("height", C.c_uint32),
                ("o0", C.c_float * 3), ("ou", C.c_float * 3), ("ov", C.c_float * 3),
                ("d0", C.c_float * 3), ("du", C.c_float * 3), ("dv", C.c_float * 3),
                ("step", C.c_float), ("ert_alpha", C.c_float), ("flags", C.c_uint32)]


class vr_image(C.Structure):
    _fields_ = [("struct_size", C.c_uint32), ("channels", C.c_uint32), ("location", C.c_uint32),
                ("reserved", C.c_uint32), ("pixels", C.c_void_p), ("row_pitch_bytes", C.c_uint64)]


class vr_stats(C.Structure):
    _fields_ = [("struct_size", C.c_uint32), ("n_bricks", C.c_uint32), ("bricks_drawn", C.c_uint32),
                ("bricks_culled", C.c_uint32), ("path", C.c_uint32), ("kernel_launches", C.c_uint32),
                ("fragments", C.c_uint64), ("h2d_bytes", C.c_uint64), ("d2h_bytes", C.c_uint64),
                ("total_kernel_launches", C.c_uint64), ("resident_bytes", C.c_uint64),
                ("zfast_copy", C.c_uint32), ("skip_variant", C.c_uint32), ("bricks_empty", C.c_uint32),
                ("quad_launches", C.c_uint32), ("macro_cells", C.c_uint64),
                ("empty_cells", C.c_uint64)]


class vr_statistics_result(C.Structure):
    _fields_ = [("n_finite", C.c_uint64), ("n_nonfinite", C.c_uint64), ("mean", C.c_double), ("stddev", C.c_double),
                ("median", C.c_float), ("reserved", C.c_uint32)]


class vr_encode_desc(C.Structure):
    _fields_ = [("struct_size", C.c_uint32), ("width", C.c_uint32), ("height", C.c_uint32), ("mode", C.c_uint32),
                ("background", C.c_float * 3), ("vmin", C.c_float), ("vmax", C.c_float)]


EXPORTS = ("vr_create_volume", "vr_destroy_volume", "vr_set_transfer_function", "vr_render",
           "vr_minmax_histogram", "vr_statistics", "vr_encode_rgba8", "vr_get_stats", "vr_set_option", "vr_last_error", "vr_version")

_lib = None


def library_path() -> str:
    return _build.LIB


def _declare(lib):
    """ctypes signatures of the entry points of include/vr.h."""
    if True:
        lib.vr_create_volume.restype = C.c_int
        lib.vr_create_volume.argtypes = [C.POINTER(vr_volume_desc), C.POINTER(C.c_void_p)]
        lib.vr_destroy_volume.restype = C.c_int
        lib.vr_destroy_volume.argtypes = [C.c_void_p]
        lib.vr_set_transfer_function.restype = C.c_int
        lib.vr_set_transfer_function.argtypes = [C.c_void_p, C.c_void_p, C.c_float, C.c_float]
        lib.vr_render.restype = C.c_int
        lib.vr_render.argtypes = [C.c_void_p, C.POINTER(vr_camera), C.c_int, C.POINTER(vr_image), C.c_void_p]
        lib.vr_minmax_histogram.restype = C.c_int
        lib.vr_minmax_histogram.argtypes = [C.c_void_p, C.c_uint32, C.c_void_p, C.c_void_p, C.c_uint32, C.c_void_p]
        lib.vr_statistics.restype = C.c_int
        lib.vr_statistics.argtypes = [C.c_void_p, C.c_void_p, C.c_uint32, C.c_void_p]
        lib.vr_encode_rgba8.restype = C.c_int
        lib.vr_encode_rgba8.argtypes = [C.c_void_p, C.POINTER(vr_encode_desc), C.POINTER(vr_image), C.c_void_p,
                                        C.c_uint64, C.c_uint32, C.c_void_p]
        lib.vr_get_stats.restype = C.c_int
        lib.vr_get_stats.argtypes = [C.c_void_p, C.POINTER(vr_stats)]
        lib.vr_set_option.restype = C.c_int
        lib.vr_set_option.argtypes = [C.c_void_p, C.c_uint32, C.c_int64]
        lib.vr_last_error.restype = C.c_char_p
        lib.vr_version.restype = C.c_char_p
    return lib


def load():
    """dlopen libvr.so (building it with nvcc first if it is missing or stale).  There is nothing else to load:
    no CPU implementation exists behind this binding."""
    global _lib
    if _lib is None:
        _lib = _declare(C.CDLL(_build.build()))
    return _lib


def _check(rc: int):
    if rc != VR_OK:
        raise VrError(rc, load().vr_last_error().decode())


def vr_version() -> str:
    return load().vr_version().decode()


def vr_last_error() -> str:
    return load().vr_last_error().decode()


def _stream_ptr(stream) -> C.c_void_p:
    if stream is None:
        import torch
        stream = torch.cuda.current_stream()
    if hasattr(stream, "cuda_stream"):
        return C.c_void_p(stream.cuda_stream)
    return C.c_void_p(int(stream))


def make_camera(cam) -> vr_camera:
    """workload.Camera (or anything with .vectors(), width, height, step, ert_alpha, flags) -> struct."""
    c = vr_camera()
    c.struct_size = C.sizeof(vr_camera)
    c.width, c.height = int(cam.width), int(cam.height)
    v = np.asarray(cam.vectors(), dtype=np.float32)
    for name, row in zip(("o0", "ou", "ov", "d0", "du", "dv"), v):
        setattr(c, name, (C.c_float * 3)(*[float(x) for x in row]))
    c.step, c.ert_alpha, c.flags = float(cam.step), float(cam.ert_alpha), int(cam.flags)
    return c


def summary_dtype(nbins: int) -> np.dtype:
    return np.dtype([("vmin", np.float32), ("vmax", np.float32), ("n_nonfinite", np.uint64),
                     ("n_below", np.uint64), ("n_above", np.uint64), ("counts", np.uint64, (nbins,))])


STATISTICS_DTYPE = np.dtype([("n_finite", np.uint64), ("n_nonfinite", np.uint64), ("mean", np.float64),
                             ("stddev", np.float64), ("median", np.float32), ("reserved", np.uint32)])


class Volume:
    """Owner of one vr_volume handle.  `data` is a CUDA float32 tensor (VR_DEVICE) or a pinned CPU
    float32 tensor (VR_HOST_PINNED); it is borrowed and kept alive by this object."""

    def __init__(self, data, dims, brick: int = 0, layout: int = VR_LINEAR, resident_bytes: int = 0,
                 n_copy_streams: int = 0):
        lib = load()
        nx, ny, nz = (int(d) for d in dims)
        self._data = data
        self.dims = (nx, ny, nz)
        d = vr_volume_desc()
        d.struct_size = C.sizeof(vr_volume_desc)
        d.nx, d.ny, d.nz, d.brick, d.layout = nx, ny, nz, int(brick), int(layout)
        d.location = VR_DEVICE if data.is_cuda else VR_HOST_PINNED
        d.n_copy_streams = int(n_copy_streams)
        d.data = data.data_ptr()
        d.resident_bytes = int(resident_bytes)
        h = C.c_void_p()
        _check(lib.vr_create_volume(C.byref(d), C.byref(h)))
        self._h = h

    def close(self):
        if getattr(self, "_h", None):
            load().vr_destroy_volume(self._h)
            self._h = None
            self._data = None

    __del__ = close

    def __enter__(self):
        return self

    def __exit__(self, *a):
        self.close()

    # -- vr_set_transfer_function
    def set_transfer_function(self, rgba, vmin: float, vmax: float):
        tab = np.ascontiguousarray(rgba, dtype=np.float32)
        assert tab.shape == (256, 4)
        _check(load().vr_set_transfer_function(self._h, tab.ctypes.data, float(vmin), float(vmax)))

    # -- vr_render
    def render(self, cam, mode: int, out=None, stream=None):
        """Enqueue one frame.  `out`: CUDA or pinned-CPU float32 tensor (H,W,4) / (H,W); allocated on
        the device if None.  Returns the tensor (valid once the stream reaches this point)."""
        import torch
        ch = 4 if mode == VR_EA else 1
        if out is None:
            shape = (cam.height, cam.width, 4) if mode == VR_EA else (cam.height, cam.width)
            out = torch.empty(shape, dtype=torch.float32, device="cuda")
        im = vr_image()
        im.struct_size = C.sizeof(vr_image)
        im.channels = ch
        im.location = VR_DEVICE if out.is_cuda else VR_HOST_PINNED
        im.pixels = out.data_ptr()
        im.row_pitch_bytes = out.stride(0) * 4
        c = cam if isinstance(cam, vr_camera) else make_camera(cam)
        _check(load().vr_render(self._h, C.byref(c), int(mode), C.byref(im), _stream_ptr(stream)))
        return out

    # -- vr_minmax_histogram
    def minmax_histogram(self, nbins: int = 256, range_=None, out=None, stream=None):
        """Enqueue the summary pass.  `out`: uint8 tensor of VR_SUMMARY_BYTES(nbins) bytes (CUDA or
        pinned CPU); allocated on the device if None.  Returns the tensor; see read_summary()."""
        import torch
        nbytes = 32 + 8 * nbins
        if out is None:
            out = torch.empty(nbytes, dtype=torch.uint8, device="cuda")
        assert out.numel() * out.element_size() >= nbytes
        rng = None
        if range_ is not None:
            rng = (C.c_float * 2)(float(range_[0]), float(range_[1]))
        _check(load().vr_minmax_histogram(self._h, int(nbins), rng, out.data_ptr(),
                                          VR_DEVICE if out.is_cuda else VR_HOST_PINNED, _stream_ptr(stream)))
        return out

    @staticmethod
    def read_summary(buf, nbins: int = 256):
        """Synchronise and decode a summary buffer into a numpy record."""
        import torch
        if buf.is_cuda:
            torch.cuda.current_stream().synchronize()
            buf = buf.cpu()
        return np.frombuffer(buf.numpy().tobytes()[: 32 + 8 * nbins], dtype=summary_dtype(nbins))[0]

    # -- vr_statistics
    def statistics(self, out=None, stream=None):
        """Enqueue the mean / standard deviation / median passes.  `out`: uint8 tensor of 40 bytes (CUDA or pinned
        CPU); allocated on the device if None.  Returns the tensor; see read_statistics()."""
        import torch
        nbytes = C.sizeof(vr_statistics_result)
        if out is None:
            out = torch.empty(nbytes, dtype=torch.uint8, device="cuda")
        assert out.numel() * out.element_size() >= nbytes
        _check(load().vr_statistics(self._h, out.data_ptr(), VR_DEVICE if out.is_cuda else VR_HOST_PINNED,
                                    _stream_ptr(stream)))
        return out

    @staticmethod
    def read_statistics(buf):
        """Synchronise and decode a statistics buffer into a numpy record."""
        import torch
        if buf.is_cuda:
            torch.cuda.current_stream().synchronize()
            buf = buf.cpu()
        return np.frombuffer(buf.numpy().tobytes()[: C.sizeof(vr_statistics_result)], dtype=STATISTICS_DTYPE)[0]

    # -- vr_encode_rgba8
    def encode_rgba8(self, image, mode: int, out, background=(0.0, 0.0, 0.0), vmin: float = 0.0, vmax: float = 1.0,
                     stream=None):
        """Enqueue the 8-bit frame of a rendered device image.  `out`: uint8 tensor (H,W,4), CUDA or pinned CPU."""
        H, W = int(image.shape[0]), int(image.shape[1])
        d = vr_encode_desc()
        d.struct_size = C.sizeof(vr_encode_desc)
        d.width, d.height, d.mode = W, H, int(mode)
        d.background = (C.c_float * 3)(*[float(x) for x in background])
        d.vmin, d.vmax = float(vmin), float(vmax)
        im = vr_image()
        im.struct_size = C.sizeof(vr_image)
        im.channels = 4 if mode == VR_EA else 1
        im.location = VR_DEVICE
        im.pixels = image.data_ptr()
        im.row_pitch_bytes = image.stride(0) * 4
        _check(load().vr_encode_rgba8(self._h, C.byref(d), C.byref(im), out.data_ptr(), out.stride(0),
                                      VR_DEVICE if out.is_cuda else VR_HOST_PINNED, _stream_ptr(stream)))
        return out

    # -- vr_set_option
    def set_option(self, option: int, value: int):
        _check(load().vr_set_option(self._h, int(option), int(value)))

    # -- vr_get_stats
    def stats(self) -> dict:
        s = vr_stats()
        s.struct_size = C.sizeof(vr_stats)
        _check(load().vr_get_stats(self._h, C.byref(s)))
        return {k: int(getattr(s, k)) for k, _ in vr_stats._fields_ if k != "struct_size"}
