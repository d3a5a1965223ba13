"""TEST INFRASTRUCTURE: loads tests/simt/libvr_simt.so (the library's sources executed on the host, see
simt_host.h) behind the product's own ctypes binding, and provides buffers that stand in for device / pinned
tensors.  Only tests import this."""
from __future__ import annotations

import contextlib
import ctypes as C
import os
import sys

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, HERE)
import build_simt  # noqa: E402

import paper_1111_6661_b200.binding as B  # noqa: E402

_lib = None


def lib():
    global _lib
    if _lib is None:
        l = B._declare(C.CDLL(build_simt.build()))
        for name in ("simt_device_alloc", "simt_pinned_alloc"):
            getattr(l, name).restype = C.c_void_p
            getattr(l, name).argtypes = [C.c_size_t]
        l.simt_free.argtypes = [C.c_void_p]
        l.simt_device_bytes_in_use.restype = C.c_size_t
        l.simt_set_device_capacity.argtypes = [C.c_size_t]
        l.simt_trace.argtypes = [C.c_int]
        l.simt_trace_stat.restype = C.c_ulonglong
        l.simt_trace_stat.argtypes = [C.c_int]
        l.simt_counter.restype = C.c_ulonglong
        l.simt_counter.argtypes = [C.c_int]
        _lib = l
    return _lib


@contextlib.contextmanager
def emulated():
    """Within the block the binding's entry points are those of the host-emulated library."""
    old = B._lib
    B._lib = lib()
    try:
        yield
    finally:
        B._lib = old


class Buffer:
    """A float32/uint8 array in emulated device memory (is_cuda) or emulated pinned host memory, with the few
    tensor attributes the binding reads.  Guard pages surround it (simt_runtime.cpp)."""

    def __init__(self, shape, dtype=np.float32, device=True, fill=None):
        self.shape = tuple(int(s) for s in np.atleast_1d(shape))
        self.dtype = np.dtype(dtype)
        self.nbytes = int(np.prod(self.shape)) * self.dtype.itemsize
        self.is_cuda = bool(device)
        self._p = (lib().simt_device_alloc if device else lib().simt_pinned_alloc)(max(self.nbytes, 1))
        assert self._p
        self.array = np.ctypeslib.as_array((C.c_ubyte * max(self.nbytes, 1)).from_address(self._p))[: self.nbytes] \
            .view(self.dtype).reshape(self.shape)
        if fill is not None:
            self.array[...] = fill

    @classmethod
    def of(cls, a, device=True):
        a = np.ascontiguousarray(a)
        b = cls(a.shape, a.dtype, device)
        b.array[...] = a
        return b

    def data_ptr(self):
        return self._p

    def stride(self, d):
        return self.array.strides[d] // self.dtype.itemsize

    def numel(self):
        return int(np.prod(self.shape))

    def element_size(self):
        return self.dtype.itemsize

    def free(self):
        if self._p:
            self.array = None
            lib().simt_free(self._p)
            self._p = None

    def __del__(self):
        try:
            self.free()
        except Exception:
            pass


def read_summary(buf: Buffer, nbins: int = 256):
    return np.frombuffer(buf.array.tobytes()[: 32 + 8 * nbins], dtype=B.summary_dtype(nbins))[0]
