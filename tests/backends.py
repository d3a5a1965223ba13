"""The two ways the parity tests execute the library's CUDA sources.

`gpu`  — the product: libvr.so (nvcc, sm_100a) on a CUDA device, tensors from torch.  Marked `gpu`.
`simt` — TEST INFRASTRUCTURE: the same .cu sources (kernels and host runtime) compiled by g++ against
         tests/simt/simt_host.h and executed thread by thread on the host (fibers, real barriers and warp
         collectives, guard pages around every device allocation).  Runs without a GPU; covers the logic,
         the addressing and the arithmetic of the kernels, not their timing.
Both go through the same ctypes binding and the same C ABI."""
from __future__ import annotations

import contextlib
import os
import sys

import numpy as np
import pytest

import paper_1111_6661_b200 as vr

sys.path.insert(0, os.path.join(os.path.dirname(os.path.abspath(__file__)), "simt"))


class GpuBackend:
    name = "gpu"
    full = True                      # run the complete case matrix

    def ctx(self):
        return contextlib.nullcontext()

    def dev(self, a):
        import torch
        return torch.from_numpy(np.ascontiguousarray(a)).cuda()

    def pinned(self, a):
        import torch
        return torch.from_numpy(np.ascontiguousarray(a)).pin_memory()

    def empty(self, shape, dtype=np.float32, device=True, fill=None):
        import torch
        t = torch.empty(tuple(shape), dtype={np.float32: torch.float32, np.uint8: torch.uint8}[dtype],
                        device="cuda" if device else "cpu")
        if not device:
            t = t.pin_memory()
        if fill is not None:
            t.fill_(fill)
        return t

    def numpy(self, t):
        import torch
        torch.cuda.synchronize()
        return t.cpu().numpy()

    stream = None                    # torch's current stream

    def sync(self):
        import torch
        torch.cuda.synchronize()


class SimtBackend:
    name = "simt"
    full = False                     # reduced case matrix: the emulation runs ~1e6 samples per second

    def ctx(self):
        import simt_lib
        return simt_lib.emulated()

    def dev(self, a):
        import simt_lib
        return simt_lib.Buffer.of(a, device=True)

    def pinned(self, a):
        import simt_lib
        return simt_lib.Buffer.of(a, device=False)

    def empty(self, shape, dtype=np.float32, device=True, fill=None):
        import simt_lib
        return simt_lib.Buffer(shape, dtype, device, fill)

    def numpy(self, t):
        return np.array(t.array, copy=True)

    stream = 0                       # the emulated runtime has no streams to pick from

    def sync(self):
        pass


def render(be, vol, cam, mode, out=None, stream=None):
    """vr_render into a (new) device image; returns it as a numpy array."""
    if out is None:
        shape = (cam.height, cam.width, 4) if mode == vr.VR_EA else (cam.height, cam.width)
        out = be.empty(shape)
    vol.render(cam, mode, out=out, stream=be.stream if stream is None else stream)
    return be.numpy(out)


def summary(be, vol, nbins=256, range_=None, device=True):
    buf = be.empty((32 + 8 * nbins,), np.uint8, device=device)
    vol.minmax_histogram(nbins, range_, out=buf, stream=be.stream)
    raw = be.numpy(buf)
    return np.frombuffer(np.ascontiguousarray(raw).tobytes()[: 32 + 8 * nbins], dtype=vr.summary_dtype(nbins))[0]


def statistics(be, vol, device=True):
    buf = be.empty((40,), np.uint8, device=device)
    vol.statistics(out=buf, stream=be.stream)
    raw = be.numpy(buf)
    return np.frombuffer(np.ascontiguousarray(raw).tobytes()[:40], dtype=vr.STATISTICS_DTYPE)[0]


BACKENDS = {"gpu": GpuBackend(), "simt": SimtBackend()}
BACKEND_PARAMS = [pytest.param("gpu", marks=pytest.mark.gpu), pytest.param("simt")]


@pytest.fixture(params=BACKEND_PARAMS)
def be(request):
    b = BACKENDS[request.param]
    with b.ctx():
        yield b
