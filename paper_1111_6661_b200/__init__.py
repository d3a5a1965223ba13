"""paper_1111_6661_b200 — B200-native bricked volume ray-casting + min/max/histogram (libvr.so).

The product is the C-ABI shared library declared in include/vr.h (CUDA kernels in csrc/);
this package is its thin Python binding.  No CPU fallback exists: importing works anywhere,
but every compute call needs the built library and a CUDA device.
"""
from .binding import (Volume, VrError, load, library_path, make_camera, summary_dtype, STATISTICS_DTYPE, vr_version, vr_last_error,
                      EXPORTS, VR_EA, VR_MIP, VR_LINEAR, VR_BRICKED_HALO1, VR_DEVICE, VR_HOST_PINNED, VR_SORT_LAST, VR_SUBSAMPLE,
                      VR_OPT_RENDER_PATH, VR_OPT_ZFAST_COPY, VR_OPT_LANE_LAG, VR_OPT_EMPTY_SKIP, VR_OPT_FORCE_WIDE, VR_OPT_ROW_LOADS, VR_OPT_TILE_SHEAR, VR_PATH_AUTO, VR_PATH_RAY_MAJOR,
                      VR_OK, VR_ERR_INVALID_ARG, VR_ERR_UNSUPPORTED, VR_ERR_OUT_OF_MEMORY, VR_ERR_CUDA,
                      VR_ERR_NOT_READY)

__all__ = ["Volume", "VrError", "load", "library_path", "make_camera", "summary_dtype", "STATISTICS_DTYPE", "vr_version",
           "vr_last_error", "EXPORTS", "VR_EA", "VR_MIP", "VR_LINEAR", "VR_BRICKED_HALO1", "VR_DEVICE",
           "VR_HOST_PINNED", "VR_SORT_LAST", "VR_SUBSAMPLE", "VR_OPT_RENDER_PATH", "VR_OPT_ZFAST_COPY", "VR_OPT_LANE_LAG", "VR_OPT_EMPTY_SKIP", "VR_OPT_FORCE_WIDE", "VR_OPT_ROW_LOADS", "VR_OPT_TILE_SHEAR", "VR_PATH_AUTO",
           "VR_PATH_RAY_MAJOR"]
