"""Seeded synthetic workloads: cubes, cameras and transfer functions.

INPUT GENERATORS ONLY — this package holds none of the method's arithmetic and
imports neither ``oracle`` nor ``paper_1111_6661_b200``.  The same bytes it
produces are handed to the CPU oracle and to the CUDA library.

Stands in for the paper's spectral cubes (Table 1), which are
not available; recipes follow BASELINE.json ``configs`` and SURVEY.md §8(d).
"""
from .cubes import (Recipe, CubeGenerator, make_cube, checksum, retile_halo, bricked_halo_elems, fill_bricked_halo_ptr,
                    build as build_generator)
from .cameras import (Camera, ortho_axis_camera, perspective_camera, orbit_camera, ortho_lookat_camera,
                      nominal_samples)
from .transfer import TF_HAZE_POINTS, TF_SOURCES_POINTS, bake_tf, tf_haze, tf_opaque, tf_sources
from .configs import CONFIGS, WorkloadConfig, get_config

__all__ = [
    "Recipe", "CubeGenerator", "make_cube", "checksum", "retile_halo", "bricked_halo_elems", "fill_bricked_halo_ptr", "build_generator",
    "Camera", "ortho_axis_camera", "perspective_camera", "orbit_camera", "ortho_lookat_camera", "nominal_samples",
    "TF_HAZE_POINTS", "TF_SOURCES_POINTS", "bake_tf", "tf_haze", "tf_opaque", "tf_sources",
    "CONFIGS", "WorkloadConfig", "get_config",
]
