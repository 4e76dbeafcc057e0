"""Seeded synthetic inputs (scenes + cameras) for the Oblique-MERF render hot path.

This package is the ONLY thing the CPU oracle (`oracle/`) and the CUDA path
(`paper_2404_09531_b200/`) have in common, and they share it as *data*: it holds none
of the method's arithmetic (no ray generation, no interpolation, no compositing,
no MLP evaluation, no pyramid, no bitfield).  It only draws random arrays with the
shapes / value distributions BASELINE.json's configs describe and places pinhole
cameras.
"""
from .scenes import (  # noqa: F401
    Scene,
    make_scene,
    make_cameras,
    config_resolution,
    custom_scene,
    look_at_camera,
    low_altitude_cameras,
    orbit_cameras,
    smoothed_bytes,
    smoothness_batch,
    CAMERA_FLOATS,
)
