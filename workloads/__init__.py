"""Seeded synthetic inputs shared by the oracle tests, the GPU tests and bench.py.

This package holds data generators only: meshes, fields, scale lists.  None of the implicit filter's
arithmetic (stiffness, areas, solves, spectra) lives here; the oracle (oracle/) and the CUDA library
(paper_2404_07398_b200/) each implement that on their own and neither imports the other.
"""
from .configs import Workload, make_config
from .fields import Waves, log_spaced, planar_wave_field, sphere_frames, sphere_velocity_field, sphere_wave_field
from .meshes import (Mesh, delaunay_mesh, equilateral_mesh, grid_mesh, icosphere, icosphere_edge, jitter_sphere,
                     land_mask, sphere_band)

__all__ = ["Workload", "make_config", "Waves", "log_spaced", "planar_wave_field", "sphere_frames", "sphere_velocity_field", "sphere_wave_field",
           "Mesh", "delaunay_mesh", "equilateral_mesh", "grid_mesh", "icosphere", "icosphere_edge", "jitter_sphere",
           "land_mask", "sphere_band"]
