"""Seeded synthetic inputs for the npFEM hot path (meshes, rest shapes, placements, forces).

This package holds INPUT GENERATORS ONLY: it contains none of the method's arithmetic (no
energies, projections, masses, system matrices or time stepping).  It is the single piece of
code that both the fp64 CPU oracle (``oracle/``) and the CUDA path
(``paper_2011_04332_b200/``) are allowed to share; it imports neither of them.

Recipe: SURVEY.md section 8(d) / DESIGN.md "Input recipe".  The paper ships
258-vertex RBC and 66-vertex PLT template meshes that are not available here; icospheres mapped
to a biconcave disc / oblate ellipsoid stand in for them.
"""
from .mesh import icosphere, mesh_counts
from .shapes import rbc_biconcave, platelet_ellipsoid, rest_shape
from .materials import default_material, MATERIAL_FIELDS
from .placement import random_rigid_placements, place_cells, quat_to_rot
from .forces import (gaussian_forces, fourier_shear_field, FourierField, cap_pull_forces,
                     cap_vertex_sets)
from .configs import CONFIGS, make_config, UNITS
from .packing import colliding_neighbours, penetration_count, vertex_normals

__all__ = [
    "icosphere", "mesh_counts", "rbc_biconcave", "platelet_ellipsoid", "rest_shape",
    "default_material", "MATERIAL_FIELDS", "random_rigid_placements", "place_cells",
    "quat_to_rot", "gaussian_forces", "fourier_shear_field", "FourierField", "cap_pull_forces",
    "cap_vertex_sets", "CONFIGS", "make_config", "UNITS", "colliding_neighbours", "penetration_count",
    "vertex_normals",
]
