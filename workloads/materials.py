"""Material parameter sets handed identically to the oracle and to the CUDA library.

PAPER.md prints no material constant (PAPER.md:181-183 defers to constraints.csv / ref [7],
both unavailable); these are the builder-chosen defaults of SURVEY.md section 8(d)
(reading A-3, A-4, A-12).  Units: um, us, pg  =>  force nN, surface modulus 1e-3 N/m.
"""
from __future__ import annotations

from .shapes import mesh_volume

# order of the C struct npfem_material / oracle_material (all doubles)
MATERIAL_FIELDS = (
    "cell_mass", "k_strain", "s_min", "s_max", "k_area", "a_min", "a_max",
    "k_bend", "w_volume", "v_min", "v_max", "c_alpha", "c_beta", "w_collision", "d_collision",
    "strain_hardening",
)

DENSITY_PG_PER_UM3 = 1.125          # 1125 kg/m^3 (A-4)


def default_material(rest_xyz, tris, **overrides) -> dict:
    """Default material of SURVEY.md 8(d): all clamp bands [1,1], cell_mass = rho * V0."""
    mat = dict(
        cell_mass=DENSITY_PG_PER_UM3 * mesh_volume(rest_xyz, tris),
        k_strain=0.1, s_min=1.0, s_max=1.0,
        k_area=0.5, a_min=1.0, a_max=1.0,
        k_bend=2e-4,
        w_volume=0.5, v_min=1.0, v_max=1.0,
        c_alpha=0.0, c_beta=0.0,
        w_collision=0.0, d_collision=0.0,
        strain_hardening=0.0,
        w_garea=0.0, ga_min=1.0, ga_max=1.0,
    )
    for k, v in overrides.items():
        if k not in mat:
            raise KeyError(k)
        mat[k] = float(v)
    return mat
