"""Rest shapes: unit-sphere meshes mapped to an RBC biconcave disc or a platelet ellipsoid.

BASELINE.json configs: RBC = "biconcave Evans-Fung disc of diameter 8 um and thickness 2 um";
platelet = "oblate ellipsoid 3.6 x 3.6 x 1 um".  The paper itself prints no shape formula
(PAPER.md:163 only says meshes come from "scripts using formulas"); SURVEY.md A-16 fixes the
reading used here.  Units: micrometres.
"""
from __future__ import annotations

import numpy as np

from .mesh import icosphere

# Evans-Fung profile coefficients (dimensionless, profile written in units of the diameter D)
_EF = (0.0518, 2.0026, -4.491)


def _ef_half_thickness(rho_over_d: np.ndarray) -> np.ndarray:
    """z/D of the unscaled Evans-Fung profile at radial distance rho/D (0 <= rho/D <= 1/2)."""
    q = rho_over_d * rho_over_d
    root = np.sqrt(np.clip(1.0 - 4.0 * q, 0.0, None))
    return root * (_EF[0] + _EF[1] * q + _EF[2] * q * q)


def rbc_biconcave(unit_verts: np.ndarray, diameter: float = 8.0,
                  thickness: float = 2.0) -> np.ndarray:
    """Map unit-sphere points to the biconcave disc.

    (X,Y,Z) -> (X*D/2, Y*D/2, sign(Z)*z(rho)), rho = (D/2)*sqrt(X^2+Y^2); the profile is
    scaled so that the maximum thickness max_rho 2 z(rho) equals `thickness` exactly.
    Equator vertices (Z == 0) land on z = 0, so the surface stays closed.
    """
    grid = np.linspace(0.0, 0.5, 200001)
    zmax = float(_ef_half_thickness(grid).max())          # in units of D
    c = (0.5 * thickness / diameter) / zmax
    x = unit_verts[:, 0] * (diameter * 0.5)
    y = unit_verts[:, 1] * (diameter * 0.5)
    rho_over_d = 0.5 * np.sqrt(unit_verts[:, 0] ** 2 + unit_verts[:, 1] ** 2)
    z = np.sign(unit_verts[:, 2]) * c * diameter * _ef_half_thickness(rho_over_d)
    return np.stack([x, y, z], axis=1)


def platelet_ellipsoid(unit_verts: np.ndarray,
                       axes: tuple[float, float, float] = (3.6, 3.6, 1.0)) -> np.ndarray:
    """Oblate ellipsoid with full axes `axes` (um): unit sphere scaled by axes/2."""
    return unit_verts * (np.asarray(axes, dtype=np.float64) * 0.5)


def mesh_volume(verts: np.ndarray, tris: np.ndarray) -> float:
    """Signed enclosed volume of a closed oriented mesh (used only to set the cell mass input)."""
    a, b, c = verts[tris[:, 0]], verts[tris[:, 1]], verts[tris[:, 2]]
    return float(np.einsum("ij,ij->i", a, np.cross(b, c)).sum() / 6.0)


def cell_diameter(verts: np.ndarray) -> float:
    """Largest axis-aligned extent of the rest shape (8 um RBC, 3.6 um platelet)."""
    return float((verts.max(axis=0) - verts.min(axis=0)).max())


def rest_shape(kind: str, level: int | None = None) -> tuple[np.ndarray, np.ndarray]:
    """(rest_xyz float64 [V,3], tris int32 [T,3]) for kind in {"rbc", "plt"}.

    Default levels follow BASELINE.json: RBC level 3 (642 vertices), platelet level 1 (42).
    """
    if kind == "rbc":
        v, t = icosphere(3 if level is None else level)
        return rbc_biconcave(v), t
    if kind == "plt":
        v, t = icosphere(1 if level is None else level)
        return platelet_ellipsoid(v), t
    raise ValueError(f"unknown cell kind {kind!r}")
