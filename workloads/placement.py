"""Random rigid placements of cells in a box ("Placement").

rotation = normalised 4-vector of seeded normals (unit quaternion); translation uniform so that
the whole cell stays inside the box.  Cells may overlap; they do not interact (collisions are out
of scope, "colliding neighbours" is a coupling input the product does not have).
"""
from __future__ import annotations

import numpy as np


def quat_to_rot(q: np.ndarray) -> np.ndarray:
    """Unit quaternions [N,4] (w,x,y,z) -> rotation matrices [N,3,3]."""
    w, x, y, z = q[:, 0], q[:, 1], q[:, 2], q[:, 3]
    r = np.empty((q.shape[0], 3, 3), dtype=np.float64)
    r[:, 0, 0] = 1 - 2 * (y * y + z * z)
    r[:, 0, 1] = 2 * (x * y - z * w)
    r[:, 0, 2] = 2 * (x * z + y * w)
    r[:, 1, 0] = 2 * (x * y + z * w)
    r[:, 1, 1] = 1 - 2 * (x * x + z * z)
    r[:, 1, 2] = 2 * (y * z - x * w)
    r[:, 2, 0] = 2 * (x * z - y * w)
    r[:, 2, 1] = 2 * (y * z + x * w)
    r[:, 2, 2] = 1 - 2 * (x * x + y * y)
    return r


def random_rigid_placements(n_cells: int, box: float, radius: float,
                            rng: np.random.Generator) -> tuple[np.ndarray, np.ndarray]:
    """(R [N,3,3], t [N,3]): seeded rotations and translations in [radius, box-radius]^3."""
    q = rng.standard_normal((n_cells, 4))
    q /= np.linalg.norm(q, axis=1, keepdims=True)
    t = rng.uniform(radius, box - radius, size=(n_cells, 3))
    return quat_to_rot(q), t


def place_cells(rest_xyz: np.ndarray, rot: np.ndarray, trans: np.ndarray,
                chunk: int = 4096) -> np.ndarray:
    """World positions float32 [N,V,3] = rest @ R^T + t, cast to fp32 once (both paths read these)."""
    n = rot.shape[0]
    out = np.empty((n, rest_xyz.shape[0], 3), dtype=np.float32)
    for s in range(0, n, chunk):
        e = min(n, s + chunk)
        out[s:e] = (np.einsum("vj,nij->nvi", rest_xyz, rot[s:e]) + trans[s:e, None, :]
                    ).astype(np.float32)
    return out
