"""Icosphere surface meshes (closed, outward-oriented triangle meshes on the unit sphere).

Stand-in for the paper's template meshes (RBC 258 vertices, PLT 66 vertices, files
not available).  Level l has V = 10*4^l + 2 vertices, T = 20*4^l triangles, E = 30*4^l edges:
level 1 = 42/80 (platelet), level 2 = 162/320, level 3 = 642/1280 (RBC).
"""
from __future__ import annotations

import functools

import numpy as np


def mesh_counts(level: int) -> tuple[int, int, int]:
    """(n_verts, n_tris, n_edges) of the level-`level` icosphere."""
    f = 4 ** level
    return 10 * f + 2, 20 * f, 30 * f


def _icosahedron() -> tuple[np.ndarray, np.ndarray]:
    phi = (1.0 + np.sqrt(5.0)) / 2.0
    v = np.array(
        [[-1, phi, 0], [1, phi, 0], [-1, -phi, 0], [1, -phi, 0],
         [0, -1, phi], [0, 1, phi], [0, -1, -phi], [0, 1, -phi],
         [phi, 0, -1], [phi, 0, 1], [-phi, 0, -1], [-phi, 0, 1]], dtype=np.float64)
    v /= np.linalg.norm(v, axis=1, keepdims=True)
    t = np.array(
        [[0, 11, 5], [0, 5, 1], [0, 1, 7], [0, 7, 10], [0, 10, 11],
         [1, 5, 9], [5, 11, 4], [11, 10, 2], [10, 7, 6], [7, 1, 8],
         [3, 9, 4], [3, 4, 2], [3, 2, 6], [3, 6, 8], [3, 8, 9],
         [4, 9, 5], [2, 4, 11], [6, 2, 10], [8, 6, 7], [9, 8, 1]], dtype=np.int32)
    return v, t


@functools.lru_cache(maxsize=8)
def _icosphere_cached(level: int):
    verts, tris = _icosahedron()
    verts = [tuple(p) for p in verts]
    for _ in range(level):
        cache: dict[tuple[int, int], int] = {}

        def midpoint(i: int, j: int) -> int:
            key = (i, j) if i < j else (j, i)
            k = cache.get(key)
            if k is None:
                m = (np.asarray(verts[i]) + np.asarray(verts[j])) * 0.5
                m /= np.linalg.norm(m)
                k = len(verts)
                verts.append(tuple(m))
                cache[key] = k
            return k

        new_tris = []
        for a, b, c in tris:
            ab, bc, ca = midpoint(a, b), midpoint(b, c), midpoint(c, a)
            new_tris += [[a, ab, ca], [b, bc, ab], [c, ca, bc], [ab, bc, ca]]
        tris = np.asarray(new_tris, dtype=np.int32)
    v = np.asarray(verts, dtype=np.float64)
    t = np.asarray(tris, dtype=np.int32)
    # orient outward: (b-a)x(c-a) . centroid > 0 on the unit sphere
    a, b, c = v[t[:, 0]], v[t[:, 1]], v[t[:, 2]]
    flip = np.einsum("ij,ij->i", np.cross(b - a, c - a), a + b + c) < 0
    t[flip] = t[flip][:, [0, 2, 1]]
    v.setflags(write=False)
    t.setflags(write=False)
    return v, t


def icosphere(level: int) -> tuple[np.ndarray, np.ndarray]:
    """Unit icosphere: (verts float64 [V,3], tris int32 [T,3]); deterministic vertex order."""
    if level < 0 or level > 6:
        raise ValueError("icosphere level must be in 0..6")
    v, t = _icosphere_cached(level)
    return v.copy(), t.copy()
