"""Colliding-neighbour input for the solid step (the coupling framework hands
"external forces & colliding neighbours" to npFEM; :129-133: the cell-packing application places
cells at random positions and orientations at their rest shape and lets the solver resolve the
overlaps).  In the paper the detection lives in the Palabos framework, outside npFEM; here it is an
input generator like the force fields: no arithmetic of the method lives in this file.

For every vertex: the nearest vertex of any OTHER cell within `cutoff`, returned as the contact
point q and that cell's outward unit vertex normal n at q (zero normal = no neighbour).
"""
from __future__ import annotations

import numpy as np
from scipy.spatial import cKDTree


def vertex_normals(pos: np.ndarray, tris: np.ndarray) -> np.ndarray:
    """Area-weighted outward unit normals per vertex, pos [N,V,3] -> [N,V,3] (float64)."""
    p = np.asarray(pos, dtype=np.float64)
    a, b, c = p[:, tris[:, 0]], p[:, tris[:, 1]], p[:, tris[:, 2]]
    fn = np.cross(b - a, c - a)                                   # [N,T,3], length 2 x area
    vn = np.zeros_like(p)
    for k in range(3):
        np.add.at(vn, (slice(None), tris[:, k]), fn)
    return vn / np.maximum(np.linalg.norm(vn, axis=2, keepdims=True), 1e-300)


def colliding_neighbours(pos: np.ndarray, tris: np.ndarray, cutoff: float):
    """(q, n) float32 [N,V,3] for positions pos [N,V,3]; vertices without a neighbour get n = 0."""
    p = np.asarray(pos, dtype=np.float64)
    n_cells, n_verts = p.shape[:2]
    flat = p.reshape(-1, 3)
    owner = np.repeat(np.arange(n_cells), n_verts)
    normals = vertex_normals(p, tris).reshape(-1, 3)
    tree = cKDTree(flat)
    q = np.zeros_like(flat)
    nrm = np.zeros_like(flat)
    # enough neighbours to get past the vertex's own cell (whose vertices are the closest ones)
    k = min(len(flat), 48)
    dist, idx = tree.query(flat, k=k, distance_upper_bound=cutoff)
    for j in range(k):
        ok = np.isfinite(dist[:, j]) & (idx[:, j] < len(flat))
        other = ok.copy()
        other[ok] &= owner[idx[ok, j]] != owner[ok]
        take = other & (nrm == 0).all(axis=1)
        q[take] = flat[idx[take, j]]
        nrm[take] = normals[idx[take, j]]
    return (q.reshape(p.shape).astype(np.float32), nrm.reshape(p.shape).astype(np.float32))


def penetration_count(pos: np.ndarray, q: np.ndarray, nrm: np.ndarray) -> int:
    """Number of vertices on the inner side of their neighbour's tangent plane (a packing metric)."""
    active = (np.asarray(nrm) != 0).any(axis=2)
    depth = ((np.asarray(pos, dtype=np.float64) - q) * nrm).sum(axis=2)
    return int((active & (depth < 0)).sum())
