"""The five BASELINE.json configurations as seeded synthetic workloads.

Units: um, us, pg (force nN, 1 pN = 1e-3); dt = 1e-7 s = 0.1 us.  The paper measures on no public
benchmark; these inputs stand in for its blood-cell suspensions (20-35 % hematocrit,
PAPER.md:113, 272).  A workload is a list of cell groups (one per cell TYPE = one shared system
matrix) plus a force recipe; everything is reproducible from (config id, cell indices).
"""
from __future__ import annotations

from dataclasses import dataclass, field
from typing import Callable

import numpy as np

from .forces import (PN, cap_pull_forces, fourier_shear_field, gaussian_forces)
from .materials import default_material
from .placement import place_cells, random_rigid_placements
from .shapes import cell_diameter, rest_shape

UNITS = {"length": "um", "time": "us", "mass": "pg", "force": "nN"}
DT = 0.1                      # 1e-7 s in us
FORCE_CHUNK = 256             # gaussian forces are drawn per (seed, step, chunk of 256 cells)

CONFIGS = {
    1: dict(name="config1_single_rbc2", groups=[("rbc", 2, 1)], box=None, seed=0,
            n_steps=1, n_iters=10, forces="gauss"),
    2: dict(name="config2_1k_rbc3_shear", groups=[("rbc", 3, 1000)], box=100.0, seed=1,
            n_steps=100, n_iters=20, forces="fourier"),
    3: dict(name="config3_mixed_rbc_plt", groups=[("rbc", 3, 1000), ("plt", 1, 500)], box=100.0,
            seed=2, n_steps=50, n_iters=20, forces="gauss"),
    4: dict(name="config4_100k_rbc3", groups=[("rbc", 3, 100_000)], box=300.0, seed=4,
            n_steps=10, n_iters=20, forces="gauss"),
    5: dict(name="config5_20k_rbc3_stretch", groups=[("rbc", 3, 20_000)], box=100.0, seed=5,
            n_steps=200, n_iters=30, forces="caps"),
}


@dataclass
class CellGroup:
    kind: str
    level: int
    rest: np.ndarray            # float64 [V,3]
    tris: np.ndarray            # int32 [T,3]
    material: dict
    diameter: float             # um; parity tolerance is 1e-4 * diameter (north_star)
    cells: np.ndarray           # global indices of the cells materialised here
    n_cells_full: int
    rot: np.ndarray             # float64 [N,3,3]
    trans: np.ndarray           # float64 [N,3]
    pos0: np.ndarray            # float32 [N,V,3]
    vel0: np.ndarray            # float32 [N,V,3] (zeros)
    seed: int = 0


@dataclass
class Workload:
    config: int
    name: str
    dt: float
    n_steps: int
    n_iters: int
    groups: list[CellGroup]
    force_fn: Callable[[int, int], np.ndarray] = field(repr=False, default=None)

    def forces(self, group: int, step: int) -> np.ndarray:
        """float32 [N,V,3] external forces on the materialised cells of `group` at `step`."""
        return self.force_fn(group, step)


def chunked_gaussian(cells: np.ndarray, n_verts: int, sigma: float, seed: int,
                     step: int) -> np.ndarray:
    """Gaussian forces for arbitrary global cell indices, identical to the full-suspension draw."""
    out = np.empty((len(cells), n_verts, 3), dtype=np.float32)
    chunks = cells // FORCE_CHUNK
    for ch in np.unique(chunks):
        block = gaussian_forces((FORCE_CHUNK, n_verts, 3), sigma, seed * 1_000_003 + int(ch), step)
        sel = np.nonzero(chunks == ch)[0]
        out[sel] = block[cells[sel] - ch * FORCE_CHUNK]
    return out


def make_config(config: int, cells: dict[int, np.ndarray] | int | None = None,
                n_steps: int | None = None) -> Workload:
    """Materialise config `config`.

    cells: None = every cell; an int k = the first k cells of every group; or
    {group index: array of global cell indices} for a parity subsample (placements and forces of
    a cell do not depend on which other cells are materialised).
    """
    spec = CONFIGS[config]
    groups: list[CellGroup] = []
    for gi, (kind, level, n_full) in enumerate(spec["groups"]):
        rest, tris = rest_shape(kind, level)
        diam = cell_diameter(rest)
        seed = spec["seed"] + gi
        if spec["box"] is None:                                   # config 1: one cell at the origin
            rot = np.eye(3)[None].repeat(n_full, axis=0)
            trans = np.zeros((n_full, 3))
        else:
            rng = np.random.Generator(np.random.PCG64([seed, 0xCE11]))
            radius = 0.5 * float(np.linalg.norm(rest, axis=1).max() * 2.0)
            rot, trans = random_rigid_placements(n_full, spec["box"], radius, rng)
        if cells is None:
            idx = np.arange(n_full)
        elif isinstance(cells, (int, np.integer)):
            idx = np.arange(min(int(cells), n_full))
        else:
            idx = np.asarray(cells.get(gi, np.arange(0)), dtype=np.int64)
        pos0 = place_cells(rest, rot[idx], trans[idx])
        groups.append(CellGroup(kind=kind, level=level, rest=rest, tris=tris,
                                material=default_material(rest, tris), diameter=diam,
                                cells=idx, n_cells_full=n_full, rot=rot[idx], trans=trans[idx],
                                pos0=pos0, vel0=np.zeros_like(pos0), seed=seed))

    kind_f = spec["forces"]
    if kind_f == "gauss":
        def force_fn(g: int, step: int) -> np.ndarray:
            grp = groups[g]
            return chunked_gaussian(grp.cells, grp.rest.shape[0], 1.0 * PN, grp.seed, step)
    elif kind_f == "fourier":
        field_ = fourier_shear_field(spec["seed"], box=spec["box"], amp=1.0 * PN)
        smooth = [field_(grp.pos0) for grp in groups]              # step-0 positions, held fixed

        def force_fn(g: int, step: int) -> np.ndarray:
            grp = groups[g]
            noise = chunked_gaussian(grp.cells, grp.rest.shape[0], 0.1 * PN, grp.seed, step)
            return (smooth[g] + noise).astype(np.float32)
    elif kind_f == "caps":
        pulls = [cap_pull_forces(grp.rest, grp.rot, 20.0 * PN) for grp in groups]

        def force_fn(g: int, step: int) -> np.ndarray:
            return pulls[g]
    else:
        raise ValueError(kind_f)

    return Workload(config=config, name=spec["name"], dt=DT,
                    n_steps=spec["n_steps"] if n_steps is None else int(n_steps),
                    n_iters=spec["n_iters"], groups=groups, force_fn=force_fn)
