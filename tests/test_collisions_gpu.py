"""NEXT-3 on the GPU: collision constraint with neighbour input (npfem_step_collide), the
cell-packing workload and the area per surface vertex (npfem_vertex_areas).

PAPER.md:103 (the coupling hands "external forces & colliding neighbours" to the solid solver),
:129-133 (cell packing: random placements at rest shape, the solver resolves the overlaps),
:145 (collisions_weight), :226 (area per surface vertex); reading A-22.
"""
import numpy as np
import pytest
import torch

import workloads as W
from oracle import npfem_oracle as O
from paper_2011_04332_b200.harness import DeviceGroup
from tests.parity_util import displacement_tolerance, max_abs_err

pytestmark = pytest.mark.gpu


class _G:
    def __init__(self, rest, pos0):
        self.rest, self.pos0 = rest, pos0


def _packed_cells(n_cells, box, seed, level=2, **mat_over):
    rest, tris = W.rest_shape("rbc", level)
    mat = W.default_material(rest, tris, **mat_over)
    rng = np.random.Generator(np.random.PCG64([seed, 3]))
    rot, trans = W.random_rigid_placements(n_cells, box, 4.0, rng)
    trans = trans + 50.0                                           # away from the origin: world offsets
    pos0 = W.place_cells(rest, rot, trans)
    return rest, tris, mat, pos0


def test_collide_step_matches_the_oracle_on_overlapping_cells():
    """12 RBC-2 cells thrown into a 14 um box overlap heavily; the neighbour input is generated once
    from the initial positions and held fixed, so both paths see identical inputs."""
    rest, tris, mat, pos0 = _packed_cells(12, 14.0, 81, w_collision=2.0, d_collision=0.05)
    q, nrm = W.colliding_neighbours(pos0, tris, cutoff=0.8)
    active = (nrm != 0).any(axis=2)
    assert 0.05 < active.mean() < 0.95                               # some vertices collide, some do not
    assert W.penetration_count(pos0, q, nrm) > 50
    vel0 = np.zeros_like(pos0)
    f = W.gaussian_forces(pos0.shape, 1e-3, 81, 0)
    dg = DeviceGroup(tris, rest, mat, 0.1, pos0, vel0)
    dg.set_forces(f)
    oc = O.OracleCell(tris, rest, mat, 0.1)
    po, vo = pos0.astype(np.float64), vel0.astype(np.float64)
    g = _G(rest, pos0)
    diam = W.shapes.cell_diameter(rest)
    for step in range(4):
        dg.step_collide(q, nrm, 12)
        prev = po
        po, vo = oc.step_collide(po, vo, f, q, nrm, 12)
        pg, vg = dg.state()
        err = max_abs_err(pg, po)
        assert err <= 1e-4 * diam, f"step {step}: {err:.3e}"
        dx_o = po - prev
        derr = np.abs(vg.astype(np.float64) * 0.1 - dx_o).max()
        assert derr <= displacement_tolerance(g, np.abs(dx_o).max(), err, step), f"step {step}: {derr:.3e}"
    # and the contacts really acted: the same run without neighbours ends somewhere else
    dg0 = DeviceGroup(tris, rest, mat, 0.1, pos0, vel0)
    dg0.set_forces(f)
    for _ in range(4):
        dg0.step(12)
    assert np.abs(dg0.state()[0] - pg).max() > 1e-3


def test_free_cell_pressed_on_a_wall_reaches_the_closed_form_gap_on_the_gpu():
    """P-23 on the CUDA path: no elasticity, force f towards the wall, every vertex has the wall as
    neighbour: equilibrium gap = d - |f| / w_c."""
    rest, tris = W.rest_shape("plt", 1)
    wc, d, fmag = 2.0, 0.05, 1e-2
    mat = W.default_material(rest, tris, k_strain=0, k_area=0, k_bend=0, w_volume=0, c_alpha=2.0,
                             w_collision=wc, d_collision=d)
    n = rest.shape[0]
    n_cells = 3
    pos0 = np.stack([rest + np.array([3.0 * c, 0.0, 0.3 - rest[:, 2].min()]) for c in range(n_cells)]).astype(np.float32)
    nrm = np.zeros((n_cells, n, 3), dtype=np.float32); nrm[..., 2] = 1.0
    q = np.zeros_like(nrm)
    f = np.zeros_like(nrm); f[..., 2] = -fmag
    dg = DeviceGroup(tris, rest, mat, 0.1, pos0, np.zeros_like(pos0))
    dg.set_forces(f)
    qd = torch.as_tensor(q); nd = torch.as_tensor(nrm)
    for _ in range(1500):
        dg.step_collide(qd, nd, 3)
    pg, vg = dg.state()
    assert np.abs(vg).max() < 1e-6
    assert np.abs(pg[..., 2] - (d - fmag / wc)).max() < 2e-5


def test_cell_packing_resolves_overlaps():
    """cells placed at random positions and orientations at their rest shape
    overlap; running the solid solver with collision neighbours (regenerated every few steps, as the
    coupling framework would) and some damping drives the interpenetration down."""
    rest, tris, mat, pos0 = _packed_cells(24, 18.0, 82, w_collision=4.0, d_collision=0.1, c_alpha=1.0)
    dg = DeviceGroup(tris, rest, mat, 0.1, pos0, np.zeros_like(pos0))
    q, nrm = W.colliding_neighbours(pos0, tris, cutoff=1.0)
    before = W.penetration_count(pos0, q, nrm)
    depth0 = -np.minimum(((pos0.astype(np.float64) - q) * nrm).sum(axis=2), 0).sum()
    assert before > 200
    for it in range(60):
        dg.step_collide(q, nrm, 10)
        if it % 5 == 4:
            q, nrm = W.colliding_neighbours(dg.state()[0], tris, cutoff=1.0)
    pg, _ = dg.state()
    q, nrm = W.colliding_neighbours(pg, tris, cutoff=1.0)
    after = W.penetration_count(pg, q, nrm)
    depth1 = -np.minimum(((pg.astype(np.float64) - q) * nrm).sum(axis=2), 0).sum()
    print(f"[packing] penetrating vertices {before} -> {after}, summed depth {depth0:.2f} -> {depth1:.2f} um")
    assert np.isfinite(pg).all()
    assert depth1 < 0.5 * depth0 and after < before


def test_vertex_areas_match_the_oracle():
    rest, tris, mat, pos0 = _packed_cells(9, 60.0, 83, level=3)
    pos0 = (pos0 * np.linspace(0.8, 1.3, 9)[:, None, None]).astype(np.float32)     # different sizes
    dg = DeviceGroup(tris, rest, mat, 0.1, pos0, np.zeros_like(pos0))
    a = dg.vertex_areas()
    oc = O.OracleCell(tris, rest, mat, 0.1)
    for c in range(9):
        ref = oc.vertex_areas(pos0[c].astype(np.float64))
        assert np.abs(a[c] - ref).max() <= 2e-5 * ref.max()
