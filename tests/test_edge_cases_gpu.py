"""GPU edge cases of the C ABI: empty and ragged inputs, strides, option variants, clamp bands,
degenerate iteration counts, the host-buffer entry point and run-to-run determinism."""
import numpy as np
import pytest
import torch

import workloads as W
from oracle import npfem_oracle as O
from paper_2011_04332_b200 import NpfemError, NpfemHandle
from paper_2011_04332_b200.harness import DeviceGroup, from_strided, to_strided
from tests.parity_util import displacement_tolerance, gpu_trajectory, max_abs_err, oracle_trajectory, position_tolerance

pytestmark = pytest.mark.gpu


def _small_workload(kind="rbc", level=2, n_cells=7, seed=7, sigma=1e-3, box=100.0, **mat_over):
    rest, tris = W.rest_shape(kind, level)
    mat = W.default_material(rest, tris, **mat_over)
    rng = np.random.Generator(np.random.PCG64([seed, 1]))
    rot, trans = W.random_rigid_placements(n_cells, box, 5.0, rng)
    pos0 = W.place_cells(rest, rot, trans)
    vel0 = (rng.standard_normal(pos0.shape) * 1e-4).astype(np.float32)
    forces = [W.gaussian_forces(pos0.shape, sigma, seed, s) for s in range(3)]
    return rest, tris, mat, pos0, vel0, forces


class _G:        # minimal stand-in for workloads.CellGroup
    def __init__(self, rest, tris, mat, pos0, vel0):
        self.rest, self.tris, self.material, self.pos0, self.vel0 = rest, tris, mat, pos0, vel0
        self.diameter = W.shapes.cell_diameter(rest)


def _parity(g, forces, n_iters, dt=0.1, **options):
    tol = position_tolerance(g)
    worst = 0.0
    for step, ((po, vo), (pg, vg)) in enumerate(zip(oracle_trajectory(g, dt, forces, n_iters),
                                                    gpu_trajectory(g, dt, forces, n_iters, **options))):
        err = max_abs_err(pg, po)
        worst = max(worst, err)
        assert err <= tol
        scale = np.abs(vo).max() * dt
        assert np.abs(vg.astype(np.float64) - vo).max() * dt <= displacement_tolerance(g, scale, err, step)
    return worst


def test_zero_cells_is_a_no_op_and_null_pointers_are_rejected():
    rest, tris, mat, pos0, vel0, forces = _small_workload(n_cells=1)
    h = NpfemHandle(tris, rest, mat, 0.1)
    h.step(0, None, None, None, 5)                       # n_cells == 0: nothing to do, no error
    with pytest.raises(NpfemError):
        h.step(1, None, None, None, 5)
    p = to_strided(pos0, h.cell_stride)
    with pytest.raises(NpfemError):
        h.step(-1, p, p, p, 5)
    with pytest.raises(NpfemError):
        h.step(1, p, p, p, -1)


def test_n_iters_zero_is_the_inertial_prediction():
    rest, tris, mat, pos0, vel0, forces = _small_workload(n_cells=3)
    g = _G(rest, tris, mat, pos0, vel0)
    (pg, vg), = list(gpu_trajectory(g, 0.1, forces[:1], 0))
    oc = O.OracleCell(tris, rest, mat, 0.1)
    m = oc.masses()[None, :, None]
    inc = 0.1 * vel0.astype(np.float64) + 0.01 * forces[0].astype(np.float64) / m
    assert np.abs(vg * 0.1 - inc).max() <= 1e-6 * np.abs(inc).max()
    assert max_abs_err(pg, pos0.astype(np.float64) + inc) <= 1e-5


@pytest.mark.parametrize("k", [1, 2, 3, 4, 5])
def test_cells_per_cta_variants_and_ragged_tails(k):
    rest, tris, mat, pos0, vel0, forces = _small_workload(n_cells=7)
    _parity(_G(rest, tris, mat, pos0, vel0), forces, 6, cells_per_cta=k)


@pytest.mark.parametrize("mode", [1, 2, 3])
def test_global_step_modes_simt_3xtf32_and_fp16_split(mode):
    rest, tris, mat, pos0, vel0, forces = _small_workload(level=3, n_cells=6)
    _parity(_G(rest, tris, mat, pos0, vel0), forces, 8, global_mode=mode)


def test_dense_operator_matches_dropped_operator():
    """inv_drop_tol = 0 keeps every entry of A_sys^-1; the default drop rule must agree with it
    far inside the parity tolerance."""
    rest, tris, mat, pos0, vel0, forces = _small_workload(level=3, n_cells=5)
    g = _G(rest, tris, mat, pos0, vel0)
    a = list(gpu_trajectory(g, 0.1, forces, 10, inv_drop_tol=0.0))
    b = list(gpu_trajectory(g, 0.1, forces, 10))
    for (pa, va), (pb, vb) in zip(a, b):
        assert np.abs(va - vb).max() * 0.1 <= 1e-5 * np.abs(va).max() * 0.1 + 1e-9
    _parity(g, forces, 10, inv_drop_tol=0.0)


def test_platelets_pack_many_cells():
    rest, tris, mat, pos0, vel0, forces = _small_workload(kind="plt", level=1, n_cells=41)
    _parity(_G(rest, tris, mat, pos0, vel0), forces, 20)


@pytest.mark.parametrize("stride_extra", [0, 1, 2, 64])
def test_custom_cell_strides_and_padding_is_preserved(stride_extra):
    """3*n floats = 8 (mod 16) bytes for every icosphere: stride 3n puts odd cells off 16-byte
    alignment; padding floats must come back untouched."""
    rest, tris, mat, pos0, vel0, forces = _small_workload(n_cells=5)
    n = rest.shape[0]
    stride = 3 * n + stride_extra
    h = NpfemHandle(tris, rest, mat, 0.1, stride, 5)
    assert h.cell_stride == stride
    pos, vel = to_strided(pos0, stride), to_strided(vel0, stride)
    fx = to_strided(forces[0], stride)
    pos[:, 3 * n:] = 123.0
    vel[:, 3 * n:] = -7.0
    h.step(5, pos, vel, fx, 10)
    torch.cuda.synchronize()
    assert (pos[:, 3 * n:] == 123.0).all() and (vel[:, 3 * n:] == -7.0).all()
    oc = O.OracleCell(tris, rest, mat, 0.1)
    po, vo = oc.step(pos0, vel0, forces[0], 10)
    assert max_abs_err(from_strided(pos, n), po) <= 1e-4 * 8.0
    assert np.abs(from_strided(vel, n) - vo).max() <= 2e-3 * np.abs(vo).max()
    with pytest.raises(NpfemError):
        NpfemHandle(tris, rest, mat, 0.1, 3 * n - 1, 5)


def test_nontrivial_clamp_bands_under_large_forces():
    """Strain band [0.9, 1.1], area band [0.95, 1.05], volume band [0.99, 1.01]: forces large
    enough that some elements sit inside, some outside their bands (exercises every clamp
    branch and the hyperbola projection)."""
    rest, tris, mat, pos0, vel0, forces = _small_workload(
        n_cells=4, sigma=2e-2, s_min=0.9, s_max=1.1, a_min=0.95, a_max=1.05, v_min=0.99,
        v_max=1.01)
    g = _G(rest, tris, mat, pos0, vel0)
    forces = [f for f in forces] * 4                     # 12 steps
    _parity(g, forces, 10)
    # the bands were really active / inactive on different elements
    oc = O.OracleCell(tris, rest, mat, 0.1)
    last = list(oracle_trajectory(g, 0.1, forces, 10))[-1][0][0]
    sv = np.array([np.linalg.svd(oc.deformation_gradient(t, last), compute_uv=False)
                   for t in range(tris.shape[0])])
    assert (sv.max(axis=1) > 1.1).any() or (sv.min(axis=1) < 0.9).any()
    assert ((sv > 0.9) & (sv < 1.1)).all(axis=1).any()


def test_shrunk_and_inflated_cells_exercise_volume_and_area_projection():
    """Start from uniformly scaled rest shapes (0.9x and 1.15x): large volume/area violations."""
    rest, tris, mat, pos0, vel0, forces = _small_workload(n_cells=2, sigma=1e-3)
    c = pos0.mean(axis=1, keepdims=True)
    pos0 = (c + (pos0 - c) * np.array([0.9, 1.15], dtype=np.float32)[:, None, None]).astype(np.float32)
    g = _G(rest, tris, mat, pos0, np.zeros_like(pos0))
    # 27 % / 52 % volume violations: the adaptive pass loop of the volume projection (A-17) runs
    # as many passes as fp32 can resolve, at DEFAULT options
    _parity(g, forces * 3, 10)


def _split_triangles(rest, tris, which):
    """1 -> 3 split of the chosen triangles (new vertex at the centroid): valence-3 vertices, and
    every corner of a split triangle gains one neighbour."""
    rest = [np.asarray(p, dtype=np.float64) for p in rest]
    out = []
    for ti, (a, b, c) in enumerate(tris.tolist()):
        if ti in which:
            m = len(rest)
            rest.append((rest[a] + rest[b] + rest[c]) / 3.0)
            out += [(a, b, m), (b, c, m), (c, a, m)]
        else:
            out.append((a, b, c))
    return np.array(rest), np.array(out, dtype=np.int32)


def test_irregular_mesh_with_valence_3_and_12_vertices():
    """Vertex fans longer than the 6 entries a thread keeps in registers (a valence-12 vertex) and
    valence-3 vertices: the overflow lists of the gather and of the volume gradient."""
    rest, tris = W.rest_shape("rbc", 2)
    rng = np.random.Generator(np.random.PCG64(11))
    hub = 17
    which = set(np.nonzero((tris == hub).any(axis=1))[0].tolist()) | set(
        rng.choice(tris.shape[0], size=18, replace=False).tolist())
    rest, tris = _split_triangles(rest, tris, which)
    assert np.bincount(tris.ravel()).max() == 12 and np.bincount(tris.ravel()).min() == 3
    mat = W.default_material(rest, tris)
    rot, trans = W.random_rigid_placements(6, 100.0, 5.0, rng)
    pos0 = W.place_cells(rest, rot, trans)
    vel0 = (rng.standard_normal(pos0.shape) * 1e-4).astype(np.float32)
    forces = [W.gaussian_forces(pos0.shape, 1e-3, 11, s) for s in range(3)]
    _parity(_G(rest, tris, mat, pos0, vel0), forces, 8)


def test_unpaired_triangles_one_element_per_triangle():
    """pair_triangles = 2: every triangle is a single-triangle element (the shared hinge is then
    evaluated half by each side, nothing is written for the fourth vertex)."""
    rest, tris, mat, pos0, vel0, forces = _small_workload(n_cells=6)
    g = _G(rest, tris, mat, pos0, vel0)
    h = NpfemHandle(tris, rest, mat, 0.1, pair_triangles=2)
    assert h.info()["n_diamonds"] == 0 and h.info()["n_elements"] == tris.shape[0]
    _parity(g, forces, 8, pair_triangles=2)
    # and it is the same computation as the paired default up to fp32 summation order
    a = list(gpu_trajectory(g, 0.1, forces, 8))[-1][0]
    b = list(gpu_trajectory(g, 0.1, forces, 8, pair_triangles=2))[-1][0]
    assert np.abs(a.astype(np.float64) - b).max() <= 4e-6


def test_step_host_matches_device_step_bit_for_bit_and_is_deterministic():
    rest, tris, mat, pos0, vel0, forces = _small_workload(level=3, n_cells=23)
    n = rest.shape[0]
    h = NpfemHandle(tris, rest, mat, 0.1)
    stride = h.cell_stride
    runs = []
    for _ in range(2):
        pos, vel, fx = (to_strided(a, stride) for a in (pos0, vel0, forces[0]))
        h.step(23, pos, vel, fx, 10)
        torch.cuda.synchronize()
        runs.append((pos.cpu().numpy().copy(), vel.cpu().numpy().copy()))
    assert np.array_equal(runs[0][0], runs[1][0]) and np.array_equal(runs[0][1], runs[1][1])
    hp = [to_strided(a, stride, device="cpu").pin_memory() for a in (pos0, vel0, forces[0])]
    h.step_host(23, hp[0], hp[1], hp[2], 10)
    assert np.array_equal(hp[0].numpy(), runs[0][0]) and np.array_equal(hp[1].numpy(), runs[0][1])


def test_step_on_a_side_stream():
    rest, tris, mat, pos0, vel0, forces = _small_workload(n_cells=5)
    dg = DeviceGroup(tris, rest, mat, 0.1, pos0, vel0)
    dg.set_forces(forces[0])
    st = torch.cuda.Stream()
    st.wait_stream(torch.cuda.current_stream())
    with torch.cuda.stream(st):
        dg.step(10, stream=st)
    st.synchronize()
    pg, vg = dg.state()
    oc = O.OracleCell(tris, rest, mat, 0.1)
    po, vo = oc.step(pos0, vel0, forces[0], 10)
    assert max_abs_err(pg, po) <= 8e-4


def test_mesh_too_large_for_one_cta_is_rejected_loudly():
    rest, tris = W.rest_shape("rbc", 4)                  # 2562 vertices > 1024
    with pytest.raises(NpfemError) as e:
        NpfemHandle(tris, rest, W.default_material(rest, tris), 0.1)
    assert e.value.code == -4


@pytest.mark.parametrize("damp", [dict(c_alpha=0.5), dict(c_beta=0.05), dict(c_alpha=0.5, c_beta=0.05)])
def test_viscoelastic_damping_matches_the_oracle(damp):
    """NEXT-2 (reading A-20): implicit Rayleigh damping
    C = c_alpha M + c_beta L_el.  The kernel folds it into the residual (diagonal, membrane and
    hinge factors) and a once-per-step constant; the oracle adds (C/h) x_n to the right-hand side
    of the damped system.  Cells start with velocities, so the damping really acts."""
    rest, tris, mat, pos0, vel0, forces = _small_workload(n_cells=7, **damp)
    vel0 = (vel0 * 50).astype(np.float32)                      # 5e-3 um/us: damping force ~ elastic force
    g = _G(rest, tris, mat, pos0, vel0)
    _parity(g, forces * 2, 10)
    # and it is not a no-op: the damped run differs from the undamped one by far more than the check resolves
    a = list(gpu_trajectory(g, 0.1, forces, 10))[-1][1]
    g0 = _G(rest, tris, W.default_material(rest, tris), pos0, vel0)
    b = list(gpu_trajectory(g0, 0.1, forces, 10))[-1][1]
    assert np.abs(a - b).max() > 0.02 * np.abs(b).max()


def test_damping_on_rbc3_and_platelets_with_world_offsets():
    for kind, level, n_cells in (("rbc", 3, 6), ("plt", 1, 37)):
        rest, tris, mat, pos0, vel0, forces = _small_workload(kind=kind, level=level, n_cells=n_cells,
                                                              c_alpha=0.3, c_beta=0.02)
        vel0 = (vel0 * 30).astype(np.float32)
        _parity(_G(rest, tris, mat, pos0, vel0), forces, 12)


def test_schedule_jitter_leaves_results_bit_identical():
    """Race check by schedule fuzzing (compute-sanitizer is closed on this pool): with
    debug_jitter every warp sleeps a pseudo-random time after every CTA barrier, so warps cross
    the kernel's phases (two shared buffers with three lives each per iteration, the temporary
    overwrite of z in the volume passes, the staging buffers) at very different times.  Any
    missing barrier would let a fast warp overwrite what a slow warp still reads; a correctly
    synchronised kernel is bit-identical for every seed."""
    cases = []
    rest, tris, mat, pos0, vel0, forces = _small_workload(n_cells=7)
    cases += [("rbc2 k=5", rest, tris, mat, pos0, vel0, forces, {}),
              ("rbc2 k=2", rest, tris, mat, pos0, vel0, forces, dict(cells_per_cta=2)),
              ("rbc2 single triangles", rest, tris, mat, pos0, vel0, forces, dict(pair_triangles=2)),
              ("rbc2 simt", rest, tris, mat, pos0, vel0, forces, dict(global_mode=1))]
    c = pos0.mean(axis=1, keepdims=True)
    shrunk = (c + (pos0 - c) * 0.9).astype(np.float32)
    cases.append(("rbc2 shrunk (volume passes)", rest, tris, mat, shrunk, np.zeros_like(pos0), forces, {}))
    matd = W.default_material(rest, tris, c_alpha=0.3, c_beta=0.03)
    cases.append(("rbc2 damped", rest, tris, matd, pos0, vel0, forces, {}))
    r3 = _small_workload(level=3, n_cells=6)
    cases.append(("rbc3", r3[0], r3[1], r3[2], r3[3], r3[4], r3[5], {}))
    pl = _small_workload(kind="plt", level=1, n_cells=23)
    cases.append(("plt", pl[0], pl[1], pl[2], pl[3], pl[4], pl[5], {}))
    for name, rest, tris, mat, pos0, vel0, forces, opt in cases:
        g = _G(rest, tris, mat, pos0, vel0)
        ref = list(gpu_trajectory(g, 0.1, forces[:2], 6, **opt))[-1]
        for seed in (1, 2, 3):
            out = list(gpu_trajectory(g, 0.1, forces[:2], 6, debug_jitter=seed, **opt))[-1]
            assert np.array_equal(ref[0], out[0]) and np.array_equal(ref[1], out[1]), (name, seed)


@pytest.mark.parametrize("damp", [{}, dict(c_alpha=0.3, c_beta=0.02)])
def test_strain_dependent_weight_matches_the_oracle(damp):
    """NEXT-4 (reading A-23): strain weight k_strain (1 + beta d^2).  Forces large
    enough to strain the membrane by several per cent, so that the hardening factor really differs
    from 1; with and without damping (both optioned kernel instantiations)."""
    rest, tris, mat, pos0, vel0, forces = _small_workload(n_cells=6, sigma=2e-2, strain_hardening=60.0, **damp)
    g = _G(rest, tris, mat, pos0, vel0)
    forces = list(forces) * 3                                     # 9 steps
    _parity(g, forces, 12)
    oc = O.OracleCell(tris, rest, mat, 0.1)
    last = list(oracle_trajectory(g, 0.1, forces, 12))[-1][0][0]
    sv = np.array([np.linalg.svd(oc.deformation_gradient(t, last), compute_uv=False) for t in range(tris.shape[0])])
    assert np.abs(sv - 1).max() > 0.03                            # beta d^2 > 5 % somewhere
    # and it is not a no-op
    a = list(gpu_trajectory(g, 0.1, forces, 12))[-1][0]
    g0 = _G(rest, tris, W.default_material(rest, tris, **damp), pos0, vel0)
    b = list(gpu_trajectory(g0, 0.1, forces, 12))[-1][0]
    assert np.abs(a.astype(np.float64) - b).max() > 1e-4
