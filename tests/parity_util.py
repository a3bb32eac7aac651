"""Helpers shared by the GPU parity tests: run a workload through the C ABI and through the oracle.

Both sides start from the same seeded fp32 inputs (workloads/) and run FREE: the oracle continues
from its own fp64 state, the CUDA path from its own fp32 state; nothing the CUDA path produced is
ever fed to the oracle.
"""
from __future__ import annotations

import numpy as np

from oracle import npfem_oracle as O


def oracle_trajectory(group, dt, forces_per_step, n_iters):
    """Yield (pos, vel) fp64 [N,V,3] after every step; forces_per_step: iterable of fp32 [N,V,3]."""
    oc = O.OracleCell(group.tris, group.rest, group.material, dt)
    pos = group.pos0.astype(np.float64)
    vel = group.vel0.astype(np.float64)
    for f in forces_per_step:
        pos, vel = oc.step(pos, vel, f, n_iters)
        yield pos, vel


def gpu_trajectory(group, dt, forces_per_step, n_iters, **options):
    """Yield (pos, vel) fp32 [N,V,3] after every step through npfem_step (device buffers)."""
    from paper_2011_04332_b200.harness import DeviceGroup
    dg = DeviceGroup(group.tris, group.rest, group.material, dt, group.pos0, group.vel0, **options)
    for f in forces_per_step:
        dg.set_forces(f)
        dg.step(n_iters)
        yield dg.state()


def max_abs_err(a, b):
    return float(np.max(np.abs(np.asarray(a, dtype=np.float64) - np.asarray(b, dtype=np.float64))))


def position_tolerance(group):
    """north_star: max abs position error 1e-4 x cell diameter after each step."""
    return 1e-4 * group.diameter


DISP_RTOL = 1e-3       # A-13: relative part of the displacement self-check


def displacement_tolerance(group, scale, err=0.0, step=0):
    """Self-imposed check (A-13 and "error budget"): per-step displacement error bound

        DISP_RTOL * max|dx_oracle| + (0.3 ulp32(|x|max) + 2 ulp32(R)) sqrt(step + 1) + 0.02 * err

    The absolute floor is the fp32 contract's own, not the kernel's:
      * the state crosses the boundary as fp32 WORLD coordinates (north_star: fp32 GPU), so after
        the first step every stored coordinate carries a rounding of up to ulp32(|x|max)/2
        (3.8e-6 um at 100 um); to the next step this is a high-frequency perturbation of the
        elastic state, answered by a displacement of about K_el/(M/h^2 + K_el) ~ 0.2-0.3 of it;
      * inside a step the iterate lives in cell-local coordinates rounded to ulp32(R)/2, R = the
        largest |coordinate| about the centroid (2.4e-7 um for an RBC).
    Both runs are FREE (never re-synchronised), so the velocity error of step k is part of the
    displacement error of step k+1: the floor accumulates like a random walk, hence sqrt(step+1).
    The last term lets the trajectories differ by what their accumulated state difference
    (err = position error so far) explains."""
    radius = float(np.abs(group.rest - group.rest.mean(axis=0)).max())
    xmax = float(np.abs(group.pos0).max())
    floor = 0.3 * float(np.spacing(np.float32(xmax))) + 2.0 * float(np.spacing(np.float32(radius)))
    return DISP_RTOL * scale + floor * np.sqrt(step + 1.0) + 0.02 * err
