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
