"""External per-vertex force fields (stand-ins for the fluid/IBM forces).

Units: nN (1 pN = 1e-3).  Every field is seeded; values are cast to fp32 once and both the oracle
and the CUDA path read those same fp32 numbers.
"""
from __future__ import annotations

from dataclasses import dataclass

import numpy as np

PN = 1e-3   # one piconewton in the harness unit (nN)


def gaussian_forces(shape, sigma: float, seed: int, step: int = 0) -> np.ndarray:
    """i.i.d. N(0, sigma^2) per component, float32 `shape`; a fresh stream per (seed, step)."""
    rng = np.random.Generator(np.random.PCG64([int(seed), int(step), 0x6E70]))
    return (rng.standard_normal(shape) * sigma).astype(np.float32)


def gaussian_forces_torch(shape, sigma: float, seed: int, step: int, device):
    """Bulk variant for configs 4/5: drawn on `device` with a seeded torch.Generator.

    The oracle's parity subsample is copied back from this tensor, so both paths see one draw.
    """
    import torch
    gen = torch.Generator(device=device)
    gen.manual_seed((int(seed) * 1_000_003 + int(step)) & 0x7FFFFFFFFFFF)
    return torch.randn(shape, generator=gen, device=device, dtype=torch.float32) * float(sigma)


@dataclass
class FourierField:
    """Smooth random field of config 2: f_c(p) = amp * sin(pi * sum_m sin(2 pi n_m.p/box + phi_mc))."""
    modes: np.ndarray      # int [M,3], entries in -2..2, not all zero
    phases: np.ndarray     # float64 [M,3] (one phase per mode and force component)
    box: float
    amp: float

    def __call__(self, pos: np.ndarray) -> np.ndarray:
        p = np.asarray(pos, dtype=np.float64)
        arg = 2.0 * np.pi * np.tensordot(p, self.modes.astype(np.float64).T, axes=1) / self.box
        phi = np.pi * np.sin(arg[..., None] + self.phases).sum(axis=-2)   # [..., 3]
        return (self.amp * np.sin(phi)).astype(np.float32)


def fourier_shear_field(seed: int, box: float = 100.0, amp: float = PN,
                        n_modes: int = 8) -> FourierField:
    rng = np.random.Generator(np.random.PCG64([int(seed), 0xF0F0]))
    modes = np.zeros((n_modes, 3), dtype=np.int64)
    for m in range(n_modes):
        while not modes[m].any():
            modes[m] = rng.integers(-2, 3, size=3)
    phases = rng.uniform(0.0, 2.0 * np.pi, size=(n_modes, 3))
    return FourierField(modes=modes, phases=phases, box=float(box), amp=float(amp))


def cap_vertex_sets(rest_xyz: np.ndarray, frac: float = 0.05) -> tuple[np.ndarray, np.ndarray]:
    """(minus_cap, plus_cap): the k = round(frac*V) vertices of smallest / largest body-frame x.

    Ties broken by a stable sort on (x, vertex index).
    """
    n = rest_xyz.shape[0]
    k = int(round(frac * n))
    order = np.lexsort((np.arange(n), rest_xyz[:, 0]))
    return order[:k].astype(np.int64), order[n - k:].astype(np.int64)


def cap_pull_forces(rest_xyz: np.ndarray, rot: np.ndarray, pull: float = 20.0 * PN,
                    frac: float = 0.05) -> np.ndarray:
    """Config 5: +-`pull` per cap vertex along the body-frame x axis rotated to world; float32 [N,V,3]."""
    minus, plus = cap_vertex_sets(rest_xyz, frac)
    n_cells, n = rot.shape[0], rest_xyz.shape[0]
    f = np.zeros((n_cells, n, 3), dtype=np.float32)
    axis = rot[:, :, 0]                                    # R e_x, [N,3]
    f[:, plus, :] = (pull * axis)[:, None, :].astype(np.float32)
    f[:, minus, :] = (-pull * axis)[:, None, :].astype(np.float32)
    return f
