"""Device-buffer plumbing around the C ABI: pad [N,V,3] arrays to the cell stride, run steps.

PyTorch is used for device memory and streams only; every step of the method runs in
libnpfem_b200.so.  No arithmetic of the method lives here.
"""
from __future__ import annotations

import numpy as np
import torch

from .binding import NpfemHandle


def to_strided(a: np.ndarray | torch.Tensor, stride: int, device="cuda") -> torch.Tensor:
    """[N,V,3] float32 -> device tensor [N,stride] (cell-major, vertex-major xyz, zero padding)."""
    t = torch.as_tensor(a, dtype=torch.float32)
    n = t.shape[0]
    flat = t.reshape(n, -1)
    out = torch.zeros((n, stride), dtype=torch.float32, device=device)
    out[:, : flat.shape[1]] = flat.to(device)
    return out


def from_strided(t: torch.Tensor, n_verts: int) -> np.ndarray:
    """device/host tensor [N,stride] -> numpy float32 [N,V,3]."""
    return t[:, : 3 * n_verts].reshape(t.shape[0], n_verts, 3).cpu().numpy()


class DeviceGroup:
    """One cell type resident on the GPU: handle + pos/vel/fext device buffers."""

    def __init__(self, tris, rest, material, dt, pos0, vel0, device="cuda", **options):
        self.handle = NpfemHandle(tris, rest, material, dt, 0, int(pos0.shape[0]), **options)
        self.n_verts = int(rest.shape[0])
        self.n_cells = int(pos0.shape[0])
        self.stride = self.handle.cell_stride
        self.device = device
        self.pos = to_strided(pos0, self.stride, device)
        self.vel = to_strided(vel0, self.stride, device)
        self.fext = torch.zeros_like(self.pos)

    def set_forces(self, f):
        if isinstance(f, torch.Tensor) and f.is_cuda and f.shape == self.fext.shape:
            self.fext = f
        else:
            self.fext = to_strided(f, self.stride, self.device)

    def step(self, n_iters: int, stream=None):
        self.handle.step(self.n_cells, self.pos, self.vel, self.fext, n_iters, stream)

    def step_collide(self, coll_q, coll_n, n_iters: int, stream=None):
        """coll_q, coll_n: [N,V,3] arrays (numpy or torch); zero normal = no neighbour."""
        q = to_strided(coll_q, self.stride, self.device)
        nn = to_strided(coll_n, self.stride, self.device)
        self.handle.step_collide(self.n_cells, self.pos, self.vel, self.fext, q, nn, n_iters, stream)
        torch.cuda.synchronize()      # q and nn are temporaries of this call

    def vertex_areas(self):
        a = torch.zeros((self.n_cells, self.n_verts), dtype=torch.float32, device=self.device)
        self.handle.vertex_areas(self.n_cells, self.pos, a)
        torch.cuda.synchronize()
        return a.cpu().numpy()

    def step_converged(self, tol: float, max_iters: int, stream=None):
        """Converged quasi-Newton step; returns (iterations, residual lengths) per cell (numpy)."""
        its = torch.zeros(self.n_cells, dtype=torch.int32, device=self.device)
        res = torch.zeros(self.n_cells, dtype=torch.float32, device=self.device)
        self.handle.step_converged(self.n_cells, self.pos, self.vel, self.fext, tol, max_iters, its, res, stream)
        torch.cuda.synchronize()
        return its.cpu().numpy(), res.cpu().numpy()

    def state(self):
        torch.cuda.synchronize()
        return (from_strided(self.pos, self.n_verts), from_strided(self.vel, self.n_verts))
