"""Phase clocks of the fused step kernel: where one iteration of one CTA spends its cycles.

Diagnostic, not part of the product path.  Builds a second copy of the library with
-DNPFEM_PHASE_CLOCKS (paper_2011_04332_b200/libnpfem_b200_diag.so; the shipped library carries
none of this), runs the config-4 recipe on `--cells` cells and prints, per global-step mode, the
clock64() ticks thread 0 of every CTA accumulated between the kernel's barriers, divided by
CTAs x iterations.  A phase is closed by a CTA barrier, and the barrier is deferred-blocking: the
wait for the slowest warp shows up in the phase that follows.

    python -m paper_2011_04332_b200.phase_clocks --cells 14800 --modes 3,2 [--masks 0,1,2]

`--masks` are ablations of the global_mode-3 operator product (results are then meaningless, the
timing is what is looked at; the owner update ignores the product's output so that the state
stays where it is): 1 no mma, 2 no shared-memory loads, 16 skip the product loop, 32 skip the
right-hand-side split.  `profiles/` quotes this command.
"""
from __future__ import annotations

import argparse
import os
import subprocess

import numpy as np
import torch

from . import binding as B
from . import build as _build

DIAG_LIB = os.path.join(_build.HERE, "libnpfem_b200_diag.so")
PHASES = ["prologue", "first element pass", "cell pipeline", "rhs split", "operator product",
          "hand-off", "owner update"]


def build_diag(force: bool = False) -> str:
    srcs = [os.path.join(_build.CSRC, s) for s in _build.SOURCES]
    deps = srcs + [h if os.path.isabs(h) else os.path.join(_build.CSRC, h) for h in _build.HEADERS]
    if not force and os.path.exists(DIAG_LIB) and all(os.path.getmtime(d) <= os.path.getmtime(DIAG_LIB) for d in deps):
        return DIAG_LIB
    cmd = [_build._nvcc(), "-O3", "-std=c++17", "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo",
           "-DNPFEM_PHASE_CLOCKS", "-Xcompiler", "-fPIC", "-shared", "-I", os.path.join(_build.ROOT, "include"),
           "-I", _build.CSRC, "-o", DIAG_LIB] + srcs
    subprocess.run(cmd, check=True)
    return DIAG_LIB


def main() -> None:
    ap = argparse.ArgumentParser(description=__doc__, formatter_class=argparse.RawDescriptionHelpFormatter)
    ap.add_argument("--cells", type=int, default=14800)
    ap.add_argument("--modes", default="3,2")
    ap.add_argument("--masks", default="0")
    ap.add_argument("--iters", type=int, default=20)
    args = ap.parse_args()
    B._lib = B.load_library(build_diag())          # every handle created below uses the diagnostic library
    import workloads as W
    from .harness import DeviceGroup

    rest, tris = W.rest_shape("rbc", 3)
    mat = W.default_material(rest, tris)
    rng = np.random.Generator(np.random.PCG64([4, 1]))
    rot, trans = W.random_rigid_placements(args.cells, 300.0, 5.0, rng)
    pos0 = W.place_cells(rest, rot, trans)
    vel0 = np.zeros_like(pos0)
    for mode in [int(x) for x in args.modes.split(",")]:
        for mask in [int(x) for x in args.masks.split(",")]:
            B.npfem_debug_phase_clocks(0x100 | mask)          # >= 0x100: set the ablation mask
            dg = DeviceGroup(tris, rest, mat, 0.1, pos0, vel0, global_mode=mode)
            gen = torch.Generator(device="cuda")
            gen.manual_seed(4)
            dg.set_forces(torch.randn(dg.pos.shape, generator=gen, device="cuda") * 1e-3)
            for _ in range(2):
                dg.step(args.iters)
            torch.cuda.synchronize()
            B.npfem_debug_phase_clocks(1)                     # read and reset
            t0, t1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            t0.record()
            dg.step(args.iters)
            t1.record()
            torch.cuda.synchronize()
            c = B.npfem_debug_phase_clocks(1)
            k = dg.handle.info()["cells_per_cta"]
            ctas = (args.cells + k - 1) // k
            per = [x / (ctas * args.iters) for x in c[1:7]]
            print(f"mode {mode} mask {mask}: {t0.elapsed_time(t1):.2f} ms per step; prologue {c[0] / ctas:.0f} cycles per CTA; "
                  "per CTA-iteration: " + ", ".join(f"{n} {p:.0f}" for n, p in zip(PHASES[1:], per)) +
                  f"; total {sum(per):.0f}", flush=True)


if __name__ == "__main__":
    main()
