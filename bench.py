"""bench.py -- throughput of the npFEM solid-phase hot path on B200 (BASELINE.json metric).

  python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--cells C]

One "step" = one npfem_step over the whole suspension: every SURVEY.md 8(a) row (inertial
prediction, n_iters x {local projections, rhs, global solve}, finalise) in ONE kernel launch.
Workload at N=1: BASELINE.json configs[3], the throughput run the metric is quoted on --
100 000 RBC-3 cells (642 vertices each), 20 iterations per step, forces redrawn per step from a
seeded N(0,(1 pN)^2) field, all state resident in HBM (2.3 GB of pos/vel/force per step: far
larger than the 126 MB L2, so no L2 flush is needed between timed steps).  N>1: weak scaling,
every rank owns its own 100 000 cells (cells are independent: no data-path collective).

The JSON line carries: value = cell-steps/s with inputs resident in HBM (CUDA events on the
launching stream, max over ranks); vertex_iterations_per_s; e2e = the same metric through
npfem_step_host with pinned HOST buffers (H2D of pos/vel/force and D2H of pos/vel inside the
timed region); roofline for the fused step kernel; cpu_baseline = the fp64 oracle timed on this
box's host cores on a bounded sample; clocks sampled during the timed region.
--impl reference times the oracle itself (this tier's reference arm).
"""
from __future__ import annotations

import argparse
import json
import os
import statistics
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

CONFIG_ID = 4
N_FORCE_FIELDS = 4          # pre-generated per-step force fields, cycled (each 771 MB at 100k cells)

# ---- algorithmic work per unit (FMA = 2 flop) -------------------------
# nnz of the nested-dissection Cholesky factor of A_sys per icosphere level
NNZ_L = {42: 573, 162: 4620, 642: 31397}
FLOP_PER_TRI = 210          # F, 2x2 SVD via F^T F, strain clamp, area hyperbola (4 Newton steps), G^T P
FLOP_PER_NEWTON = 23        # one Newton step on the hyperbola stationarity (g, g', quotient, update)
FLOP_PER_HINGE = 60         # k = sum K_i x_i, normalise, scatter 4 x 3
FLOP_VOL_PER_TRI, FLOP_VOL_PER_VERT, VOL_INNER = 45, 15, 2
FLOP_RHS_PER_VERT = 10


def flops_per_cell_iteration(n_verts: int, n_tris: int, vol_passes: int = VOL_INNER,
                             newton_steps: int = 4) -> float:
    """Algorithmic flops of one local/global iteration of one cell (defaults: the count DESIGN.md
    states).  vol_passes / newton_steps let the caller count what the kernel really executes on
    a near-rest suspension: one volume pass and one Newton step per triangle (A-17, A-18)."""
    n_h = 3 * n_tris // 2
    nnz_l = NNZ_L.get(n_verts, int(49 * n_verts))
    local = (FLOP_PER_TRI - (4 - newton_steps) * FLOP_PER_NEWTON) * n_tris + FLOP_PER_HINGE * n_h
    volume = vol_passes * (FLOP_VOL_PER_TRI * n_tris + FLOP_VOL_PER_VERT * n_verts)
    solve = 12 * nnz_l + 6 * n_verts            # 3 rhs x (forward + backward) x 2 flop per entry
    return float(local + volume + solve + FLOP_RHS_PER_VERT * n_verts)


def hbm_bytes_per_cell_step(n_verts: int) -> int:
    return 5 * 3 * n_verts * 4                   # read x, v, f; write x, v


FP32_PEAK_TFLOPS_NOMINAL = 148 * 128 * 2 * 1.965e9 / 1e12   # SMs x FP32 lanes x FMA x max clock


TRAFFIC_CAPTURE = "r2_dram_traffic.csv"     # newest committed `ncu --set full` capture (profiles/)


def measured_dram_traffic(n_verts: int, n_cells: int):
    """(DRAM bytes per launch, provenance) of the step kernel: dram__bytes_read.sum +
    dram__bytes_write.sum from the newest committed `ncu --set full` capture.  The csv holds the
    bytes per cell measured there and the commit of the kernel it was taken on; a launch moves
    that times its cells.  (None, reason) without a capture for this mesh size."""
    path = os.path.join(ROOT, "profiles", TRAFFIC_CAPTURE)
    if not os.path.exists(path):
        return None, "no capture committed"
    with open(path) as fh:
        rows = [ln.strip().split(",") for ln in fh if ln.strip() and not ln.startswith("#")]
    rec = dict(zip(rows[0], rows[1]))
    if int(rec["n_verts"]) != n_verts:
        return None, "capture is for another mesh size"
    return float(rec["dram_bytes_per_cell"]) * n_cells, (
        f"profiles/{TRAFFIC_CAPTURE}: {rec['dram_bytes_per_cell']} B per cell at "
        f"{rec.get('n_cells', '?')} cells, kernel of commit {rec.get('commit', '?')}")


def load_peaks() -> dict:
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        with open(path) as fh:
            p = json.load(fh)
        p["source"] = "measured"
        return p
    return {"hbm_gbs": 6650.0, "bf16_tflops": 1590.0, "sm_max_mhz": 1965.0, "source": "fallback"}


# ---- clocks -----------------------------------------------------------------------------------
class ClockSampler:
    """nvidia-smi clock / throttle-reason samples taken DURING the timed region."""
    FIELDS = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
              "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
              "clocks_event_reasons.sw_power_cap")

    def __init__(self, gpu_index: int):
        self.gpu, self.rows, self.proc, self.thread = gpu_index, [], None, None

    def start(self):
        try:
            self.proc = subprocess.Popen(
                ["nvidia-smi", f"--id={self.gpu}", f"--query-gpu={self.FIELDS}",
                 "--format=csv,noheader,nounits", "-lms", "100"],
                stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
        except OSError:
            self.proc = None
            return
        self.thread = threading.Thread(target=self._read, daemon=True)
        self.thread.start()

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append((time.time(), [c.strip() for c in line.split(",")]))

    def stop(self, t0: float, t1: float) -> dict:
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except subprocess.TimeoutExpired:
            self.proc.kill()
        rows = [r for t, r in self.rows if t0 <= t <= t1 + 0.1] or [r for _, r in self.rows]
        sm, smax, power, reasons = [], [], [], set()
        names = ("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap")
        for r in rows:
            try:
                sm.append(float(r[0])); smax.append(float(r[1])); power.append(float(r[2]))
            except (ValueError, IndexError):
                continue
            for name, val in zip(names, r[3:7]):
                if val.lower().startswith("active"):
                    reasons.add(name)
        return {"sm_mhz": statistics.median(sm) if sm else None,
                "sm_max_mhz": max(smax) if smax else None,
                "power_w_max": max(power) if power else None,
                "samples": len(sm), "reasons": sorted(reasons)}


# ---- the oracle, timed (cpu_baseline leg and --impl reference arm) ----------------------------
def _oracle_sample(n_cells: int, seed_step: int = 0):
    """(oracle cell type, pos0, vel0, forces, workload) for the first n_cells of config 4."""
    import workloads as W
    from oracle import npfem_oracle as O
    w = W.make_config(CONFIG_ID, cells=n_cells)
    g = w.groups[0]
    oc = O.OracleCell(g.tris, g.rest, g.material, w.dt)
    return oc, g, w


def time_oracle(budget_s: float = 15.0, steps: int = 1) -> dict:
    """Time the fp64 oracle, as it stands, on this box's host cores on a bounded sample of the
    bench workload (first cells of config 4, `steps` steps x 20 iterations).  The sample is
    sized from a short calibration call so that the timed part is about `budget_s` seconds."""
    from oracle import npfem_oracle as O
    cores = O.num_threads()
    oc, g, w = _oracle_sample(cores)
    f = w.forces(0, 0)
    oc.step(g.pos0, g.vel0, f, 1)                         # page in the factor, spin up OpenMP
    t = time.perf_counter()
    oc.step(g.pos0, g.vel0, f, w.n_iters)
    t_cal = time.perf_counter() - t                       # one batch of `cores` cells, one step
    batches = max(1, min(256, int(budget_s / max(t_cal * steps, 1e-3))))
    n_cells = cores * batches
    oc, g, w = _oracle_sample(n_cells)
    pos, vel = g.pos0.astype(np.float64), g.vel0.astype(np.float64)
    forces = [w.forces(0, s) for s in range(steps)]
    t = time.perf_counter()
    for s in range(steps):
        pos, vel = oc.step(pos, vel, forces[s], w.n_iters)
    dt = time.perf_counter() - t
    n = g.rest.shape[0]
    return {"value": n_cells * steps / dt, "unit": "cell-steps/s", "cores": cores, "kind": "oracle",
            "vertex_iterations_per_s": n_cells * steps * n * w.n_iters / dt,
            "sample": f"first {n_cells} cells of config 4 (RBC-3, 642 vertices), {steps} step(s) x "
                      f"{w.n_iters} iterations, fp64, OpenMP over cells, {dt:.1f} s",
            "seconds": dt, "n_cells": n_cells, "steps": steps}


def run_reference(args) -> None:
    """--impl reference: the oracle as the reference arm, rank 0 only."""
    if int(os.environ.get("RANK", "0")) != 0:
        return
    per_step = []
    total = args.steps + args.warmup
    budget = max(2.0, min(20.0, 150.0 / max(total, 1)))
    res = None
    for i in range(total):
        res = time_oracle(budget_s=budget, steps=1)
        if i >= args.warmup:
            per_step.append(res)
    cells = sum(r["n_cells"] for r in per_step)
    secs = sum(r["seconds"] for r in per_step)
    value = cells / secs
    line = {"impl": "reference", "metric": "cell-steps/s", "value": value, "unit": "cell-steps/s",
            "n_gpus": args.gpus, "steps": args.steps, "warmup": args.warmup,
            "ms_per_step": 1e3 * secs / max(len(per_step), 1), "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": "config4: RBC-3 (642 vertices), 20 iterations per step; each "
                                   "reference step is a bounded sample of the 100000-cell suspension",
                       "n_iters": 20, "sample_cells_per_step": per_step[-1]["n_cells"]},
            "cpu_baseline": {"value": value, "unit": "cell-steps/s", "cores": res["cores"],
                             "kind": "oracle", "sample": res["sample"]},
            "e2e": {"value": value, "unit": "cell-steps/s", "h2d_bytes_per_step": 0,
                    "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line))


# ---- the CUDA arm -------------------------------------------------------------------------------
def roofline_of(n, T, n_iters, n_cells, launch_ms, peak_measured, peaks, clocks=None, traffic=True):
    """Roofline object of the fused step kernel for one workload: the path is
    bound by plain FP32 issue, so achieved = algorithmic flops per launch / launch duration, against
    the FFMA rate measured in this run (npfem_measure_fp32_peak) and, for reference, the nominal one."""
    f_alg = flops_per_cell_iteration(n, T) * n_iters * n_cells
    f_exe = flops_per_cell_iteration(n, T, vol_passes=1, newton_steps=1) * n_iters * n_cells
    b_alg = hbm_bytes_per_cell_step(n) * n_cells
    sec = launch_ms * 1e-3
    achieved = f_alg / sec / 1e12
    r = {"bound": "alu", "achieved": achieved, "peak": peak_measured, "unit": "TFLOP/s",
         "frac": achieved / peak_measured, "kernel": "npfem_step_kernel",
         "peak_source": "measured in this run: npfem_measure_fp32_peak(FFMA), best of 4 launches",
         "peak_measured": peak_measured, "peak_nominal": FP32_PEAK_TFLOPS_NOMINAL,
         "frac_of_nominal": achieved / FP32_PEAK_TFLOPS_NOMINAL,
         "peak_nominal_source": "derived: 148 SMs x 128 FP32 lanes x 2 x 1.965 GHz",
         "algorithmic_flops_per_launch": f_alg, "launch_ms": launch_ms,
         "executed_equivalent": {
             "flops_per_launch": f_exe, "achieved": f_exe / sec / 1e12,
             "frac": f_exe / sec / 1e12 / peak_measured,
             "note": "the same count with the 1 volume pass and 1 area-Newton step per triangle "
                     "that the adaptive loops really take on a near-rest suspension (A-17, A-18); "
                     "the algorithmic count charges 2 passes and 4 steps"},
         "hbm": {"achieved_gbs": b_alg / sec / 1e9, "peak_gbs": peaks["hbm_gbs"],
                 "frac": b_alg / sec / 1e9 / peaks["hbm_gbs"], "peak_source": peaks["source"],
                 "algorithmic_bytes_per_launch": b_alg}}
    if traffic:
        r["traffic"], r["traffic_source"] = measured_dram_traffic(n, n_cells)
    if clocks and clocks.get("sm_mhz"):
        at_clock = 148 * 128 * 2 * clocks["sm_mhz"] * 1e6 / 1e12
        r["frac_at_observed_clock"] = achieved / at_clock
    return r


def time_extra_workload(W, NpfemHandle, to_strided, dev, name, kind, level, n_cells, n_iters,
                        force_kind, seed, steps, warmup, peak_measured, peaks):
    """Device-resident timing of one non-headline workload (other cell types / config 5)."""
    import torch
    rest, tris = W.rest_shape(kind, level)
    mat = W.default_material(rest, tris)
    n, T = rest.shape[0], tris.shape[0]
    rng = np.random.Generator(np.random.PCG64(seed))
    radius = float(np.linalg.norm(rest, axis=1).max())
    rot, trans = W.random_rigid_placements(n_cells, 300.0, radius, rng)
    pos0 = W.place_cells(rest, rot, trans)
    h = NpfemHandle(tris, rest, mat, W.configs.DT, 0, n_cells)
    stride = h.cell_stride
    pos = to_strided(pos0, stride, dev)
    vel = torch.zeros_like(pos)
    f = torch.zeros((n_cells, stride), dtype=torch.float32, device=dev)
    if force_kind == "caps":        # config 5: +-20 pN on the two diametric caps, constant in time
        fc = W.forces.cap_pull_forces(rest, rot, 20e-3)
        f[:, : 3 * n] = torch.as_tensor(fc.reshape(n_cells, 3 * n), device=dev)
    else:
        f[:, : 3 * n] = W.forces.gaussian_forces_torch((n_cells, 3 * n), 1e-3, seed, 0, dev)
    stream = torch.cuda.current_stream()
    for _ in range(warmup):
        h.step(n_cells, pos, vel, f, n_iters, stream)
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    torch.cuda.synchronize()
    ev0.record(stream)
    for _ in range(steps):
        h.step(n_cells, pos, vel, f, n_iters, stream)
    ev1.record(stream)
    torch.cuda.synchronize()
    ms = ev0.elapsed_time(ev1) / steps
    info = h.info()
    finite = bool(torch.isfinite(pos).all().item())
    del h, pos, vel, f
    torch.cuda.empty_cache()
    r = roofline_of(n, T, n_iters, n_cells, ms, peak_measured, peaks, traffic=False)
    return {"workload": name, "n_cells": n_cells, "n_verts": n, "n_iters": n_iters, "steps": steps,
            "warmup": warmup, "ms_per_step": ms, "cell_steps_per_s": n_cells / (ms * 1e-3),
            "vertex_iterations_per_s": n_cells * n * n_iters / (ms * 1e-3),
            "cells_per_cta": info["cells_per_cta"], "threads_per_cta": info["threads_per_cta"],
            "frac": r["frac"], "frac_executed_equivalent": r["executed_equivalent"]["frac"],
            "achieved_tflops": r["achieved"], "hbm_frac": r["hbm"]["frac"], "state_finite": finite}


def run_ours(args) -> None:
    import torch
    import torch.distributed as dist
    import workloads as W
    from paper_2011_04332_b200 import NpfemHandle, npfem_measure_fp32_peak
    from paper_2011_04332_b200.harness import to_strided
    from paper_2011_04332_b200.multi import max_over_ranks, rank_seed

    if not torch.cuda.is_available():
        raise RuntimeError("bench.py needs a CUDA device: the npFEM path has no CPU fallback")
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)
    if world > 1:
        dist.init_process_group("nccl", device_id=dev)

    # ---- the roofline denominator, measured on this GPU before the timed region
    peak_measured = npfem_measure_fp32_peak(0)
    peak_variants = {"ffma": peak_measured}
    if rank == 0 and not args.kernel_only:
        peak_variants.update({"ffma2": npfem_measure_fp32_peak(1), "fadd": npfem_measure_fp32_peak(2),
                              "ffma_fadd_mix": npfem_measure_fp32_peak(3)})

    # ---- workload: config 4, this rank's own cells (weak scaling: fixed cells per GPU)
    spec = W.CONFIGS[CONFIG_ID]
    kind, level, n_full = spec["groups"][0]
    n_cells = args.cells or n_full
    n_iters = spec["n_iters"]
    rest, tris = W.rest_shape(kind, level)
    mat = W.default_material(rest, tris)
    n, T = rest.shape[0], tris.shape[0]
    rng = np.random.Generator(np.random.PCG64(rank_seed(spec["seed"], rank)))
    radius = float(np.linalg.norm(rest, axis=1).max())
    rot, trans = W.random_rigid_placements(n_cells, spec["box"], radius, rng)
    pos0 = W.place_cells(rest, rot, trans)                                 # fp32 [N,V,3]
    opts = {}
    if args.global_mode:
        opts["global_mode"] = args.global_mode
    if args.cells_per_cta:
        opts["cells_per_cta"] = args.cells_per_cta
    if args.drop_tol is not None:
        opts["inv_drop_tol"] = args.drop_tol
    h = NpfemHandle(tris, rest, mat, W.configs.DT, 0, n_cells, **opts)
    info = h.info()
    stride = h.cell_stride
    pos = to_strided(pos0, stride, dev)
    vel = torch.zeros_like(pos)
    fields = []
    for s in range(min(N_FORCE_FIELDS, args.steps + args.warmup)):
        f = torch.zeros((n_cells, stride), dtype=torch.float32, device=dev)
        f[:, : 3 * n] = W.forces.gaussian_forces_torch((n_cells, 3 * n), 1e-3,
                                                       spec["seed"] + 7919 * rank, s, dev)
        fields.append(f)
    stream = torch.cuda.current_stream()

    def barrier():
        torch.cuda.synchronize()
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    # ---- device-resident timing
    for s in range(args.warmup):
        h.step(n_cells, pos, vel, fields[s % len(fields)], n_iters, stream)
    barrier()
    sampler = ClockSampler(local_rank)
    if rank == 0:
        sampler.start()
        time.sleep(0.3)
    ev = [torch.cuda.Event(enable_timing=True) for _ in range(args.steps + 1)]
    t_wall0 = time.time()
    ev[0].record(stream)
    for s in range(args.steps):
        h.step(n_cells, pos, vel, fields[(args.warmup + s) % len(fields)], n_iters, stream)
        ev[s + 1].record(stream)
    barrier()
    t_wall1 = time.time()
    clocks = sampler.stop(t_wall0, t_wall1) if rank == 0 else None
    per_launch_ms = [ev[s].elapsed_time(ev[s + 1]) for s in range(args.steps)]
    total_ms = ev[0].elapsed_time(ev[-1])
    total_ms = max_over_ranks(total_ms, dev)
    finite = bool(torch.isfinite(pos).all().item())

    # ---- end to end through the host-buffer entry point (pinned host memory): every step copies
    #      pos / vel / that step's own force field host -> device and pos / vel back
    e2e = None
    e2e_steps = 0 if args.kernel_only else max(1, min(args.steps, 10))
    field_bytes = n_cells * stride * 4
    if e2e_steps:
        hp = to_strided(pos0, stride, "cpu").pin_memory()
        hv = torch.zeros_like(hp).pin_memory()
        hfs = [f.cpu().pin_memory() for f in fields]
        h.step_host(n_cells, hp, hv, hfs[0], n_iters)                      # warm-up
        barrier()
        t0 = time.perf_counter()
        for s in range(e2e_steps):
            h.step_host(n_cells, hp, hv, hfs[(s + 1) % len(hfs)], n_iters)  # blocking
        torch.cuda.synchronize()
        t_e2e = time.perf_counter() - t0
        t_e2e = max_over_ranks(t_e2e, dev)
        e2e = {"value": world * n_cells * e2e_steps / t_e2e, "unit": "cell-steps/s",
               "h2d_bytes_per_step": 3 * field_bytes, "d2h_bytes_per_step": 2 * field_bytes,
               "steps": e2e_steps, "ms_per_step": 1e3 * t_e2e / e2e_steps,
               "force_fields_cycled": len(hfs),
               "api": "npfem_step_host (pinned host buffers, chunked 3-stream pipeline)"}
        del hp, hv, hfs

    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return

    # ---- roofline of the fused step kernel (the only kernel of a step)
    peaks = load_peaks()
    launch_ms = statistics.mean(per_launch_ms)
    roofline = roofline_of(n, T, n_iters, n_cells, launch_ms, peak_measured, peaks, clocks)
    roofline["fp32_pipe_tflops_measured"] = peak_variants

    # ---- the other cell types and the large-deformation config through the same kernel
    #      (not the headline: BASELINE.json configs 3 and 5; SURVEY.md H8 many-small-cells packing)
    others = []
    if world == 1 and not args.kernel_only and not args.cells:
        del pos, vel, fields, h
        torch.cuda.empty_cache()
        for name, kind2, level2, nc2, it2, fk in (
                ("400000 PLT-1 cells (42 vertices), 20 iterations, N(0,(1 pN)^2) forces", "plt", 1, 400000, 20, "gauss"),
                ("200000 RBC-2 cells (162 vertices), 20 iterations, N(0,(1 pN)^2) forces", "rbc", 2, 200000, 20, "gauss"),
                ("config5: 20000 RBC-3 cells, 30 iterations, +-20 pN cap pulls (first steps of the stretch)", "rbc", 3, 20000, 30, "caps")):
            others.append(time_extra_workload(W, NpfemHandle, to_strided, dev, name, kind2, level2, nc2,
                                              it2, fk, 900 + len(others), 5, 3, peak_measured, peaks))

    cpu = time_oracle(budget_s=12.0, steps=1) if world == 1 and not args.kernel_only else None
    value = world * n_cells * args.steps / (total_ms * 1e-3)
    line = {"metric": "cell-steps/s", "value": value, "unit": "cell-steps/s", "n_gpus": world,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": total_ms / args.steps,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f32",
            "data": "synthetic",
            "vertex_iterations_per_s": value * n * n_iters,
            "config": {"workload": f"config4: {n_cells} RBC-3 cells per GPU (642 vertices, 1280 "
                                   "triangles), random rigid placements in a 300 um cube, 20 "
                                   "iterations per step, N(0,(1 pN)^2) forces redrawn per step",
                       "n_cells_per_gpu": n_cells, "n_verts": n, "n_iters": n_iters,
                       "cells_per_cta": info["cells_per_cta"], "threads_per_cta": info["threads_per_cta"],
                       "smem_bytes": info["smem_bytes"], "global_mode": info["global_mode"],
                       "op_blocks": info["n_op_blocks"], "op_blocks_tf32x1": info["n_op_blocks_tf32x1"],
                       "op_blocks_f16x1": info["n_op_blocks_f16x1"],
                       "ctas_per_sm": info["ctas_per_sm"], "tmem_columns": info["tmem_columns"],
                       "elements_per_cell": info["n_elements"],
                       "l2": "inputs (2.3 GB per step) exceed L2; no flush needed"},
            "e2e": e2e, "gpu_launches": args.steps, "roofline": roofline, "clocks": clocks,
            "state_finite": finite}
    if others:
        line["other_workloads"] = others
    if cpu is not None:
        line["cpu_baseline"] = {k: cpu[k] for k in ("value", "unit", "cores", "kind", "sample")}
    print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()


def main() -> None:
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", choices=["ours", "reference"], default="ours")
    ap.add_argument("--cells", type=int, default=0, help="cells per GPU (default: config 4's 100000)")
    ap.add_argument("--global-mode", type=int, default=0, help="npfem_options.global_mode (0 = default)")
    ap.add_argument("--cells-per-cta", type=int, default=0, help="npfem_options.cells_per_cta (0 = auto)")
    ap.add_argument("--drop-tol", type=float, default=None, help="npfem_options.inv_drop_tol")
    ap.add_argument("--kernel-only", action="store_true",
                    help="tuning runs: skip the e2e and cpu_baseline legs (not a bench line)")
    args = ap.parse_args()
    if args.impl == "reference":
        run_reference(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
