"""ctypes binding with the same names as include/npfem.h (argument marshalling only).

PyTorch is used by callers for device memory and streams; this module accepts raw device
pointers (ints) or anything with ``data_ptr()``, and numpy arrays / pointers for host buffers.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

from . import build as _build

MATERIAL_FIELDS = ("cell_mass", "k_strain", "s_min", "s_max", "k_area", "a_min", "a_max",
                   "k_bend", "w_volume", "v_min", "v_max", "c_alpha", "c_beta", "w_collision",
                   "d_collision", "strain_hardening", "w_garea", "ga_min", "ga_max")

QUERY = {"perm": (1, np.int32), "mass": (2, np.float64), "system": (3, np.float64),
         "operator": (4, np.float64), "hinge_verts": (5, np.int32), "hinge_K": (6, np.float64),
         "hinge_wr": (7, np.float64), "tri_dminv": (8, np.float64), "tri_area": (9, np.float64),
         "operator_x1": (10, np.float64), "operator_f16": (11, np.float64),
         "operator_f16x1": (12, np.float64), "operator_stream": (13, np.float64),
         "stream_shape": (14, np.int32), "stream_val": (15, np.int32), "stream_desc": (16, np.int32),
         "stream_rows": (17, np.int32), "row_scale": (18, np.float64)}

ERROR_NAMES = {0: "NPFEM_OK", -1: "NPFEM_EINVAL", -2: "NPFEM_ENOMEM", -3: "NPFEM_ECUDA",
               -4: "NPFEM_ELIMIT"}


class Material(C.Structure):
    _fields_ = [(f, C.c_double) for f in MATERIAL_FIELDS]


class Options(C.Structure):
    _fields_ = [("inv_drop_tol", C.c_double), ("volume_inner_iters", C.c_int),
                ("cells_per_cta", C.c_int), ("global_mode", C.c_int), ("pair_triangles", C.c_int),
                ("debug_jitter", C.c_int)]


class Info(C.Structure):
    _fields_ = [(f, C.c_int) for f in (
        "n_verts", "n_tris", "n_hinges", "cell_stride", "cells_per_cta", "threads_per_cta",
        "smem_bytes", "n_vblocks", "n_op_blocks", "op_nnz", "global_mode",
        "volume_inner_iters", "n_op_blocks_tf32x1", "n_elements", "n_diamonds", "n_op_blocks_f16x1", "tmem_columns", "ctas_per_sm",
        "ctas_per_sm_limiter")] + [(f, C.c_double) for f in ("rest_volume", "total_mass",
                                                            "inv_drop_tol")]

    def as_dict(self) -> dict:
        return {f: getattr(self, f) for f, _ in self._fields_}


class NpfemError(RuntimeError):
    def __init__(self, code: int, message: str):
        super().__init__(f"{ERROR_NAMES.get(code, code)}: {message}")
        self.code = code


_lib = None


def load_library(path: str | None = None):
    """Load (building if stale) libnpfem_b200.so and declare every symbol of include/npfem.h."""
    global _lib
    if _lib is not None and path is None:
        return _lib
    lib = C.CDLL(path or _build.build())
    vp, ip, dp, fp = C.c_void_p, C.POINTER(C.c_int32), C.POINTER(C.c_double), C.c_void_p
    lib.npfem_create.restype = C.c_int
    lib.npfem_create.argtypes = [C.c_int, C.c_int, ip, dp, C.POINTER(Material), C.c_double,
                                 C.c_int, C.c_int, C.POINTER(Options), C.POINTER(vp)]
    lib.npfem_step.restype = C.c_int
    lib.npfem_step.argtypes = [vp, C.c_int, fp, fp, fp, C.c_int, vp]
    lib.npfem_step_collide.restype = C.c_int
    lib.npfem_step_collide.argtypes = [vp, C.c_int, fp, fp, fp, fp, fp, C.c_int, vp]
    lib.npfem_vertex_areas.restype = C.c_int
    lib.npfem_vertex_areas.argtypes = [vp, C.c_int, fp, fp, vp]
    lib.npfem_step_converged.restype = C.c_int
    lib.npfem_step_converged.argtypes = [vp, C.c_int, fp, fp, fp, C.c_double, C.c_int, vp, vp, vp]
    lib.npfem_step_host.restype = C.c_int
    lib.npfem_step_host.argtypes = [vp, C.c_int, fp, fp, fp, C.c_int]
    lib.npfem_destroy.restype = C.c_int
    lib.npfem_destroy.argtypes = [vp]
    lib.npfem_last_error.restype = C.c_char_p
    lib.npfem_last_error.argtypes = []
    lib.npfem_cell_stride.restype = C.c_int
    lib.npfem_cell_stride.argtypes = [vp]
    lib.npfem_get_info.restype = C.c_int
    lib.npfem_get_info.argtypes = [vp, C.POINTER(Info)]
    lib.npfem_plan_create.restype = C.c_int
    lib.npfem_plan_create.argtypes = [C.c_int, C.c_int, ip, dp, C.POINTER(Material), C.c_double,
                                      C.POINTER(Options), C.POINTER(vp)]
    lib.npfem_plan_destroy.restype = C.c_int
    lib.npfem_plan_destroy.argtypes = [vp]
    lib.npfem_plan_info.restype = C.c_int
    lib.npfem_plan_info.argtypes = [vp, C.POINTER(Info)]
    lib.npfem_plan_query.restype = C.c_int
    lib.npfem_plan_query.argtypes = [vp, C.c_int, vp, C.c_int]
    lib.npfem_measure_fp32_peak.restype = C.c_int
    lib.npfem_measure_fp32_peak.argtypes = [C.c_int, dp]
    lib.npfem_debug_phase_clocks.restype = C.c_int
    lib.npfem_debug_phase_clocks.argtypes = [C.POINTER(C.c_ulonglong), C.c_int]
    if path is None:
        _lib = lib
    return lib


def npfem_measure_fp32_peak(variant: int = 0) -> float:
    """TFLOP/s of the FP32 pipe on the current device (0 FFMA, 1 FFMA2, 2 FADD, 3 FFMA+FADD)."""
    out = C.c_double(0.0)
    _check(load_library().npfem_measure_fp32_peak(int(variant), C.byref(out)))
    return float(out.value)


def npfem_debug_phase_clocks(reset: bool = True) -> list:
    """Diagnostic builds only (-DNPFEM_PHASE_CLOCKS): the 16 per-phase tick counters of the step kernel."""
    out = (C.c_ulonglong * 16)()
    _check(load_library().npfem_debug_phase_clocks(out, int(reset)))
    return [int(x) for x in out]


def npfem_last_error() -> str:
    return load_library().npfem_last_error().decode()


def _check(rc: int):
    if rc < 0:
        raise NpfemError(rc, npfem_last_error())
    return rc


def _material(mat: dict) -> Material:
    return Material(**{k: float(mat.get(k, 0.0)) for k in MATERIAL_FIELDS})


def _options(inv_drop_tol=None, volume_inner_iters=0, cells_per_cta=0, global_mode=0,
             pair_triangles=0, debug_jitter=0) -> Options:
    return Options(-1.0 if inv_drop_tol is None else float(inv_drop_tol), int(volume_inner_iters),
                   int(cells_per_cta), int(global_mode), int(pair_triangles), int(debug_jitter))


def _mesh_args(tris, rest_xyz):
    tris = np.ascontiguousarray(tris, dtype=np.int32)
    rest = np.ascontiguousarray(rest_xyz, dtype=np.float64)
    if tris.ndim != 2 or tris.shape[1] != 3 or rest.ndim != 2 or rest.shape[1] != 3:
        raise ValueError("tris must be [T,3] and rest_xyz [V,3]")
    return tris, rest


def _ptr(x) -> int:
    """Raw address of a device tensor (data_ptr), a numpy array, or an int."""
    if x is None:
        return 0
    if hasattr(x, "data_ptr"):
        return int(x.data_ptr())
    if isinstance(x, np.ndarray):
        return int(x.ctypes.data)
    return int(x)


def npfem_create(tris, rest_xyz, material: dict, dt: float, cell_stride_floats: int = 0,
                 max_cells: int = 0, **options) -> "NpfemHandle":
    return NpfemHandle(tris, rest_xyz, material, dt, cell_stride_floats, max_cells, **options)


def npfem_step(handle: "NpfemHandle", n_cells: int, pos, vel, fext, n_iters: int, stream=None):
    return handle.step(n_cells, pos, vel, fext, n_iters, stream)


def npfem_step_collide(handle: "NpfemHandle", n_cells: int, pos, vel, fext, coll_q, coll_n,
                       n_iters: int, stream=None):
    handle.step_collide(n_cells, pos, vel, fext, coll_q, coll_n, n_iters, stream)


def npfem_vertex_areas(handle: "NpfemHandle", n_cells: int, pos, areas, stream=None):
    handle.vertex_areas(n_cells, pos, areas, stream)


def npfem_step_converged(handle: "NpfemHandle", n_cells: int, pos, vel, fext, tol: float,
                         max_iters: int, iters_out=None, res_out=None, stream=None):
    handle.step_converged(n_cells, pos, vel, fext, tol, max_iters, iters_out, res_out, stream)


def npfem_step_host(handle: "NpfemHandle", n_cells: int, pos, vel, fext, n_iters: int):
    return handle.step_host(n_cells, pos, vel, fext, n_iters)


def npfem_destroy(handle: "NpfemHandle"):
    handle.destroy()


def npfem_cell_stride(handle: "NpfemHandle") -> int:
    return handle.cell_stride


class NpfemHandle:
    """Owns one npfem_handle (one cell TYPE).  Raises NpfemError if CUDA is unavailable."""

    def __init__(self, tris, rest_xyz, material: dict, dt: float, cell_stride_floats: int = 0,
                 max_cells: int = 0, **options):
        lib = load_library()
        tris, rest = _mesh_args(tris, rest_xyz)
        m, o = _material(material), _options(**options)
        h = C.c_void_p()
        _check(lib.npfem_create(rest.shape[0], tris.shape[0],
                                tris.ctypes.data_as(C.POINTER(C.c_int32)),
                                rest.ctypes.data_as(C.POINTER(C.c_double)), C.byref(m), float(dt),
                                int(cell_stride_floats), int(max_cells), C.byref(o), C.byref(h)))
        self._h = h
        self.n_verts = rest.shape[0]
        self.cell_stride = int(lib.npfem_cell_stride(h))

    def info(self) -> dict:
        i = Info()
        _check(load_library().npfem_get_info(self._h, C.byref(i)))
        return i.as_dict()

    def step(self, n_cells: int, pos, vel, fext, n_iters: int, stream=None):
        """Asynchronous on `stream` (a torch.cuda.Stream, a raw cudaStream_t int, or None)."""
        s = 0 if stream is None else int(getattr(stream, "cuda_stream", stream))
        _check(load_library().npfem_step(self._h, int(n_cells), _ptr(pos), _ptr(vel), _ptr(fext),
                                         int(n_iters), s))

    def step_collide(self, n_cells: int, pos, vel, fext, coll_q, coll_n, n_iters: int, stream=None):
        """npfem_step with one colliding neighbour (point, outward normal; zero normal = none) per vertex."""
        s = 0 if stream is None else int(getattr(stream, "cuda_stream", stream))
        _check(load_library().npfem_step_collide(self._h, int(n_cells), _ptr(pos), _ptr(vel), _ptr(fext),
                                                 _ptr(coll_q), _ptr(coll_n), int(n_iters), s))

    def vertex_areas(self, n_cells: int, pos, areas, stream=None):
        s = 0 if stream is None else int(getattr(stream, "cuda_stream", stream))
        _check(load_library().npfem_vertex_areas(self._h, int(n_cells), _ptr(pos), _ptr(areas), s))

    def step_converged(self, n_cells: int, pos, vel, fext, tol: float, max_iters: int,
                       iters_out=None, res_out=None, stream=None):
        """Converged quasi-Newton step (npfem_step_converged); iters_out int32 / res_out float32
        device arrays [n_cells] or None.  Asynchronous on `stream`."""
        s = 0 if stream is None else int(getattr(stream, "cuda_stream", stream))
        _check(load_library().npfem_step_converged(
            self._h, int(n_cells), _ptr(pos), _ptr(vel), _ptr(fext), float(tol), int(max_iters),
            _ptr(iters_out) if iters_out is not None else None,
            _ptr(res_out) if res_out is not None else None, s))

    def step_host(self, n_cells: int, pos, vel, fext, n_iters: int):
        _check(load_library().npfem_step_host(self._h, int(n_cells), _ptr(pos), _ptr(vel),
                                              _ptr(fext), int(n_iters)))

    def destroy(self):
        if getattr(self, "_h", None) is not None:
            load_library().npfem_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.destroy()
        except Exception:
            pass


class NpfemPlan:
    """Host-only create step (no CUDA): used by the CPU tests to inspect create-time data."""

    def __init__(self, tris, rest_xyz, material: dict, dt: float, **options):
        lib = load_library()
        tris, rest = _mesh_args(tris, rest_xyz)
        m, o = _material(material), _options(**options)
        p = C.c_void_p()
        _check(lib.npfem_plan_create(rest.shape[0], tris.shape[0],
                                     tris.ctypes.data_as(C.POINTER(C.c_int32)),
                                     rest.ctypes.data_as(C.POINTER(C.c_double)), C.byref(m),
                                     float(dt), C.byref(o), C.byref(p)))
        self._p = p

    def info(self) -> dict:
        i = Info()
        _check(load_library().npfem_plan_info(self._p, C.byref(i)))
        return i.as_dict()

    def query(self, what: str) -> np.ndarray:
        code, dtype = QUERY[what]
        lib = load_library()
        n = _check(lib.npfem_plan_query(self._p, code, None, 0))
        out = np.empty(n, dtype=dtype)
        _check(lib.npfem_plan_query(self._p, code, out.ctypes.data, n))
        return out

    def __del__(self):
        p = getattr(self, "_p", None)
        if p is not None and _lib is not None:
            _lib.npfem_plan_destroy(p)
            self._p = None
