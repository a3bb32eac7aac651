"""B200-native npFEM solid-phase hot path (arXiv 2011.04332): thin ctypes binding over the C ABI.

Every step of the method runs inside libnpfem_b200.so (hand-written CUDA for sm_100a); this
package only marshals arguments.  There is no CPU fallback: creating a handle without a CUDA
device raises.
"""
from .binding import (NpfemError, NpfemHandle, NpfemPlan, load_library, npfem_create,
                      npfem_destroy, npfem_step, npfem_step_collide, npfem_step_converged, npfem_step_host,
                      npfem_vertex_areas, npfem_last_error,
                      npfem_cell_stride, npfem_measure_fp32_peak, MATERIAL_FIELDS, QUERY)

__all__ = ["NpfemError", "NpfemHandle", "NpfemPlan", "load_library", "npfem_create",
           "npfem_destroy", "npfem_step", "npfem_step_collide", "npfem_step_converged", "npfem_step_host",
           "npfem_vertex_areas", "npfem_last_error",
           "npfem_cell_stride", "npfem_measure_fp32_peak", "MATERIAL_FIELDS", "QUERY"]
