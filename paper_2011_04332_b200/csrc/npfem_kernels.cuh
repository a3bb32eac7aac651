// npfem_kernels.cuh -- launch interface between the C ABI (npfem_api.cu) and the step kernel.
#pragma once
#include <cuda_runtime.h>

#include "npfem_internal.h"

namespace npfem {

// Everything the fused step kernel needs, passed by value.  Pointers are device pointers.
struct DevParams {
  int n, T, nvb, k, n_cells, cell_stride, n_iters, vol_iters;
  float h, w_volume, V0, Vmin, Vmax;       // Vmin/Vmax = v_min*V0, v_max*V0
  float s_min, s_max, a_min, a_max;
  const uint16_t* perm;                    // [n] internal -> caller vertex
  const uint16_t* tri_ids;                 // [6][T]  structure of arrays
  const float* tri_f;                      // [17][T] structure of arrays
  const float* h2_over_m;                  // [n]
  const float* m_over_h2;                  // [n]
  const uint16_t* inc_ptr;                 // [n+1]
  const uint16_t* inc_out;                 // [3T]
  const uint16_t* inc_ring;                // [3T]
  const int* blk_ptr;                      // [nvb+1]
  const uint16_t* blk_col;                 // [n_op_blocks]
  const float* blk_val;                    // [n_op_blocks][64]
  float* pos;
  float* vel;
  const float* fext;
  SmemLayout L;
};

// Opt the kernels into their dynamic shared memory once per process.  Returns a cudaError_t.
cudaError_t configure_kernels(int smem_bytes);

// Enqueue one step on `stream`.  threads = CTA size (multiple of 32), mode 1 = SIMT, 2 = 3xTF32.
cudaError_t launch_step(const DevParams& p, int threads, int smem_bytes, int mode,
                        cudaStream_t stream);

}  // namespace npfem
