// npfem_kernels.cuh -- launch interface between the C ABI (npfem_api.cu) and the step kernel.
#pragma once
#include <cuda_runtime.h>

#include "npfem_internal.h"

namespace npfem {

// The volume projection stops iterating once the violation |V - V*| it has just corrected to first
// order is below kVolTol * V0: the step converges quadratically, so the remaining violation is
// then below the fp32 resolution of V itself (A-17).
constexpr float kVolTol = 2e-4f;
// Later passes stop once the last one changed the projection by less than kVolDTol * V0^(1/3)
// (rms per vertex): below the fp32 resolution of the cell-local coordinates.
constexpr float kVolDTol = 5e-8f;

// Everything the fused step kernel needs, passed by value.  Pointers are device pointers.
struct DevParams {
  int n, E, nvb, k, n_cells, cell_stride, n_iters, vol_iters;
  float h, w_volume, V0, Vmin, Vmax;       // Vmin/Vmax = v_min*V0, v_max*V0
  float s_min, s_max, a_min, a_max;
  float cbh;                               // c_beta / h (stiffness-proportional damping, A-20)
  int damped;                              // c_alpha != 0 or c_beta != 0
  int jitter;                              // debug: seed of the per-warp sleeps after every barrier (0 = off)
  int dbg;                                 // diagnostic builds: ablation mask of the MODE 3 product (0 in the shipped library)
  const uint16_t* perm;                    // [NP] internal -> caller vertex (padding: 0)
  const float4* elem_c;                    // [kElemGroups][E] element constants (npfem_api.cu)
  const float* h2_over_m;                  // [NP]
  const float* m_over_h2;                  // [NP] m (1/h^2 + c_alpha/h)
  const float* damp_m;                     // [NP] m c_alpha / h
  const uint4* vrole;                      // [NP][2] vertex-role constants (npfem_api.cu)
  const uint16_t* inc_ptr;                 // [n+1]
  const uint16_t* inc_off;                 // byte offsets into the element result buffer
  const uint16_t* ring_ptr;                // [n+1]
  const uint16_t* ring_off;                // byte offsets into one cell's z4
  const int* blk_ptr;                      // [nvb][3]: first 3xTF32 block, first 1xTF32 block, end
  const uint16_t* blk_col;                 // [n_blocks_padded]
  const float* blk_val;                    // [n_blocks_padded][64]
  // global_mode 3: per-warp operator streams of uniform shape (npfem_internal.h)
  const uint4* hs_val;                     // [warps][hs_slots][32]: B fragments, 16 bytes per lane and slot
  const uint4* hs_desc;                    // [warps][32 lanes]: descriptors of slots lane (x, y) and lane + 32 (z, w)
  int hs_slots;                            // slots per warp (<= 64)
  int hs_na[4], hs_nb[4];                  // per row slot: three-product slots, one-product slots
  uint8_t hs_rows[4 * 32];                 // [row slot][warp] -> output block row, 255 = none
  const float* hp_scale;                   // [NP] 2^-k of the operator row's scaling
  float* pos;
  float* vel;
  const float* fext;
  const float* coll_q;                     // [n_cells][cell_stride] colliding neighbour point per vertex, or NULL
  const float* coll_n;                     // [n_cells][cell_stride] its outward unit normal (0 = none), or NULL
  float w_coll, d_coll;                    // collision weight, contact distance (A-22)
  float hard;                              // strain hardening beta (A-23)
  SmemLayout L;
};

// Diagnostic builds only (-DNPFEM_PHASE_CLOCKS): accumulated clock64() ticks per phase of the step
// kernel, summed over CTAs and iterations; cudaErrorNotSupported in the shipped library.
cudaError_t read_phase_clocks(unsigned long long* out16, int reset);

// Opt the kernels into their dynamic shared memory once per process.  Returns a cudaError_t.
cudaError_t configure_kernels(int smem_bytes);

// Enqueue one step on `stream`.  threads = CTA size (multiple of 32), mode 1 = SIMT, 2 = 3xTF32.
cudaError_t launch_step(const DevParams& p, int threads, int smem_bytes, int mode,
                        cudaStream_t stream);

// Area per surface vertex at the current positions: areas [n_cells][n] in caller order.
cudaError_t launch_vertex_areas(const DevParams& p, int threads, float* areas, cudaStream_t stream);

// Converged quasi-Newton step (npfem_converged.cu): one CTA per cell; p.k must be 1 and p.L the
// shared-memory layout for k = 1.  iters_out / res_out: device arrays [n_cells] or NULL.
cudaError_t configure_converged_kernels();
cudaError_t launch_converged(const DevParams& p, int threads, int smem_bytes, float tol, int max_iters,
                             int* iters_out, float* res_out, cudaStream_t stream);

}  // namespace npfem
