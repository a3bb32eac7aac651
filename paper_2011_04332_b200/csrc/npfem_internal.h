// npfem_internal.h -- data shared between the host-side create step (npfem_plan.cpp), the C ABI
// (npfem_api.cu) and the kernels (npfem_kernels.cu).  Not installed; the public boundary is
// include/npfem.h.  Algorithm and citations: DESIGN.md.
#pragma once
#include <cstdint>
#include <string>
#include <vector>

#include "npfem.h"

namespace npfem {

constexpr int kMaxVerts = 1024;       // one CTA owns whole cells; blockDim <= 1024
constexpr int kMaxCellsPerCta = 5;    // 5 cells x 3 coordinates = 15 right-hand sides (+1 pad = 16)
constexpr int kRhs = 16;              // right-hand sides per CTA in the global step
constexpr int kTriFloats = 17;        // per-triangle float constants (see TriConst below)
constexpr int kTrisPerThread = 2;     // register-resident triangle constants per thread
constexpr int kSmemMaxDynamic = 232448 - 1024;   // 227 KB opt-in limit per CTA minus static shared memory

// Per-triangle constants, all in INTERNAL vertex numbering.
//   ids:  a, b, c  own vertices;  f0, f1, f2  the vertices across edges (a,b), (b,c), (c,a).
//   f[0..2]  D_m^-1 = [[i00, i01], [0, i11]]      f[3], f[4]  w_s = k_strain*A_t, w_a = k_area*A_t
//   f[5+4e .. 8+4e], e = 0,1,2: the hinge on edge e seen from this triangle, scaled by sqrt(w_h):
//       Kp, Kq (edge endpoints in the triangle's cyclic order), Ko (own opposite vertex), r' =
//       sqrt(w_h) * r_h.  The coefficient of the far vertex is -(Kp + Kq + Ko) (rows of K sum to 0).
struct TriConst {
  uint16_t ids[6];
  float f[kTriFloats];
};

struct Plan {
  int n = 0, T = 0, H = 0;
  double h = 0.0;
  npfem_material mat{};
  npfem_options opt{};
  double V0 = 0.0, total_mass = 0.0;

  // caller-order fp64 data kept for npfem_plan_query
  std::vector<int32_t> tris_ext;     // [T][3]
  std::vector<double> mass;          // [n]
  std::vector<double> A;             // [n][n] A_sys
  std::vector<int32_t> hinge_verts;  // [H][4]
  std::vector<double> hinge_K;       // [H][4]
  std::vector<double> hinge_wr;      // [H][2]
  std::vector<double> tri_dminv;     // [T][3]
  std::vector<double> tri_area;      // [T]

  // device-bound data (internal numbering)
  std::vector<int32_t> perm;         // internal -> caller vertex
  std::vector<int32_t> iperm;        // caller -> internal
  std::vector<TriConst> tri;         // [T] in internal triangle order
  std::vector<float> h2_over_m;      // [n]
  std::vector<float> m_over_h2;      // [n]
  std::vector<uint16_t> inc_ptr;     // [n+1] CSR over incident triangles, cyclically ordered
  std::vector<uint16_t> inc_out;     // [3T] float offset of the vertex's 3-vector in the out buffer
  std::vector<uint16_t> inc_ring;    // [3T] internal id of the ring neighbour r_i (triangle i = v, r_i, r_i+1)
  int nvb = 0;                       // number of 8-vertex blocks
  std::vector<int32_t> blk_ptr;      // [nvb+1] kept operator blocks per OUTPUT block
  std::vector<uint16_t> blk_col;     // [n_op_blocks] source block index
  std::vector<float> blk_val;        // [n_op_blocks][64] in mma B-fragment order
  int op_nnz = 0;

  // launch configuration decided at create time
  int threads = 0, cells_per_cta = 0, smem_bytes = 0, global_mode = 0;
};

// Builds the plan on the host in fp64.  Returns NPFEM_OK or an error code and fills `err`.
int build_plan(int n_verts, int n_tris, const int32_t* tris, const double* rest_xyz,
               const npfem_material* mat, double dt, const npfem_options* opts, Plan* plan,
               std::string* err);

// Shared-memory carve-up used by both the host (to size the launch) and the kernel.
struct SmemLayout {
  int z, s, d, r, out, red, total;   // byte offsets
};
inline SmemLayout smem_layout(int n, int T, int nvb, int k) {
  auto up16 = [](int x) { return (x + 15) & ~15; };
  SmemLayout L{};
  int field = up16(k * n * 3 * 4);
  int off = 0;
  L.z = off; off += field;
  L.s = off; off += field;
  L.d = off; off += field;
  L.r = off; off += up16(2 * nvb * 8 * 8 * 4);
  int out_bytes = T * 9 * 4;
  if (out_bytes < k * n * 3 * 4) out_bytes = k * n * 3 * 4;   // doubles as scratch for the volume step
  L.out = off; off += up16(out_bytes);
  L.red = off; off += up16(kMaxCellsPerCta * 32 * 4 * 4);
  L.total = off;
  return L;
}

}  // namespace npfem
