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
constexpr int kRhs = 16;              // right-hand sides per CTA in the global step (mma M)
constexpr int kElemFloats = 31;       // per-element float constants (see ElemConst below)
constexpr int kRegList = 6;           // incidence / ring entries a vertex thread keeps in registers
constexpr int kMaxOpSlots = 64;       // global_mode 3: slots per warp whose descriptors fit four registers per lane
constexpr int kSmemMaxDynamic = 232448 - 1024;   // 227 KB opt-in limit per CTA minus static shared memory

// One ELEMENT = the work of one thread in the local step: a "diamond" of two triangles
// t1 = (a,b,c) and t2 = (b,a,d) sharing the edge (a,b), or a single triangle t1 whose t2 carries
// zero weights.  All vertex ids are INTERNAL numbers.
//   ids:  a, b, c, d  own vertices;  f1..f4 the vertices across the outer edges
//         (b,c), (c,a), (a,d), (d,b).
//   f[0..4]   t1: D_m^-1 = [[i00, i01], [0, i11]] for the vertex order (a,b,c); w_s, w_a
//   f[5..9]   t2: the same for the vertex order (b,a,d)
//   f[10+4e .. 13+4e], e = 0..4: hinge e scaled by sqrt(w_h): Kp, Kq (edge endpoints), Ko (the
//         element's own opposite vertex), r' = sqrt(w_h) r_h; the coefficient of the vertex
//         across is -(Kp+Kq+Ko).  e = 0 the shared edge (a,b | c ; d); e = 1 (b,c | a ; f1);
//         e = 2 (c,a | b ; f2); e = 3 (a,d | b ; f3); e = 4 (d,b | a ; f4).
//   f[30]     he: 1 for a diamond (the shared hinge is evaluated once, in full), 0.5 for a single
//         triangle (its neighbour evaluates the other half; nothing goes to d).
// Outer hinges are evaluated by both elements that see them, each adding half of the end-point
// terms and all of its own opposite vertex's term, so that every hinge counts exactly once.
struct ElemConst {
  uint16_t ids[8];
  float f[kElemFloats];
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
  int E = 0;                         // number of elements (diamonds + single triangles)
  int n_diamonds = 0;
  std::vector<ElemConst> elem;       // [E]
  std::vector<int32_t> elem_tris;    // [E][2] caller triangle ids (second = -1 for a single)
  std::vector<float> h2_over_m;      // [n]
  std::vector<float> m_over_h2;      // [n] m (1/h^2 + c_alpha/h)
  std::vector<float> damp_m;         // [n] m c_alpha/h
  bool damped = false;               // c_alpha != 0 or c_beta != 0 (reading A-20)
  std::vector<uint16_t> inc_ptr;     // [n+1] CSR over the element slots a vertex gathers from
  std::vector<uint16_t> inc_off;     // byte offset of the slot's float4 in the out buffer
  std::vector<uint16_t> ring_ptr;    // [n+1] CSR over the cyclically ordered ring neighbours
  std::vector<uint16_t> ring_off;    // byte offset (16 * internal id) of the neighbour in z4
  int nvb = 0;                       // number of 8-vertex blocks
  std::vector<int32_t> blk_ptr;      // [nvb][3] per OUTPUT block row: first 3xTF32 block, first 1xTF32 block, end
  std::vector<uint16_t> blk_col;     // [n_blocks_padded] source block index
  std::vector<float> blk_val;        // [n_blocks_padded][64] in mma B-fragment order
  // The same operator for global_mode 3 (two-term fp16 split, mma m16n8k16): the kept blocks of an
  // OUTPUT block row grouped in PAIRS of source blocks (one mma covers K = 16 = two source blocks):
  // first the pairs applied with three products (hi*hi + hi*lo + lo*hi), then the pairs whose
  // blocks are so small that the hi*hi product alone is exact to fp32 rounding of the row sum.
  // Rows are scaled by a power of two (hp_scale) so that their entries sit in the fp16 range.
  // Every warp of the step kernel owns up to 4 output block rows ("row slots" j = 0..3) and consumes
  // ONE contiguous stream of 512-byte SLOTS (16 bytes per lane) in a fixed order that is the same
  // for all warps: per row slot j first hs_na[j] three-product slots (one pair each: B fragment hi,
  // lo), then hs_nb[j] one-product slots (two pairs each: hi, hi).  Rows are sorted by cost and
  // dealt to the row slots so that the rows of a slot have similar lengths; shorter rows are padded
  // with zero pairs (the phase ends at a CTA barrier, so the longest row of a slot sets the time
  // anyway).  Uniform shapes make every branch of the product loop warp-uniform at compile time.
  // A slot's descriptor holds the byte offsets of its pairs' source blocks in the right-hand-side
  // buffer: x = pair 0 (low / high 16 bits: kb 512 | (kb & 7) << 5, the kernel's bank swizzle),
  // y = pair 1 (one-product slots); absent blocks point at block 0 with zero values.
  int hs_na[4] = {0, 0, 0, 0}, hs_nb[4] = {0, 0, 0, 0};
  int hs_slots = 0;                  // slots per warp = sum_j hs_na[j] + hs_nb[j]
  std::vector<uint8_t> hs_rows;      // [4][32] output block row of (row slot, warp), 255 = none
  std::vector<uint32_t> hs_desc;     // [warps][32 lanes][4]: descriptors of slots lane (words 0, 1) and lane + 32 (words 2, 3)
  std::vector<uint32_t> hs_val;      // [warps][hs_slots][32 lanes][4]
  std::vector<int32_t> hp_ptr;       // [nvb][4] pair ranges for npfem_plan_query: three-product [0],[1]), one-product [2],[3])
  std::vector<uint32_t> hp_col_a;    // [pairs A] source blocks kb1 | kb2 << 16 (0xffff = none)
  std::vector<uint32_t> hp_val_a;    // [pairs A][32 lanes][4]: B fragment hi (2 words), lo (2 words)
  std::vector<uint32_t> hp_col_b;    // [pairs B]
  std::vector<uint32_t> hp_val_b;    // [pairs B][32 lanes][2]: B fragment hi
  std::vector<float> hp_scale;       // [n] 2^-k of the row's scaling 2^k (internal numbering)
  int n_op_blocks_h1 = 0;            // kept blocks applied as one fp16 product
  int n_op_blocks = 0;               // kept blocks (without the zero padding blocks)
  int n_op_blocks_x1 = 0;            // of those, blocks applied as one TF32 product
  int op_nnz = 0;

  // launch configuration decided at create time
  int threads = 0, cells_per_cta = 0, smem_bytes = 0, global_mode = 0;
};

// Builds the plan on the host in fp64.  Returns NPFEM_OK or an error code and fills `err`.
int build_plan(int n_verts, int n_tris, const int32_t* tris, const double* rest_xyz,
               const npfem_material* mat, double dt, const npfem_options* opts, Plan* plan,
               std::string* err);

// Shared-memory carve-up used by both the host (to size the launch) and the kernel.
//   z4   [k][NP] float4   current iterate z = s + d, cell-local coordinates (w unused)
//   ec   [9][E] float4    element constants (kElemGroups groups of 4 words, see npfem_api.cu)
//   ra   max(E*64, NP*64) element results `out` [4][E] float4 of the ODD cells during the local
//                         step, then the tf32 high parts of the right-hand sides in mma
//                         A-fragment order ([nvb][32] float4)
//   rb   max(E*64, NP*64) element results of the EVEN cells during the local step, then the
//                         tf32 low parts of the right-hand sides, then the increments of d
//   red  [5][32] float4   per-warp partial sums of the volume reductions, then [5] float4 centroids,
//                         then [5] uint32: bits of max |r| per cell (global_mode 3: fp16 scaling)
// The inertial prediction s and the correction d are private to the thread that owns the vertex
// and live in tensor memory (TMEM), 32 columns per group of 4 warps.
constexpr int kElemGroups = 9;
struct SmemLayout {
  int z4, ec, ra, rb, red, total;   // byte offsets
};
inline SmemLayout smem_layout(int n, int E, int nvb, int k) {
  (void)n;
  const int NP = nvb * 8;
  SmemLayout L{};
  int off = 0;
  L.z4 = off; off += k * NP * 16;
  L.ec = off; off += kElemGroups * E * 16;
  const int rbuf = E * 64 > NP * 64 ? E * 64 : NP * 64;   // both buffers hold [4][E] element results
  L.ra = off; off += rbuf;
  L.rb = off; off += rbuf;
  L.red = off; off += kMaxCellsPerCta * 32 * 16 + kMaxCellsPerCta * 16 + 32;   // + the cells' centroids + residual maxima (global_mode 3)
  L.total = off;
  return L;
}

}  // namespace npfem
