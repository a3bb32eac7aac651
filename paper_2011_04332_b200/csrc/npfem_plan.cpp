// npfem_plan.cpp -- host-side, fp64 "create" step of the npFEM hot path.
//
// Builds, once per cell TYPE, everything the step kernel treats as constant:
//   rest operators D_m^-1, rest areas and corner cotangents   (per-element energies
//   lumped masses                                              with a weight and parameters; :66
//   hinge rows K, weights w_h, rest magnitudes r_h             mass lumping; readings A-2..A-4)
//   A_sys = M/h^2 + sum w A^T A + w_volume I                   (north_star: the shared SPD system)
//   T = A_sys^-1 in fp64, a locality ordering of the vertices, and T cut into 8x8 blocks with the
//   numerically negligible ones dropped.
// No CUDA here: this file is plain C++ so that the CPU tests can exercise it through
// npfem_plan_create / npfem_plan_query.
#include <algorithm>
#include <array>
#include <cmath>
#include <cstring>
#include <deque>
#include <numeric>

#include "npfem_internal.h"

namespace npfem {
namespace {

struct V3 {
  double x, y, z;
};
inline V3 operator-(V3 a, V3 b) { return {a.x - b.x, a.y - b.y, a.z - b.z}; }
inline V3 operator+(V3 a, V3 b) { return {a.x + b.x, a.y + b.y, a.z + b.z}; }
inline V3 operator*(double s, V3 a) { return {s * a.x, s * a.y, s * a.z}; }
inline double dot(V3 a, V3 b) { return a.x * b.x + a.y * b.y + a.z * b.z; }
inline V3 cross(V3 a, V3 b) {
  return {a.y * b.z - a.z * b.y, a.z * b.x - a.x * b.z, a.x * b.y - a.y * b.x};
}
inline double norm(V3 a) { return std::sqrt(dot(a, a)); }

// cotangent of the angle at p between (q - p) and (r - p)
inline double cot_corner(V3 p, V3 q, V3 r) {
  V3 u = q - p, v = r - p;
  return dot(u, v) / norm(cross(u, v));
}

// ---------------------------------------------------------------- vertex ordering
// Recursive graph bisection: inside a vertex subset, breadth-first distances from a
// pseudo-peripheral vertex split the subset into a near and a far half (the cut is moved to a
// multiple of 8 when the subset is large enough), recursively.  Consecutive groups of 8/16/32
// internal indices are then compact surface patches, which is what keeps the 8x8 blocks of the
// numerically sparse A_sys^-1 few.
// fp32 -> fp16 bits, round to nearest even (subnormals included); |f| < 65520 by construction.
uint16_t half_bits(float f) {
  uint32_t x;
  std::memcpy(&x, &f, 4);
  const uint16_t sign = (uint16_t)((x >> 16) & 0x8000u);
  x &= 0x7fffffffu;
  if (x >= 0x477ff000u) return (uint16_t)(sign | 0x7c00u);   // rounds to >= 65536: infinity
  if (x < 0x38800000u) {                                      // below 2^-14: fp16 subnormal, unit 2^-24
    float a;
    std::memcpy(&a, &x, 4);
    return (uint16_t)(sign | (uint32_t)std::nearbyint(a * 16777216.0f));
  }
  uint32_t hb = (((x >> 23) - 112u) << 10) | ((x & 0x7fffffu) >> 13);
  const uint32_t rem = x & 0x1fffu;
  if (rem > 0x1000u || (rem == 0x1000u && (hb & 1u))) ++hb;   // a carry into the exponent is the right result
  return (uint16_t)(sign | hb);
}
float half_value(uint16_t hb) {
  const int e = (hb >> 10) & 0x1f, m = hb & 0x3ff;
  const float v = e == 0 ? std::ldexp((float)m, -24) : std::ldexp((float)(m | 0x400), e - 25);
  return (hb & 0x8000u) ? -v : v;
}

struct Bisector {
  const std::vector<std::vector<int>>& adj;
  std::vector<int> mark, dist;
  int stamp = 0;
  explicit Bisector(const std::vector<std::vector<int>>& a)
      : adj(a), mark(a.size(), 0), dist(a.size(), 0) {}

  // BFS restricted to vertices with mark == tag; returns visit order
  std::vector<int> bfs(int src, int tag, const std::vector<int>& tagv) {
    std::vector<int> order;
    ++stamp;
    std::deque<int> q;
    q.push_back(src);
    dist[src] = stamp;
    order.push_back(src);
    while (!q.empty()) {
      int u = q.front();
      q.pop_front();
      for (int v : adj[u]) {
        if (tagv[v] == tag && dist[v] != stamp) {
          dist[v] = stamp;
          q.push_back(v);
          order.push_back(v);
        }
      }
    }
    return order;
  }

  void run(std::vector<int> verts, std::vector<int>& tagv, int& next_tag, std::vector<int>& out) {
    if (verts.size() <= 1) {
      for (int v : verts) out.push_back(v);
      return;
    }
    int tag = next_tag++;
    for (int v : verts) tagv[v] = tag;
    int a = verts[0];
    std::vector<int> order;
    for (int sweep = 0; sweep < 4; ++sweep) {
      order = bfs(a, tag, tagv);
      a = order.back();
    }
    if (order.size() < verts.size()) {   // disconnected remainder: append in given order
      ++stamp;
      for (int v : order) dist[v] = stamp;
      for (int v : verts)
        if (dist[v] != stamp) order.push_back(v);
    }
    size_t half = order.size() / 2;
    if (order.size() >= 16) {
      size_t h8 = (half + 7) / 8 * 8;
      if (h8 < order.size()) half = h8;
    }
    std::vector<int> left(order.begin(), order.begin() + half), right(order.begin() + half, order.end());
    run(std::move(left), tagv, next_tag, out);
    run(std::move(right), tagv, next_tag, out);
  }
};

}  // namespace

int build_plan(int n, int T, const int32_t* tris, const double* X, const npfem_material* mat,
               double dt, const npfem_options* opts, Plan* P, std::string* err) {
  auto fail = [&](int code, const char* msg) {
    if (err) *err = msg;
    return code;
  };
  if (!tris || !X || !mat || !P) return fail(NPFEM_EINVAL, "null argument");
  if (n < 4 || T < 4) return fail(NPFEM_EINVAL, "mesh needs at least 4 vertices and 4 triangles");
  if (!(dt > 0.0)) return fail(NPFEM_EINVAL, "dt must be positive");
  if (n > kMaxVerts) return fail(NPFEM_ELIMIT, "n_verts exceeds 1024 (one CTA owns whole cells)");
  if (mat->s_min > mat->s_max || mat->a_min > mat->a_max || mat->v_min > mat->v_max)
    return fail(NPFEM_EINVAL, "clamp band with min > max");
  if (!(mat->c_alpha >= 0.0) || !(mat->c_beta >= 0.0))
    return fail(NPFEM_EINVAL, "damping coefficients c_alpha, c_beta must be >= 0 (DESIGN.md A-20)");
  if (!(mat->strain_hardening >= 0.0))
    return fail(NPFEM_EINVAL, "strain_hardening must be >= 0 (DESIGN.md A-23)");
  if (mat->w_garea != 0.0)
    return fail(NPFEM_EINVAL, "the global-area term (w_garea != 0) exists in the oracle only (DESIGN.md A-24)");
  if (!(mat->w_collision >= 0.0) || !(mat->d_collision >= 0.0))
    return fail(NPFEM_EINVAL, "collision weight and contact distance must be >= 0 (DESIGN.md A-22)");
  if (!(mat->cell_mass > 0.0)) return fail(NPFEM_EINVAL, "cell_mass must be positive");
  if (mat->k_strain < 0 || mat->k_area < 0 || mat->k_bend < 0 || mat->w_volume < 0)
    return fail(NPFEM_EINVAL, "negative weight");
  if ((3 * T) % 2) return fail(NPFEM_EINVAL, "odd number of triangle edges: mesh is not closed");
  for (int i = 0; i < 3 * T; ++i)
    if (tris[i] < 0 || tris[i] >= n) return fail(NPFEM_EINVAL, "triangle index out of range");

  P->n = n; P->T = T; P->H = 3 * T / 2; P->h = dt; P->mat = *mat;
  npfem_options o{};
  o.inv_drop_tol = std::ldexp(1.0, -24);
  if (opts) {
    if (opts->inv_drop_tol >= 0.0) o.inv_drop_tol = opts->inv_drop_tol;   // < 0 (or NaN) = default
    o.volume_inner_iters = opts->volume_inner_iters;
    o.cells_per_cta = opts->cells_per_cta;
    o.global_mode = opts->global_mode;
    o.pair_triangles = opts->pair_triangles;
    o.debug_jitter = opts->debug_jitter;
  }
  if (o.volume_inner_iters <= 0) o.volume_inner_iters = 8;
  if (o.volume_inner_iters > 32) o.volume_inner_iters = 32;
  if (o.cells_per_cta < 0 || o.cells_per_cta > kMaxCellsPerCta)
    return fail(NPFEM_EINVAL, "cells_per_cta must be 0..5");
  if (o.global_mode < 0 || o.global_mode > 3) return fail(NPFEM_EINVAL, "global_mode must be 0..3");
  if (o.pair_triangles < 0 || o.pair_triangles > 2) return fail(NPFEM_EINVAL, "pair_triangles must be 0..2");
  P->tris_ext.assign(tris, tris + 3 * T);
  auto Xv = [&](int v) { return V3{X[3 * v], X[3 * v + 1], X[3 * v + 2]}; };

  // ---- A-14: closed, consistently oriented 2-manifold: every directed edge once, its reverse once
  std::vector<int32_t> etri((size_t)n * n, -1);   // triangle holding directed edge u->v
  std::vector<int8_t> eslot((size_t)n * n, 0);    // slot of u in that triangle
  for (int t = 0; t < T; ++t)
    for (int e = 0; e < 3; ++e) {
      int u = tris[3 * t + e], v = tris[3 * t + (e + 1) % 3];
      if (u == v) return fail(NPFEM_EINVAL, "degenerate triangle (repeated vertex)");
      if (etri[(size_t)u * n + v] != -1)
        return fail(NPFEM_EINVAL, "directed edge used twice: inconsistent orientation or non-manifold");
      etri[(size_t)u * n + v] = t;
      eslot[(size_t)u * n + v] = (int8_t)e;
    }
  for (int t = 0; t < T; ++t)
    for (int e = 0; e < 3; ++e) {
      int u = tris[3 * t + e], v = tris[3 * t + (e + 1) % 3];
      if (etri[(size_t)v * n + u] == -1) return fail(NPFEM_EINVAL, "open edge: mesh is not closed");
    }
  auto opposite = [&](int u, int v) {   // vertex opposite the directed edge u->v
    int t = etri[(size_t)u * n + v];
    int s = eslot[(size_t)u * n + v];
    return (int)tris[3 * t + (s + 2) % 3];
  };

  // ---- per-triangle rest data
  P->tri_dminv.resize(3 * (size_t)T);
  P->tri_area.resize(T);
  std::vector<double> cotc(3 * (size_t)T);   // rest cotangent at corner slot s of triangle t
  double total_area = 0.0;
  for (int t = 0; t < T; ++t) {
    V3 a = Xv(tris[3 * t]), b = Xv(tris[3 * t + 1]), c = Xv(tris[3 * t + 2]);
    V3 e1 = b - a, e2 = c - a, nn = cross(e1, e2);
    double twoA = norm(nn), l1 = norm(e1);
    if (!(twoA > 0.0) || !(l1 > 0.0)) return fail(NPFEM_EINVAL, "degenerate rest triangle");
    // local frame t1 = e1/|e1|, t2 = n x t1:  D_m = [[|e1|, e2.t1], [0, e2.t2]]
    double d00 = l1, d01 = dot(e2, e1) / l1, d11 = twoA / l1;
    P->tri_dminv[3 * t + 0] = 1.0 / d00;
    P->tri_dminv[3 * t + 1] = -d01 / (d00 * d11);
    P->tri_dminv[3 * t + 2] = 1.0 / d11;
    P->tri_area[t] = 0.5 * twoA;
    total_area += 0.5 * twoA;
    cotc[3 * t + 0] = cot_corner(a, b, c);
    cotc[3 * t + 1] = cot_corner(b, c, a);
    cotc[3 * t + 2] = cot_corner(c, a, b);
  }

  // ---- lumped masses (A-4) and rest volume
  P->mass.assign(n, 0.0);
  for (int t = 0; t < T; ++t)
    for (int e = 0; e < 3; ++e) P->mass[tris[3 * t + e]] += P->tri_area[t] / 3.0;
  for (int v = 0; v < n; ++v) {
    if (!(P->mass[v] > 0.0)) return fail(NPFEM_EINVAL, "vertex without triangles");
    P->mass[v] *= mat->cell_mass / total_area;
  }
  P->total_mass = mat->cell_mass;
  double V0 = 0.0;
  for (int t = 0; t < T; ++t)
    V0 += dot(Xv(tris[3 * t]), cross(Xv(tris[3 * t + 1]), Xv(tris[3 * t + 2])));
  V0 /= 6.0;
  if (!(V0 > 0.0)) return fail(NPFEM_EINVAL, "rest volume is not positive (inward orientation?)");
  P->V0 = V0;

  // ---- hinges, one per undirected edge, increasing (min, max)
  const int H = P->H;
  P->hinge_verts.resize(4 * (size_t)H);
  P->hinge_K.resize(4 * (size_t)H);
  P->hinge_wr.resize(2 * (size_t)H);
  std::vector<int32_t> hinge_of((size_t)n * n, -1);   // undirected lookup (both orders)
  int hc = 0;
  for (int u = 0; u < n; ++u)
    for (int v = u + 1; v < n; ++v) {
      if (etri[(size_t)u * n + v] == -1) continue;
      if (hc >= H) return fail(NPFEM_EINVAL, "edge count does not match 3T/2");
      int x2 = opposite(u, v), x3 = opposite(v, u);
      V3 p0 = Xv(u), p1 = Xv(v), p2 = Xv(x2), p3 = Xv(x3);
      double c01 = cot_corner(p0, p1, p2), c02 = cot_corner(p0, p1, p3);
      double c03 = cot_corner(p1, p0, p2), c04 = cot_corner(p1, p0, p3);
      double K[4] = {c03 + c04, c01 + c02, -c01 - c03, -c02 - c04};
      double A0 = 0.5 * norm(cross(p1 - p0, p2 - p0)), A1 = 0.5 * norm(cross(p1 - p0, p3 - p0));
      double wh = mat->k_bend * 3.0 / (A0 + A1);
      V3 kv = K[0] * p0 + K[1] * p1 + K[2] * p2 + K[3] * p3;
      int32_t* hv = &P->hinge_verts[4 * (size_t)hc];
      hv[0] = u; hv[1] = v; hv[2] = x2; hv[3] = x3;
      for (int i = 0; i < 4; ++i) P->hinge_K[4 * (size_t)hc + i] = K[i];
      P->hinge_wr[2 * (size_t)hc] = wh;
      P->hinge_wr[2 * (size_t)hc + 1] = norm(kv);
      hinge_of[(size_t)u * n + v] = hinge_of[(size_t)v * n + u] = hc;
      ++hc;
    }
  if (hc != H) return fail(NPFEM_EINVAL, "edge count does not match 3T/2");

  // ---- A_sys (caller order) = (1/h^2 + c_alpha/h) M + (1 + c_beta/h) L_el + (w_volume + w_collision) I, where
  //      L_el = sum_t (w_s + w_a) G^T G + sum_h w_h K^T K.  c_alpha = c_beta = 0: the undamped
  //      system; otherwise the implicit Rayleigh damping of reading A-20
  const double ih2 = 1.0 / (dt * dt);
  const double mass_scale = ih2 + mat->c_alpha / dt, el_scale = 1.0 + mat->c_beta / dt;
  P->A.assign((size_t)n * n, 0.0);
  std::vector<double>& A = P->A;
  for (int t = 0; t < T; ++t) {
    double i00 = P->tri_dminv[3 * t], i01 = P->tri_dminv[3 * t + 1], i11 = P->tri_dminv[3 * t + 2];
    // columns of G = D_m^-T [[-1,1,0],[-1,0,1]]: vertex b -> (i00, i01), c -> (0, i11), a -> -(b + c)
    double G[3][2] = {{-i00, -i01 - i11}, {i00, i01}, {0.0, i11}};
    double w = (mat->k_strain + mat->k_area) * P->tri_area[t];
    for (int p = 0; p < 3; ++p)
      for (int q = 0; q < 3; ++q)
        A[(size_t)tris[3 * t + p] * n + tris[3 * t + q]] += w * (G[p][0] * G[q][0] + G[p][1] * G[q][1]);
  }
  for (int hh = 0; hh < H; ++hh) {
    const int32_t* hv = &P->hinge_verts[4 * (size_t)hh];
    const double* K = &P->hinge_K[4 * (size_t)hh];
    double wh = P->hinge_wr[2 * (size_t)hh];
    for (int p = 0; p < 4; ++p)
      for (int q = 0; q < 4; ++q) A[(size_t)hv[p] * n + hv[q]] += wh * K[p] * K[q];
  }
  for (double& a : A) a *= el_scale;
  for (int v = 0; v < n; ++v) A[(size_t)v * n + v] += P->mass[v] * mass_scale + mat->w_volume + mat->w_collision;

  // ---- T = A_sys^-1 (fp64): Cholesky A = L L^T, M = L^-1, T = M^T M
  std::vector<double> L((size_t)n * n, 0.0), M((size_t)n * n, 0.0), Tinv((size_t)n * n, 0.0);
  for (int j = 0; j < n; ++j) {
    for (int i = j; i < n; ++i) {
      double s = A[(size_t)i * n + j];
      const double *li = &L[(size_t)i * n], *lj = &L[(size_t)j * n];
      for (int k = 0; k < j; ++k) s -= li[k] * lj[k];
      if (i == j) {
        if (!(s > 0.0)) return fail(NPFEM_EINVAL, "system matrix is not positive definite");
        L[(size_t)j * n + j] = std::sqrt(s);
      } else {
        L[(size_t)i * n + j] = s / L[(size_t)j * n + j];
      }
    }
  }
  for (int i = 0; i < n; ++i) {
    double* mi = &M[(size_t)i * n];
    mi[i] = 1.0;
    for (int k = 0; k < i; ++k) {
      double lik = L[(size_t)i * n + k];
      if (lik == 0.0) continue;
      const double* mk = &M[(size_t)k * n];
      for (int j = 0; j <= k; ++j) mi[j] -= lik * mk[j];
    }
    double inv = 1.0 / L[(size_t)i * n + i];
    for (int j = 0; j <= i; ++j) mi[j] *= inv;
  }
  for (int k = 0; k < n; ++k) {
    const double* mk = &M[(size_t)k * n];
    for (int i = 0; i <= k; ++i) {
      double mki = mk[i];
      if (mki == 0.0) continue;
      double* ti = &Tinv[(size_t)i * n];
      for (int j = 0; j <= i; ++j) ti[j] += mki * mk[j];
    }
  }
  for (int i = 0; i < n; ++i)
    for (int j = 0; j < i; ++j) Tinv[(size_t)j * n + i] = Tinv[(size_t)i * n + j];
  L.clear(); L.shrink_to_fit(); M.clear(); M.shrink_to_fit();

  // ---- locality ordering
  std::vector<std::vector<int>> adj(n);
  for (int u = 0; u < n; ++u)
    for (int v = 0; v < n; ++v)
      if (etri[(size_t)u * n + v] != -1) adj[u].push_back(v);
  {
    Bisector bis(adj);
    std::vector<int> all(n), tagv(n, 0), order;
    std::iota(all.begin(), all.end(), 0);
    int next_tag = 1;
    order.reserve(n);
    bis.run(all, tagv, next_tag, order);
    P->perm.assign(order.begin(), order.end());
    P->iperm.assign(n, -1);
    for (int i = 0; i < n; ++i) P->iperm[P->perm[i]] = i;
    for (int v = 0; v < n; ++v)
      if (P->iperm[v] < 0) return fail(NPFEM_EINVAL, "internal: ordering is not a permutation");
  }

  // ---- drop rule on T (per row: smallest entries first while dropped l1 mass <= tol * ||row||_1),
  //      symmetrised, then 8x8 blocks in internal numbering; kept blocks store ALL their entries
  const int nvb = (n + 7) / 8;
  P->nvb = nvb;
  std::vector<uint8_t> keep((size_t)n * n, 0);
  {
    std::vector<int> idx(n);
    for (int i = 0; i < n; ++i) {
      const double* ti = &Tinv[(size_t)i * n];
      double l1 = 0.0;
      for (int j = 0; j < n; ++j) l1 += std::fabs(ti[j]);
      std::iota(idx.begin(), idx.end(), 0);
      std::sort(idx.begin(), idx.end(), [&](int p, int q) {
        double ap = std::fabs(ti[p]), aq = std::fabs(ti[q]);
        return ap != aq ? ap < aq : p < q;
      });
      double dropped = 0.0;
      int m = 0;
      while (m < n && dropped + std::fabs(ti[idx[m]]) <= o.inv_drop_tol * l1 && idx[m] != i) {
        dropped += std::fabs(ti[idx[m]]);
        ++m;
      }
      for (int q = m; q < n; ++q) keep[(size_t)i * n + idx[q]] = 1;
      keep[(size_t)i * n + i] = 1;
    }
  }
  int nnz = 0;
  std::vector<uint8_t> bmask((size_t)nvb * nvb, 0);
  for (int i = 0; i < n; ++i)
    for (int j = 0; j < n; ++j)
      if (keep[(size_t)i * n + j] || keep[(size_t)j * n + i]) {
        ++nnz;
        bmask[(size_t)(P->iperm[i] / 8) * nvb + P->iperm[j] / 8] = 1;
      }
  P->op_nnz = nnz;
  // Per output block row: first the blocks applied with 3xTF32, then the blocks whose entries are
  // so small that ONE TF32 product is exact to fp32 rounding of the row sum: a TF32 product of
  // truncated operands errs by < 2^-9 relative, so blocks are moved to the second run, smallest
  // first, while their l1 mass stays <= 2^-15 of the l1 norm of EVERY row of the block row
  // (product error <= 2^-24 ||row||_1 |r|_max, the size of one fp32 rounding).  Each run is padded
  // with all-zero blocks to a multiple of 4 for the kernel's unrolled, software-pipelined loop.
  auto Tint = [&](int i, int j) {   // operator entry in internal numbering, 0 outside
    return (i < n && j < n) ? Tinv[(size_t)P->perm[i] * n + P->perm[j]] : 0.0;
  };
  // Kept source blocks of output block row ib (`cols`) and which of them may take the cheap single
  // product (`single`): blocks are moved to that tier, smallest first (by their largest row mass),
  // while the tier's l1 mass stays <= tier_tol of the l1 norm of EVERY row of the block row; the
  // diagonal block never moves.
  auto tier_split = [&](int ib, double tier_tol, std::vector<int>& cols, std::vector<uint8_t>& single) {
    cols.clear();
    for (int jb = 0; jb < nvb; ++jb)
      if (bmask[(size_t)ib * nvb + jb]) cols.push_back(jb);
    std::vector<std::array<double, 8>> mass(cols.size());
    std::array<double, 8> rowl1{};
    for (size_t q = 0; q < cols.size(); ++q)
      for (int r = 0; r < 8; ++r) {
        double m = 0.0;
        for (int cc = 0; cc < 8; ++cc) m += std::fabs(Tint(ib * 8 + r, cols[q] * 8 + cc));
        mass[q][r] = m;
        rowl1[r] += m;
      }
    std::vector<int> order(cols.size());
    std::iota(order.begin(), order.end(), 0);
    auto bmax = [&](int q) { return *std::max_element(mass[q].begin(), mass[q].end()); };
    std::sort(order.begin(), order.end(), [&](int p, int q) {
      double mp = bmax(p), mq = bmax(q);
      return mp != mq ? mp < mq : p < q;
    });
    single.assign(cols.size(), 0);
    std::array<double, 8> cum{};
    for (int q : order) {
      bool ok = cols[q] != ib;
      for (int r = 0; r < 8 && ok; ++r)
        if (rowl1[r] > 0.0 && cum[r] + mass[q][r] > tier_tol * rowl1[r]) ok = false;
      if (!ok) break;
      for (int r = 0; r < 8; ++r) cum[r] += mass[q][r];
      single[q] = 1;
    }
  };
  P->blk_ptr.assign(3 * (size_t)nvb, 0);
  P->blk_col.clear();
  P->blk_val.clear();
  P->n_op_blocks = 0;
  P->n_op_blocks_x1 = 0;
  {
    const double tier_tol = std::ldexp(1.0, -15);
    auto emit = [&](int ib, int jb, bool zero) {
      P->blk_col.push_back((uint16_t)jb);
      size_t base = P->blk_val.size();
      P->blk_val.resize(base + 64, 0.0f);
      if (zero) return;
      for (int l = 0; l < 32; ++l)
        for (int r = 0; r < 2; ++r) {
          int j = jb * 8 + (l & 3) + 4 * r;   // source vertex (k index of the mma B fragment)
          int i = ib * 8 + (l >> 2);          // output vertex (n index)
          P->blk_val[base + 2 * l + r] = (float)Tint(i, j);
        }
    };
    for (int ib = 0; ib < nvb; ++ib) {
      std::vector<int> cols;
      std::vector<uint8_t> single;
      tier_split(ib, tier_tol, cols, single);
      for (int pass = 0; pass < 2; ++pass) {
        P->blk_ptr[3 * (size_t)ib + pass] = (int32_t)P->blk_col.size();
        int run_blocks = 0;
        for (size_t q = 0; q < cols.size(); ++q) {
          if ((int)single[q] != pass) continue;
          emit(ib, cols[q], false);
          ++run_blocks;
          ++P->n_op_blocks;
          P->n_op_blocks_x1 += pass;
        }
        while (run_blocks % 4) {
          emit(ib, ib, true);
          ++run_blocks;
        }
      }
      P->blk_ptr[3 * (size_t)ib + 2] = (int32_t)P->blk_col.size();
    }
  }

  // ---- the same operator for global_mode 3: two-term fp16 split on mma m16n8k16 (K = 16 = a PAIR
  //      of source blocks per instruction).  x = hi + lo with hi = fp16(x), lo = fp16(x - hi)
  //      represents x to 2^-24 relative, so hi*hi + hi*lo + lo*hi with fp32 accumulation is
  //      fp32-equivalent (the dropped lo*lo is 2^-24 of the product).  A product of the hi parts
  //      alone errs by <= 2^-11 relative (each operand rounded to 11 bits), so blocks are moved to
  //      the one-product run, smallest first, while their l1 mass stays <= 2^-13 of the l1 norm of
  //      every row of the block row: total error <= 2^-24 ||row||_1 |r|_max, one fp32 rounding.
  //      Row i is scaled by 2^k_i so that its largest entry lies in [2^13, 2^14) (fp16 normal range
  //      reaches down to 2^-14: 27 binades below, more than the 24 the drop rule leaves); the
  //      kernel scales the right-hand sides likewise per cell and undoes both with hp_scale.
  //      A run with an odd number of blocks ends with a half-empty pair.
  {
    const double tier_tol = std::ldexp(1.0, -13);
    std::vector<int> kexp(nvb * 8, 0);
    P->hp_scale.assign(n, 1.0f);
    for (int i = 0; i < n; ++i) {
      double mx = 0.0;
      for (int j = 0; j < n; ++j) mx = std::max(mx, std::fabs(Tint(i, j)));
      int e = 0;
      if (mx > 0.0) std::frexp(mx, &e);   // mx = f 2^e, f in [0.5, 1)
      kexp[i] = 14 - e;                   // mx 2^k in [2^13, 2^14)
      P->hp_scale[i] = (float)std::ldexp(1.0, -kexp[i]);
    }
    P->hp_ptr.assign(4 * (size_t)nvb, 0);
    P->hp_col_a.clear(); P->hp_val_a.clear(); P->hp_col_b.clear(); P->hp_val_b.clear();
    P->n_op_blocks_h1 = 0;
    // B fragment of mma.m16n8k16 (col): lane = 4 g + t holds b0 = (k = 2t, 2t+1; n = g) from the first
    // source block and b1 = (k = 2t+8, 2t+9; n = g) from the second; low half = lower k.
    auto emit_pair = [&](int ib, int jb1, int jb2, bool full) {
      std::vector<uint32_t>& val = full ? P->hp_val_a : P->hp_val_b;
      (full ? P->hp_col_a : P->hp_col_b)
          .push_back((uint32_t)(jb1 < 0 ? 0xffff : jb1) | ((uint32_t)(jb2 < 0 ? 0xffff : jb2)) << 16);
      const int words = full ? 4 : 2;
      size_t base = val.size();
      val.resize(base + 32 * (size_t)words, 0u);
      for (int l = 0; l < 32; ++l) {
        const int g = l >> 2, t = l & 3, i = ib * 8 + g;
        for (int half = 0; half < 2; ++half) {
          const int jb = half ? jb2 : jb1;
          if (jb < 0) continue;
          uint32_t hi = 0, lo = 0;
          for (int q = 0; q < 2; ++q) {
            const float x = (float)std::ldexp(Tint(i, jb * 8 + 2 * t + q), i < n ? kexp[i] : 0);
            const uint16_t hb = half_bits(x);
            const uint16_t lb = half_bits(x - half_value(hb));
            hi |= (uint32_t)hb << (16 * q);
            lo |= (uint32_t)lb << (16 * q);
          }
          val[base + (size_t)l * words + half] = hi;
          if (full) val[base + (size_t)l * words + 2 + half] = lo;
        }
      }
    };
    for (int ib = 0; ib < nvb; ++ib) {
      std::vector<int> cols;
      std::vector<uint8_t> single;
      tier_split(ib, tier_tol, cols, single);
      for (int pass = 0; pass < 2; ++pass) {
        std::vector<uint32_t>& colv = pass ? P->hp_col_b : P->hp_col_a;
        P->hp_ptr[4 * (size_t)ib + 2 * pass] = (int32_t)colv.size();
        std::vector<int> run;
        for (size_t q = 0; q < cols.size(); ++q)
          if ((int)single[q] == pass) run.push_back(cols[q]);
        P->n_op_blocks_h1 += pass ? (int)run.size() : 0;
        int run_pairs = 0;
        for (size_t q = 0; q < run.size(); q += 2, ++run_pairs)
          emit_pair(ib, run[q], q + 1 < run.size() ? run[q + 1] : -1, pass == 0);
        (void)run_pairs;
        P->hp_ptr[4 * (size_t)ib + 2 * pass + 1] = (int32_t)colv.size();
      }
    }
  }

  // ---- per-vertex constants (internal numbering)
  P->h2_over_m.resize(n);
  P->m_over_h2.resize(n);
  P->damp_m.resize(n);
  for (int i = 0; i < n; ++i) {
    double m = P->mass[P->perm[i]];
    P->h2_over_m[i] = (float)(dt * dt / m);
    P->m_over_h2[i] = (float)(m * mass_scale);          // inertial + mass-proportional damping diagonal
    P->damp_m[i] = (float)(m * mat->c_alpha / dt);      // (c_alpha/h) m: acts on the predicted increment
  }
  P->damped = mat->c_alpha != 0.0 || mat->c_beta != 0.0;

  // ---- elements: pair triangles across shared edges (a matching of the dual graph, which is
  //      cubic and bridgeless for a closed manifold, so a perfect matching exists; greedy by
  //      fewest free neighbours, then augmenting paths; whatever stays unmatched becomes a
  //      single-triangle element).  Triangle neighbour across edge slot e: the triangle holding
  //      the reversed directed edge.
  auto tnbr = [&](int t, int e) {
    int u = tris[3 * t + e], v = tris[3 * t + (e + 1) % 3];
    return (int)etri[(size_t)v * n + u];
  };
  std::vector<int> mate(T, -1);
  {
    auto tkey = [&](int t) {
      int a = P->iperm[tris[3 * t]], b = P->iperm[tris[3 * t + 1]], c = P->iperm[tris[3 * t + 2]];
      return std::make_pair(std::min(a, std::min(b, c)), a + b + c);
    };
    std::vector<int> order(T);
    std::iota(order.begin(), order.end(), 0);
    std::sort(order.begin(), order.end(), [&](int p, int q) {
      auto kp = tkey(p), kq = tkey(q);
      return kp != kq ? kp < kq : p < q;
    });
    auto free_nbrs = [&](int t) {
      int c = 0;
      for (int e = 0; e < 3; ++e) {
        int u = tnbr(t, e);
        if (u != t && mate[u] < 0) ++c;
      }
      return c;
    };
    for (int t : order) {
      if (mate[t] >= 0) continue;
      int best = -1, bestc = 99;
      for (int e = 0; e < 3; ++e) {
        int u = tnbr(t, e);
        if (u == t || mate[u] >= 0) continue;
        mate[t] = t;   // count u's free neighbours without t
        int c = free_nbrs(u);
        mate[t] = -1;
        if (c < bestc) { bestc = c; best = u; }
      }
      if (best >= 0) { mate[t] = best; mate[best] = t; }
    }
    // augmenting paths (alternating BFS without blossom handling: a heuristic that only ever
    // increases the matching; correctness does not depend on it being maximum)
    for (int root : order) {
      if (mate[root] >= 0) continue;
      std::vector<int> parent(T, -1), seen(T, 0);
      std::deque<int> q;
      q.push_back(root);
      seen[root] = 1;
      int found = -1;
      while (!q.empty() && found < 0) {
        int t = q.front();
        q.pop_front();
        for (int e = 0; e < 3 && found < 0; ++e) {
          int u = tnbr(t, e);
          if (u == t || seen[u]) continue;
          seen[u] = 1;
          parent[u] = t;
          if (mate[u] < 0) { found = u; break; }
          int w = mate[u];
          if (!seen[w]) { seen[w] = 1; parent[w] = u; q.push_back(w); }
        }
      }
      if (found < 0) continue;
      // flip along the path found <- parent ... <- root
      int u = found;
      while (u != root) {
        int t = parent[u];          // t is an "even" vertex: (t,u) becomes matched
        int prev = mate[t];         // t's old mate (or -1 for the root)
        mate[t] = u; mate[u] = t;
        if (t == root) break;
        u = prev;                   // prev's new partner is parent[prev]... continue flipping
        mate[u] = -1;
      }
    }
    if (o.pair_triangles == 2) std::fill(mate.begin(), mate.end(), -1);
    // sanity: mate must be an involution
    for (int t = 0; t < T; ++t)
      if (mate[t] >= 0 && (mate[t] == t || mate[mate[t]] != t)) {
        for (int q2 = 0; q2 < T; ++q2) mate[q2] = -1;   // give up pairing: all single triangles
        break;
      }
  }

  // ---- element constants.  dminv of a triangle for an arbitrary cyclic vertex order (p0,p1,p2):
  //      frame t1 = e1/|e1|, t2 = n x t1, D_m = [[|e1|, e2.t1], [0, e2.t2]]  (same construction as
  //      tri_dminv above; a cyclic shift only rotates F on the right, which no energy sees).
  auto dminv_of = [&](int p0, int p1, int p2, double out3[3]) {
    V3 a = Xv(p0), b = Xv(p1), c = Xv(p2);
    V3 e1 = b - a, e2 = c - a;
    double twoA = norm(cross(e1, e2)), l1 = norm(e1);
    double d00 = l1, d01 = dot(e2, e1) / l1, d11 = twoA / l1;
    out3[0] = 1.0 / d00;
    out3[1] = -d01 / (d00 * d11);
    out3[2] = 1.0 / d11;
  };
  // hinge on the undirected edge (p,q) seen from the element whose own opposite vertex is oo
  auto hinge_consts = [&](int p, int q, int oo, float out4[4]) {
    int hh = hinge_of[(size_t)p * n + q];
    const int32_t* hv = &P->hinge_verts[4 * (size_t)hh];
    const double* K = &P->hinge_K[4 * (size_t)hh];
    double sw = std::sqrt(P->hinge_wr[2 * (size_t)hh]);
    auto Kof = [&](int vtx) {
      for (int i = 0; i < 4; ++i)
        if (hv[i] == vtx) return K[i];
      return 0.0;
    };
    out4[0] = (float)(sw * Kof(p));
    out4[1] = (float)(sw * Kof(q));
    out4[2] = (float)(sw * Kof(oo));
    out4[3] = (float)(sw * P->hinge_wr[2 * (size_t)hh + 1]);
  };
  struct Proto { int t1, t2, a, b, c, d; };
  std::vector<Proto> protos;
  {
    std::vector<uint8_t> done(T, 0);
    for (int t = 0; t < T; ++t) {
      if (done[t]) continue;
      done[t] = 1;
      Proto pr{};
      pr.t1 = t;
      int eshared = 0;
      if (mate[t] >= 0) {
        for (int e = 0; e < 3; ++e)
          if (tnbr(t, e) == mate[t]) { eshared = e; break; }
        pr.t2 = mate[t];
        done[mate[t]] = 1;
      } else {
        pr.t2 = -1;
      }
      pr.a = tris[3 * t + eshared];
      pr.b = tris[3 * t + (eshared + 1) % 3];
      pr.c = tris[3 * t + (eshared + 2) % 3];
      pr.d = opposite(pr.b, pr.a);
      protos.push_back(pr);
    }
  }
  // element order: by smallest internal vertex id, then by the id sum (locality in shared memory)
  std::sort(protos.begin(), protos.end(), [&](const Proto& x, const Proto& y) {
    auto key = [&](const Proto& p) {
      int a = P->iperm[p.a], b = P->iperm[p.b], c = P->iperm[p.c];
      return std::make_pair(std::min(a, std::min(b, c)), a + b + c);
    };
    auto kx = key(x), ky = key(y);
    return kx != ky ? kx < ky : x.t1 < y.t1;
  });
  const int E = (int)protos.size();
  if (E > 1024) return fail(NPFEM_ELIMIT, "mesh needs more than 1024 elements per cell");
  P->E = E;
  P->n_diamonds = 0;
  P->elem.assign(E, ElemConst{});
  P->elem_tris.assign(2 * (size_t)E, -1);
  std::vector<std::vector<uint16_t>> inc(n);   // per internal vertex: out-slot byte offsets
  for (int e = 0; e < E; ++e) {
    const Proto& pr = protos[e];
    ElemConst& ec = P->elem[e];
    const bool diamond = pr.t2 >= 0;
    P->n_diamonds += diamond ? 1 : 0;
    P->elem_tris[2 * (size_t)e] = pr.t1;
    P->elem_tris[2 * (size_t)e + 1] = pr.t2;
    const int a = pr.a, b = pr.b, c = pr.c, d = pr.d;
    const int f1 = opposite(c, b), f2 = opposite(a, c);
    const int f3 = diamond ? opposite(d, a) : a, f4 = diamond ? opposite(b, d) : a;
    const int idv[8] = {a, b, c, d, f1, f2, f3, f4};
    for (int s = 0; s < 8; ++s) ec.ids[s] = (uint16_t)P->iperm[idv[s]];
    double dm[3];
    dminv_of(a, b, c, dm);
    ec.f[0] = (float)dm[0]; ec.f[1] = (float)dm[1]; ec.f[2] = (float)dm[2];
    ec.f[3] = (float)(mat->k_strain * P->tri_area[pr.t1]);
    ec.f[4] = (float)(mat->k_area * P->tri_area[pr.t1]);
    dminv_of(b, a, d, dm);   // the real neighbour triangle even for a single: finite arithmetic
    ec.f[5] = (float)dm[0]; ec.f[6] = (float)dm[1]; ec.f[7] = (float)dm[2];
    ec.f[8] = diamond ? (float)(mat->k_strain * P->tri_area[pr.t2]) : 0.0f;
    ec.f[9] = diamond ? (float)(mat->k_area * P->tri_area[pr.t2]) : 0.0f;
    hinge_consts(a, b, c, &ec.f[10]);
    hinge_consts(b, c, a, &ec.f[14]);
    hinge_consts(c, a, b, &ec.f[18]);
    if (diamond) {
      hinge_consts(a, d, b, &ec.f[22]);
      hinge_consts(d, b, a, &ec.f[26]);
    } else {
      for (int q = 22; q < 30; ++q) ec.f[q] = 0.0f;
    }
    ec.f[30] = diamond ? 1.0f : 0.5f;
    const int nslots = diamond ? 4 : 3;
    for (int s = 0; s < nslots; ++s)
      inc[P->iperm[idv[s]]].push_back((uint16_t)((s * E + e) * 16));
  }
  P->inc_ptr.assign(n + 1, 0);
  P->inc_off.clear();
  for (int i = 0; i < n; ++i) {
    for (uint16_t o16 : inc[i]) P->inc_off.push_back(o16);
    P->inc_ptr[i + 1] = (uint16_t)P->inc_off.size();
  }

  // ---- ring neighbours of every vertex in cyclic (counter-clockwise seen from outside) order:
  //      triangle i of the fan is (v, r_i, r_i+1); grad V at v = 1/6 sum_i (r_i - v) x (r_i+1 - v)
  P->ring_ptr.assign(n + 1, 0);
  P->ring_off.clear();
  for (int i = 0; i < n; ++i) {
    int ve = P->perm[i];
    int t0 = -1, s0 = 0;
    for (int w : adj[ve]) {
      t0 = etri[(size_t)ve * n + w];
      s0 = eslot[(size_t)ve * n + w];
      break;
    }
    int t = t0, s = s0, count = 0;
    do {
      int r0 = tris[3 * t + (s + 1) % 3], r1 = tris[3 * t + (s + 2) % 3];
      P->ring_off.push_back((uint16_t)(P->iperm[r0] * 16));
      // next triangle around ve holds the directed edge ve -> r1
      int tn = etri[(size_t)ve * n + r1];
      s = eslot[(size_t)ve * n + r1];
      t = tn;
      if (++count > T) return fail(NPFEM_EINVAL, "non-manifold vertex fan");
    } while (t != t0);
    if (count != (int)adj[ve].size()) return fail(NPFEM_EINVAL, "non-manifold vertex (several fans)");
    P->ring_ptr[i + 1] = (uint16_t)P->ring_off.size();
  }

  // ---- launch configuration: one thread per element and per (padded) vertex
  int need = std::max(nvb * 8, E);
  P->threads = (need + 31) / 32 * 32;
  if (P->threads > 1024) return fail(NPFEM_ELIMIT, "mesh needs more than 1024 threads per cell");
  if (P->damped && P->threads > 768)   // 80 tensor-memory columns per 4 warps: 6 groups fit the 512
    return fail(NPFEM_ELIMIT, "damping needs more tensor-memory columns than a CTA of more than 768 threads has");
  const int smem_max = kSmemMaxDynamic;
  int k = o.cells_per_cta ? o.cells_per_cta : kMaxCellsPerCta;
  while (k > 1 && smem_layout(n, E, nvb, k).total > smem_max) {
    if (o.cells_per_cta) return fail(NPFEM_ELIMIT, "requested cells_per_cta does not fit shared memory");
    --k;
  }
  if (smem_layout(n, E, nvb, k).total > smem_max)
    return fail(NPFEM_ELIMIT, "cell state does not fit the shared memory of one SM");
  P->cells_per_cta = k;
  P->smem_bytes = smem_layout(n, E, nvb, k).total;

  // ---- global_mode 3: per-warp operator streams of uniform shape (npfem_internal.h)
  {
    const int W = P->threads / 32;
    const int J = (nvb + W - 1) / W;
    if (J > 4 || W > 32) return fail(NPFEM_ELIMIT, "internal: more than 4 operator block rows per warp");
    auto pairs_a = [&](int ib) { return P->hp_ptr[4 * (size_t)ib + 1] - P->hp_ptr[4 * (size_t)ib]; };
    auto pairs_b = [&](int ib) { return P->hp_ptr[4 * (size_t)ib + 3] - P->hp_ptr[4 * (size_t)ib + 2]; };
    std::vector<int> order(nvb);
    std::iota(order.begin(), order.end(), 0);
    std::stable_sort(order.begin(), order.end(), [&](int p, int q) {   // by mma count, longest first
      return 3 * pairs_a(p) + pairs_b(p) > 3 * pairs_a(q) + pairs_b(q);
    });
    P->hs_rows.assign(4 * 32, 255);
    for (int j = 0; j < 4; ++j) { P->hs_na[j] = 0; P->hs_nb[j] = 0; }
    for (int r = 0; r < nvb; ++r) {
      const int j = r / W, w = r % W, ib = order[r];
      P->hs_rows[(size_t)j * 32 + w] = (uint8_t)ib;
      P->hs_na[j] = std::max(P->hs_na[j], pairs_a(ib));
      P->hs_nb[j] = std::max(P->hs_nb[j], (pairs_b(ib) + 1) / 2);
    }
    P->hs_slots = 0;
    for (int j = 0; j < 4; ++j) P->hs_slots += P->hs_na[j] + P->hs_nb[j];
    const int Q = P->hs_slots;
    P->hs_desc.assign((size_t)W * 128, 0u);
    auto dword = [&](int w, int q, int x) -> uint32_t& {   // descriptor word x of slot q of warp w
      return P->hs_desc[((size_t)w * 32 + (q & 31)) * 4 + 2 * ((q >> 5) & 1) + x];
    };
    P->hs_val.assign((size_t)W * Q * 128, 0u);
    auto colword = [](uint32_t kb) { return kb == 0xffffu ? 0u : (kb << 9 | (kb & 7u) << 5); };
    for (int w = 0; w < W; ++w) {
      int q0 = 0;
      for (int j = 0; j < 4; ++j) {
        const int ib = P->hs_rows[(size_t)j * 32 + w];
        if (ib != 255) {
          const int a0 = P->hp_ptr[4 * (size_t)ib], b0 = P->hp_ptr[4 * (size_t)ib + 2];
          for (int u = 0; u < pairs_a(ib); ++u) {
            const size_t slot = (size_t)w * Q + q0 + u;
            const uint32_t c = P->hp_col_a[a0 + u];
            if (q0 + u < kMaxOpSlots) dword(w, q0 + u, 0) = colword(c & 0xffffu) | colword(c >> 16) << 16;
            for (int l = 0; l < 32; ++l)
              for (int x = 0; x < 4; ++x)
                P->hs_val[(slot * 32 + l) * 4 + x] = P->hp_val_a[((size_t)(a0 + u) * 32 + l) * 4 + x];
          }
          for (int u = 0; u < pairs_b(ib); ++u) {
            const size_t slot = (size_t)w * Q + q0 + P->hs_na[j] + u / 2;
            const uint32_t c = P->hp_col_b[b0 + u];
            if (q0 + P->hs_na[j] + u / 2 < kMaxOpSlots)
              dword(w, q0 + P->hs_na[j] + u / 2, u & 1) = colword(c & 0xffffu) | colword(c >> 16) << 16;
            for (int l = 0; l < 32; ++l)
              for (int x = 0; x < 2; ++x)
                P->hs_val[(slot * 32 + l) * 4 + 2 * (u & 1) + x] = P->hp_val_b[((size_t)(b0 + u) * 32 + l) * 2 + x];
          }
        }
        q0 += P->hs_na[j] + P->hs_nb[j];
      }
    }
  }
  if (o.global_mode == 3 && P->hs_slots > kMaxOpSlots)
    o.global_mode = 2;   // more slots per warp than the descriptor registers hold: 3xTF32 blocks
  // default: the fp16-split streams where they apply (measured 7 % faster per step than 3xTF32 on
  // config 4), else the 3xTF32 blocks
  P->global_mode = o.global_mode ? o.global_mode : (P->hs_slots <= kMaxOpSlots ? 3 : 2);
  o.cells_per_cta = k;
  o.global_mode = P->global_mode;
  P->opt = o;
  return NPFEM_OK;
}

}  // namespace npfem
