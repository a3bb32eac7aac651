// npfem_api.cu -- the C ABI of include/npfem.h: argument checks, handle ownership, uploads,
// launches and the host-buffer pipeline.  No arithmetic of the method lives here (create-time
// math: npfem_plan.cpp; step math: npfem_kernels.cu).
#include <cuda_runtime.h>

#include <cmath>
#include <cstdio>
#include <cstring>
#include <new>
#include <string>

#include "npfem_internal.h"
#include "npfem_kernels.cuh"

using namespace npfem;

struct npfem_plan_s {
  Plan plan;
};

struct npfem_handle_s {
  Plan plan;
  int device = 0;
  int cell_stride = 0;
  int max_cells = 0;
  DevParams dev{};            // device pointers + scalars (pos/vel/fext/n_cells/n_iters set per call)
  void* blob = nullptr;       // one device allocation holding every constant table
  // host-buffer pipeline (npfem_step_host)
  static constexpr int kStages = 3;
  int chunk_cells = 0;
  float* stage[kStages][3] = {};   // device staging: pos, vel, fext per stage
  cudaStream_t streams[kStages] = {};
  bool pipeline_ready = false;
};

namespace {

thread_local char g_err[512] = "";

int set_err(int code, const std::string& msg) {
  std::snprintf(g_err, sizeof(g_err), "%s", msg.c_str());
  return code;
}
int cuda_err(cudaError_t e, const char* what) {
  std::snprintf(g_err, sizeof(g_err), "%s: %s", what, cudaGetErrorString(e));
  return NPFEM_ECUDA;
}

void fill_info(const Plan& P, int cell_stride, npfem_info* o) {
  o->n_verts = P.n; o->n_tris = P.T; o->n_hinges = P.H;
  o->cell_stride = cell_stride;
  o->cells_per_cta = P.cells_per_cta;
  o->threads_per_cta = P.threads;
  o->smem_bytes = P.smem_bytes;
  o->n_vblocks = P.nvb;
  o->n_op_blocks = P.n_op_blocks;
  o->n_op_blocks_tf32x1 = P.n_op_blocks_x1;
  o->n_elements = P.E;
  o->n_diamonds = P.n_diamonds;
  o->n_op_blocks_f16x1 = P.n_op_blocks_h1;
  {   // occupancy of the fixed-count step kernel (the same arithmetic as its tcgen05.alloc)
    const int groups = (P.threads / 32 + 3) / 4;
    int cols = 64;
    while (cols < (P.damped ? 80 : 64) * groups) cols <<= 1;
    o->tmem_columns = cols;
    const int by_smem = (227 * 1024) / (P.smem_bytes + 1024);   // + static shared memory and the per-CTA reserve
    const int by_tmem = 512 / cols, by_threads = 2048 / P.threads;
    int best = by_smem, lim = 1;
    if (by_tmem < best) { best = by_tmem; lim = 2; }
    if (by_threads < best) { best = by_threads; lim = 3; }
    o->ctas_per_sm = best < 1 ? 1 : best;
    o->ctas_per_sm_limiter = lim;
  }
  o->op_nnz = P.op_nnz;
  o->global_mode = P.global_mode;
  o->volume_inner_iters = P.opt.volume_inner_iters;
  o->rest_volume = P.V0;
  o->total_mass = P.total_mass;
  o->inv_drop_tol = P.opt.inv_drop_tol;
}

size_t align_up(size_t x, size_t a) { return (x + a - 1) / a * a; }

// Makes the handle's device current for the lifetime of the guard (the handle's tables, streams
// and staging ring live on the device that was current in npfem_create).
struct DeviceGuard {
  int prev = -1;
  bool switched = false;
  cudaError_t err = cudaSuccess;
  explicit DeviceGuard(int device) {
    err = cudaGetDevice(&prev);
    if (err == cudaSuccess && prev != device) {
      err = cudaSetDevice(device);
      switched = err == cudaSuccess;
    }
  }
  ~DeviceGuard() {
    if (switched) cudaSetDevice(prev);
  }
};

void destroy_pipeline(npfem_handle_s* h) {
  for (int sidx = 0; sidx < npfem_handle_s::kStages; ++sidx) {
    for (int f = 0; f < 3; ++f) {
      if (h->stage[sidx][f]) cudaFree(h->stage[sidx][f]);
      h->stage[sidx][f] = nullptr;
    }
    if (h->streams[sidx]) cudaStreamDestroy(h->streams[sidx]);
    h->streams[sidx] = nullptr;
  }
  h->pipeline_ready = false;
}

// Streams and device staging ring of npfem_step_host: chunks of a whole number of CTAs' worth of
// cells, about 32 MB per field, never more than `cells_hint` cells (0 = no hint).  Everything
// created so far is released again when a later allocation fails.
int create_pipeline(npfem_handle_s* h, int cells_hint) {
  if (h->pipeline_ready) return NPFEM_OK;
  const size_t cell_bytes = (size_t)h->cell_stride * sizeof(float);
  const int k = h->plan.cells_per_cta;
  int chunk = (int)((32u << 20) / cell_bytes);
  if (cells_hint > 0 && chunk > cells_hint) chunk = cells_hint;
  chunk = (chunk + k - 1) / k * k;
  if (chunk < k) chunk = k;
  h->chunk_cells = chunk;
  for (int sidx = 0; sidx < npfem_handle_s::kStages; ++sidx) {
    cudaError_t e = cudaStreamCreateWithFlags(&h->streams[sidx], cudaStreamNonBlocking);
    if (e != cudaSuccess) { h->streams[sidx] = nullptr; destroy_pipeline(h); return cuda_err(e, "cudaStreamCreate"); }
    for (int f = 0; f < 3; ++f) {
      e = cudaMalloc(&h->stage[sidx][f], (size_t)chunk * cell_bytes);
      if (e != cudaSuccess) { h->stage[sidx][f] = nullptr; destroy_pipeline(h); return cuda_err(e, "cudaMalloc(staging ring)"); }
    }
  }
  h->pipeline_ready = true;
  return NPFEM_OK;
}

}  // namespace

extern "C" {

const char* npfem_last_error(void) { return g_err; }

int npfem_plan_create(int n_verts, int n_tris, const int32_t* tris, const double* rest_xyz,
                      const npfem_material* mat, double dt, const npfem_options* opts,
                      npfem_plan* out) {
  if (!out) return set_err(NPFEM_EINVAL, "out is NULL");
  *out = nullptr;
  npfem_plan_s* p = new (std::nothrow) npfem_plan_s;
  if (!p) return set_err(NPFEM_ENOMEM, "out of host memory");
  std::string err;
  int rc;
  try {
    rc = build_plan(n_verts, n_tris, tris, rest_xyz, mat, dt, opts, &p->plan, &err);
  } catch (const std::bad_alloc&) {
    delete p;
    return set_err(NPFEM_ENOMEM, "out of host memory");
  }
  if (rc != NPFEM_OK) {
    delete p;
    return set_err(rc, err);
  }
  *out = p;
  return NPFEM_OK;
}

int npfem_plan_destroy(npfem_plan p) {
  delete p;
  return NPFEM_OK;
}

int npfem_plan_info(npfem_plan p, npfem_info* out) {
  if (!p || !out) return set_err(NPFEM_EINVAL, "null argument");
  fill_info(p->plan, (3 * p->plan.n + 3) / 4 * 4, out);
  return NPFEM_OK;
}

int npfem_plan_query(npfem_plan p, int what, void* dst, int dst_elems) {
  if (!p) return set_err(NPFEM_EINVAL, "null plan");
  const Plan& P = p->plan;
  const int n = P.n;
  auto copy_out = [&](const void* src, size_t elems, size_t elem_size) -> int {
    if (!dst) return (int)elems;
    if ((size_t)dst_elems < elems) return set_err(NPFEM_EINVAL, "destination too small");
    std::memcpy(dst, src, elems * elem_size);
    return (int)elems;
  };
  switch (what) {
    case NPFEM_Q_PERM: return copy_out(P.perm.data(), n, sizeof(int32_t));
    case NPFEM_Q_MASS: return copy_out(P.mass.data(), n, sizeof(double));
    case NPFEM_Q_SYSTEM: return copy_out(P.A.data(), (size_t)n * n, sizeof(double));
    case NPFEM_Q_HINGE_VERTS: return copy_out(P.hinge_verts.data(), 4 * (size_t)P.H, sizeof(int32_t));
    case NPFEM_Q_HINGE_K: return copy_out(P.hinge_K.data(), 4 * (size_t)P.H, sizeof(double));
    case NPFEM_Q_HINGE_WR: return copy_out(P.hinge_wr.data(), 2 * (size_t)P.H, sizeof(double));
    case NPFEM_Q_TRI_DMINV: return copy_out(P.tri_dminv.data(), 3 * (size_t)P.T, sizeof(double));
    case NPFEM_Q_TRI_AREA: return copy_out(P.tri_area.data(), (size_t)P.T, sizeof(double));
    case NPFEM_Q_OPERATOR:
    case NPFEM_Q_OPERATOR_X1: {
      const size_t elems = (size_t)n * n;
      if (!dst) return (int)elems;
      if ((size_t)dst_elems < elems) return set_err(NPFEM_EINVAL, "destination too small");
      double* D = static_cast<double*>(dst);
      std::memset(D, 0, elems * sizeof(double));
      for (int ib = 0; ib < P.nvb; ++ib)
        for (int b = P.blk_ptr[3 * ib + (what == NPFEM_Q_OPERATOR_X1 ? 1 : 0)]; b < P.blk_ptr[3 * ib + 2]; ++b) {
          const int jb = P.blk_col[b];
          for (int l = 0; l < 32; ++l)
            for (int r = 0; r < 2; ++r) {
              const int j = jb * 8 + (l & 3) + 4 * r, i = ib * 8 + (l >> 2);
              if (i < n && j < n)
                D[(size_t)P.perm[i] * n + P.perm[j]] += (double)P.blk_val[(size_t)b * 64 + 2 * l + r];
            }
        }
      return (int)elems;
    }
    case NPFEM_Q_OPERATOR_F16:
    case NPFEM_Q_OPERATOR_F16X1: {
      const size_t elems = (size_t)n * n;
      if (!dst) return (int)elems;
      if ((size_t)dst_elems < elems) return set_err(NPFEM_EINVAL, "destination too small");
      double* D = static_cast<double*>(dst);
      std::memset(D, 0, elems * sizeof(double));
      auto hv = [](uint32_t w, int q) {   // value of half q of a packed word
        const uint32_t hb = (w >> (16 * q)) & 0xffffu;
        const int e = (hb >> 10) & 0x1f, m = hb & 0x3ff;
        const double v = e == 0 ? std::ldexp((double)m, -24) : std::ldexp((double)(m | 0x400), e - 25);
        return (hb & 0x8000u) ? -v : v;
      };
      for (int ib = 0; ib < P.nvb; ++ib)
        for (int pass = (what == NPFEM_Q_OPERATOR_F16X1 ? 1 : 0); pass < 2; ++pass) {
          const std::vector<uint32_t>& col = pass ? P.hp_col_b : P.hp_col_a;
          const std::vector<uint32_t>& val = pass ? P.hp_val_b : P.hp_val_a;
          const int words = pass ? 2 : 4;
          for (int pr = P.hp_ptr[4 * ib + 2 * pass]; pr < P.hp_ptr[4 * ib + 2 * pass + 1]; ++pr)
            for (int l = 0; l < 32; ++l)
              for (int half = 0; half < 2; ++half) {
                const int jb = (int)((col[pr] >> (16 * half)) & 0xffffu);
                if (jb == 0xffff) continue;
                for (int q = 0; q < 2; ++q) {
                  const int i = ib * 8 + (l >> 2), j = jb * 8 + 2 * (l & 3) + q;
                  if (i >= n || j >= n) continue;
                  double x = hv(val[((size_t)pr * 32 + l) * words + half], q);
                  if (!pass) x += hv(val[((size_t)pr * 32 + l) * words + 2 + half], q);
                  D[(size_t)P.perm[i] * n + P.perm[j]] += x * (double)P.hp_scale[i];
                }
              }
        }
      return (int)elems;
    }
    case NPFEM_Q_STREAM_SHAPE: {
      int32_t shape[10] = {P.threads / 32, P.hs_slots, P.hs_na[0], P.hs_na[1], P.hs_na[2], P.hs_na[3],
                           P.hs_nb[0], P.hs_nb[1], P.hs_nb[2], P.hs_nb[3]};
      return copy_out(shape, 10, sizeof(int32_t));
    }
    case NPFEM_Q_STREAM_VAL: return copy_out(P.hs_val.data(), P.hs_val.size(), sizeof(uint32_t));
    case NPFEM_Q_STREAM_DESC: return copy_out(P.hs_desc.data(), P.hs_desc.size(), sizeof(uint32_t));
    case NPFEM_Q_STREAM_ROWS: {
      int32_t rows[4 * 32];
      for (int i = 0; i < 4 * 32; ++i) rows[i] = P.hs_rows[i];
      return copy_out(rows, 4 * 32, sizeof(int32_t));
    }
    case NPFEM_Q_ROW_SCALE: {
      std::vector<double> sc(P.hp_scale.begin(), P.hp_scale.end());
      return copy_out(sc.data(), sc.size(), sizeof(double));
    }
    case NPFEM_Q_OPERATOR_STREAM: {
      // walk the streams exactly as the kernel does: warp w, row slot j, first hs_na[j] three-product
      // slots (one pair: words 0,1 hi, 2,3 lo), then hs_nb[j] one-product slots (two pairs: hi, hi)
      const size_t elems = (size_t)n * n;
      if (!dst) return (int)elems;
      if ((size_t)dst_elems < elems) return set_err(NPFEM_EINVAL, "destination too small");
      if (P.hs_slots > kMaxOpSlots) return set_err(NPFEM_EINVAL, "no streams: more slots per warp than the kernel supports");
      double* D = static_cast<double*>(dst);
      std::memset(D, 0, elems * sizeof(double));
      auto hv = [](uint32_t w, int q) {
        const uint32_t hb = (w >> (16 * q)) & 0xffffu;
        const int e = (hb >> 10) & 0x1f, m = hb & 0x3ff;
        const double v = e == 0 ? std::ldexp((double)m, -24) : std::ldexp((double)(m | 0x400), e - 25);
        return (hb & 0x8000u) ? -v : v;
      };
      const int W = P.threads / 32, Q = P.hs_slots;
      for (int w = 0; w < W; ++w) {
        int q = 0;
        for (int j = 0; j < 4; ++j) {
          const int ib = P.hs_rows[(size_t)j * 32 + w];
          for (int u = 0; u < P.hs_na[j] + P.hs_nb[j]; ++u, ++q) {
            if (ib == 255) continue;
            const bool full = u < P.hs_na[j];
            for (int pr = 0; pr < (full ? 1 : 2); ++pr) {
              const uint32_t dw = P.hs_desc[((size_t)w * 32 + (q & 31)) * 4 + 2 * ((q >> 5) & 1) + pr];
              for (int l = 0; l < 32; ++l)
                for (int half = 0; half < 2; ++half) {
                  const uint32_t off = (dw >> (16 * half)) & 0xffffu;
                  const int jb = (int)(off >> 9);
                  if ((off & 0x1ffu) != ((uint32_t)(jb & 7) << 5)) return set_err(NPFEM_EINVAL, "internal: descriptor swizzle bits");
                  const uint32_t* val = &P.hs_val[(((size_t)w * Q + q) * 32 + l) * 4];
                  for (int e2 = 0; e2 < 2; ++e2) {
                    const int i = ib * 8 + (l >> 2), jv = jb * 8 + 2 * (l & 3) + e2;
                    if (i >= n || jv >= n) continue;
                    double x = full ? hv(val[half], e2) + hv(val[2 + half], e2) : hv(val[2 * pr + half], e2);
                    D[(size_t)P.perm[i] * n + P.perm[jv]] += x * (double)P.hp_scale[i];
                  }
                }
            }
          }
        }
      }
      return (int)elems;
    }
    default: return set_err(NPFEM_EINVAL, "unknown query");
  }
}

int npfem_create(int n_verts, int n_tris, const int32_t* tris, const double* rest_xyz,
                 const npfem_material* mat, double dt, int cell_stride_floats, int max_cells,
                 const npfem_options* opts, npfem_handle* out) {
  if (!out) return set_err(NPFEM_EINVAL, "out is NULL");
  *out = nullptr;
  if (max_cells < 0) return set_err(NPFEM_EINVAL, "max_cells is negative");
  int stride = cell_stride_floats;
  if (stride == 0) stride = (3 * n_verts + 3) / 4 * 4;
  if (stride < 3 * n_verts) return set_err(NPFEM_EINVAL, "cell_stride_floats < 3*n_verts");

  npfem_handle_s* H = new (std::nothrow) npfem_handle_s;
  if (!H) return set_err(NPFEM_ENOMEM, "out of host memory");
  std::string err;
  int rc;
  try {
    rc = build_plan(n_verts, n_tris, tris, rest_xyz, mat, dt, opts, &H->plan, &err);
  } catch (const std::bad_alloc&) {
    delete H;
    return set_err(NPFEM_ENOMEM, "out of host memory");
  }
  if (rc != NPFEM_OK) {
    delete H;
    return set_err(rc, err);
  }
  Plan& P = H->plan;
  H->cell_stride = stride;
  H->max_cells = max_cells;

  cudaError_t e = cudaGetDevice(&H->device);
  if (e != cudaSuccess) { delete H; return cuda_err(e, "cudaGetDevice (no CUDA device: there is no CPU fallback)"); }
  e = configure_kernels(P.smem_bytes);
  if (e == cudaSuccess) e = configure_converged_kernels();
  if (e != cudaSuccess) { delete H; return cuda_err(e, "cudaFuncSetAttribute(shared memory)"); }

  // ---- one blob for all constant tables, 256-byte aligned sections
  const int n = P.n, E = P.E, NP = P.nvb * 8;
  std::vector<uint16_t> perm16(NP, 0);
  // element constants as kElemGroups groups of 4 words, group-major ([group][E] float4):
  //   0: packed byte offsets 16*id of (a,b) (c,d) (f1,f2) (f3,f4)   1: t1 i00 i01 i11 w_s
  //   2: t2 i00 i01 i11 w_s      3: t1 w_a, t2 w_a, he, 0           4..8: hinge e: Kp Kq Ko r'
  std::vector<uint32_t> elem_c((size_t)kElemGroups * E * 4, 0u);
  std::vector<float> h2m(NP, 0.0f), mh2(NP, 0.0f), dmp(NP, 0.0f), hps(NP, 0.0f);
  for (int i = 0; i < n; ++i) {
    perm16[i] = (uint16_t)P.perm[i];
    h2m[i] = P.h2_over_m[i];
    mh2[i] = P.m_over_h2[i];
    dmp[i] = P.damp_m[i];
    hps[i] = P.hp_scale[i];
  }
  auto fbits = [](float x) { uint32_t u; std::memcpy(&u, &x, 4); return u; };
  for (int e = 0; e < E; ++e) {
    const ElemConst& ec = P.elem[e];
    auto W = [&](int g, int w) -> uint32_t& { return elem_c[((size_t)g * E + e) * 4 + w]; };
    for (int q = 0; q < 4; ++q)
      W(0, q) = (uint32_t)ec.ids[2 * q] * 16u | ((uint32_t)ec.ids[2 * q + 1] * 16u) << 16;
    for (int q = 0; q < 4; ++q) { W(1, q) = fbits(ec.f[q]); W(2, q) = fbits(ec.f[5 + q]); }
    W(3, 0) = fbits(ec.f[4]); W(3, 1) = fbits(ec.f[9]); W(3, 2) = fbits(ec.f[30]);
    for (int hgi = 0; hgi < 5; ++hgi)
      for (int q = 0; q < 4; ++q) W(4 + hgi, q) = fbits(ec.f[10 + 4 * hgi + q]);
  }
  // vertex-role constants, two uint4 per (padded) vertex, fetched by the owner thread just before
  // its vertex phase: [0] = first 6 element-slot byte offsets (u16 pairs), icnt | rcnt << 8;
  // [1] = first 6 ring byte offsets (u16 pairs), bits of m/h^2.  Longer lists continue in
  // inc_off / ring_off.
  std::vector<uint32_t> vrole((size_t)NP * 8, 0u);
  for (int i = 0; i < n; ++i) {
    const int i0 = P.inc_ptr[i], icnt = P.inc_ptr[i + 1] - i0;
    const int r0 = P.ring_ptr[i], rcnt = P.ring_ptr[i + 1] - r0;
    uint32_t* w = &vrole[(size_t)i * 8];
    for (int q = 0; q < kRegList; ++q) {
      if (q < icnt) w[q >> 1] |= (uint32_t)P.inc_off[i0 + q] << (16 * (q & 1));
      if (q < rcnt) w[4 + (q >> 1)] |= (uint32_t)P.ring_off[r0 + q] << (16 * (q & 1));
    }
    w[3] = (uint32_t)(icnt > 255 ? 255 : icnt) | (uint32_t)(rcnt > 255 ? 255 : rcnt) << 8;
    w[7] = fbits(P.m_over_h2[i]);
  }
  struct Sec { const void* src; size_t bytes; size_t off; };
  Sec secs[] = {
      {perm16.data(), perm16.size() * 2, 0},          {elem_c.data(), elem_c.size() * 4, 0},
      {vrole.data(), vrole.size() * 4, 0},            {h2m.data(), h2m.size() * 4, 0},
      {mh2.data(), mh2.size() * 4, 0},                {P.inc_ptr.data(), P.inc_ptr.size() * 2, 0},
      {P.inc_off.data(), P.inc_off.size() * 2, 0},    {P.ring_ptr.data(), P.ring_ptr.size() * 2, 0},
      {P.ring_off.data(), P.ring_off.size() * 2, 0},  {P.blk_ptr.data(), P.blk_ptr.size() * 4, 0},
      {P.blk_col.data(), P.blk_col.size() * 2, 0},    {P.blk_val.data(), P.blk_val.size() * 4, 0},
      {dmp.data(), dmp.size() * 4, 0},
      {P.hs_val.data(), P.hs_val.size() * 4, 0},      {hps.data(), hps.size() * 4, 0},
      {P.hs_desc.data(), P.hs_desc.size() * 4, 0},
  };
  size_t total = 0;
  for (auto& sct : secs) { sct.off = total; total += align_up(sct.bytes, 256); }
  e = cudaMalloc(&H->blob, total);
  if (e != cudaSuccess) { delete H; return cuda_err(e, "cudaMalloc(constants)"); }
  for (auto& sct : secs) {
    if (!sct.bytes) continue;
    e = cudaMemcpy(static_cast<char*>(H->blob) + sct.off, sct.src, sct.bytes, cudaMemcpyHostToDevice);
    if (e != cudaSuccess) { cudaFree(H->blob); delete H; return cuda_err(e, "cudaMemcpy(constants)"); }
  }
  char* base = static_cast<char*>(H->blob);
  DevParams& D = H->dev;
  D.n = n; D.E = E; D.nvb = P.nvb; D.k = P.cells_per_cta; D.cell_stride = stride;
  D.vol_iters = P.opt.volume_inner_iters;
  D.h = (float)P.h; D.w_volume = (float)P.mat.w_volume; D.V0 = (float)P.V0;
  D.Vmin = (float)(P.mat.v_min * P.V0); D.Vmax = (float)(P.mat.v_max * P.V0);
  D.s_min = (float)P.mat.s_min; D.s_max = (float)P.mat.s_max;
  D.a_min = (float)P.mat.a_min; D.a_max = (float)P.mat.a_max;
  D.perm = reinterpret_cast<const uint16_t*>(base + secs[0].off);
  D.elem_c = reinterpret_cast<const float4*>(base + secs[1].off);
  D.vrole = reinterpret_cast<const uint4*>(base + secs[2].off);
  D.h2_over_m = reinterpret_cast<const float*>(base + secs[3].off);
  D.m_over_h2 = reinterpret_cast<const float*>(base + secs[4].off);
  D.inc_ptr = reinterpret_cast<const uint16_t*>(base + secs[5].off);
  D.inc_off = reinterpret_cast<const uint16_t*>(base + secs[6].off);
  D.ring_ptr = reinterpret_cast<const uint16_t*>(base + secs[7].off);
  D.ring_off = reinterpret_cast<const uint16_t*>(base + secs[8].off);
  D.blk_ptr = reinterpret_cast<const int*>(base + secs[9].off);
  D.blk_col = reinterpret_cast<const uint16_t*>(base + secs[10].off);
  D.blk_val = reinterpret_cast<const float*>(base + secs[11].off);
  D.damp_m = reinterpret_cast<const float*>(base + secs[12].off);
  D.hs_val = reinterpret_cast<const uint4*>(base + secs[13].off);
  D.hp_scale = reinterpret_cast<const float*>(base + secs[14].off);
  D.hs_desc = reinterpret_cast<const uint4*>(base + secs[15].off);
  D.hs_slots = P.hs_slots;
  for (int j = 0; j < 4; ++j) { D.hs_na[j] = P.hs_na[j]; D.hs_nb[j] = P.hs_nb[j]; }
  std::memcpy(D.hs_rows, P.hs_rows.data(), sizeof(D.hs_rows));
  D.cbh = (float)(P.mat.c_beta / P.h);
  D.damped = P.damped ? 1 : 0;
  D.jitter = P.opt.debug_jitter;
  D.dbg = 0;
  D.coll_q = nullptr; D.coll_n = nullptr;
  D.w_coll = (float)P.mat.w_collision; D.d_coll = (float)P.mat.d_collision;
  D.hard = (float)P.mat.strain_hardening;
  D.L = smem_layout(n, E, P.nvb, P.cells_per_cta);
  if (max_cells > 0) {   // everything any later step entry point needs exists now
    rc = create_pipeline(H, max_cells);
    if (rc != NPFEM_OK) { cudaFree(H->blob); delete H; return rc; }
  }
  *out = H;
  return NPFEM_OK;
}

int npfem_debug_phase_clocks(unsigned long long* out16, int reset) {
  if (!out16) return set_err(NPFEM_EINVAL, "null argument");
  cudaError_t e = read_phase_clocks(out16, reset);
  if (e == cudaErrorNotSupported) return set_err(NPFEM_EINVAL, "library built without -DNPFEM_PHASE_CLOCKS");
  if (e != cudaSuccess) return cuda_err(e, "npfem_debug_phase_clocks");
  return NPFEM_OK;
}

int npfem_get_info(npfem_handle h, npfem_info* out) {
  if (!h || !out) return set_err(NPFEM_EINVAL, "null argument");
  fill_info(h->plan, h->cell_stride, out);
  return NPFEM_OK;
}

int npfem_cell_stride(npfem_handle h) {
  if (!h) return set_err(NPFEM_EINVAL, "null handle");
  return h->cell_stride;
}

int npfem_step(npfem_handle h, int n_cells, float* pos, float* vel, const float* fext,
               int n_iters, void* cuda_stream) {
  if (!h) return set_err(NPFEM_EINVAL, "null handle");
  if (n_cells < 0 || n_iters < 0) return set_err(NPFEM_EINVAL, "negative n_cells or n_iters");
  if (n_cells == 0) return NPFEM_OK;
  if (!pos || !vel || !fext) return set_err(NPFEM_EINVAL, "null device pointer");
  if (h->max_cells > 0 && n_cells > h->max_cells) return set_err(NPFEM_EINVAL, "n_cells exceeds the max_cells given to npfem_create");
  DeviceGuard guard(h->device);
  if (guard.err != cudaSuccess) return cuda_err(guard.err, "cudaSetDevice(handle device)");
  DevParams p = h->dev;
  p.n_cells = n_cells; p.n_iters = n_iters;
  p.pos = pos; p.vel = vel; p.fext = fext;
  cudaError_t e = launch_step(p, h->plan.threads, h->plan.smem_bytes, h->plan.global_mode,
                              static_cast<cudaStream_t>(cuda_stream));
  if (e != cudaSuccess) return cuda_err(e, "npfem_step launch");
  return NPFEM_OK;
}

int npfem_step_collide(npfem_handle h, int n_cells, float* pos, float* vel, const float* fext,
                       const float* coll_q, const float* coll_n, int n_iters, void* cuda_stream) {
  if (!h) return set_err(NPFEM_EINVAL, "null handle");
  if (n_cells < 0 || n_iters < 0) return set_err(NPFEM_EINVAL, "negative n_cells or n_iters");
  if (n_cells == 0) return NPFEM_OK;
  if (!pos || !vel || !fext || !coll_q || !coll_n) return set_err(NPFEM_EINVAL, "null device pointer");
  if (h->max_cells > 0 && n_cells > h->max_cells) return set_err(NPFEM_EINVAL, "n_cells exceeds the max_cells given to npfem_create");
  DeviceGuard guard(h->device);
  if (guard.err != cudaSuccess) return cuda_err(guard.err, "cudaSetDevice(handle device)");
  DevParams p = h->dev;
  p.n_cells = n_cells; p.n_iters = n_iters;
  p.pos = pos; p.vel = vel; p.fext = fext;
  p.coll_q = coll_q; p.coll_n = coll_n;
  cudaError_t e = launch_step(p, h->plan.threads, h->plan.smem_bytes, h->plan.global_mode,
                              static_cast<cudaStream_t>(cuda_stream));
  if (e != cudaSuccess) return cuda_err(e, "npfem_step_collide launch");
  return NPFEM_OK;
}

int npfem_vertex_areas(npfem_handle h, int n_cells, const float* pos, float* areas, void* cuda_stream) {
  if (!h) return set_err(NPFEM_EINVAL, "null handle");
  if (n_cells < 0) return set_err(NPFEM_EINVAL, "negative n_cells");
  if (n_cells == 0) return NPFEM_OK;
  if (!pos || !areas) return set_err(NPFEM_EINVAL, "null device pointer");
  DeviceGuard guard(h->device);
  if (guard.err != cudaSuccess) return cuda_err(guard.err, "cudaSetDevice(handle device)");
  DevParams p = h->dev;
  p.n_cells = n_cells;
  p.pos = const_cast<float*>(pos);
  cudaError_t e = launch_vertex_areas(p, h->plan.threads, areas, static_cast<cudaStream_t>(cuda_stream));
  if (e != cudaSuccess) return cuda_err(e, "npfem_vertex_areas launch");
  return NPFEM_OK;
}

int npfem_step_converged(npfem_handle h, int n_cells, float* pos, float* vel, const float* fext,
                         double tol, int max_iters, int32_t* iters_out, float* res_out,
                         void* cuda_stream) {
  if (!h) return set_err(NPFEM_EINVAL, "null handle");
  if (n_cells < 0 || max_iters < 0 || !(tol >= 0.0)) return set_err(NPFEM_EINVAL, "negative n_cells, max_iters or tol");
  if (n_cells == 0) return NPFEM_OK;
  if (!pos || !vel || !fext) return set_err(NPFEM_EINVAL, "null device pointer");
  if (h->max_cells > 0 && n_cells > h->max_cells) return set_err(NPFEM_EINVAL, "n_cells exceeds the max_cells given to npfem_create");
  if (h->plan.damped) return set_err(NPFEM_EINVAL, "the converged solve does not support damping yet (c_alpha, c_beta must be 0)");
  if (h->plan.mat.w_collision != 0.0) return set_err(NPFEM_EINVAL, "the converged solve does not support collisions yet (w_collision must be 0)");
  DeviceGuard guard(h->device);
  if (guard.err != cudaSuccess) return cuda_err(guard.err, "cudaSetDevice(handle device)");
  DevParams p = h->dev;
  p.n_cells = n_cells; p.n_iters = max_iters;
  p.pos = pos; p.vel = vel; p.fext = fext;
  p.k = 1;                                               // one CTA owns one cell
  p.L = smem_layout(h->plan.n, h->plan.E, h->plan.nvb, 1);
  cudaError_t e = launch_converged(p, h->plan.threads, p.L.total, (float)tol, max_iters, iters_out, res_out,
                                   static_cast<cudaStream_t>(cuda_stream));
  if (e != cudaSuccess) return cuda_err(e, "npfem_step_converged launch");
  return NPFEM_OK;
}

int npfem_step_host(npfem_handle h, int n_cells, float* pos, float* vel, const float* fext,
                    int n_iters) {
  if (!h) return set_err(NPFEM_EINVAL, "null handle");
  if (n_cells < 0 || n_iters < 0) return set_err(NPFEM_EINVAL, "negative n_cells or n_iters");
  if (n_cells == 0) return NPFEM_OK;
  if (!pos || !vel || !fext) return set_err(NPFEM_EINVAL, "null host pointer");
  if (h->max_cells > 0 && n_cells > h->max_cells) return set_err(NPFEM_EINVAL, "n_cells exceeds the max_cells given to npfem_create");
  DeviceGuard guard(h->device);
  if (guard.err != cudaSuccess) return cuda_err(guard.err, "cudaSetDevice(handle device)");
  const size_t cell_bytes = (size_t)h->cell_stride * sizeof(float);
  if (!h->pipeline_ready) {   // handle created with max_cells = 0: the ring is sized on first use
    int rc = create_pipeline(h, 0);
    if (rc != NPFEM_OK) return rc;
  }
  const int chunk = h->chunk_cells;
  cudaError_t e = cudaSuccess;
  int rc = NPFEM_OK, idx = 0;
  const char* what = "";
  for (int c0 = 0; c0 < n_cells && rc == NPFEM_OK && e == cudaSuccess; c0 += chunk, ++idx) {
    const int sidx = idx % npfem_handle_s::kStages;
    const int nc = (n_cells - c0 < chunk) ? (n_cells - c0) : chunk;
    const size_t off = (size_t)c0 * h->cell_stride, bytes = (size_t)nc * cell_bytes;
    cudaStream_t st = h->streams[sidx];
    // stream order serialises reuse of this stage's buffers with its previous chunk
    what = "cudaMemcpyAsync(H2D)";
    e = cudaMemcpyAsync(h->stage[sidx][0], pos + off, bytes, cudaMemcpyHostToDevice, st);
    if (e == cudaSuccess) e = cudaMemcpyAsync(h->stage[sidx][1], vel + off, bytes, cudaMemcpyHostToDevice, st);
    if (e == cudaSuccess) e = cudaMemcpyAsync(h->stage[sidx][2], fext + off, bytes, cudaMemcpyHostToDevice, st);
    if (e != cudaSuccess) break;
    rc = npfem_step(h, nc, h->stage[sidx][0], h->stage[sidx][1], h->stage[sidx][2], n_iters, st);
    if (rc != NPFEM_OK) break;
    what = "cudaMemcpyAsync(D2H)";
    e = cudaMemcpyAsync(pos + off, h->stage[sidx][0], bytes, cudaMemcpyDeviceToHost, st);
    if (e == cudaSuccess) e = cudaMemcpyAsync(vel + off, h->stage[sidx][1], bytes, cudaMemcpyDeviceToHost, st);
  }
  // success or not, nothing may still be writing into the caller's buffers when this returns
  for (int sidx = 0; sidx < npfem_handle_s::kStages; ++sidx) {
    cudaError_t es = cudaStreamSynchronize(h->streams[sidx]);
    if (e == cudaSuccess && rc == NPFEM_OK && es != cudaSuccess) { e = es; what = "cudaStreamSynchronize"; }
  }
  if (rc != NPFEM_OK) return rc;
  if (e != cudaSuccess) return cuda_err(e, what);
  return NPFEM_OK;
}

int npfem_destroy(npfem_handle h) {
  if (!h) return NPFEM_OK;
  {
    DeviceGuard guard(h->device);
    destroy_pipeline(h);
    if (h->blob) cudaFree(h->blob);
  }
  delete h;
  return NPFEM_OK;
}

}  // extern "C"
