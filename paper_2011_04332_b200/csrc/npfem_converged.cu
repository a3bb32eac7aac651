// npfem_converged.cu -- converged npFEM step on sm_100a (NEXT-1; reading A-21).
//
// "Our approach follows the redesigned projective dynamics approach as described in
// Liu et al. [11] ... we provide a converged solution"; :133: "unconditional stability for
// arbitrary time steps".  One CTA owns ONE cell and minimises the implicit-Euler objective
//   g(x) = 1/2 ||x - s||^2_M / h^2 + E_el(x),   grad g(x) = M (x - s)/h^2 - f_int(x),
// by L-BFGS (history kHist = 3) seeded with the prefactored operator T = A_sys^-1, a backtracking
// (halving) line search on g, and a per-cell on-device stop flag
//   res(x) = max_v || (h^2/m_v) grad g(x)_v ||_inf <= tol.
// Everything runs in one launch; no host round trip (north_star (d)).
//
// Work mapping: as in the fused fixed-count kernel (npfem_kernels.cu) for one cell -- thread e owns
// an element, thread v a vertex; f_int and the element energies come from the same element pass
// (the energy rides in the unused fourth word of the element results and is summed by the vertex
// gather); the dot products of the two-loop recursion, the energy and the residual are CTA
// reductions; the operator product is the same tensor-core block product with 3 of the 16
// right-hand-side columns in use.  All per-vertex vectors are private to the owner thread: s, x,
// grad g, the direction and u0 in registers, the three (s_k, y_k) pairs in tensor memory.
#include <cstdint>

#include "npfem_device.cuh"

namespace npfem {
namespace {

constexpr int kHist = 3;

__device__ __forceinline__ void tmem_st8(uint32_t a, const float (&v)[8]) {
  asm volatile("tcgen05.st.sync.aligned.32x32b.x8.b32 [%0], {%1,%2,%3,%4,%5,%6,%7,%8};"
               :: "r"(a), "f"(v[0]), "f"(v[1]), "f"(v[2]), "f"(v[3]), "f"(v[4]), "f"(v[5]), "f"(v[6]), "f"(v[7])
               : "memory");
  asm volatile("tcgen05.wait::st.sync.aligned;" ::: "memory");
}
__device__ __forceinline__ void tmem_ld8(uint32_t a, float (&v)[8]) {
  asm volatile("tcgen05.ld.sync.aligned.32x32b.x8.b32 {%0,%1,%2,%3,%4,%5,%6,%7}, [%8];"
               : "=f"(v[0]), "=f"(v[1]), "=f"(v[2]), "=f"(v[3]), "=f"(v[4]), "=f"(v[5]), "=f"(v[6]), "=f"(v[7])
               : "r"(a)
               : "memory");
  asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
}
__device__ __forceinline__ float warp_max(float v) {
  v = fmaxf(v, __shfl_xor_sync(0xffffffffu, v, 16));
  v = fmaxf(v, __shfl_xor_sync(0xffffffffu, v, 8));
  v = fmaxf(v, __shfl_xor_sync(0xffffffffu, v, 4));
  v = fmaxf(v, __shfl_xor_sync(0xffffffffu, v, 2));
  v = fmaxf(v, __shfl_xor_sync(0xffffffffu, v, 1));
  return v;
}

// TMEM columns of the owner thread (per group of 4 warps: 64 columns): the pairs at 0, 8, 16
constexpr int kColHist = 0;

template <int MAXT>
__global__ void __launch_bounds__(MAXT, 1) npfem_converged_kernel(const DevParams P, const float tol,
                                                                   const int max_iters, int* iters_out,
                                                                   float* res_out) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  unsigned char* const z4b = smem_raw + P.L.z4;                        // [NP] float4 trial iterate z
  const float4* const ecs = reinterpret_cast<const float4*>(smem_raw + P.L.ec);
  float* const ra = reinterpret_cast<float*>(smem_raw + P.L.ra);
  unsigned char* const rbb = smem_raw + P.L.rb;
  float* const rb = reinterpret_cast<float*>(rbb);
  float4* const red = reinterpret_cast<float4*>(smem_raw + P.L.red);   // [32] partial sums
  __shared__ uint32_t tmem_base_s;

  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5, nwarps = blockDim.x >> 5;
  const int n = P.n, E = P.E, nvb = P.nvb, NP = nvb * 8;
  const int cell = blockIdx.x;

  uint32_t tmem_cols = 64;
  while (tmem_cols < 64u * ((nwarps + 3) >> 2)) tmem_cols <<= 1;
  if (warp == 0) {
    const uint32_t sa = (uint32_t)__cvta_generic_to_shared(&tmem_base_s);
    asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" :: "r"(sa), "r"(tmem_cols) : "memory");
    asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
  }
  const bool is_e = tid < E, isv = tid < n, isvp = tid < NP;
  const int v = isvp ? tid : 0;
  const float h = P.h;
  const int fbase = ((v >> 3) * 32 + (v & 3)) * 4 + 2 * ((v & 7) >> 2);
  for (int i = tid; i < kElemGroups * E; i += blockDim.x)
    reinterpret_cast<float4*>(smem_raw + P.L.ec)[i] = P.elem_c[i];
  for (int i = tid; i < NP; i += blockDim.x) reinterpret_cast<float4*>(z4b)[i] = make_float4(0.f, 0.f, 0.f, 0.f);
  asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
  __syncthreads();
  asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
  const uint32_t ta = tmem_base_s + ((uint32_t)(32 * (warp & 3)) << 16) + (uint32_t)((warp >> 2) * 64);

  // CTA reductions: every warp reduces the same partials in the same order, so the result (and
  // every decision taken on it) is CTA-uniform
  auto cta_sum4 = [&](float4 a) -> float4 {
    a.x = warp_sum(a.x); a.y = warp_sum(a.y); a.z = warp_sum(a.z); a.w = warp_sum(a.w);
    if (lane == 0) red[warp] = a;
    __syncthreads();
    float4 p4 = lane < nwarps ? red[lane] : make_float4(0.f, 0.f, 0.f, 0.f);
    p4.x = warp_sum(p4.x); p4.y = warp_sum(p4.y); p4.z = warp_sum(p4.z); p4.w = warp_sum(p4.w);
    __syncthreads();
    return p4;
  };
  auto cta_max = [&](float a) -> float {
    a = warp_max(a);
    if (lane == 0) red[warp].x = a;
    __syncthreads();
    float p = lane < nwarps ? red[lane].x : 0.f;
    p = warp_max(p);
    __syncthreads();
    return p;
  };

  // ---- prologue: stage the cell, centroid, local coordinates, inertial prediction
  const int vext3 = 3 * (int)P.perm[v];
  const float h2m = P.h2_over_m[v];
  const float mh2 = __uint_as_float(P.vrole[2 * v + 1].w);
  F3 s3 = {0.f, 0.f, 0.f}, u3 = s3;
  {
    float* const st = rb;
    const int n3 = 3 * n;
    const size_t g = (size_t)cell * P.cell_stride;
    for (int i = tid; i < n3; i += blockDim.x) { st[i] = P.pos[g + i]; st[n3 + i] = P.vel[g + i]; st[2 * n3 + i] = P.fext[g + i]; }
    __syncthreads();
    F3 x3 = {0.f, 0.f, 0.f};
    if (isv) {
      x3 = {st[vext3], st[vext3 + 1], st[vext3 + 2]};
      u3 = {fmaf(h, st[n3 + vext3], h2m * st[2 * n3 + vext3]), fmaf(h, st[n3 + vext3 + 1], h2m * st[2 * n3 + vext3 + 1]),
            fmaf(h, st[n3 + vext3 + 2], h2m * st[2 * n3 + vext3 + 2])};
    }
    __syncthreads();
    const float4 c4 = cta_sum4(make_float4(x3.x, x3.y, x3.z, 0.f));
    const float invn = 1.0f / (float)n;
    if (isv) s3 = {(x3.x - c4.x * invn) + u3.x, (x3.y - c4.y * invn) + u3.y, (x3.z - c4.z * invn) + u3.z};
    if (isv) reinterpret_cast<float4*>(z4b)[v] = make_float4(s3.x, s3.y, s3.z, 0.f);
    __syncthreads();
  }

  const float vol_tol = kVolTol * P.V0;
  const float vol_dlen = kVolDTol * cbrtf(P.V0);
  const float vol_dtol2 = (float)n * vol_dlen * vol_dlen;
  const bool use_vol = P.w_volume > 0.0f;

  // ---- f_int and E_el at the iterate in z4: element pass, vertex gather, volume projection.
  //      Returns this vertex's elastic residual ev and its share en of g (inertial term included).
  auto evaluate = [&](F3 zv, F3& ev, float& en) {
    if (is_e) element_residual<3, true>(ecs + tid, E, z4b, P, reinterpret_cast<float4*>(rbb) + tid);
    const uint4 vr0 = P.vrole[2 * v];
    const uint4 vr1 = P.vrole[2 * v + 1];
    const int icnt = vr0.w & 0xff, rcnt = (vr0.w >> 8) & 0xff;
    F3 g = {0.f, 0.f, 0.f};
    float S1 = 0.f, S2 = 0.f;
    if (use_vol && isv) {
      g = ring_gradient(z4b, zv, rcnt, vr1.x, vr1.y, vr1.z, P, v);
      S1 = dot(zv, g); S2 = dot(g, g);
    }
    __syncthreads();                       // element results complete
    ev = {0.f, 0.f, 0.f}; en = 0.f;
    if (isv) {
      const uint32_t ioff[kRegList / 2] = {vr0.x, vr0.y, vr0.z};
#pragma unroll
      for (int i = 0; i < kRegList; ++i)
        if (i < icnt) {
          const float4 o = *reinterpret_cast<const float4*>(rbb + ((i & 1) ? (ioff[i >> 1] >> 16) : (ioff[i >> 1] & 0xffffu)));
          ev = ev + xyz(o); en += o.w;
        }
      if (icnt > kRegList) {
        const uint16_t* inc_tail = P.inc_off + P.inc_ptr[v];
        for (int i = kRegList; i < icnt; ++i) {
          const float4 o = *reinterpret_cast<const float4*>(rbb + inc_tail[i]);
          ev = ev + xyz(o); en += o.w;
        }
      }
    }
    if (use_vol) {                         // D = lambda grad V(z + D), iterated as in the fused kernel (A-17)
      float4 p4 = cta_sum4(make_float4(S1, S2, 0.f, 0.f));
      const float V = p4.x * (1.0f / 3.0f);
      const float vstar = fminf(fmaxf(V, P.Vmin), P.Vmax);
      float C = V - vstar;
      const bool active = (V != vstar);
      float lambda = (active && p4.y > 0.f) ? -C / p4.y : 0.f;
      F3 D = lambda * g;
      bool more = fabsf(C) > vol_tol, moved = false;
      float D2prev = lambda * lambda * p4.y;
      for (int pass = 1; pass < P.vol_iters && active && more; ++pass) {
        const F3 zz = zv + D;
        if (isv) reinterpret_cast<float4*>(z4b)[v] = make_float4(zz.x, zz.y, zz.z, 0.f);
        moved = true;
        __syncthreads();
        float T1 = 0.f, T2 = 0.f, T3 = 0.f;
        if (isv) {
          g = ring_gradient(z4b, zz, rcnt, vr1.x, vr1.y, vr1.z, P, v);
          T1 = dot(zz, g); T2 = dot(g, g); T3 = dot(g, D);
        }
        p4 = cta_sum4(make_float4(T1, T2, T3, 0.f));
        C = p4.x * (1.0f / 3.0f) - vstar;
        lambda = p4.y > 0.f ? (p4.z - C) / p4.y : 0.f;
        D = lambda * g;
        const float D2new = lambda * lambda * p4.y;
        more = (D2new + D2prev - 2.0f * lambda * p4.z) > vol_dtol2;
        D2prev = D2new;
      }
      if (moved && isv) reinterpret_cast<float4*>(z4b)[v] = make_float4(zv.x, zv.y, zv.z, 0.f);
      ev = fma3(P.w_volume, D, ev);
      en = fmaf(0.5f * P.w_volume, dot(D, D), en);
    }
    const F3 dz = zv - s3;
    en = fmaf(0.5f * mh2, dot(dz, dz), en);
    if (!isv) { ev = {0.f, 0.f, 0.f}; en = 0.f; }
    __syncthreads();                       // the element results are consumed: rb may be reused
  };

  // ---- r = T q for the 3 columns of this cell (tensor-core block product; columns 3..15 are zero)
  auto apply_operator = [&](F3 q) -> F3 {
    if (isvp) {
#pragma unroll
      for (int m = 0; m < kRhs; ++m) {
        const int idx = fbase + (m & 7) * 16 + (m >> 3);
        const float x = m == 0 ? q.x : m == 1 ? q.y : m == 2 ? q.z : 0.0f;
        const float hi = __uint_as_float((__float_as_uint(x) + 0x1000u) & 0xffffe000u);
        ra[idx] = hi;
        rb[idx] = x - hi;
      }
    }
    __syncthreads();
    const int g8 = lane >> 2, t4 = lane & 3;
    float acc[4][4];
#pragma unroll
    for (int j = 0; j < 4; ++j) {
      acc[j][0] = acc[j][1] = acc[j][2] = acc[j][3] = 0.f;
      const int ib = warp + j * nwarps;
      if (ib < nvb) {
        const int b0 = P.blk_ptr[3 * ib], bm = P.blk_ptr[3 * ib + 1], b1 = P.blk_ptr[3 * ib + 2];
        const unsigned char* const Ahi = reinterpret_cast<const unsigned char*>(ra) + lane * 16;
        const float2* const tv = reinterpret_cast<const float2*>(P.blk_val) + lane;
        float accx[4] = {0.f, 0.f, 0.f, 0.f};
        block_run<true>(acc[j], accx, tv, P.blk_col, b0, bm, Ahi, P.L.rb - P.L.ra, lane);
        block_run<false>(acc[j], accx, tv, P.blk_col, bm, b1, Ahi, 0, lane);
#pragma unroll
        for (int q2 = 0; q2 < 4; ++q2) acc[j][q2] += accx[q2];
      }
    }
    __syncthreads();
#pragma unroll
    for (int j = 0; j < 4; ++j) {
      const int ib = warp + j * nwarps;
      if (ib < nvb && g8 < 3)
        *reinterpret_cast<float2*>(rb + g8 * NP + ib * 8 + 2 * t4) = make_float2(acc[j][0], acc[j][1]);
    }
    __syncthreads();
    const F3 r = {rb[v], rb[NP + v], rb[2 * NP + v]};
    __syncthreads();
    return isv ? r : F3{0.f, 0.f, 0.f};
  };

  // ---- initial state: x = s
  F3 x3 = s3, g3, ev;
  float en;
  evaluate(x3, ev, en);
  g3 = mh2 * (x3 - s3) - ev;
  float gval = cta_sum4(make_float4(en, 0.f, 0.f, 0.f)).x;
  float res = cta_max(isv ? fmaxf(fmaxf(fabsf(g3.x), fabsf(g3.y)), fabsf(g3.z)) * h2m : 0.f);
  float rho0 = 0.f, rho1 = 0.f, rho2 = 0.f;        // 1/(s_j . y_j) of the pair in slot j (CTA-uniform)
  auto rho_of = [&](int j) { return j == 0 ? rho0 : j == 1 ? rho1 : rho2; };
  int npairs = 0, k = 0;

  while (k < max_iters && res > tol) {
    // -- direction by the two-loop recursion (pair of age a sits in slot (k - 1 - a) % kHist)
    F3 r3;
    float slope, alpha0 = 0.f, alpha1 = 0.f, alpha2 = 0.f;
    for (;;) {
      F3 q = g3;
#pragma unroll
      for (int a = 0; a < kHist; ++a) {
        if (a < npairs) {
          const int j = (k - 1 - a) % kHist;
          float hp[8];
          tmem_ld8(ta + kColHist + 8 * j, hp);
          const float sq = cta_sum4(make_float4(hp[0] * q.x + hp[1] * q.y + hp[2] * q.z, 0.f, 0.f, 0.f)).x;
          const float al = rho_of(j) * sq;
          if (a == 0) alpha0 = al; else if (a == 1) alpha1 = al; else alpha2 = al;
          q = {fmaf(-al, hp[3], q.x), fmaf(-al, hp[4], q.y), fmaf(-al, hp[5], q.z)};
        }
      }
      r3 = apply_operator(q);
#pragma unroll
      for (int a = kHist - 1; a >= 0; --a) {
        if (a < npairs) {
          const int j = (k - 1 - a) % kHist;
          float hp[8];
          tmem_ld8(ta + kColHist + 8 * j, hp);
          const float yr = cta_sum4(make_float4(hp[3] * r3.x + hp[4] * r3.y + hp[5] * r3.z, 0.f, 0.f, 0.f)).x;
          const float cfa = (a == 0 ? alpha0 : a == 1 ? alpha1 : alpha2) - rho_of(j) * yr;
          r3 = {fmaf(hp[0], cfa, r3.x), fmaf(hp[1], cfa, r3.y), fmaf(hp[2], cfa, r3.z)};
        }
      }
      slope = -cta_sum4(make_float4(dot(g3, r3), 0.f, 0.f, 0.f)).x;
      if (slope < 0.0f || npairs == 0) break;
      npairs = 0;    // not a descent direction (piecewise-smooth energies): drop the history
    }
    // -- backtracking line search on g
    float step = 1.0f, gtry;
    F3 xt, gn;
    for (;;) {
      xt = {fmaf(-step, r3.x, x3.x), fmaf(-step, r3.y, x3.y), fmaf(-step, r3.z, x3.z)};
      if (isv) reinterpret_cast<float4*>(z4b)[v] = make_float4(xt.x, xt.y, xt.z, 0.f);
      __syncthreads();
      evaluate(xt, ev, en);
      gtry = cta_sum4(make_float4(en, 0.f, 0.f, 0.f)).x;
      if (gtry <= gval + 1e-4f * step * slope + 8.0f * 1.1920929e-7f * fabsf(gval) || step < 1e-3f) break;
      step *= 0.5f;
    }
    gn = mh2 * (xt - s3) - ev;
    // -- history update
    {
      const int j = k % kHist;
      const F3 sk = xt - x3, yk = gn - g3;
      const float sy = cta_sum4(make_float4(dot(sk, yk), 0.f, 0.f, 0.f)).x;
      if (sy > 1e-30f) {
        const float hp[8] = {sk.x, sk.y, sk.z, yk.x, yk.y, yk.z, 0.f, 0.f};
        tmem_st8(ta + kColHist + 8 * j, hp);
        if (j == 0) rho0 = 1.0f / sy; else if (j == 1) rho1 = 1.0f / sy; else rho2 = 1.0f / sy;
        npairs = min(npairs + 1, kHist);
      } else {
        npairs = 0;
      }
    }
    x3 = xt; g3 = gn; gval = gtry;
    res = cta_max(isv ? fmaxf(fmaxf(fabsf(g3.x), fabsf(g3.y)), fabsf(g3.z)) * h2m : 0.f);
    ++k;
  }

  // ---- epilogue: x_n+1 = x_n + (u0 + x - s), v_n+1 = (u0 + x - s)/h
  {
    float* const st = rb;
    const int n3 = 3 * n;
    const size_t g = (size_t)cell * P.cell_stride;
    __syncthreads();
    for (int i = tid; i < n3; i += blockDim.x) st[i] = P.pos[g + i];
    __syncthreads();
    if (isv) {
      const F3 inc = u3 + (x3 - s3);
      const float invh = 1.0f / h;
      st[vext3] += inc.x; st[vext3 + 1] += inc.y; st[vext3 + 2] += inc.z;
      st[n3 + vext3] = inc.x * invh; st[n3 + vext3 + 1] = inc.y * invh; st[n3 + vext3 + 2] = inc.z * invh;
    }
    __syncthreads();
    for (int i = tid; i < n3; i += blockDim.x) { P.pos[g + i] = st[i]; P.vel[g + i] = st[n3 + i]; }
    if (tid == 0) {
      if (iters_out) iters_out[cell] = k;
      if (res_out) res_out[cell] = res;
    }
  }
  asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
  __syncthreads();
  if (warp == 0)
    asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" :: "r"(tmem_base_s), "r"(tmem_cols) : "memory");
}

}  // namespace

cudaError_t configure_converged_kernels() {
  cudaError_t e = cudaFuncSetAttribute(npfem_converged_kernel<672>, cudaFuncAttributeMaxDynamicSharedMemorySize, kSmemMaxDynamic);
  if (e != cudaSuccess) return e;
  return cudaFuncSetAttribute(npfem_converged_kernel<1024>, cudaFuncAttributeMaxDynamicSharedMemorySize, kSmemMaxDynamic);
}

cudaError_t launch_converged(const DevParams& p, int threads, int smem_bytes, float tol, int max_iters,
                             int* iters_out, float* res_out, cudaStream_t stream) {
  if (p.n_cells <= 0) return cudaSuccess;
  if (threads <= 672) npfem_converged_kernel<672><<<p.n_cells, threads, smem_bytes, stream>>>(p, tol, max_iters, iters_out, res_out);
  else npfem_converged_kernel<1024><<<p.n_cells, threads, smem_bytes, stream>>>(p, tol, max_iters, iters_out, res_out);
  return cudaGetLastError();
}

}  // namespace npfem
