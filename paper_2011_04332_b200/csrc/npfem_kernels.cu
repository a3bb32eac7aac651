// npfem_kernels.cu -- the fused npFEM step kernel for sm_100a.
//
// One CTA owns k <= 5 whole cells for a whole time step: it stages their state into shared
// memory, runs ALL n_iters local/global iterations there and writes positions and velocities
// back (north_star (b)-(d): no host round trip, no global-memory traffic between iterations
// except the read-only, L2-resident operator blocks).
//
// Arithmetic (fp32, increment form -- DESIGN.md "fp32 formulation"):
//   c      = centroid of x_n                      y = x_n - c        (cell-local coordinates)
//   u0     = h v_n + (h^2/m) f                    s = y + u0         (inertial prediction)
//   z^k    = s + d^k,  d^0 = 0                                        (current iterate)
//   e^k    = sum_el w A^T (p(z^k) - A z^k) + w_vol D(z^k)             (local step: elastic residual)
//   d^k+1  = d^k + T (e^k - (m/h^2) d^k),  T = A_sys^-1               (global step)
//   x_n+1  = x_n + (u0 + d),  v_n+1 = (u0 + d)/h
// which is algebraically the oracle's  x^{k+1} = A_sys^-1 (M/h^2 s + sum w A^T p)  (PAPER.md:90-95
// lineage), but never differences world coordinates.
#include <cstdint>

#include "npfem_kernels.cuh"

namespace npfem {
namespace {

struct F3 {
  float x, y, z;
};
__device__ __forceinline__ F3 operator+(F3 a, F3 b) { return {a.x + b.x, a.y + b.y, a.z + b.z}; }
__device__ __forceinline__ F3 operator-(F3 a, F3 b) { return {a.x - b.x, a.y - b.y, a.z - b.z}; }
__device__ __forceinline__ F3 operator*(float s, F3 a) { return {s * a.x, s * a.y, s * a.z}; }
__device__ __forceinline__ float dot(F3 a, F3 b) { return fmaf(a.x, b.x, fmaf(a.y, b.y, a.z * b.z)); }
__device__ __forceinline__ F3 cross(F3 a, F3 b) {
  return {fmaf(a.y, b.z, -a.z * b.y), fmaf(a.z, b.x, -a.x * b.z), fmaf(a.x, b.y, -a.y * b.x)};
}
__device__ __forceinline__ F3 fma3(float s, F3 a, F3 b) {
  return {fmaf(s, a.x, b.x), fmaf(s, a.y, b.y), fmaf(s, a.z, b.z)};
}
__device__ __forceinline__ F3 ld3(const float* p) { return {p[0], p[1], p[2]}; }
__device__ __forceinline__ void st3(float* p, F3 v) { p[0] = v.x; p[1] = v.y; p[2] = v.z; }

// MUFU-based approximations (<= 2 ulp): the local step's inputs carry the rounding of fp32
// cell-local positions, far above these, and IEEE division / sqrt
// cost 8-12 instructions each on the FMA pipe.
__device__ __forceinline__ float fdiv(float a, float b) { return __fdividef(a, b); }
__device__ __forceinline__ float frcp(float a) {
  float r;
  asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(a));
  return r;
}
__device__ __forceinline__ float fsqrt(float a) {
  float r;
  asm("sqrt.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(a));
  return r;
}
__device__ __forceinline__ float frsqrt(float a) {
  float r;
  asm("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(a));
  return r;
}

__device__ __forceinline__ float warp_sum(float v) {
  v += __shfl_xor_sync(0xffffffffu, v, 16);
  v += __shfl_xor_sync(0xffffffffu, v, 8);
  v += __shfl_xor_sync(0xffffffffu, v, 4);
  v += __shfl_xor_sync(0xffffffffu, v, 2);
  v += __shfl_xor_sync(0xffffffffu, v, 1);
  return v;
}

// Register-resident constants of one triangle (npfem_internal.h: TriConst).
struct TriReg {
  uint32_t ab, cf0, f12;   // packed internal vertex ids: (a,b), (c,f0), (f1,f2)
  float f[kTriFloats];
};

// Closest point of the hyperbola branch {t1*t2 = q^2, t > 0} to (s1, s2), s1 >= s2 > 0, written
// as (q p, q / p) with p >= 1: root of  g(p) = q p^4 - s1 p^3 + s2 p - q  (stationarity of the
// squared distance), bracketed in [1, max(s1/q, q/s2)] where g changes sign from <= 0 to >= 0.
// Newton from the same-ratio point sqrt(s1/s2), bisection whenever Newton leaves the bracket.
__device__ __forceinline__ float hyperbola_p(float s1, float s2, float q) {
  float lo = 1.0f, hi = fmaxf(fdiv(s1, q), fdiv(q, s2));
  float p = fsqrt(fdiv(s1, s2));
  p = fminf(fmaxf(p, lo), hi);
  for (int it = 0; it < 24; ++it) {
    float p2 = p * p;
    float g = fmaf(fmaf(q, p, -s1), p2 * p, fmaf(s2, p, -q));
    float dg = fmaf(fmaf(4.0f * q, p, -3.0f * s1), p2, s2);
    if (g < 0.0f) lo = p; else hi = p;
    float pn = p - fdiv(g, dg);
    if (!(dg > 0.0f) || !(pn >= lo) || !(pn <= hi)) pn = 0.5f * (lo + hi);
    float step = fabsf(pn - p);
    p = pn;
    if (step <= 2.4e-7f * p) break;
  }
  return p;
}

// Local step for one triangle: elastic residual forces on its three vertices from
//   - triangle strain   w_s ||F - P_s||^2/2,  P_s = U clamp(Sigma,[s_min,s_max]) V^T
//   - triangle area     w_a ||F - P_a||^2/2,  P_a = U Sigma' V^T, sigma1' sigma2' = clamp(sigma1 sigma2)
//   - the three hinges on its edges (each hinge is evaluated by both of its triangles; endpoint
//     contributions are halved so that every hinge counts once)
// (DESIGN.md "local step").  z = the cell's current iterate in shared memory.
__device__ __forceinline__ void triangle_residual(const TriReg& tr, const float* __restrict__ z,
                                                  const DevParams& P, float* __restrict__ out9) {
  const int ia = tr.ab & 0xffff, ib = tr.ab >> 16, ic = tr.cf0 & 0xffff;
  const int i0 = tr.cf0 >> 16, i1 = tr.f12 & 0xffff, i2 = tr.f12 >> 16;
  const F3 za = ld3(z + 3 * ia), zb = ld3(z + 3 * ib), zc = ld3(z + 3 * ic);
  const F3 zf0 = ld3(z + 3 * i0), zf1 = ld3(z + 3 * i1), zf2 = ld3(z + 3 * i2);
  const F3 eab = zb - za, eac = zc - za, ebc = zc - zb;

  // ---- membrane: F = [eab eac] D_m^-1, C = F^T F, singular values from tr and det
  const float i00 = tr.f[0], i01 = tr.f[1], i11 = tr.f[2];
  const F3 F0 = i00 * eab;
  const F3 F1 = fma3(i01, eab, i11 * eac);
  const float C11 = dot(F0, F0), C12 = dot(F0, F1), C22 = dot(F1, F1);
  const F3 Nn = cross(F0, F1);
  const float J = fsqrt(dot(Nn, Nn));                         // sigma1 * sigma2
  const float tau = fsqrt(C11 + C22 + 2.0f * J);              // sigma1 + sigma2
  const float dC = C11 - C22;
  const float Delta = fsqrt(fmaf(dC, dC, 4.0f * C12 * C12));  // sigma1^2 - sigma2^2
  const float delta = fdiv(Delta, fmaxf(tau, 1e-30f));             // sigma1 - sigma2
  const float s1 = 0.5f * (tau + delta);
  const float s2 = fmaxf(0.5f * (tau - delta), 1e-30f);
  // g_i = sum_terms w (projected sigma_i - sigma_i) / sigma_i   (residual form: P - F = F V diag(g) V^T)
  const float r1 = frcp(s1), r2 = frcp(s2);
  float g1 = tr.f[3] * (fminf(fmaxf(s1, P.s_min), P.s_max) - s1) * r1;
  float g2 = tr.f[3] * (fminf(fmaxf(s2, P.s_min), P.s_max) - s2) * r2;
  const float astar = fminf(fmaxf(J, P.a_min), P.a_max);
  if (J != astar) {
    const float q = fsqrt(astar);
    const float p = hyperbola_p(s1, s2, q);
    g1 = fmaf(tr.f[4], (q * p - s1) * r1, g1);
    g2 = fmaf(tr.f[4], (fdiv(q, p) - s2) * r2, g2);
  }
  const float gbar = 0.5f * (g1 + g2);
  const float rho = fdiv(g1 - g2, fmaxf(Delta, 1e-30f));
  const float S00 = fmaf(rho, 0.5f * dC, gbar), S11 = fmaf(-rho, 0.5f * dC, gbar), S01 = rho * C12;
  const F3 Q0 = fma3(S00, F0, S01 * F1);
  const F3 Q1 = fma3(S01, F0, S11 * F1);
  F3 fb = fma3(i00, Q0, i01 * Q1);
  F3 fc = i11 * Q1;
  F3 fa = {-(fb.x + fc.x), -(fb.y + fc.y), -(fb.z + fc.z)};

  // ---- bending hinges.  edge 0 = (a,b) opp c far f0; edge 1 = (b,c) opp a far f1; edge 2 = (c,a) opp b far f2
  {
    const float Kp = tr.f[5], Kq = tr.f[6], Ko = tr.f[7], rp = tr.f[8];
    const float Kf = -(Kp + Kq + Ko);
    F3 kv = fma3(Kq, eab, fma3(Ko, eac, Kf * (zf0 - za)));
    const float nk2 = dot(kv, kv);
    const float cf = nk2 > 1e-30f ? fmaf(rp, frsqrt(nk2), -1.0f) : 0.0f;
    kv = cf * kv;
    fa = fma3(0.5f * Kp, kv, fa); fb = fma3(0.5f * Kq, kv, fb); fc = fma3(Ko, kv, fc);
  }
  {
    const float Kp = tr.f[9], Kq = tr.f[10], Ko = tr.f[11], rp = tr.f[12];
    const float Kf = -(Kp + Kq + Ko);
    F3 kv = fma3(Kq, ebc, fma3(-Ko, eab, Kf * (zf1 - zb)));   // za - zb = -eab
    const float nk2 = dot(kv, kv);
    const float cf = nk2 > 1e-30f ? fmaf(rp, frsqrt(nk2), -1.0f) : 0.0f;
    kv = cf * kv;
    fb = fma3(0.5f * Kp, kv, fb); fc = fma3(0.5f * Kq, kv, fc); fa = fma3(Ko, kv, fa);
  }
  {
    const float Kp = tr.f[13], Kq = tr.f[14], Ko = tr.f[15], rp = tr.f[16];
    const float Kf = -(Kp + Kq + Ko);
    F3 kv = fma3(-Kq, eac, fma3(-Ko, ebc, Kf * (zf2 - zc)));  // za - zc = -eac, zb - zc = -ebc
    const float nk2 = dot(kv, kv);
    const float cf = nk2 > 1e-30f ? fmaf(rp, frsqrt(nk2), -1.0f) : 0.0f;
    kv = cf * kv;
    fc = fma3(0.5f * Kp, kv, fc); fa = fma3(0.5f * Kq, kv, fa); fb = fma3(Ko, kv, fb);
  }
  st3(out9, fa); st3(out9 + 3, fb); st3(out9 + 6, fc);
}

__device__ __forceinline__ uint32_t to_tf32(float x) {
  uint32_t r;
  asm("cvt.rna.tf32.f32 %0, %1;" : "=r"(r) : "f"(x));
  return r;
}
__device__ __forceinline__ void mma_tf32(float (&c)[4], const uint32_t (&a)[4], const uint32_t (&b)[2]) {
  asm volatile(
      "mma.sync.aligned.m16n8k8.row.col.f32.tf32.tf32.f32 {%0,%1,%2,%3}, {%4,%5,%6,%7}, {%8,%9}, "
      "{%0,%1,%2,%3};"
      : "+f"(c[0]), "+f"(c[1]), "+f"(c[2]), "+f"(c[3])
      : "r"(a[0]), "r"(a[1]), "r"(a[2]), "r"(a[3]), "r"(b[0]), "r"(b[1]));
}


// ------------------------------------------------------------------------------------------
// The fused step kernel.  MODE 1: global step with fp32 FMAs; MODE 2: 3xTF32 mma.sync.
// ------------------------------------------------------------------------------------------
template <int MODE, int MAXT>
__global__ void __launch_bounds__(MAXT, 1) npfem_step_kernel(const DevParams P) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  float* const z = reinterpret_cast<float*>(smem_raw + P.L.z);      // [k][n][3] current iterate (local coords)
  float* const s = reinterpret_cast<float*>(smem_raw + P.L.s);      // [k][n][3] inertial prediction
  float* const d = reinterpret_cast<float*>(smem_raw + P.L.d);      // [k][n][3] correction d^k
  float* const r = reinterpret_cast<float*>(smem_raw + P.L.r);      // [2][nvb*8][8] right-hand sides
  float* const out = reinterpret_cast<float*>(smem_raw + P.L.out);  // [T][9] triangle results / scratch
  float* const red = reinterpret_cast<float*>(smem_raw + P.L.red);  // [5][32][4] reduction partials
  __shared__ float vstar_s[kMaxCellsPerCta];
  __shared__ int vactive_s[kMaxCellsPerCta];

  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5, nwarps = blockDim.x >> 5;
  const int n = P.n, T = P.T, nvb = P.nvb;
  const int cell0 = blockIdx.x * P.k;
  const int kact = min(P.k, P.n_cells - cell0);
  const int n3 = 3 * n;

  // ---- per-thread constants: up to two triangles and one vertex
  TriReg tr[kTrisPerThread];
#pragma unroll
  for (int j = 0; j < kTrisPerThread; ++j) {
    const int t = tid + j * blockDim.x;
    if (t < T) {
      tr[j].ab = P.tri_ids[t] | (uint32_t(P.tri_ids[T + t]) << 16);
      tr[j].cf0 = P.tri_ids[2 * T + t] | (uint32_t(P.tri_ids[3 * T + t]) << 16);
      tr[j].f12 = P.tri_ids[4 * T + t] | (uint32_t(P.tri_ids[5 * T + t]) << 16);
#pragma unroll
      for (int q = 0; q < kTriFloats; ++q) tr[j].f[q] = P.tri_f[q * T + t];
    } else {
      tr[j].ab = tr[j].cf0 = tr[j].f12 = 0;
#pragma unroll
      for (int q = 0; q < kTriFloats; ++q) tr[j].f[q] = 0.0f;
    }
  }
  const bool isv = tid < n;
  const int v = isv ? tid : 0;
  const int vext = P.perm[v];
  const float h2m = P.h2_over_m[v], mh2 = P.m_over_h2[v];
  const int inc0 = P.inc_ptr[v], inc1 = P.inc_ptr[v + 1];
  const float h = P.h;

  // zero the right-hand-side buffer once: padding vertices, the 16th column and the columns of
  // missing cells are never written afterwards
  for (int i = tid; i < 2 * nvb * 64; i += blockDim.x) r[i] = 0.0f;

  // ---- prologue: load state, centroid, local coordinates, inertial prediction
  for (int c = 0; c < kact; ++c) {
    float sx = 0.f, sy = 0.f, sz = 0.f;
    if (isv) {
      const float* px = P.pos + (size_t)(cell0 + c) * P.cell_stride + 3 * vext;
      sx = px[0]; sy = px[1]; sz = px[2];
    }
    sx = warp_sum(sx); sy = warp_sum(sy); sz = warp_sum(sz);
    if (lane == 0) { float* q = red + (c * 32 + warp) * 4; q[0] = sx; q[1] = sy; q[2] = sz; }
  }
  __syncthreads();
  for (int c = 0; c < kact; ++c) {
    const float* q = red + (c * 32 + lane) * 4;
    float cx = lane < nwarps ? q[0] : 0.f, cy = lane < nwarps ? q[1] : 0.f, cz = lane < nwarps ? q[2] : 0.f;
    cx = warp_sum(cx); cy = warp_sum(cy); cz = warp_sum(cz);
    const float invn = 1.0f / (float)n;
    cx *= invn; cy *= invn; cz *= invn;
    if (isv) {
      const size_t g = (size_t)(cell0 + c) * P.cell_stride + 3 * vext;
      const F3 x = ld3(P.pos + g), vv = ld3(P.vel + g), ff = ld3(P.fext + g);
      const F3 u0 = {fmaf(h, vv.x, h2m * ff.x), fmaf(h, vv.y, h2m * ff.y), fmaf(h, vv.z, h2m * ff.z)};
      const F3 y = {x.x - cx, x.y - cy, x.z - cz};
      const F3 sv = y + u0;
      const int o = c * n3 + 3 * v;
      st3(s + o, sv); st3(z + o, sv);
      d[o] = 0.f; d[o + 1] = 0.f; d[o + 2] = 0.f;
    }
  }
  __syncthreads();

  // ---- iterations
  for (int it = 0; it < P.n_iters; ++it) {
    // local step, elastic part: triangles -> out, vertices gather -> r = e - (m/h^2) d
    for (int c = 0; c < kact; ++c) {
      const float* zc = z + c * n3;
#pragma unroll
      for (int j = 0; j < kTrisPerThread; ++j) {
        const int t = tid + j * blockDim.x;
        if (t < T) triangle_residual(tr[j], zc, P, out + 9 * t);
      }
      __syncthreads();
      if (isv) {
        float ex = 0.f, ey = 0.f, ez = 0.f;
        for (int i = inc0; i < inc1; ++i) {
          const float* o = out + P.inc_out[i];
          ex += o[0]; ey += o[1]; ez += o[2];
        }
        const int o = c * n3 + 3 * v;
        const int m = 3 * c;
        float* rr = r + (size_t)v * 8;
        const int half = nvb * 64;
        rr[((m) >> 3) * half + ((m) & 7)] = fmaf(-mh2, d[o], ex);
        rr[((m + 1) >> 3) * half + ((m + 1) & 7)] = fmaf(-mh2, d[o + 1], ey);
        rr[((m + 2) >> 3) * half + ((m + 2) & 7)] = fmaf(-mh2, d[o + 2], ez);
      }
      __syncthreads();
    }

    // local step, volume part: D = lambda * grad V(z + D), vol_iters fixed-point sweeps
    // (D <- ((g.D - C)/(g.g)) g; grad V at a vertex = 1/6 sum of ring cross products,
    //  V = 1/3 sum_v x_v . g_v for the closed surface).  out[] is free now and holds D / g.
    if (P.w_volume > 0.0f) {
      float* const scr = out;   // [k][n][3]
      for (int vi = 0; vi < P.vol_iters; ++vi) {
        for (int c = 0; c < kact; ++c) {
          float S1 = 0.f, S2 = 0.f, S3 = 0.f;
          if (isv && (vi == 0 || vactive_s[c])) {
            const float* zc = z + c * n3;
            const int o = c * n3 + 3 * v;
            const F3 zv = ld3(zc + 3 * v);
            F3 g = {0.f, 0.f, 0.f};
            F3 eprev = ld3(zc + 3 * P.inc_ring[inc1 - 1]) - zv;
            for (int i = inc0; i < inc1; ++i) {
              const F3 e = ld3(zc + 3 * P.inc_ring[i]) - zv;
              const F3 cr = cross(eprev, e);
              g = g + cr;
              eprev = e;
            }
            g = (1.0f / 6.0f) * g;
            S1 = dot(zv, g);
            S2 = dot(g, g);
            if (vi > 0) S3 = dot(g, ld3(scr + o));
            st3(scr + o, g);
          }
          S1 = warp_sum(S1); S2 = warp_sum(S2); S3 = warp_sum(S3);
          if (lane == 0) { float* q = red + (c * 32 + warp) * 4; q[0] = S1; q[1] = S2; q[2] = S3; }
        }
        __syncthreads();
        for (int c = 0; c < kact; ++c) {
          const float* q = red + (c * 32 + lane) * 4;
          float S1 = lane < nwarps ? q[0] : 0.f, S2 = lane < nwarps ? q[1] : 0.f, S3 = lane < nwarps ? q[2] : 0.f;
          S1 = warp_sum(S1); S2 = warp_sum(S2); S3 = warp_sum(S3);
          const float V = S1 * (1.0f / 3.0f);
          float vstar;
          bool active;
          if (vi == 0) {
            vstar = fminf(fmaxf(V, P.Vmin), P.Vmax);
            active = (V != vstar);
          } else {
            vstar = vstar_s[c];
            active = vactive_s[c] != 0;
          }
          const float lambda = (active && S2 > 0.f) ? (S3 - (V - vstar)) / S2 : 0.f;
          if (isv) {
            const int o = c * n3 + 3 * v;
            const F3 D = lambda * ld3(scr + o);
            st3(scr + o, D);
            if (vi + 1 < P.vol_iters && active) {
              const F3 zz = (ld3(s + o) + ld3(d + o)) + D;
              st3(z + o, zz);
            }
          }
          if (vi == 0 && tid == 0) { vstar_s[c] = vstar; vactive_s[c] = active ? 1 : 0; }
        }
        __syncthreads();
      }
      if (isv) {
        const int half = nvb * 64;
        float* rr = r + (size_t)v * 8;
        for (int c = 0; c < kact; ++c) {
          const int o = c * n3 + 3 * v;
          const int m = 3 * c;
          // residual of the volume term: w_vol (P_v - z) = w_vol D
          rr[((m) >> 3) * half + ((m) & 7)] += P.w_volume * scr[o];
          rr[((m + 1) >> 3) * half + ((m + 1) & 7)] += P.w_volume * scr[o + 1];
          rr[((m + 2) >> 3) * half + ((m + 2) & 7)] += P.w_volume * scr[o + 2];
        }
      }
      __syncthreads();
    }

    // global step: d += T r, with T in 8x8 blocks; one warp per block of 8 output vertices
    const int mlim = 3 * kact;
    if (MODE == 1) {
      const int g = lane >> 2, q4 = lane & 3;
      const float* rbase0 = r + (q4 >> 1) * nvb * 64 + (q4 & 1) * 4;
      for (int ib = warp; ib < nvb; ib += nwarps) {
        float a0 = 0.f, a1 = 0.f, a2 = 0.f, a3 = 0.f;
        const int b1 = P.blk_ptr[ib + 1];
        for (int b = P.blk_ptr[ib]; b < b1; ++b) {
          const int jb = P.blk_col[b];
          const float4* tv = reinterpret_cast<const float4*>(P.blk_val + (size_t)b * 64 + g * 8);
          const float4 t0 = __ldg(tv), t1 = __ldg(tv + 1);
          const float tk[8] = {t0.x, t0.z, t1.x, t1.z, t0.y, t0.w, t1.y, t1.w};   // k = 0..7
          const float* rb = rbase0 + jb * 64;
#pragma unroll
          for (int kk = 0; kk < 8; ++kk) {
            const float4 r4 = *reinterpret_cast<const float4*>(rb + kk * 8);
            a0 = fmaf(tk[kk], r4.x, a0); a1 = fmaf(tk[kk], r4.y, a1);
            a2 = fmaf(tk[kk], r4.z, a2); a3 = fmaf(tk[kk], r4.w, a3);
          }
        }
        const int i = ib * 8 + g;
        const float acc[4] = {a0, a1, a2, a3};
        if (i < n) {
#pragma unroll
          for (int e = 0; e < 4; ++e) {
            const int m = 4 * q4 + e;
            if (m < mlim) {
              const int c = m / 3, comp = m - 3 * c;
              const int o = c * n3 + 3 * i + comp;
              const float dn = d[o] + acc[e];
              d[o] = dn;
              z[o] = s[o] + dn;
            }
          }
        }
      }
    } else {
      const int g = lane >> 2, t4 = lane & 3;
      const int half = nvb * 64;
      for (int ib = warp; ib < nvb; ib += nwarps) {
        float acc[4] = {0.f, 0.f, 0.f, 0.f};
        const int b1 = P.blk_ptr[ib + 1];
        for (int b = P.blk_ptr[ib]; b < b1; ++b) {
          const int jb = P.blk_col[b];
          const float2 tb = __ldg(reinterpret_cast<const float2*>(P.blk_val + (size_t)b * 64) + lane);
          const float* rb = r + jb * 64 + t4 * 8 + g;
          const float av[4] = {rb[0], rb[half], rb[32], rb[half + 32]};
          uint32_t ahi[4], alo[4], bhi[2], blo[2];
#pragma unroll
          for (int e = 0; e < 4; ++e) {
            ahi[e] = to_tf32(av[e]);
            alo[e] = to_tf32(av[e] - __uint_as_float(ahi[e]));
          }
          bhi[0] = to_tf32(tb.x); blo[0] = to_tf32(tb.x - __uint_as_float(bhi[0]));
          bhi[1] = to_tf32(tb.y); blo[1] = to_tf32(tb.y - __uint_as_float(bhi[1]));
          mma_tf32(acc, alo, bhi);
          mma_tf32(acc, ahi, blo);
          mma_tf32(acc, ahi, bhi);
        }
#pragma unroll
        for (int e = 0; e < 4; ++e) {
          const int m = g + ((e & 2) ? 8 : 0);
          const int i = ib * 8 + 2 * t4 + (e & 1);
          if (m < mlim && i < n) {
            const int c = m / 3, comp = m - 3 * c;
            const int o = c * n3 + 3 * i + comp;
            const float dn = d[o] + acc[e];
            d[o] = dn;
            z[o] = s[o] + dn;
          }
        }
      }
    }
    __syncthreads();
  }

  // ---- epilogue: x_n+1 = x_n + (u0 + d), v_n+1 = (u0 + d)/h
  if (isv) {
    for (int c = 0; c < kact; ++c) {
      const size_t g = (size_t)(cell0 + c) * P.cell_stride + 3 * vext;
      const F3 x = ld3(P.pos + g), vv = ld3(P.vel + g), ff = ld3(P.fext + g);
      const int o = c * n3 + 3 * v;
      const F3 inc = {fmaf(h, vv.x, h2m * ff.x) + d[o], fmaf(h, vv.y, h2m * ff.y) + d[o + 1],
                      fmaf(h, vv.z, h2m * ff.z) + d[o + 2]};
      st3(P.pos + g, x + inc);
      const F3 vn = {inc.x / h, inc.y / h, inc.z / h};
      st3(P.vel + g, vn);
    }
  }
}

}  // namespace

cudaError_t configure_kernels(int smem_bytes) {
  cudaError_t e;
  (void)smem_bytes;
  smem_bytes = kSmemMaxDynamic;   // opt in once to the largest carve-out any cell type may need
#define NPFEM_CFG(MODE, MAXT)                                                                   \
  e = cudaFuncSetAttribute(npfem_step_kernel<MODE, MAXT>,                                       \
                           cudaFuncAttributeMaxDynamicSharedMemorySize, smem_bytes);            \
  if (e != cudaSuccess) return e;
  NPFEM_CFG(1, 704) NPFEM_CFG(1, 1024) NPFEM_CFG(2, 704) NPFEM_CFG(2, 1024)
#undef NPFEM_CFG
  return cudaSuccess;
}

cudaError_t launch_step(const DevParams& p, int threads, int smem_bytes, int mode,
                        cudaStream_t stream) {
  if (p.n_cells <= 0) return cudaSuccess;
  const int grid = (p.n_cells + p.k - 1) / p.k;
  if (threads <= 704) {
    if (mode == 2) npfem_step_kernel<2, 704><<<grid, threads, smem_bytes, stream>>>(p);
    else npfem_step_kernel<1, 704><<<grid, threads, smem_bytes, stream>>>(p);
  } else {
    if (mode == 2) npfem_step_kernel<2, 1024><<<grid, threads, smem_bytes, stream>>>(p);
    else npfem_step_kernel<1, 1024><<<grid, threads, smem_bytes, stream>>>(p);
  }
  return cudaGetLastError();
}

}  // namespace npfem
