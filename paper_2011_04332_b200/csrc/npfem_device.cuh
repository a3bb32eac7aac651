// npfem_device.cuh -- device functions shared by the step kernels (npfem_kernels.cu: fixed-count
// fused step; npfem_converged.cu: converged quasi-Newton step): small vector helpers, MUFU
// approximations, the element-level local step (membrane + hinge residuals), the volume gradient,
// the tensor-core block product of the global step and the tensor-memory scratch accessors.
// Algorithm and citations: DESIGN.md.
#pragma once
#include <cstdint>

#include "npfem_kernels.cuh"

namespace npfem {
namespace {

// Diagnostic builds (-DNPFEM_PHASE_CLOCKS): ablation mask of the MODE 3 operator product, a kernel
// parameter (DevParams::dbg): 1 no mma, 2 no shared loads, 4 no stream loads, 8 no descriptor loads.
#ifdef NPFEM_PHASE_CLOCKS
#define NPFEM_DBG(bit) (dbg & (bit))
#else
#define NPFEM_DBG(bit) 0
#endif

struct F3 {
  float x, y, z;
};
__device__ __forceinline__ F3 operator+(F3 a, F3 b) { return {a.x + b.x, a.y + b.y, a.z + b.z}; }
__device__ __forceinline__ F3 operator-(F3 a, F3 b) { return {a.x - b.x, a.y - b.y, a.z - b.z}; }
__device__ __forceinline__ F3 operator*(float s, F3 a) { return {s * a.x, s * a.y, s * a.z}; }
__device__ __forceinline__ float dot(F3 a, F3 b) { return fmaf(a.x, b.x, fmaf(a.y, b.y, a.z * b.z)); }
// acc + a x b
__device__ __forceinline__ F3 cross_acc(F3 a, F3 b, F3 acc) {
  return {fmaf(a.y, b.z, fmaf(-a.z, b.y, acc.x)), fmaf(a.z, b.x, fmaf(-a.x, b.z, acc.y)),
          fmaf(a.x, b.y, fmaf(-a.y, b.x, acc.z))};
}
__device__ __forceinline__ F3 fma3(float s, F3 a, F3 b) {
  return {fmaf(s, a.x, b.x), fmaf(s, a.y, b.y), fmaf(s, a.z, b.z)};
}
__device__ __forceinline__ F3 xyz(float4 v) { return {v.x, v.y, v.z}; }
__device__ __forceinline__ F3 lds3(const unsigned char* base, uint32_t byte_off) {
  return xyz(*reinterpret_cast<const float4*>(base + byte_off));
}

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


// Closest point of the hyperbola branch {t1*t2 = q^2, t > 0} to (s1, s2), s1 >= s2 > 0, written
// as (q p, q / p) with p >= 1: root of  g(p) = q p^4 - s1 p^3 + s2 p - q  (stationarity of the
// squared distance).  Start: the same-ratio point p0 = sqrt(s1/s2), where g(p0) = (p0^4 - 1)
// (q - sqrt(s1 s2)) is already small for nearly isotropic or nearly area-preserving states.
// Safeguarded variant: bracket [1, max(s1/q, q/s2)] (g goes from <= 0 to >= 0), Newton with
// bisection whenever Newton leaves the bracket.
__device__ __noinline__ float hyperbola_p_safe(float s1, float s2, float q, float p) {
  float lo = 1.0f, hi = fmaxf(fdiv(s1, q), fdiv(q, s2));
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
// Fast variant for moderate deformations (s1/s2 < 1.5 and |s1 s2 - q^2| < 0.4 q^2): plain Newton
// steps from p0, quadratically convergent there (start error < 0.1 => < 1e-7 after 3).  When the
// first step is already below 2e-4 p the error after it is below fp32 resolution (6e-8 p): one
// step is all a cell near its rest state needs.
__device__ __forceinline__ float hyperbola_p(float s1, float s2, float q, float ratio, float J) {
  float p = fsqrt(ratio);
  const float q2 = q * q;
  if (ratio < 1.5f && fabsf(J - q2) < 0.4f * q2) {
    float step;
    {
      const float p2 = p * p;
      const float g = fmaf(fmaf(q, p, -s1), p2 * p, fmaf(s2, p, -q));
      const float dg = fmaf(fmaf(4.0f * q, p, -3.0f * s1), p2, s2);
      step = g * frcp(dg);
      p -= step;
    }
    if (fabsf(step) > 2e-4f * p) {
#pragma unroll
      for (int it = 0; it < 2; ++it) {
        const float p2 = p * p;
        const float g = fmaf(fmaf(q, p, -s1), p2 * p, fmaf(s2, p, -q));
        const float dg = fmaf(fmaf(4.0f * q, p, -3.0f * s1), p2, s2);
        p = fmaf(-g, frcp(dg), p);
      }
    }
    return p;
  }
  return hyperbola_p_safe(s1, s2, q, p);
}

// Membrane part of the local step for one triangle (p0,p1,p2) with edges e1 = z1 - z0,
// e2 = z2 - z0:  F = [e1 e2] D_m^-1, singular values from tr(F^T F) and det; residual forces of
//   - triangle strain   w_s ||F - P_s||^2/2,  P_s = U clamp(Sigma,[s_min,s_max]) V^T
//   - triangle area     w_a ||F - P_a||^2/2,  P_a = U Sigma' V^T, sigma1' sigma2' = clamp(sigma1 sigma2)
// on vertices 1 and 2 (vertex 0 receives -(f1 + f2)).  SURVEY.md 8(c) step 2.
// KIND 1 (damped, reading A-20): the stiffness-proportional damping adds -(c_beta/h)(w_s + w_a) G^T F,
// i.e. a shift of both g_i.  KIND 2: the linear operator alone, +(c_beta/h)(w_s + w_a) G^T F (used
// once per step on y = x_n - c to form the constant part of the damping force).
// KIND 3: residual as KIND 0, and the triangle's energy 1/2 w_s dist^2(F, strain set) +
// 1/2 w_a dist^2(F, area set) is added to `en` (converged solve: the line search needs g).
// HARD: strain-dependent strain weight w_s (1 + beta d^2) (reading A-23), beta = P.hard at run time.
template <int KIND, bool HARD>
__device__ __forceinline__ void membrane(F3 e1, F3 e2, float i00, float i01, float i11, float ws,
                                         float wa, const DevParams& P, F3& f1, F3& f2, float& en) {
  if (KIND == 2) {
    const float coef = P.cbh * (ws + wa);
    const F3 Q0 = (coef * i00) * e1;
    const F3 Q1 = coef * fma3(i01, e1, i11 * e2);
    f1 = fma3(i00, Q0, i01 * Q1);
    f2 = i11 * Q1;
    return;
  }
  const F3 F0 = i00 * e1;
  const F3 F1 = fma3(i01, e1, i11 * e2);
  const float C11 = dot(F0, F0), C12 = dot(F0, F1), C22 = dot(F1, F1);
  const float J = fsqrt(fmaxf(fmaf(C11, C22, -C12 * C12), 0.0f));   // sigma1 * sigma2 = sqrt(det F^T F)
  const float tau = fsqrt(C11 + C22 + 2.0f * J);              // sigma1 + sigma2
  const float dC = C11 - C22;
  const float Delta = fsqrt(fmaf(dC, dC, 4.0f * C12 * C12));  // sigma1^2 - sigma2^2
  const float delta = Delta * frcp(fmaxf(tau, 1e-30f));       // sigma1 - sigma2
  const float s1 = 0.5f * (tau + delta);
  const float s2 = fmaxf(0.5f * (tau - delta), 1e-30f);
  // g_i = sum_terms w (projected sigma_i - sigma_i) / sigma_i   (residual form: P - F = F V diag(g) V^T)
  const float rJ = frcp(fmaxf(s1 * s2, 1e-30f));
  const float r1 = s2 * rJ, r2 = s1 * rJ;                     // 1/sigma1, 1/sigma2
  const float d1 = fminf(fmaxf(s1, P.s_min), P.s_max) - s1, d2 = fminf(fmaxf(s2, P.s_min), P.s_max) - s2;
  float g1 = ws * d1 * r1;
  float g2 = ws * d2 * r2;
  if (HARD) {
    g1 *= fmaf(P.hard, d1 * d1, 1.0f);
    g2 *= fmaf(P.hard, d2 * d2, 1.0f);
  }
  if (KIND == 3) {
    const float q1 = d1 * d1, q2 = d2 * d2;
    en = fmaf(0.5f * ws, HARD ? fmaf(0.5f * P.hard, fmaf(q1, q1, q2 * q2), q1 + q2) : q1 + q2, en);
  }
  const float astar = fminf(fmaxf(J, P.a_min), P.a_max);
  if (J != astar) {
    const float q = fsqrt(astar);
    const float p = hyperbola_p(s1, s2, q, s1 * r2, J);
    const float a1 = fmaf(q, p, -s1), a2 = fmaf(q, frcp(p), -s2);
    g1 = fmaf(wa, a1 * r1, g1);
    g2 = fmaf(wa, a2 * r2, g2);
    if (KIND == 3) en = fmaf(0.5f * wa, fmaf(a1, a1, a2 * a2), en);
  }
  if (KIND == 1) {
    const float shift = P.cbh * (ws + wa);
    g1 -= shift; g2 -= shift;
  }
  const float gbar = 0.5f * (g1 + g2);
  const float rho = (g1 - g2) * frcp(fmaxf(Delta, 1e-30f));
  const float S00 = fmaf(rho, 0.5f * dC, gbar), S11 = fmaf(-rho, 0.5f * dC, gbar), S01 = rho * C12;
  const F3 Q0 = fma3(S00, F0, S01 * F1);
  const F3 Q1 = fma3(S01, F0, S11 * F1);
  f1 = fma3(i00, Q0, i01 * Q1);
  f2 = i11 * Q1;
}

// Bending hinge on the edge (p,q) with own opposite vertex o and the vertex f across:
// kv = sum K_i z_i written with edges from p (rows of K sum to 0), scaled so that adding
// K_i * kv to vertex i applies the residual  w_h K_i (r_h k/|k| - k)  (bending).
// KIND 1: with the damping term -(c_beta/h) w_h K_i k the factor becomes r/|k| - 1 - c_beta/h;
// KIND 2: the linear operator alone, factor +c_beta/h.
// KIND 3: `en` += wgt * 1/2 (|k| - r)^2 (the rows are pre-scaled by sqrt(w_h)).
template <int KIND>
__device__ __forceinline__ F3 hinge_vec(float Kq, float Ko, float Kf, float rp, F3 epq, F3 epo, F3 epf,
                                        float cbh, float wgt, float& en) {
  const F3 kv = fma3(Kq, epq, fma3(Ko, epo, Kf * epf));
  if (KIND == 2) return cbh * kv;
  const float nk2 = fmaxf(dot(kv, kv), 1e-30f);
  const float rs = frsqrt(nk2);
  const float cf = fmaf(rp, rs, KIND == 1 ? -1.0f - cbh : -1.0f);
  if (KIND == 3) {
    const float dk = fmaf(nk2, rs, -rp);
    en = fmaf(0.5f * wgt, dk * dk, en);
  }
  return cf * kv;
}

__device__ __forceinline__ void mma_tf32(float (&c)[4], const uint32_t (&a)[4], const uint32_t (&b)[2]) {
  asm volatile(
      "mma.sync.aligned.m16n8k8.row.col.f32.tf32.tf32.f32 {%0,%1,%2,%3}, {%4,%5,%6,%7}, {%8,%9}, "
      "{%0,%1,%2,%3};"
      : "+f"(c[0]), "+f"(c[1]), "+f"(c[2]), "+f"(c[3])
      : "r"(a[0]), "r"(a[1]), "r"(a[2]), "r"(a[3]), "r"(b[0]), "r"(b[1]));
}

// global_mode 3: D(16 rhs columns x 8 output vertices) += A(16 x 16 fp16) B(16 x 8 fp16), fp32 accumulate
__device__ __forceinline__ void mma_f16(float (&c)[4], uint32_t a0, uint32_t a1, uint32_t a2, uint32_t a3,
                                        uint32_t b0, uint32_t b1, int dbg = 0) {
  if (NPFEM_DBG(1)) { c[0] += __uint_as_float(a0 ^ b0); c[1] += __uint_as_float(a1 ^ b1); c[2] += __uint_as_float(a2); c[3] += __uint_as_float(a3); return; }
  asm volatile(
      "mma.sync.aligned.m16n8k16.row.col.f32.f16.f16.f32 {%0,%1,%2,%3}, {%4,%5,%6,%7}, {%8,%9}, "
      "{%0,%1,%2,%3};"
      : "+f"(c[0]), "+f"(c[1]), "+f"(c[2]), "+f"(c[3])
      : "r"(a0), "r"(a1), "r"(a2), "r"(a3), "r"(b0), "r"(b1));
}

// Operator blocks stream from L2 once per use: keep them out of L1, which holds the register spills.
__device__ __forceinline__ float2 ldg_stream(const float2* p) {
  float2 v;
  asm volatile("ld.global.nc.L1::no_allocate.v2.f32 {%0, %1}, [%2];" : "=f"(v.x), "=f"(v.y) : "l"(p));
  return v;
}

__device__ __forceinline__ uint4 ldg_stream(const uint4* p) {
  uint4 v;
  asm volatile("ld.global.nc.L1::no_allocate.v4.u32 {%0, %1, %2, %3}, [%4];"
               : "=r"(v.x), "=r"(v.y), "=r"(v.z), "=r"(v.w) : "l"(p));
  return v;
}
__device__ __forceinline__ uint2 ldg_stream(const uint2* p) {
  uint2 v;
  asm volatile("ld.global.nc.L1::no_allocate.v2.u32 {%0, %1}, [%2];" : "=r"(v.x), "=r"(v.y) : "l"(p));
  return v;
}

// ---- tensor memory as per-thread scratch: thread (warp w, lane l) owns TMEM lane 32*(w%4) + l;
//      a 32x32b.x16 access moves 16 consecutive columns of that lane to / from 16 registers.
__device__ __forceinline__ void tmem_st16(uint32_t a, const float (&v)[16]) {
  asm volatile(
      "tcgen05.st.sync.aligned.32x32b.x16.b32 [%0], {%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15,%16};"
      :: "r"(a), "f"(v[0]), "f"(v[1]), "f"(v[2]), "f"(v[3]), "f"(v[4]), "f"(v[5]), "f"(v[6]), "f"(v[7]),
         "f"(v[8]), "f"(v[9]), "f"(v[10]), "f"(v[11]), "f"(v[12]), "f"(v[13]), "f"(v[14]), "f"(v[15])
      : "memory");
  asm volatile("tcgen05.wait::st.sync.aligned;" ::: "memory");
}
__device__ __forceinline__ void tmem_st4(uint32_t a, float v0, float v1, float v2, float v3) {
  asm volatile("tcgen05.st.sync.aligned.32x32b.x4.b32 [%0], {%1,%2,%3,%4};"
               :: "r"(a), "f"(v0), "f"(v1), "f"(v2), "f"(v3) : "memory");
  asm volatile("tcgen05.wait::st.sync.aligned;" ::: "memory");
}
__device__ __forceinline__ void tmem_ld4(uint32_t a, float& v0, float& v1, float& v2, float& v3) {
  asm volatile("tcgen05.ld.sync.aligned.32x32b.x4.b32 {%0,%1,%2,%3}, [%4];"
               : "=f"(v0), "=f"(v1), "=f"(v2), "=f"(v3) : "r"(a) : "memory");
  asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
}
__device__ __forceinline__ void tmem_ld16(uint32_t a, float (&v)[16]) {
  asm volatile(
      "tcgen05.ld.sync.aligned.32x32b.x16.b32 {%0,%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15}, [%16];"
      : "=f"(v[0]), "=f"(v[1]), "=f"(v[2]), "=f"(v[3]), "=f"(v[4]), "=f"(v[5]), "=f"(v[6]), "=f"(v[7]),
        "=f"(v[8]), "=f"(v[9]), "=f"(v[10]), "=f"(v[11]), "=f"(v[12]), "=f"(v[13]), "=f"(v[14]), "=f"(v[15])
      : "r"(a)
      : "memory");
  asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
}

// Local step of one element for one cell: membrane residuals of its two triangles and the five
// hinges it sees, summed per own vertex (a,b,c,d) into out4[slot * E].  ec = the element's
// constants in shared memory (group g at ec[g * E], npfem_api.cu), zc = the cell's z4 array.
template <int KIND, bool HARD = false>
__device__ __forceinline__ void element_residual(const float4* __restrict__ ec, int E,
                                                 const unsigned char* __restrict__ zc,
                                                 const DevParams& P, float4* __restrict__ out4) {
  const float4 idw = ec[0];
  const uint32_t id_ab = __float_as_uint(idw.x), id_cd = __float_as_uint(idw.y);
  const uint32_t id_f12 = __float_as_uint(idw.z), id_f34 = __float_as_uint(idw.w);
  const F3 za = lds3(zc, id_ab & 0xffffu), zb = lds3(zc, id_ab >> 16);
  const F3 zc3 = lds3(zc, id_cd & 0xffffu), zd = lds3(zc, id_cd >> 16);
  const F3 eab = zb - za, eac = zc3 - za, ebc = zc3 - zb, ead = zd - za, ebd = zd - zb;
  const F3 eba = {-eab.x, -eab.y, -eab.z};

  F3 fa = {0.f, 0.f, 0.f}, fb = fa, fc = fa, fd = fa;
  float en = 0.0f;   // KIND 3: the element's share of E_el (outer hinges count half: both sides see them)
  const float4 m3 = ec[3 * E];
  // ---- shared hinge (a,b | c ; d): once in full for a diamond, the element's half for a single
  {
    const float4 hk = ec[4 * E];
    const float Kp = hk.x, Kq = hk.y, Ko = hk.z;
    const float Kf = -(Kp + Kq + Ko), he = m3.z, hf = fmaf(2.0f, he, -1.0f);
    const F3 kv = hinge_vec<KIND>(Kq, Ko, Kf, hk.w, eab, eac, ead, P.cbh, he, en);
    fa = fma3(he * Kp, kv, fa); fb = fma3(he * Kq, kv, fb);
    fc = fma3(Ko, kv, fc);      fd = fma3(hf * Kf, kv, fd);
  }
  // ---- outer hinges: half of the end-point terms, all of the own opposite vertex's term
  {   // (b,c | a ; f1)
    const float4 hk = ec[5 * E];
    const F3 zf = lds3(zc, id_f12 & 0xffffu);
    const F3 kv = hinge_vec<KIND>(hk.y, hk.z, -(hk.x + hk.y + hk.z), hk.w, ebc, eba, zf - zb, P.cbh, 0.5f, en);
    fb = fma3(0.5f * hk.x, kv, fb); fc = fma3(0.5f * hk.y, kv, fc); fa = fma3(hk.z, kv, fa);
  }
  {   // (c,a | b ; f2)
    const float4 hk = ec[6 * E];
    const F3 zf = lds3(zc, id_f12 >> 16);
    const F3 eca = {-eac.x, -eac.y, -eac.z}, ecb = {-ebc.x, -ebc.y, -ebc.z};
    const F3 kv = hinge_vec<KIND>(hk.y, hk.z, -(hk.x + hk.y + hk.z), hk.w, eca, ecb, zf - zc3, P.cbh, 0.5f, en);
    fc = fma3(0.5f * hk.x, kv, fc); fa = fma3(0.5f * hk.y, kv, fa); fb = fma3(hk.z, kv, fb);
  }
  {   // (a,d | b ; f3)
    const float4 hk = ec[7 * E];
    const F3 zf = lds3(zc, id_f34 & 0xffffu);
    const F3 kv = hinge_vec<KIND>(hk.y, hk.z, -(hk.x + hk.y + hk.z), hk.w, ead, eab, zf - za, P.cbh, 0.5f, en);
    fa = fma3(0.5f * hk.x, kv, fa); fd = fma3(0.5f * hk.y, kv, fd); fb = fma3(hk.z, kv, fb);
  }
  {   // (d,b | a ; f4)
    const float4 hk = ec[8 * E];
    const F3 zf = lds3(zc, id_f34 >> 16);
    const F3 edb = {-ebd.x, -ebd.y, -ebd.z}, eda = {-ead.x, -ead.y, -ead.z};
    const F3 kv = hinge_vec<KIND>(hk.y, hk.z, -(hk.x + hk.y + hk.z), hk.w, edb, eda, zf - zd, P.cbh, 0.5f, en);
    fd = fma3(0.5f * hk.x, kv, fd); fb = fma3(0.5f * hk.y, kv, fb); fa = fma3(hk.z, kv, fa);
  }
  // ---- membranes, last (the hinge pass is over, few values are live): t1 = (a,b,c) from a;
  //      t2 = (b,a,d) from b
  {
    const float4 m1 = ec[E], m2 = ec[2 * E];
    F3 t1b, t1c, t2a, t2d;
    membrane<KIND, HARD>(eab, eac, m1.x, m1.y, m1.z, m1.w, m3.x, P, t1b, t1c, en);
    membrane<KIND, HARD>(eba, ebd, m2.x, m2.y, m2.z, m2.w, m3.y, P, t2a, t2d, en);
    fa = fa + (t2a - (t1b + t1c));
    fb = fb + (t1b - (t2a + t2d));
    fc = fc + t1c;
    fd = fd + t2d;
  }
  out4[0] = make_float4(fa.x, fa.y, fa.z, KIND == 3 ? en : 0.0f);
  out4[E] = make_float4(fb.x, fb.y, fb.z, 0.0f);
  out4[2 * E] = make_float4(fc.x, fc.y, fc.z, 0.0f);
  out4[3 * E] = make_float4(fd.x, fd.y, fd.z, 0.0f);
}

// grad V at a vertex = 1/6 sum over its fan of (r_i - z) x (r_i+1 - z); the first kRegList ring
// offsets come from registers, longer fans continue from the global list.
__device__ __forceinline__ F3 ring_gradient(const unsigned char* zc, F3 zv, int rcnt,
                                            uint32_t roff0, uint32_t roff1, uint32_t roff2,
                                            const DevParams& P, int v) {
  const uint32_t roff[kRegList / 2] = {roff0, roff1, roff2};
  const F3 e0 = lds3(zc, roff[0] & 0xffffu) - zv;
  F3 ep = e0, g = {0.f, 0.f, 0.f};
#pragma unroll
  for (int i = 1; i < kRegList; ++i) {
    if (i < rcnt) {
      const F3 e = lds3(zc, (i & 1) ? (roff[i >> 1] >> 16) : (roff[i >> 1] & 0xffffu)) - zv;
      g = cross_acc(ep, e, g);
      ep = e;
    }
  }
  if (rcnt > kRegList) {
    const uint16_t* ring_tail = P.ring_off + P.ring_ptr[v];
    for (int i = kRegList; i < rcnt; ++i) {
      const F3 e = lds3(zc, ring_tail[i]) - zv;
      g = cross_acc(ep, e, g);
      ep = e;
    }
  }
  g = cross_acc(ep, e0, g);
  return (1.0f / 6.0f) * g;
}

// One run of operator blocks [b0, b1) of an output block row (a multiple of 4 blocks), software-
// pipelined in two stages of 4 blocks: the operator blocks stream from L2 (one float2 per lane
// and block, mma B-fragment order), the A fragments come by LDS.128 from the right-hand sides
// at the source block's byte offset.  FULL: 3xTF32 -- the block is split in registers (the
// tensor core ignores the low 13 mantissa bits) and the two correction terms go to a second
// accumulator (two dependency chains).  !FULL: blocks whose share of the row's l1 mass is below
// 2^-15 (npfem_plan.cpp): a single TF32 product is then exact to fp32 rounding of the row sum.
template <bool FULL>
__device__ __forceinline__ void block_run(float (&acc)[4], float (&accx)[4], const float2* tv,
                                          const uint16_t* __restrict__ blk_col, int b0, int b1,
                                          const unsigned char* Ahi, int lo_off, int lane) {
  tv += (size_t)b0 * 32;
  auto mma4 = [&](const float2 (&tb)[4], int colv, int jbase) {
#pragma unroll
    for (int u = 0; u < 4; ++u) {
      const int col = __shfl_sync(0xffffffffu, colv, jbase + u);
      const float4 ah = *reinterpret_cast<const float4*>(Ahi + col);
      const uint32_t ahi[4] = {__float_as_uint(ah.x), __float_as_uint(ah.y),
                               __float_as_uint(ah.z), __float_as_uint(ah.w)};
      if (FULL) {
        const float4 al = *reinterpret_cast<const float4*>(Ahi + col + lo_off);
        const uint32_t alo[4] = {__float_as_uint(al.x), __float_as_uint(al.y),
                                 __float_as_uint(al.z), __float_as_uint(al.w)};
        const uint32_t bx = __float_as_uint(tb[u].x) & 0xffffe000u;
        const uint32_t by = __float_as_uint(tb[u].y) & 0xffffe000u;
        const uint32_t bhi[2] = {bx, by};
        const uint32_t blo[2] = {__float_as_uint(tb[u].x - __uint_as_float(bx)),
                                 __float_as_uint(tb[u].y - __uint_as_float(by))};
        mma_tf32(accx, alo, bhi);
        mma_tf32(accx, ahi, blo);
        mma_tf32(acc, ahi, bhi);
      } else {
        const uint32_t braw[2] = {__float_as_uint(tb[u].x), __float_as_uint(tb[u].y)};
        mma_tf32(accx, ahi, braw);
      }
    }
  };
  for (int bb = b0; bb < b1; bb += 32) {
    const int nb = min(32, b1 - bb);          // multiple of 4 (runs are padded)
    const int colv = lane < nb ? (int)blk_col[bb + lane] * 512 : 0;   // byte offset of block jb
    float2 t0[4], t1[4];
#pragma unroll
    for (int u = 0; u < 4; ++u) { t0[u] = ldg_stream(tv + u * 32); t1[u] = t0[u]; }
    for (int jj = 0; jj < nb; jj += 8) {
      if (jj + 4 < nb) {
#pragma unroll
        for (int u = 0; u < 4; ++u) t1[u] = ldg_stream(tv + 128 + u * 32);
      }
      mma4(t0, colv, jj);
      tv += 256;
      if (jj + 4 < nb) {
        if (jj + 8 < nb) {
#pragma unroll
          for (int u = 0; u < 4; ++u) t0[u] = ldg_stream(tv + u * 32);
        }
        mma4(t1, colv, jj + 4);
      } else {
        tv -= 128;
      }
    }
  }
}

// global_mode 3: the products of one slot of a warp's operator stream (npfem_internal.h).  A pair
// = two source blocks = K = 16 of one mma.m16n8k16; the A fragment halves come from the right-hand
// sides in shared memory: source block kb sits at A + 512 kb, hi plane then (256 bytes further) lo
// plane, each 32 chunks of 8 bytes {col g, col g+8} x vertices (2t, 2t+1), chunk index
// (4 g + t) ^ 4 (kb & 7) (bank swizzle of the split pass), so a lane's address is lane8 ^ the
// descriptor's half word.  Three-product slot: hi*hi -> acc, lo*hi + hi*lo -> accx.
__device__ __forceinline__ uint2 lds64(const unsigned char* p) { return *reinterpret_cast<const uint2*>(p); }
__device__ __forceinline__ void slot_mma3(float (&acc)[4], float (&accx)[4], uint4 b, uint32_t w,
                                          const unsigned char* A, uint32_t lane8, int dbg = 0) {
  const unsigned char* A1 = A + ((w & 0xffffu) ^ lane8);
  const unsigned char* A2 = A + ((w >> 16) ^ lane8);
  uint2 h1, h2, l1, l2;
  if (NPFEM_DBG(2)) { h1 = make_uint2(w, lane8); h2 = h1; l1 = h1; l2 = h1; }
  else { h1 = lds64(A1); h2 = lds64(A2); l1 = lds64(A1 + 256); l2 = lds64(A2 + 256); }
  mma_f16(accx, l1.x, l1.y, l2.x, l2.y, b.x, b.y, dbg);
  mma_f16(accx, h1.x, h1.y, h2.x, h2.y, b.z, b.w, dbg);
  mma_f16(acc, h1.x, h1.y, h2.x, h2.y, b.x, b.y, dbg);
}
// One-product slot: two pairs, hi*hi each, one per accumulator chain.
__device__ __forceinline__ void slot_mma1(float (&acc)[4], float (&accx)[4], uint4 b, uint2 d,
                                          const unsigned char* A, uint32_t lane8, int dbg = 0) {
  uint2 h1, h2, h3, h4;
  if (NPFEM_DBG(2)) { h1 = make_uint2(d.x, lane8); h2 = h1; h3 = h1; h4 = h1; }
  else {
    h1 = lds64(A + ((d.x & 0xffffu) ^ lane8)); h2 = lds64(A + ((d.x >> 16) ^ lane8));
    h3 = lds64(A + ((d.y & 0xffffu) ^ lane8)); h4 = lds64(A + ((d.y >> 16) ^ lane8));
  }
  mma_f16(acc, h1.x, h1.y, h2.x, h2.y, b.x, b.y, dbg);
  mma_f16(accx, h3.x, h3.y, h4.x, h4.y, b.z, b.w, dbg);
}

}  // namespace
}  // namespace npfem
