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
//
// Work mapping per iteration and cell: thread e < E owns one ELEMENT (two triangles sharing an
// edge, npfem_internal.h; its constants are staged once in shared memory) and writes one float4
// per own vertex; thread v < n owns one VERTEX, gathers its element slots, evaluates grad V on
// its ring and forms the right-hand side; the global step then multiplies all 16 right-hand-side
// columns of the CTA by the block-sparse inverse on the tensor cores (3xTF32 split, fp32
// accumulate).  s, d, the elastic residual and u0, private to the owner thread, live in tensor
// memory (TMEM).
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
template <int KIND>
__device__ __forceinline__ void membrane(F3 e1, F3 e2, float i00, float i01, float i11, float ws,
                                         float wa, const DevParams& P, F3& f1, F3& f2) {
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
  float g1 = ws * (fminf(fmaxf(s1, P.s_min), P.s_max) - s1) * r1;
  float g2 = ws * (fminf(fmaxf(s2, P.s_min), P.s_max) - s2) * r2;
  const float astar = fminf(fmaxf(J, P.a_min), P.a_max);
  if (J != astar) {
    const float q = fsqrt(astar);
    const float p = hyperbola_p(s1, s2, q, s1 * r2, J);
    g1 = fmaf(wa, fmaf(q, p, -s1) * r1, g1);
    g2 = fmaf(wa, fmaf(q, frcp(p), -s2) * r2, g2);
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
template <int KIND>
__device__ __forceinline__ F3 hinge_vec(float Kq, float Ko, float Kf, float rp, F3 epq, F3 epo, F3 epf,
                                        float cbh) {
  const F3 kv = fma3(Kq, epq, fma3(Ko, epo, Kf * epf));
  if (KIND == 2) return cbh * kv;
  const float nk2 = fmaxf(dot(kv, kv), 1e-30f);
  const float cf = fmaf(rp, frsqrt(nk2), KIND == 1 ? -1.0f - cbh : -1.0f);
  return cf * kv;
}

__device__ __forceinline__ void mma_tf32(float (&c)[4], const uint32_t (&a)[4], const uint32_t (&b)[2]) {
  asm volatile(
      "mma.sync.aligned.m16n8k8.row.col.f32.tf32.tf32.f32 {%0,%1,%2,%3}, {%4,%5,%6,%7}, {%8,%9}, "
      "{%0,%1,%2,%3};"
      : "+f"(c[0]), "+f"(c[1]), "+f"(c[2]), "+f"(c[3])
      : "r"(a[0]), "r"(a[1]), "r"(a[2]), "r"(a[3]), "r"(b[0]), "r"(b[1]));
}

// Operator blocks stream from L2 once per use: keep them out of L1, which holds the register spills.
__device__ __forceinline__ float2 ldg_stream(const float2* p) {
  float2 v;
  asm volatile("ld.global.nc.L1::no_allocate.v2.f32 {%0, %1}, [%2];" : "=f"(v.x), "=f"(v.y) : "l"(p));
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
template <int KIND>
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
  const float4 m3 = ec[3 * E];
  // ---- shared hinge (a,b | c ; d): once in full for a diamond, the element's half for a single
  {
    const float4 hk = ec[4 * E];
    const float Kp = hk.x, Kq = hk.y, Ko = hk.z;
    const float Kf = -(Kp + Kq + Ko), he = m3.z, hf = fmaf(2.0f, he, -1.0f);
    const F3 kv = hinge_vec<KIND>(Kq, Ko, Kf, hk.w, eab, eac, ead, P.cbh);
    fa = fma3(he * Kp, kv, fa); fb = fma3(he * Kq, kv, fb);
    fc = fma3(Ko, kv, fc);      fd = fma3(hf * Kf, kv, fd);
  }
  // ---- outer hinges: half of the end-point terms, all of the own opposite vertex's term
  {   // (b,c | a ; f1)
    const float4 hk = ec[5 * E];
    const F3 zf = lds3(zc, id_f12 & 0xffffu);
    const F3 kv = hinge_vec<KIND>(hk.y, hk.z, -(hk.x + hk.y + hk.z), hk.w, ebc, eba, zf - zb, P.cbh);
    fb = fma3(0.5f * hk.x, kv, fb); fc = fma3(0.5f * hk.y, kv, fc); fa = fma3(hk.z, kv, fa);
  }
  {   // (c,a | b ; f2)
    const float4 hk = ec[6 * E];
    const F3 zf = lds3(zc, id_f12 >> 16);
    const F3 eca = {-eac.x, -eac.y, -eac.z}, ecb = {-ebc.x, -ebc.y, -ebc.z};
    const F3 kv = hinge_vec<KIND>(hk.y, hk.z, -(hk.x + hk.y + hk.z), hk.w, eca, ecb, zf - zc3, P.cbh);
    fc = fma3(0.5f * hk.x, kv, fc); fa = fma3(0.5f * hk.y, kv, fa); fb = fma3(hk.z, kv, fb);
  }
  {   // (a,d | b ; f3)
    const float4 hk = ec[7 * E];
    const F3 zf = lds3(zc, id_f34 & 0xffffu);
    const F3 kv = hinge_vec<KIND>(hk.y, hk.z, -(hk.x + hk.y + hk.z), hk.w, ead, eab, zf - za, P.cbh);
    fa = fma3(0.5f * hk.x, kv, fa); fd = fma3(0.5f * hk.y, kv, fd); fb = fma3(hk.z, kv, fb);
  }
  {   // (d,b | a ; f4)
    const float4 hk = ec[8 * E];
    const F3 zf = lds3(zc, id_f34 >> 16);
    const F3 edb = {-ebd.x, -ebd.y, -ebd.z}, eda = {-ead.x, -ead.y, -ead.z};
    const F3 kv = hinge_vec<KIND>(hk.y, hk.z, -(hk.x + hk.y + hk.z), hk.w, edb, eda, zf - zd, P.cbh);
    fd = fma3(0.5f * hk.x, kv, fd); fb = fma3(0.5f * hk.y, kv, fb); fa = fma3(hk.z, kv, fa);
  }
  // ---- membranes, last (the hinge pass is over, few values are live): t1 = (a,b,c) from a;
  //      t2 = (b,a,d) from b
  {
    const float4 m1 = ec[E], m2 = ec[2 * E];
    F3 t1b, t1c, t2a, t2d;
    membrane<KIND>(eab, eac, m1.x, m1.y, m1.z, m1.w, m3.x, P, t1b, t1c);
    membrane<KIND>(eba, ebd, m2.x, m2.y, m2.z, m2.w, m3.y, P, t2a, t2d);
    fa = fa + (t2a - (t1b + t1c));
    fb = fb + (t1b - (t2a + t2d));
    fc = fc + t1c;
    fd = fd + t2d;
  }
  out4[0] = make_float4(fa.x, fa.y, fa.z, 0.0f);
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

// ------------------------------------------------------------------------------------------
// The fused step kernel.  MODE 1: global step with fp32 FMAs (comparison path); MODE 2: 3xTF32
// mma.sync on the block-sparse inverse.
// ------------------------------------------------------------------------------------------
template <int MODE, int MAXT, bool DAMP>
__global__ void __launch_bounds__(MAXT, 1) npfem_step_kernel(const DevParams P) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  unsigned char* const z4b = smem_raw + P.L.z4;                        // [k][NP] float4 iterate z
  const float4* const ecs = reinterpret_cast<const float4*>(smem_raw + P.L.ec);   // element constants
  float* const ra = reinterpret_cast<float*>(smem_raw + P.L.ra);       // rhs, A-fragment order (fp32 / hi)
  unsigned char* const rab = smem_raw + P.L.ra;                        // element results (odd cells) / rhs hi
  unsigned char* const rbb = smem_raw + P.L.rb;                        // element results (even cells) / rhs lo / delta d
  float* const rb = reinterpret_cast<float*>(rbb);
  float4* const red = reinterpret_cast<float4*>(smem_raw + P.L.red);   // [5][32] partial sums
  __shared__ uint32_t tmem_base_s;

  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5, nwarps = blockDim.x >> 5;
  const int n = P.n, E = P.E, nvb = P.nvb, NP = nvb * 8;
  const int cell0 = blockIdx.x * P.k;
  const int kact = min(P.k, P.n_cells - cell0);
  const int cellz = NP * 16;                      // bytes of one cell's z4

  // ---- tensor memory: 64 columns per group of 4 warps (s: 0..14, d: 16..30, rhs: 32..47, u0: 48..62);
  //      with damping 16 more (64..78: the part of the damping force that is constant over a step)
  constexpr uint32_t kTmemGroup = DAMP ? 80u : 64u;
  uint32_t tmem_cols = 64;
  while (tmem_cols < kTmemGroup * ((nwarps + 3) >> 2)) tmem_cols <<= 1;
  if (warp == 0) {
    const uint32_t sa = (uint32_t)__cvta_generic_to_shared(&tmem_base_s);
    asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" :: "r"(sa), "r"(tmem_cols) : "memory");
    asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
  }

  // ---- per-thread constants of the vertex role
  const bool is_e = tid < E, isv = tid < n, isvp = tid < NP;
  const int v = isvp ? tid : 0;
  const float h = P.h;
  // float index of (vertex v, rhs column 0) in the A-fragment layout:
  //   block jb = v/8 holds 32 lanes x float4; lane = (m&7)*4 + (v&3), component = 2*((v&7)>>2) + (m>>3)
  const int fbase = ((v >> 3) * 32 + (v & 3)) * 4 + 2 * ((v & 7) >> 2);

  // ---- stage the element constants; zero what padding vertices / missing cells never write
  for (int i = tid; i < kElemGroups * E; i += blockDim.x)
    reinterpret_cast<float4*>(smem_raw + P.L.ec)[i] = P.elem_c[i];
  for (int i = tid; i < NP * 16; i += blockDim.x) ra[i] = 0.0f;
  for (int i = tid; i < P.k * NP; i += blockDim.x)
    reinterpret_cast<float4*>(z4b)[i] = make_float4(0.f, 0.f, 0.f, 0.f);

  asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
  __syncthreads();
  asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
  const uint32_t ta = tmem_base_s + ((uint32_t)(32 * (warp & 3)) << 16) + (uint32_t)((warp >> 2) * kTmemGroup);

  // ---- prologue: stage each cell's pos / vel / fext rows through shared memory with coalesced
  //      loads, hand every vertex to its owner thread, centroid, local coordinates, prediction
  const int vext3 = 3 * (int)P.perm[v];
  {
    const float h2m = P.h2_over_m[v];
    float* const st = rb;                    // [3][3n] staging (the element buffer is idle)
    const int n3 = 3 * n;
    float xr[16], ur[16], sreg[16], zero16[16];
#pragma unroll
    for (int i = 0; i < 16; ++i) { xr[i] = 0.f; ur[i] = 0.f; sreg[i] = 0.f; zero16[i] = 0.f; }
#pragma unroll
    for (int c = 0; c < kMaxCellsPerCta; ++c) {
      if (c < kact) {
        const size_t g = (size_t)(cell0 + c) * P.cell_stride;
        for (int i = tid; i < n3; i += blockDim.x) {
          st[i] = P.pos[g + i]; st[n3 + i] = P.vel[g + i]; st[2 * n3 + i] = P.fext[g + i];
        }
        __syncthreads();
        float sx = 0.f, sy = 0.f, sz = 0.f;
        if (isv) {
#pragma unroll
          for (int q = 0; q < 3; ++q) {
            xr[3 * c + q] = st[vext3 + q];
            ur[3 * c + q] = fmaf(h, st[n3 + vext3 + q], h2m * st[2 * n3 + vext3 + q]);
          }
          sx = xr[3 * c]; sy = xr[3 * c + 1]; sz = xr[3 * c + 2];
        }
        sx = warp_sum(sx); sy = warp_sum(sy); sz = warp_sum(sz);
        if (lane == 0) red[c * 32 + warp] = make_float4(sx, sy, sz, 0.f);
        __syncthreads();   // staging is reused by the next cell; partial sums complete
      }
    }
#pragma unroll
    for (int c = 0; c < kMaxCellsPerCta; ++c) {
      if (c < kact) {
        const float4 p4 = lane < nwarps ? red[c * 32 + lane] : make_float4(0.f, 0.f, 0.f, 0.f);
        const float invn = 1.0f / (float)n;
        const float cx = warp_sum(p4.x) * invn, cy = warp_sum(p4.y) * invn, cz = warp_sum(p4.z) * invn;
        if (isv) {
          const float sx = (xr[3 * c] - cx) + ur[3 * c];
          const float sy = (xr[3 * c + 1] - cy) + ur[3 * c + 1];
          const float sz = (xr[3 * c + 2] - cz) + ur[3 * c + 2];
          sreg[3 * c] = sx; sreg[3 * c + 1] = sy; sreg[3 * c + 2] = sz;
          reinterpret_cast<float4*>(z4b)[c * NP + v] = make_float4(sx, sy, sz, 0.f);
        }
      }
    }
    tmem_st16(ta, sreg);
    tmem_st16(ta + 16, zero16);
    tmem_st16(ta + 32, zero16);
    tmem_st16(ta + 48, ur);
    __syncthreads();
    if (DAMP) {
      // Rayleigh damping, implicit (reading A-20): the damping force -(C/h)(x - x_n),
      // C = c_alpha M + c_beta L_el, with x - x_n = u0 + d and L_el (u0 + d) = L_el z - L_el y:
      //   -(c_alpha/h) m d      -> folded into the diagonal m (1/h^2 + c_alpha/h) of the residual
      //   -(c_beta/h) L_el z    -> folded into the element pass (a shift of the membrane factors and
      //                            of the hinge factor)
      //   Q = (c_beta/h) L_el y - (c_alpha/h) m u0   -> constant over the step: formed here, once,
      //                            by one pass of the linear operator over y, and parked in TMEM.
      float qreg[16];
#pragma unroll
      for (int i = 0; i < 16; ++i) qreg[i] = 0.f;
      const float dm = P.damp_m[v];
      if (P.cbh != 0.0f) {
        const uint4 vr0q = P.vrole[2 * v];
        const int icnt = vr0q.w & 0xff;
#pragma unroll
        for (int c = 0; c < kMaxCellsPerCta; ++c) {
          if (c < kact) {
            float4* z4c = reinterpret_cast<float4*>(z4b) + c * NP;
            if (isv) z4c[v] = make_float4(sreg[3 * c] - ur[3 * c], sreg[3 * c + 1] - ur[3 * c + 1],
                                          sreg[3 * c + 2] - ur[3 * c + 2], 0.f);        // y = s - u0
            __syncthreads();
            if (tid < E)
              element_residual<2>(ecs + tid, E, z4b + c * cellz, P, reinterpret_cast<float4*>(rbb) + tid);
            __syncthreads();
            if (isv) {
              F3 q = {0.f, 0.f, 0.f};
              const uint32_t ioff[kRegList / 2] = {vr0q.x, vr0q.y, vr0q.z};
#pragma unroll
              for (int i = 0; i < kRegList; ++i)
                if (i < icnt) q = q + lds3(rbb, (i & 1) ? (ioff[i >> 1] >> 16) : (ioff[i >> 1] & 0xffffu));
              if (icnt > kRegList) {
                const uint16_t* inc_tail = P.inc_off + P.inc_ptr[v];
                for (int i = kRegList; i < icnt; ++i) q = q + lds3(rbb, inc_tail[i]);
              }
              qreg[3 * c] = q.x; qreg[3 * c + 1] = q.y; qreg[3 * c + 2] = q.z;
              z4c[v] = make_float4(sreg[3 * c], sreg[3 * c + 1], sreg[3 * c + 2], 0.f);   // back to z = s
            }
            __syncthreads();
          }
        }
      }
#pragma unroll
      for (int i = 0; i < 15; ++i) qreg[i] = fmaf(-dm, ur[i], qreg[i]);
      tmem_st16(ta + 64, qreg);
    }
  }

  // ---- iterations
  const float vol_tol = kVolTol * P.V0;
  const float vol_dlen = kVolDTol * cbrtf(P.V0);
  const float vol_dtol2 = (float)n * vol_dlen * vol_dlen;
  const bool use_vol = P.w_volume > 0.0f;
  const float4* const ec_t = ecs + (is_e ? tid : 0);
  for (int it = 0; it < P.n_iters; ++it) {
    // local step.  Pipeline over the CTA's cells, one barrier per cell:
    //   [elements(0) -> out B; volume gradient(0), partial sums] |
    //   [vertices(c): gather out(c), volume multiplier, residual -> TMEM; elements(c+1) -> the other
    //    out buffer; volume gradient(c+1), partial sums] | ...
    // The volume gradient only reads z, so every warp runs its share right after its elements:
    // warps that finish the element pass early keep working instead of waiting at the barrier.
    // Vertex-role constants (npfem_api.cu: vrole) are fetched just before they are needed instead
    // of living in registers across the element pass: [0] = element-slot offsets 0..5 (3 words) +
    // counts, [1] = ring offsets 0..5 (3 words) + m/h^2.
    F3 g = {0.f, 0.f, 0.f}, zv = {0.f, 0.f, 0.f};
    uint4 vr0;
    // element results alternate between two buffers (rb, and ra, which is idle until the split),
    // so the vertex phase of cell c and the element pass of cell c+1 share one barrier interval
    auto elements_and_gradient = [&](int cc) {
      const unsigned char* zcc = z4b + cc * cellz;
      if (is_e) element_residual<DAMP ? 1 : 0>(ec_t, E, zcc, P, reinterpret_cast<float4*>((cc & 1) ? rab : rbb) + tid);
      vr0 = P.vrole[2 * v];
      if (use_vol) {
        float S1 = 0.f, S2 = 0.f;
        if (isv) {
          const uint4 vr1 = P.vrole[2 * v + 1];
          zv = lds3(zcc, v * 16);
          g = ring_gradient(zcc, zv, (vr0.w >> 8) & 0xff, vr1.x, vr1.y, vr1.z, P, v);
          S1 = dot(zv, g);
          S2 = dot(g, g);
        }
        S1 = warp_sum(S1); S2 = warp_sum(S2);
        if (lane == 0) red[cc * 32 + warp] = make_float4(S1, S2, 0.f, 0.f);
      }
    };
    elements_and_gradient(0);
    __syncthreads();
    for (int c = 0; c < kact; ++c) {
      const unsigned char* zc = z4b + c * cellz;
      const unsigned char* outb = (c & 1) ? rab : rbb;
      const int icnt = vr0.w & 0xff, rcnt = (vr0.w >> 8) & 0xff;
      F3 ev = {0.f, 0.f, 0.f};
      float S1, S2;
      if (isv) {
        const uint32_t ioff[kRegList / 2] = {vr0.x, vr0.y, vr0.z};
#pragma unroll
        for (int i = 0; i < kRegList; ++i) {
          if (i < icnt) {
            const F3 o = lds3(outb, (i & 1) ? (ioff[i >> 1] >> 16) : (ioff[i >> 1] & 0xffffu));
            ev = ev + o;
          }
        }
        if (icnt > kRegList) {
          const uint16_t* inc_tail = P.inc_off + P.inc_ptr[v];
          for (int i = kRegList; i < icnt; ++i) ev = ev + lds3(outb, inc_tail[i]);
        }
      }

      // finish(c): D = lambda grad V(z + D), iterated (D <- ((g.D - C)/(g.g)) g,
      // V = 1/3 sum_v z_v . g_v for the closed surface)
      F3 D = {0.f, 0.f, 0.f};
      if (use_vol) {
        float4 p4 = lane < nwarps ? red[c * 32 + lane] : make_float4(0.f, 0.f, 0.f, 0.f);
        S1 = warp_sum(p4.x); S2 = warp_sum(p4.y);
        const float V = S1 * (1.0f / 3.0f);
        const float vstar = fminf(fmaxf(V, P.Vmin), P.Vmax);
        float C = V - vstar;
        const bool active = (V != vstar);
        float lambda = (active && S2 > 0.f) ? -C / S2 : 0.f;
        D = lambda * g;
        bool moved = false;
        // Another pass only while it can still matter: after the first, first-order correction the
        // remaining error is second order in the violation (kVolTol); later, when the last pass
        // moved D by less than vol_dtol (rms per vertex).  |D_j+1 - D_j|^2 follows from the sums
        // already reduced: |D_j+1|^2 + |D_j|^2 - 2 lambda_j+1 (g_j+1 . D_j).
        bool more = fabsf(C) > vol_tol;
        float D2prev = lambda * lambda * S2;
        for (int pass = 1; pass < P.vol_iters && active && more; ++pass) {
          // CTA-uniform branch: every warp reduced the same partial sums in the same order
          float4* z4c = reinterpret_cast<float4*>(z4b + c * cellz);
          const F3 zz = zv + D;
          if (isv) z4c[v] = make_float4(zz.x, zz.y, zz.z, 0.f);
          moved = true;
          __syncthreads();
          float S3 = 0.f;
          S1 = 0.f; S2 = 0.f;
          if (isv) {
            const uint4 vr1 = P.vrole[2 * v + 1];
            g = ring_gradient(zc, zz, rcnt, vr1.x, vr1.y, vr1.z, P, v);
            S1 = dot(zz, g); S2 = dot(g, g); S3 = dot(g, D);
          }
          S1 = warp_sum(S1); S2 = warp_sum(S2); S3 = warp_sum(S3);
          if (lane == 0) red[c * 32 + warp] = make_float4(S1, S2, S3, 0.f);
          __syncthreads();
          p4 = lane < nwarps ? red[c * 32 + lane] : make_float4(0.f, 0.f, 0.f, 0.f);
          S1 = warp_sum(p4.x); S2 = warp_sum(p4.y); S3 = warp_sum(p4.z);
          C = S1 * (1.0f / 3.0f) - vstar;
          lambda = S2 > 0.f ? (S3 - C) / S2 : 0.f;
          D = lambda * g;
          const float D2new = lambda * lambda * S2;
          more = (D2new + D2prev - 2.0f * lambda * S3) > vol_dtol2;
          D2prev = D2new;
          __syncthreads();   // red[c] is rewritten by the next pass
        }
        if (moved && isv) reinterpret_cast<float4*>(z4b + c * cellz)[v] = make_float4(zv.x, zv.y, zv.z, 0.f);
      }
      // elastic residual of the cell's vertices, e = sum of element results + w_vol D, parked in
      // the owner's TMEM columns 32 + 3c .. (the fourth column written belongs to the next cell,
      // which overwrites it later in this same pass)
      tmem_st4(ta + 32 + 3 * c, fmaf(P.w_volume, D.x, ev.x), fmaf(P.w_volume, D.y, ev.y),
               fmaf(P.w_volume, D.z, ev.z), 0.0f);
      if (c + 1 < kact) elements_and_gradient(c + 1);
      __syncthreads();   // out(c) consumed; out(c+1) and the partial sums of cell c+1 complete
    }

    // right-hand sides of the global step, r = e - (m/h^2) d, split into tf32 high and low parts and
    // written in mma A-fragment order (hi -> ra, lo -> rb; both element buffers are dead now).
    // Round-to-nearest on the 13 dropped mantissa bits; lo = x - hi is exact.
    {
      float ee[16], dd[16];
      tmem_ld16(ta + 32, ee);
      if (DAMP) {
        tmem_ld16(ta + 64, dd);
#pragma unroll
        for (int m = 0; m < 15; ++m) ee[m] += dd[m];
      }
      tmem_ld16(ta + 16, dd);
      const float nmh2 = -__uint_as_float(P.vrole[2 * v + 1].w);
      if (isvp) {
#pragma unroll
        for (int m = 0; m < kRhs; ++m) {
          const int idx = fbase + (m & 7) * 16 + (m >> 3);
          const float x = m < 15 ? fmaf(nmh2, dd[m], ee[m]) : 0.0f;
          const float hi = __uint_as_float((__float_as_uint(x) + 0x1000u) & 0xffffe000u);
          ra[idx] = hi;
          rb[idx] = x - hi;
        }
      }
    }
    __syncthreads();

    // global step: delta d = T r with T = A_sys^-1 in 8x8 blocks.  One warp per block row of 8
    // output vertices (up to 4 rows per warp): mma m16n8k8, M = the 16 right-hand-side columns,
    // N = 8 output vertices, K = 8 source vertices per operator block (block_run above).
    const int g8 = lane >> 2, t4 = lane & 3;
    float acc[4][4];
#pragma unroll
    for (int j = 0; j < 4; ++j) {
      acc[j][0] = acc[j][1] = acc[j][2] = acc[j][3] = 0.f;
      const int ib = warp + j * nwarps;
      if (ib < nvb) {
        const int b0 = P.blk_ptr[3 * ib], bm = P.blk_ptr[3 * ib + 1], b1 = P.blk_ptr[3 * ib + 2];
        if (MODE == 2) {
          const unsigned char* const Ahi = reinterpret_cast<const unsigned char*>(ra) + lane * 16;
          const float2* const tv = reinterpret_cast<const float2*>(P.blk_val) + lane;
          float accx[4] = {0.f, 0.f, 0.f, 0.f};
          block_run<true>(acc[j], accx, tv, P.blk_col, b0, bm, Ahi, P.L.rb - P.L.ra, lane);
          block_run<false>(acc[j], accx, tv, P.blk_col, bm, b1, Ahi, 0, lane);
#pragma unroll
          for (int q = 0; q < 4; ++q) acc[j][q] += accx[q];
        } else {
          // fp32 comparison path: the same sums with plain FMAs, operands re-read per term
          for (int b = b0; b < b1; ++b) {
            const int col = (int)P.blk_col[b] * 32;
            const float* hi = ra + col * 4;
            const float* lo = rb + col * 4;
            const float* tb = P.blk_val + (size_t)b * 64;
#pragma unroll
            for (int kk = 0; kk < 8; ++kk) {
              // A(m, kk) sits in lane (m&7)*4 + (kk&3), component 2*(kk>>2) + (m>>3)
              const int ia = (g8 * 4 + (kk & 3)) * 4 + 2 * (kk >> 2);
              const float a0 = hi[ia] + lo[ia], a1 = hi[ia + 1] + lo[ia + 1];
              // B(kk, i) sits at 2*((i<<2) | (kk&3)) + (kk>>2)
              const float bq0 = __ldg(tb + 2 * (((2 * t4) << 2) | (kk & 3)) + (kk >> 2));
              const float bq1 = __ldg(tb + 2 * (((2 * t4 + 1) << 2) | (kk & 3)) + (kk >> 2));
              acc[j][0] = fmaf(a0, bq0, acc[j][0]); acc[j][1] = fmaf(a0, bq1, acc[j][1]);
              acc[j][2] = fmaf(a1, bq0, acc[j][2]); acc[j][3] = fmaf(a1, bq1, acc[j][3]);
            }
          }
        }
      }
    }
    __syncthreads();   // every warp is done reading the right-hand sides

    // hand the increments to the vertex owners: dd[m][NP] over the dead lo buffer
#pragma unroll
    for (int j = 0; j < 4; ++j) {
      const int ib = warp + j * nwarps;
      if (ib < nvb) {
        const int i0 = ib * 8 + 2 * t4;
        *reinterpret_cast<float2*>(rb + g8 * NP + i0) = make_float2(acc[j][0], acc[j][1]);
        if (g8 < 7) *reinterpret_cast<float2*>(rb + (g8 + 8) * NP + i0) = make_float2(acc[j][2], acc[j][3]);
      }
    }
    __syncthreads();

    // owner update: d += delta d, z = s + d
    {
      float sv[16], dv[16];
      tmem_ld16(ta, sv);
      tmem_ld16(ta + 16, dv);
#pragma unroll
      for (int m = 0; m < 15; ++m) dv[m] += rb[m * NP + v];
      if (isvp) {
#pragma unroll
        for (int c = 0; c < kMaxCellsPerCta; ++c)
          if (c < P.k)
            reinterpret_cast<float4*>(z4b)[c * NP + v] =
                make_float4(sv[3 * c] + dv[3 * c], sv[3 * c + 1] + dv[3 * c + 1], sv[3 * c + 2] + dv[3 * c + 2], 0.f);
      }
      tmem_st16(ta + 16, dv);
    }
    __syncthreads();
  }

  // ---- epilogue: x_n+1 = x_n + (u0 + d), v_n+1 = (u0 + d)/h, staged in caller order through
  //      shared memory so that the loads of x_n and the stores to pos / vel are coalesced
  {
    float dv[16], ur[16];
    tmem_ld16(ta + 16, dv);
    tmem_ld16(ta + 48, ur);
    float* const st = rb;                    // [2][3n]
    const int n3 = 3 * n;
    const float invh = 1.0f / h;
#pragma unroll
    for (int c = 0; c < kMaxCellsPerCta; ++c) {
      if (c < kact) {
        const size_t g = (size_t)(cell0 + c) * P.cell_stride;
        for (int i = tid; i < n3; i += blockDim.x) st[i] = P.pos[g + i];
        __syncthreads();
        if (isv) {
#pragma unroll
          for (int q = 0; q < 3; ++q) {
            const float inc = ur[3 * c + q] + dv[3 * c + q];
            st[vext3 + q] += inc;
            st[n3 + vext3 + q] = inc * invh;
          }
        }
        __syncthreads();
        for (int i = tid; i < n3; i += blockDim.x) { P.pos[g + i] = st[i]; P.vel[g + i] = st[n3 + i]; }
        __syncthreads();
      }
    }
  }
  asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
  __syncthreads();
  if (warp == 0)
    asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" :: "r"(tmem_base_s), "r"(tmem_cols) : "memory");
}

}  // namespace

cudaError_t configure_kernels(int smem_bytes) {
  cudaError_t e;
  (void)smem_bytes;
  smem_bytes = kSmemMaxDynamic;   // opt in once to the largest carve-out any cell type may need
#define NPFEM_CFG(MODE, MAXT, DAMP)                                                             \
  e = cudaFuncSetAttribute(npfem_step_kernel<MODE, MAXT, DAMP>,                                 \
                           cudaFuncAttributeMaxDynamicSharedMemorySize, smem_bytes);            \
  if (e != cudaSuccess) return e;
  NPFEM_CFG(1, 672, false) NPFEM_CFG(1, 1024, false) NPFEM_CFG(2, 672, false) NPFEM_CFG(2, 1024, false)
  NPFEM_CFG(1, 672, true) NPFEM_CFG(1, 1024, true) NPFEM_CFG(2, 672, true) NPFEM_CFG(2, 1024, true)
#undef NPFEM_CFG
  return cudaSuccess;
}

cudaError_t launch_step(const DevParams& p, int threads, int smem_bytes, int mode,
                        cudaStream_t stream) {
  if (p.n_cells <= 0) return cudaSuccess;
  const int grid = (p.n_cells + p.k - 1) / p.k;
#define NPFEM_LAUNCH(MODE, MAXT)                                                                \
  do {                                                                                          \
    if (p.damped) npfem_step_kernel<MODE, MAXT, true><<<grid, threads, smem_bytes, stream>>>(p); \
    else npfem_step_kernel<MODE, MAXT, false><<<grid, threads, smem_bytes, stream>>>(p);        \
  } while (0)
  if (threads <= 672) {
    if (mode == 2) NPFEM_LAUNCH(2, 672); else NPFEM_LAUNCH(1, 672);
  } else {
    if (mode == 2) NPFEM_LAUNCH(2, 1024); else NPFEM_LAUNCH(1, 1024);
  }
#undef NPFEM_LAUNCH
  return cudaGetLastError();
}

}  // namespace npfem
