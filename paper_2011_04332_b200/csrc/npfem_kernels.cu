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
#include <cstring>

#include <cuda_fp16.h>

#include "npfem_device.cuh"

namespace npfem {
namespace {

// Debug option `debug_jitter` (npfem_options): every warp sleeps a pseudo-random time after every
// CTA barrier, so that warps cross each phase at very different times.  A missing barrier between
// a phase that writes a shared buffer and one that reads it then changes the result, while a
// correctly synchronised kernel stays bit-identical (tests/test_edge_cases_gpu.py) -- the stand-in
// for compute-sanitizer racecheck, which is closed on this pool.
__device__ __forceinline__ void jitter_sleep(int seed, int phase, int warp) {
  unsigned hsh = ((unsigned)seed * 2654435761u) ^ ((unsigned)phase * 40503u) ^ ((unsigned)warp * 9176u + blockIdx.x * 7u);
  hsh ^= hsh >> 13; hsh *= 0x5bd1e995u; hsh ^= hsh >> 15;
  __nanosleep(hsh & 2047u);
}
// Diagnostic build (-DNPFEM_PHASE_CLOCKS, never the shipped library): thread 0 of every CTA adds the
// clock64() ticks between marks to g_phase[] (one slot per phase of an iteration), read back with
// npfem_debug_phase_clocks (profiles/ quotes these as "phase clocks").
#ifdef NPFEM_PHASE_CLOCKS
__device__ unsigned long long g_phase[16];
#define NPFEM_PHASE(i)                                                          \
  do {                                                                          \
    if (tid == 0) {                                                             \
      const long long t_now = clock64();                                        \
      atomicAdd(&g_phase[i], (unsigned long long)(t_now - t_phase));            \
      t_phase = t_now;                                                          \
    }                                                                           \
  } while (0)
#define NPFEM_PDBG(bit) (P.dbg & (bit))
#else
#define NPFEM_PHASE(i) do { } while (0)
#define NPFEM_PDBG(bit) 0
#endif
#ifndef NPFEM_OP_DEPTH
#define NPFEM_OP_DEPTH 4
#endif
constexpr int kOpDepth = NPFEM_OP_DEPTH;   // slots of the operator stream a warp loads per batch (MODE 3)

#define NPFEM_SYNC()                                                    \
  do {                                                                  \
    __syncthreads();                                                    \
    if (OPT && P.jitter) jitter_sleep(P.jitter, ++jphase, warp);        \
  } while (0)

// ------------------------------------------------------------------------------------------
// The fused step kernel.  MODE 1: global step with fp32 FMAs (comparison path); MODE 2: 3xTF32
// mma.sync on the block-sparse inverse.
// ------------------------------------------------------------------------------------------
// FEAT 0: the lean kernel of the headline path; FEAT 1: damping (compile-time) plus the run-time
// options; FEAT 2: undamped with the run-time options (collision neighbours, strain hardening,
// debug_jitter).
template <int MODE, int MAXT, int FEAT>
__global__ void __launch_bounds__(MAXT, 1) npfem_step_kernel(const DevParams P) {
  constexpr bool DAMP = FEAT == 1, OPT = FEAT != 0;
  extern __shared__ __align__(16) unsigned char smem_raw[];
  unsigned char* const z4b = smem_raw + P.L.z4;                        // [k][NP] float4 iterate z
  const float4* const ecs = reinterpret_cast<const float4*>(smem_raw + P.L.ec);   // element constants
  float* const ra = reinterpret_cast<float*>(smem_raw + P.L.ra);       // rhs, A-fragment order (fp32 / hi)
  unsigned char* const rab = smem_raw + P.L.ra;                        // element results (odd cells) / rhs hi
  unsigned char* const rbb = smem_raw + P.L.rb;                        // element results (even cells) / rhs lo / delta d
  float* const rb = reinterpret_cast<float*>(rbb);
  float4* const red = reinterpret_cast<float4*>(smem_raw + P.L.red);   // [5][32] partial sums
  // MODE 3: bits of max |r| per cell (the right-hand sides are scaled into the fp16 range per cell)
  uint32_t* const smax = reinterpret_cast<uint32_t*>(smem_raw + P.L.red + kMaxCellsPerCta * 33 * 16);
  __shared__ uint32_t tmem_base_s;

  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5, nwarps = blockDim.x >> 5;
  int jphase = 0;   // barrier counter of the schedule-jitter debug option
#ifdef NPFEM_PHASE_CLOCKS
  long long t_phase = clock64();
#endif
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
  if (tid < 8) smax[tid] = 0u;

  asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
  NPFEM_SYNC();
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
        NPFEM_SYNC();
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
        NPFEM_SYNC();   // staging is reused by the next cell; partial sums complete
      }
    }
#pragma unroll
    for (int c = 0; c < kMaxCellsPerCta; ++c) {
      if (c < kact) {
        const float4 p4 = lane < nwarps ? red[c * 32 + lane] : make_float4(0.f, 0.f, 0.f, 0.f);
        const float invn = 1.0f / (float)n;
        const float cx = warp_sum(p4.x) * invn, cy = warp_sum(p4.y) * invn, cz = warp_sum(p4.z) * invn;
        if (OPT && tid == 0) red[kMaxCellsPerCta * 32 + c] = make_float4(cx, cy, cz, 0.f);   // kept for the collision planes
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
    NPFEM_SYNC();
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
            NPFEM_SYNC();
            if (tid < E)
              element_residual<2>(ecs + tid, E, z4b + c * cellz, P, reinterpret_cast<float4*>(rbb) + tid);
            NPFEM_SYNC();
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
            NPFEM_SYNC();
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
  const float nmh2 = -__uint_as_float(P.vrole[2 * v + 1].w);   // -(m/h^2) (with damping: -m (1/h^2 + c_alpha/h))
  NPFEM_PHASE(0);   // prologue
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
    if (MODE == 3 && tid < kMaxCellsPerCta) smax[tid] = 0u;   // read last by the owner update, before its barrier
    // element results alternate between two buffers (rb, and ra, which is idle until the split),
    // so the vertex phase of cell c and the element pass of cell c+1 share one barrier interval
    auto elements_and_gradient = [&](int cc) {
      const unsigned char* zcc = z4b + cc * cellz;
      if (is_e) element_residual<DAMP ? 1 : 0, OPT>(ec_t, E, zcc, P, reinterpret_cast<float4*>((cc & 1) ? rab : rbb) + tid);
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
    NPFEM_SYNC();
    NPFEM_PHASE(1);   // element pass + volume gradient of the first cell
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
          NPFEM_SYNC();
          float S3 = 0.f;
          S1 = 0.f; S2 = 0.f;
          if (isv) {
            const uint4 vr1 = P.vrole[2 * v + 1];
            g = ring_gradient(zc, zz, rcnt, vr1.x, vr1.y, vr1.z, P, v);
            S1 = dot(zz, g); S2 = dot(g, g); S3 = dot(g, D);
          }
          S1 = warp_sum(S1); S2 = warp_sum(S2); S3 = warp_sum(S3);
          if (lane == 0) red[c * 32 + warp] = make_float4(S1, S2, S3, 0.f);
          NPFEM_SYNC();
          p4 = lane < nwarps ? red[c * 32 + lane] : make_float4(0.f, 0.f, 0.f, 0.f);
          S1 = warp_sum(p4.x); S2 = warp_sum(p4.y); S3 = warp_sum(p4.z);
          C = S1 * (1.0f / 3.0f) - vstar;
          lambda = S2 > 0.f ? (S3 - C) / S2 : 0.f;
          D = lambda * g;
          const float D2new = lambda * lambda * S2;
          more = (D2new + D2prev - 2.0f * lambda * S3) > vol_dtol2;
          D2prev = D2new;
          NPFEM_SYNC();   // red[c] is rewritten by the next pass
        }
        if (moved && isv) reinterpret_cast<float4*>(z4b + c * cellz)[v] = make_float4(zv.x, zv.y, zv.z, 0.f);
      }
      // colliding neighbour of this vertex (reading A-22): the half space (x - q).n >= d, residual
      // w_c max(d - (z - q).n, 0) n; q arrives in world coordinates, the iterate is cell-local
      if (OPT && P.coll_n != nullptr && isv) {
        const size_t gq = (size_t)(cell0 + c) * P.cell_stride + vext3;
        const F3 nn = {P.coll_n[gq], P.coll_n[gq + 1], P.coll_n[gq + 2]};
        if (nn.x != 0.f || nn.y != 0.f || nn.z != 0.f) {
          const float4 cen = red[kMaxCellsPerCta * 32 + c];
          const F3 ql = {P.coll_q[gq] - cen.x, P.coll_q[gq + 1] - cen.y, P.coll_q[gq + 2] - cen.z};
          const F3 zc3 = lds3(zc, v * 16);
          const float t = P.d_coll - dot(zc3 - ql, nn);
          if (t > 0.f) ev = fma3(P.w_coll * t, nn, ev);
        }
      }
      // right-hand side of the global step for the cell's vertices, r = e - (m/h^2) d with the
      // elastic residual e = sum of element results + w_vol D, parked in the owner's TMEM columns
      // 32 + 3c .. (the fourth column written belongs to the next cell, which overwrites it later
      // in this same pass)
      {
        float d0, d1, d2, d3;
        tmem_ld4(ta + 16 + 3 * c, d0, d1, d2, d3);
        float rx = fmaf(nmh2, d0, fmaf(P.w_volume, D.x, ev.x));
        float ry = fmaf(nmh2, d1, fmaf(P.w_volume, D.y, ev.y));
        float rz = fmaf(nmh2, d2, fmaf(P.w_volume, D.z, ev.z));
        if (DAMP) {
          tmem_ld4(ta + 64 + 3 * c, d0, d1, d2, d3);
          rx += d0; ry += d1; rz += d2;
        }
        tmem_st4(ta + 32 + 3 * c, rx, ry, rz, 0.0f);
        if (MODE == 3) {   // max |r| of the cell: the fp16 split below scales by a power of two
          uint32_t mb = __float_as_uint(fmaxf(fmaxf(fabsf(rx), fabsf(ry)), fabsf(rz)));
          mb = __reduce_max_sync(0xffffffffu, mb);
          if (lane == 0) atomicMax(&smax[c], mb);
        }
      }
      if (c + 1 < kact) elements_and_gradient(c + 1);
      NPFEM_SYNC();   // out(c) consumed; out(c+1) and the partial sums of cell c+1 complete
    }

    NPFEM_PHASE(2);   // vertex phase(c) + element pass(c+1), one barrier per cell
    // right-hand sides of the global step: r, split into a high and a low part and written in mma
    // A-fragment order (both element buffers are dead now).
    // MODE 1/2: tf32 hi -> ra, lo -> rb; round-to-nearest on the 13 dropped mantissa bits, lo = x - hi
    // is exact.  MODE 3: scaled by the cell's 2^k so that max |r| lands in [2^13, 2^14), then
    // hi = fp16(x), lo = fp16(x - hi) (x to 2^-24 relative), both into ra: source block kb holds a hi
    // plane and, 256 bytes further, a lo plane of 32 chunks of 8 bytes {col g, col g+8}, each word
    // the vertices 2t, 2t+1 of the block; chunk index (4 g + t) ^ 4 (kb & 7): the xor keeps the
    // 16-bit stores of a warp (4 source blocks x 4 t) on distinct banks.
    {
      float rr[16];
      tmem_ld16(ta + 32, rr);
      if (MODE == 3) {
        if (isvp && !NPFEM_PDBG(32)) {
          float sc[kMaxCellsPerCta];
#pragma unroll
          for (int c = 0; c < kMaxCellsPerCta; ++c) {
            const uint32_t ec_ = min(max(smax[c] >> 23, 14u), 254u);
            sc[c] = __uint_as_float((267u - ec_) << 23);
          }
          const uint32_t sw = ((uint32_t)(v >> 3) & 7u) * 32u;
          unsigned char* const wb = rab + (v >> 3) * 512 + ((v & 7) >> 1) * 8 + (v & 1) * 2;
#pragma unroll
          for (int m = 0; m < kRhs; ++m) {
            const float x = m < 15 ? rr[m] * sc[m / 3] : 0.0f;
            const __half hi = __float2half_rn(x);
            const __half lo = __float2half_rn(x - __half2float(hi));
            unsigned char* const w = wb + (((uint32_t)(m & 7) * 32u) ^ sw) + (m >> 3) * 4;
            *reinterpret_cast<__half*>(w) = hi;
            *reinterpret_cast<__half*>(w + 256) = lo;
          }
        }
      } else if (isvp) {
#pragma unroll
        for (int m = 0; m < kRhs; ++m) {
          const int idx = fbase + (m & 7) * 16 + (m >> 3);
          const float x = m < 15 ? rr[m] : 0.0f;
          const float hi = __uint_as_float((__float_as_uint(x) + 0x1000u) & 0xffffe000u);
          ra[idx] = hi;
          rb[idx] = x - hi;
        }
      }
    }
    NPFEM_SYNC();

    NPFEM_PHASE(3);   // split + barrier
    // global step: delta d = T r with T = A_sys^-1 in 8x8 blocks.  One warp per block row of 8
    // output vertices (up to 4 rows per warp): mma m16n8k8, M = the 16 right-hand-side columns,
    // N = 8 output vertices, K = 8 source vertices per operator block (block_run above).
    int tid_p = tid;
    asm volatile("" : "+r"(tid_p));   // everything the product derives from the thread index is formed here, per
                                      // iteration, instead of being hoisted and kept live across the element pass
    const int lane_p = tid_p & 31, warp_p = tid_p >> 5;
    const int g8 = lane_p >> 2, t4 = lane_p & 3;
    if constexpr (MODE == 3) {
      // the warp's operator stream: slots of 512 bytes of B fragments, consumed in order.  The
      // stream has the same shape for every warp (per row slot j: hs_na[j] three-product slots,
      // then hs_nb[j] one-product slots), so every branch below is uniform; the slot descriptors
      // (<= 64 slots per warp) sit in four registers, lane l holding those of slots l and l + 32,
      // and are broadcast by shuffle; a finished block row goes straight to the owners' hand-off
      // buffer (rb is not read in this phase)
      const int Q = NPFEM_PDBG(16) ? 0 : P.hs_slots;
      const uint4* const vp = P.hs_val + (size_t)warp_p * Q * 32 + lane_p;
      // (x, y) slot lane, (z, w) slot lane + 32.  The identity shuffles re-home the four words from
      // the load's scoreboard to registers no pending load guards: ptxas otherwise makes every
      // later read of them wait for the newest stream loads as well (measured: the whole L2
      // latency per slot).
      uint4 dreg = __ldg(P.hs_desc + warp_p * 32 + lane_p);
      dreg.x = __shfl_sync(0xffffffffu, dreg.x, lane_p); dreg.y = __shfl_sync(0xffffffffu, dreg.y, lane_p);
      dreg.z = __shfl_sync(0xffffffffu, dreg.z, lane_p); dreg.w = __shfl_sync(0xffffffffu, dreg.w, lane_p);
      const uint32_t lane8 = (uint32_t)lane_p * 8u;
      // Batches of kOpDepth slots: all loads of a batch are issued back to back, then the batch is
      // consumed.  No load is in flight while a warp computes -- deliberately: ptxas guards every
      // register a load wrote with a scoreboard that later loads re-use, so that in a software-
      // pipelined ring the consumer of the OLDEST load also waits for the newest (measured: one
      // whole L2 latency per slot, whatever the depth).  The latency of a batch is covered by the
      // other warps of the sub-partition, which sit in other batches.  (Measured in isolation: the
      // loop is bound by the SM's load/store data path, which the 512-byte stream loads (5.8 cycles
      // each) and the 256-byte right-hand-side loads (2 cycles each) share; starting the warps of a
      // sub-partition staggered changed nothing.)
      {
        float acc[4] = {0.f, 0.f, 0.f, 0.f}, accx[4] = {0.f, 0.f, 0.f, 0.f};
        int j = 0, qa_end = P.hs_na[0], q_end = P.hs_na[0] + P.hs_nb[0];
        for (int q = 0; q < Q; q += kOpDepth) {
          uint4 rv[kOpDepth];
#pragma unroll
          for (int u = 0; u < kOpDepth; ++u) {
            // the zero is never consumed (same guard below), but without it ptxas takes rv[] for
            // live from the kernel's entry ("maybe uninitialised") and the ELEMENT PASS spills:
            // 40 bytes of spill stores at kOpDepth 4, 0 with this line
            rv[u] = make_uint4(0u, 0u, 0u, 0u);
            if (q + u < Q) rv[u] = ldg_stream(vp + (q + u) * 32);
          }
#pragma unroll
          for (int u = 0; u < kOpDepth; ++u) {
            if (q + u < Q) {
              uint2 d;
              d.x = __shfl_sync(0xffffffffu, q + u < 32 ? dreg.x : dreg.z, (q + u) & 31);
              d.y = q + u < qa_end ? 0u : __shfl_sync(0xffffffffu, q + u < 32 ? dreg.y : dreg.w, (q + u) & 31);
              if (q + u < qa_end) slot_mma3(acc, accx, rv[u], d.x, rab, lane8, NPFEM_PDBG(0xff));
              else slot_mma1(acc, accx, rv[u], d, rab, lane8, NPFEM_PDBG(0xff));
              if (q + u + 1 == q_end) {
                const int ib = P.hs_rows[j * 32 + warp_p];
                if (ib != 255) {
                  const int i0 = ib * 8 + 2 * t4;
                  *reinterpret_cast<float2*>(rb + g8 * NP + i0) = make_float2(acc[0] + accx[0], acc[1] + accx[1]);
                  if (g8 < 7)
                    *reinterpret_cast<float2*>(rb + (g8 + 8) * NP + i0) = make_float2(acc[2] + accx[2], acc[3] + accx[3]);
                }
#pragma unroll
                for (int x = 0; x < 4; ++x) { acc[x] = 0.f; accx[x] = 0.f; }
                ++j;
                if (j < 4) { qa_end = q_end + P.hs_na[j]; q_end = qa_end + P.hs_nb[j]; }
              }
            }
          }
        }
      }
      NPFEM_PHASE(4);   // operator product, warp 0's own rows
    } else {
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
    NPFEM_PHASE(4);   // operator product, warp 0's own rows
    NPFEM_SYNC();   // every warp is done reading the right-hand sides

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
    }
    NPFEM_SYNC();
    NPFEM_PHASE(5);   // hand-off + wait for the slowest warp of the product
    // owner update: d += delta d, z = s + d
    {
      float sv[16], dv[16];
      tmem_ld16(ta, sv);
      tmem_ld16(ta + 16, dv);
      if (MODE == 3) {   // undo the scaling of the operator row (2^-k_v) and of the cell's right-hand sides
        const float hs = NPFEM_PDBG(0xff) ? 0.0f : P.hp_scale[v];   // ablation runs leave d alone
        float fac[kMaxCellsPerCta];
#pragma unroll
        for (int c = 0; c < kMaxCellsPerCta; ++c) {
          const uint32_t ec_ = min(max(smax[c] >> 23, 14u), 254u);
          fac[c] = hs * __uint_as_float((ec_ - 13u) << 23);
        }
#pragma unroll
        for (int m = 0; m < 15; ++m) dv[m] = fmaf(rb[m * NP + v], fac[m / 3], dv[m]);
      } else {
#pragma unroll
        for (int m = 0; m < 15; ++m) dv[m] += rb[m * NP + v];
      }
      if (isvp) {
#pragma unroll
        for (int c = 0; c < kMaxCellsPerCta; ++c)
          if (c < P.k)
            reinterpret_cast<float4*>(z4b)[c * NP + v] =
                make_float4(sv[3 * c] + dv[3 * c], sv[3 * c + 1] + dv[3 * c + 1], sv[3 * c + 2] + dv[3 * c + 2], 0.f);
      }
      tmem_st16(ta + 16, dv);
    }
    NPFEM_SYNC();
    NPFEM_PHASE(6);   // owner update
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
        NPFEM_SYNC();
        if (isv) {
#pragma unroll
          for (int q = 0; q < 3; ++q) {
            const float inc = ur[3 * c + q] + dv[3 * c + q];
            st[vext3 + q] += inc;
            st[n3 + vext3 + q] = inc * invh;
          }
        }
        NPFEM_SYNC();
        for (int i = tid; i < n3; i += blockDim.x) { P.pos[g + i] = st[i]; P.vel[g + i] = st[n3 + i]; }
        NPFEM_SYNC();
      }
    }
  }
  asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
  NPFEM_SYNC();
  if (warp == 0)
    asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" :: "r"(tmem_base_s), "r"(tmem_cols) : "memory");
}

// Area per surface vertex (the IBM needs it): a_v = 1/3 of the areas of the triangles
// around v = 1/6 sum over the fan of |(r_i - x_v) x (r_i+1 - x_v)|.  One CTA per cell, thread =
// vertex (internal numbering: ring lists), positions straight from global memory.
__global__ void npfem_area_kernel(const DevParams P, float* __restrict__ areas) {
  const int v = threadIdx.x, cell = blockIdx.x;
  if (v >= P.n) return;
  const float* x = P.pos + (size_t)cell * P.cell_stride;
  auto at = [&](int internal) { const int e = 3 * (int)P.perm[internal]; return F3{x[e], x[e + 1], x[e + 2]}; };
  const F3 xv = at(v);
  const int r0 = P.ring_ptr[v], r1 = P.ring_ptr[v + 1];
  const F3 e0 = at(P.ring_off[r0] >> 4) - xv;
  F3 ep = e0;
  float a = 0.f;
  for (int i = r0 + 1; i <= r1; ++i) {
    const F3 e = i < r1 ? at(P.ring_off[i] >> 4) - xv : e0;
    const F3 cr = cross_acc(ep, e, F3{0.f, 0.f, 0.f});
    a += sqrtf(dot(cr, cr));
    ep = e;
  }
  areas[(size_t)cell * P.n + P.perm[v]] = a * (1.0f / 6.0f);
}

}  // namespace

cudaError_t launch_vertex_areas(const DevParams& p, int threads, float* areas, cudaStream_t stream) {
  if (p.n_cells <= 0) return cudaSuccess;
  npfem_area_kernel<<<p.n_cells, threads, 0, stream>>>(p, areas);
  return cudaGetLastError();
}

#ifdef NPFEM_PHASE_CLOCKS
static int g_dbg_host = 0;
#endif
cudaError_t read_phase_clocks(unsigned long long* out16, int reset) {
#ifdef NPFEM_PHASE_CLOCKS
  if (reset >= 0x100) {   // diagnostic: set the ablation mask of the operator product (low byte)
    g_dbg_host = reset & 0xff;
    return cudaSuccess;
  }
  cudaError_t e = cudaMemcpyFromSymbol(out16, g_phase, sizeof(unsigned long long) * 16);
  if (e != cudaSuccess) return e;
  if (reset) {
    unsigned long long zero[16] = {};
    e = cudaMemcpyToSymbol(g_phase, zero, sizeof(zero));
  }
  return e;
#else
  (void)out16; (void)reset;
  return cudaErrorNotSupported;
#endif
}

cudaError_t configure_kernels(int smem_bytes) {
  cudaError_t e;
  (void)smem_bytes;
  smem_bytes = kSmemMaxDynamic;   // opt in once to the largest carve-out any cell type may need
#define NPFEM_CFG(MODE, MAXT, FEAT)                                                             \
  e = cudaFuncSetAttribute(npfem_step_kernel<MODE, MAXT, FEAT>,                                 \
                           cudaFuncAttributeMaxDynamicSharedMemorySize, smem_bytes);            \
  if (e != cudaSuccess) return e;
  NPFEM_CFG(1, 672, 0) NPFEM_CFG(1, 1024, 0) NPFEM_CFG(2, 672, 0) NPFEM_CFG(2, 1024, 0)
  NPFEM_CFG(1, 672, 1) NPFEM_CFG(1, 1024, 1) NPFEM_CFG(2, 672, 1) NPFEM_CFG(2, 1024, 1)
  NPFEM_CFG(1, 672, 2) NPFEM_CFG(1, 1024, 2) NPFEM_CFG(2, 672, 2) NPFEM_CFG(2, 1024, 2)
  NPFEM_CFG(3, 672, 0) NPFEM_CFG(3, 1024, 0) NPFEM_CFG(3, 672, 1) NPFEM_CFG(3, 1024, 1)
  NPFEM_CFG(3, 672, 2) NPFEM_CFG(3, 1024, 2)
#undef NPFEM_CFG
  return cudaSuccess;
}

cudaError_t launch_step(const DevParams& p_in, int threads, int smem_bytes, int mode,
                        cudaStream_t stream) {
  if (p_in.n_cells <= 0) return cudaSuccess;
#ifdef NPFEM_PHASE_CLOCKS
  DevParams p = p_in;
  p.dbg = g_dbg_host;
#else
  const DevParams& p = p_in;
#endif
  const int grid = (p.n_cells + p.k - 1) / p.k;
  const int feat = p.damped ? 1 : (p.coll_n != nullptr || p.jitter != 0 || p.hard != 0.0f) ? 2 : 0;
#define NPFEM_LAUNCH(MODE, MAXT)                                                                  \
  do {                                                                                            \
    if (feat == 1) npfem_step_kernel<MODE, MAXT, 1><<<grid, threads, smem_bytes, stream>>>(p);    \
    else if (feat == 2) npfem_step_kernel<MODE, MAXT, 2><<<grid, threads, smem_bytes, stream>>>(p); \
    else npfem_step_kernel<MODE, MAXT, 0><<<grid, threads, smem_bytes, stream>>>(p);              \
  } while (0)
  if (threads <= 672) {
    if (mode == 3) NPFEM_LAUNCH(3, 672); else if (mode == 2) NPFEM_LAUNCH(2, 672); else NPFEM_LAUNCH(1, 672);
  } else {
    if (mode == 3) NPFEM_LAUNCH(3, 1024); else if (mode == 2) NPFEM_LAUNCH(2, 1024); else NPFEM_LAUNCH(1, 1024);
  }
#undef NPFEM_LAUNCH
  return cudaGetLastError();
}

}  // namespace npfem
