/*
 * npfem.h -- C ABI of the B200-native npFEM solid-phase hot path.
 *
 * What the library computes: one nodal projective-FEM time step for many deformable blood cells
 * of ONE type at once (same surface-mesh topology, rest shape, material, time step).  The step is
 * the one BASELINE.json's north_star names and PAPER.md describes in words only:
 *   - PAPER.md:56-60 (Introduction, eq. 2)  elastodynamics of each body, Newton's 2nd law;
 *   - PAPER.md:66, :70                      "mass-lumped linear FE solver" on triangular surface
 *                                           meshes, implicit time integration;
 *   - PAPER.md:90-95 (Implementation)       projective dynamics (ShapeOp lineage), time stepping
 *                                           after Liu et al.: alternate a LOCAL step (project every
 *                                           elemental constraint) and a GLOBAL step (solve the
 *                                           prefactored SPD system shared by all cells of a type);
 *   - PAPER.md:181                          the energy of a body is a sum of per-element energies,
 *                                           each with a weight and parameters;
 *   - PAPER.md:103, :159-163                what crosses the boundary every step (forces in,
 *                                           positions + velocities out) and the precedent of a
 *                                           dynamic library driven through ctypes.
 * The energies themselves (triangle strain, triangle area, bending hinge, cell volume), the
 * weights and every other point the paper leaves open are the readings A-1..A-16 of DESIGN.md.
 *
 * Conventions
 *   - every function returns NPFEM_OK (0) or a negative error code; no exception crosses the ABI;
 *     npfem_last_error() returns a thread-local, statically stored message for the last failure;
 *   - "host" / "device" on each pointer says where the memory lives;
 *   - units: any consistent system (the harness uses um, us, pg => force nN);
 *   - vertex order is the CALLER's; the library never renumbers what the caller sees (its internal
 *     fill/locality permutation is private);
 *   - npfem_step is asynchronous on the given CUDA stream and allocates nothing.
 */
#ifndef NPFEM_H_
#define NPFEM_H_

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define NPFEM_OK 0
#define NPFEM_EINVAL (-1) /* bad argument, non-closed / inconsistently oriented mesh, V0 <= 0,    */
                          /* degenerate rest triangle, band with min > max, negative damping      */
#define NPFEM_ENOMEM (-2) /* host allocation failed                                               */
#define NPFEM_ECUDA (-3)  /* a CUDA call failed (message holds the CUDA error string)             */
#define NPFEM_ELIMIT (-4) /* mesh larger than one CTA can hold (n_verts > 1024 or shared memory;   */
                          /* with damping: more than 768 threads per cell)                         */

typedef struct npfem_handle_s* npfem_handle; /* opaque; one per cell TYPE */
typedef struct npfem_plan_s* npfem_plan;     /* opaque; host-only create-time data (no CUDA)      */

/* Material of one cell type (A-2..A-5, A-12).  All doubles, caller's unit system.      */
typedef struct {
  double cell_mass;              /* total mass, lumped to vertices by rest-area share */
  double k_strain, s_min, s_max; /* triangle strain weight per rest area; singular-value band       */
  double k_area, a_min, a_max;   /* triangle area weight per rest area; band on sigma1*sigma2       */
  double k_bend;                 /* hinge weight, multiplies 3/(A0+A1)                              */
  double w_volume, v_min, v_max; /* per-cell volume weight; band on V/V0                            */
  double c_alpha, c_beta;        /* viscoelastic damping (PAPER.md:60, :145, :183 Calpha / Cbeta),   */
                                 /* >= 0: implicit Rayleigh damping f_d = -(c_alpha M + c_beta L_el) */
                                 /* v_{n+1}, L_el = the strain + area + bending stiffness (A-20);    */
                                 /* c_alpha in 1/time, c_beta in time                                */
  double w_collision;            /* collision weight per vertex (PAPER.md:145 collisions_weight), >= 0; */
  double d_collision;            /* contact distance >= 0: a vertex with a colliding neighbour (q, n)   */
                                 /* is kept at (x - q).n >= d_collision (reading A-22); both 0 = off   */
  double strain_hardening;       /* beta >= 0: strain-dependent strain weight k_strain (1 + beta d^2),  */
                                 /* d = clamp(sigma) - sigma (reading A-23: "a weight */
                                 /* and various parameters ... stiffer or softer"); 0 = constant weight */
  double w_garea, ga_min, ga_max; /* global-area term (reading A-24): weight and band on the total      */
                                 /* surface area A/A0.  Implemented in the ORACLE only (its closest-   */
                                 /* point projection needs a Newton solve with the dense area Hessian); */
                                 /* npfem_create rejects w_garea != 0 with NPFEM_EINVAL                 */
} npfem_material;

/* Tuning knobs that do not change what is computed beyond fp32 rounding.  Pass NULL for defaults. */
typedef struct {
  double inv_drop_tol;    /* entries of A_sys^-1 are dropped, smallest first, while the dropped     */
                          /* l1 mass of a row stays <= inv_drop_tol * ||row||_1.  Default 2^-24     */
                          /* (below fp32 rounding of the kept sum); < 0 = that default;             */
                          /* 0 = keep everything (dense operator).                                  */
  int volume_inner_iters; /* cap on the passes of the volume projection per local step (>= 1,      */
                          /* <= 32); default 8.  The pass loop is adaptive: a pass is skipped once  */
                          /* it cannot change the result at fp32 resolution (A-17), so    */
                          /* near-rest cells take one pass whatever the cap                         */
  int cells_per_cta;      /* 1..5 cells share one CTA and every fetched operator block; 0 = auto   */
  int global_mode;        /* 0 = auto (3 where it applies, else 2), 1 = fp32 SIMT blocks,           */
                          /* 2 = 3xTF32 tensor-core blocks, 3 = two-term fp16 split (hi*hi + hi*lo  */
                          /* + lo*hi, fp32 accumulate; like 3xTF32 exact to fp32 rounding) on       */
                          /* mma.m16n8k16, two blocks per product, per-warp operator streams        */
  int pair_triangles;     /* local-step work items: 0 = auto / 1 = pairs of triangles across a shared */
                          /* edge wherever the matching finds one, 2 = one triangle per item        */
  int debug_jitter;       /* 0 = off; otherwise a seed: every warp of the step kernel sleeps a      */
                          /* pseudo-random time (< 2 us) after every CTA barrier.  Results must be  */
                          /* bit-identical to debug_jitter = 0; a difference means a missing barrier */
                          /* (schedule-fuzz race check; costs time, never use it in production)     */
} npfem_options;

/*
 * npfem_create: build everything that depends only on the cell TYPE (rest
 * operators D_m^-1, rest areas, lumped masses, hinge rows K, rest volume, A_sys = M/h^2 +
 * sum w A^T A, its inverse in fp64, locality ordering, block-sparse fp32 operator) and upload it.
 *   n_verts, n_tris  mesh size; closed, consistently oriented 2-manifold (A-14); n_verts <= 1024
 *   tris             host, int32 [n_tris][3], vertex indices in the caller's numbering
 *   rest_xyz         host, double [n_verts][3]
 *   mat              host
 *   dt               time step h > 0
 *   cell_stride_floats  floats between consecutive cells in pos/vel/fext; >= 3*n_verts; 0 = the
 *                    default padded stride (3*n_verts rounded up to a multiple of 4)
 *   max_cells        upper bound on n_cells of any later npfem_step / npfem_step_host call; > 0:
 *                    the bound is enforced (NPFEM_EINVAL beyond it) and the streams and the
 *                    device staging ring of npfem_step_host are allocated now (3 stages x 3 fields
 *                    x min(max_cells, ~32 MB worth of cells)), so that no step entry point ever
 *                    allocates; 0: no bound, npfem_step_host sizes its ring on first use
 *   opts             host, may be NULL
 *   out              receives the handle; the handle owns all device memory it allocates
 * Errors: NPFEM_EINVAL, NPFEM_ENOMEM, NPFEM_ELIMIT, NPFEM_ECUDA (also when no CUDA device exists:
 * there is no CPU fallback).
 */
int npfem_create(int n_verts, int n_tris, const int32_t* tris, const double* rest_xyz,
                 const npfem_material* mat, double dt, int cell_stride_floats, int max_cells,
                 const npfem_options* opts, npfem_handle* out);

/*
 * npfem_step: advance n_cells cells of this type by ONE time step of n_iters local/global
 * iterations, entirely on the device (one kernel launch, no host round trip; north_star (d)).
 *   pos, vel  device, float, in/out, [n_cells][cell_stride]; inside a cell vertex-major xyz
 *             ([n_verts][3]); padding floats are neither read nor written
 *   fext      device, float, in, same layout: external force per vertex (the fluid/IBM forces of
 *             PAPER.md:103, generated inputs here)
 *   n_iters   >= 0 (0 = pure inertial prediction)
 *   cuda_stream  a cudaStream_t (NULL = default stream); the call only enqueues work
 * Result: x_{n+1} = x_n + inc, v_{n+1} = inc/h with inc = h v_n + h^2 f/m + d, d the projective-
 * dynamics correction after n_iters iterations; with c_alpha, c_beta != 0 the
 * iterations minimise the damped implicit-Euler objective (A-20).  Errors: NPFEM_EINVAL,
 * NPFEM_ECUDA (launch failure).
 */
int npfem_step(npfem_handle h, int n_cells, float* pos, float* vel, const float* fext,
               int n_iters, void* cuda_stream);

/*
 * npfem_step_collide: npfem_step with colliding neighbours (the coupling hands
 * "external forces & colliding neighbours" to the solid solver; :129-133 cell packing; :145
 * collisions_weight; reading A-22).  Per vertex at most one neighbour: a point q on the
 * other body and that body's outward unit normal n at q; the vertex is kept on the outer side,
 * (x - q).n >= d_collision, by a projective constraint of weight w_collision (both in the
 * material given to npfem_create; w_collision sits on the diagonal of A_sys for every vertex, so
 * contacts may come and go without touching the prefactored system).  Neighbour detection is the
 * caller's (the paper's framework does it outside npFEM); q and n are held fixed over the step.
 *   coll_q, coll_n  device, float, in, [n_cells][cell_stride], vertex-major xyz like pos;
 *                   n = (0,0,0) marks a vertex without neighbour
 * Everything else as npfem_step.
 */
int npfem_step_collide(npfem_handle h, int n_cells, float* pos, float* vel, const float* fext,
                       const float* coll_q, const float* coll_n, int n_iters, void* cuda_stream);

/*
 * npfem_vertex_areas: area per surface vertex at the given positions, a_v = 1/3 of the areas of the
 * triangles around v -- what the immersed-boundary coupling needs from the solid side
 * (PAPER.md:226).  One small kernel, asynchronous on the stream.
 *   pos     device, float, in, [n_cells][cell_stride]
 *   areas   device, float, out, [n_cells][n_verts] (caller's vertex order)
 */
int npfem_vertex_areas(npfem_handle h, int n_cells, const float* pos, float* areas, void* cuda_stream);

/*
 * npfem_step_converged: advance n_cells cells by ONE time step solved to convergence (PAPER.md:94-95
 * "redesigned projective dynamics approach as described in Liu et al. ... we provide a converged
 * solution"; :133 "unconditional stability for arbitrary time steps"; reading A-21): per
 * cell, L-BFGS (3 pairs) seeded with the prefactored A_sys^-1 and a backtracking line search on the
 * implicit-Euler objective g(x) = 1/2 ||x - s||^2_M/h^2 + E_el(x), until
 *     res = max_v || (h^2/m_v) grad g(x)_v ||_inf <= tol      (a length, caller's unit)
 * or max_iters iterations.  One kernel launch, one CTA per cell, the stop flag lives on the device.
 *   pos, vel, fext  device, as for npfem_step
 *   tol             >= 0; fp32 resolves about 1e-7 x the cell radius
 *   max_iters       >= 0
 *   iters_out       device, int32 [n_cells] or NULL: iterations each cell took
 *   res_out         device, float [n_cells] or NULL: final residual length of each cell
 *   cuda_stream     as for npfem_step
 * Errors: NPFEM_EINVAL (also: handle created with damping or collisions, not supported here yet),
 * NPFEM_ECUDA.
 */
int npfem_step_converged(npfem_handle h, int n_cells, float* pos, float* vel, const float* fext,
                         double tol, int max_iters, int32_t* iters_out, float* res_out,
                         void* cuda_stream);

/*
 * npfem_step_host: the same step with HOST buffers (pinned or pageable): cells are cut into
 * chunks that flow host->device, through the step kernel and device->host on three streams so
 * copies overlap compute.  Blocking: returns when pos/vel hold the new state (also on error: no
 * copy is left in flight).  Uses the device staging ring owned by the handle (allocated by
 * npfem_create when max_cells > 0, else on first use).
 *   pos, vel  host, float, in/out, [n_cells][cell_stride];  fext host, in
 * Bytes moved per call: 3 fields in, 2 fields out, n_cells*cell_stride*4 bytes each.
 */
int npfem_step_host(npfem_handle h, int n_cells, float* pos, float* vel, const float* fext,
                    int n_iters);

int npfem_destroy(npfem_handle h);

const char* npfem_last_error(void); /* thread-local, static storage; never NULL                   */
int npfem_cell_stride(npfem_handle h); /* floats per cell actually used                           */

/*
 * npfem_measure_fp32_peak: same-run measurement of the FP32 pipe rate that bounds the step kernel
 * (SURVEY.md 8(d) asks for a measured FMA peak beside the nominal one).
 * Runs a register-resident arithmetic loop on every SM of the current device and returns the best
 * of 4 timed launches (CUDA events) in TFLOP/s.  Blocking; allocates 4 bytes for its own use.
 *   variant  0 = FFMA (2 flop), 1 = packed FFMA2 (4 flop), 2 = FADD (1 flop),
 *            3 = FFMA and FADD alternating (1.5 flop per instruction on average)
 *   out_tflops  host, receives the rate.  Errors: NPFEM_EINVAL, NPFEM_ECUDA.
 */
int npfem_measure_fp32_peak(int variant, double* out_tflops);

/*
 * npfem_debug_phase_clocks: diagnostic builds only (nvcc -DNPFEM_PHASE_CLOCKS; the shipped library
 * returns NPFEM_EINVAL).  Copies 16 counters of clock64() ticks that thread 0 of every CTA of the
 * step kernel accumulates per phase of an iteration (0 prologue, 1 first element pass, 2 cell
 * pipeline, 3 right-hand-side split, 4 operator product, 5 hand-off, 6 owner update), summed over
 * CTAs and iterations since the last reset.  Blocking.
 *   out16  host, receives 16 counters;  reset  1..255: zero the counters after reading; >= 0x100:
 *          nothing is read, the low byte becomes the ablation mask of the global_mode-3 operator
 *          product for later launches (1 no mma, 2 no shared-memory operand loads, 16 skip the
 *          product loop, 32 skip the right-hand-side split; results are then meaningless)
 */
int npfem_debug_phase_clocks(unsigned long long* out16, int reset);

/* Introspection of a handle (all host-side, cheap): what the create step decided.               */
typedef struct {
  int n_verts, n_tris, n_hinges;
  int cell_stride;     /* floats */
  int cells_per_cta;   /* k */
  int threads_per_cta;
  int smem_bytes;      /* dynamic shared memory per CTA */
  int n_vblocks;       /* ceil(n_verts/8): operator is stored as 8x8 blocks */
  int n_op_blocks;     /* kept 8x8 blocks of A_sys^-1 */
  int op_nnz;          /* entries of A_sys^-1 kept by the drop rule (before blocking) */
  int global_mode;     /* 1 = SIMT, 2 = 3xTF32, 3 = two-term fp16 split */
  int volume_inner_iters;
  int n_op_blocks_tf32x1; /* of n_op_blocks, blocks applied as ONE TF32 product: their share of   */
                          /* every row's l1 mass is <= 2^-15, so the product error stays below   */
                          /* fp32 rounding of the row sum; all other blocks use 3xTF32            */
  int n_elements;         /* threads' work items of the local step: pairs of triangles sharing an  */
  int n_diamonds;         /* edge (n_diamonds of them) plus triangles left single by the matching  */
  int n_op_blocks_f16x1;  /* global_mode 3: of n_op_blocks, blocks applied as ONE fp16 product (hi   */
                          /* parts only): their share of every row's l1 mass is <= 2^-13            */
  int tmem_columns;       /* tensor-memory columns one CTA of the fixed-count step kernel allocates    */
                          /* (64 per 4 warps, 80 with damping, rounded up to a power of two)          */
  int ctas_per_sm;        /* resident CTAs per SM = min over shared memory (227 KB), tensor memory    */
  int ctas_per_sm_limiter; /* (512 columns) and threads (2048); limiter: 1 shared memory, 2 tensor     */
                          /* memory, 3 threads.  Small meshes (platelets) are limited by tensor       */
                          /* memory, not by the shared memory the plan sizes                          */
  double rest_volume, total_mass, inv_drop_tol;
} npfem_info;
int npfem_get_info(npfem_handle h, npfem_info* out);

/*
 * Host-only half of npfem_create (no CUDA call): used by the CPU tests to check the create-time
 * logic against the oracle, and by npfem_create itself.  npfem_plan_query copies create-time
 * arrays out; each `what` below states shape and type.  Returns the number of elements written,
 * or the number required when `dst` is NULL, or a negative error code.
 */
int npfem_plan_create(int n_verts, int n_tris, const int32_t* tris, const double* rest_xyz,
                      const npfem_material* mat, double dt, const npfem_options* opts,
                      npfem_plan* out);
int npfem_plan_destroy(npfem_plan p);
int npfem_plan_info(npfem_plan p, npfem_info* out);
#define NPFEM_Q_PERM 1        /* int32 [n_verts]: internal index -> caller vertex                 */
#define NPFEM_Q_MASS 2        /* double [n_verts]: lumped masses, caller order                     */
#define NPFEM_Q_SYSTEM 3      /* double [n_verts^2]: A_sys, caller order, row-major                */
#define NPFEM_Q_OPERATOR 4    /* double [n_verts^2]: the block-sparse fp32 operator expanded back  */
                              /* to a dense matrix in caller order (dropped entries = 0)           */
#define NPFEM_Q_HINGE_VERTS 5 /* int32 [n_hinges][4]: (x0,x1,x2,x3) in DESIGN.md's enumeration     */
#define NPFEM_Q_HINGE_K 6     /* double [n_hinges][4]: cotangent rows                              */
#define NPFEM_Q_HINGE_WR 7    /* double [n_hinges][2]: (w_h, r_h)                                  */
#define NPFEM_Q_TRI_DMINV 8   /* double [n_tris][3]: (i00, i01, i11) of D_m^-1                     */
#define NPFEM_Q_TRI_AREA 9    /* double [n_tris]                                                   */
#define NPFEM_Q_OPERATOR_X1 10 /* double [n_verts^2]: like NPFEM_Q_OPERATOR, only the blocks that are    */
                              /* applied as one TF32 product (npfem_info.n_op_blocks_tf32x1)       */
#define NPFEM_Q_OPERATOR_F16 11 /* double [n_verts^2]: the global_mode-3 operator (hi + lo fp16 parts,  */
                              /* row scaling undone) expanded to a dense matrix in caller order;   */
                              /* one-product blocks contribute their hi part only                  */
#define NPFEM_Q_OPERATOR_F16X1 12 /* double [n_verts^2]: only the blocks applied as one fp16 product */
#define NPFEM_Q_OPERATOR_STREAM 13 /* double [n_verts^2]: the same operator as NPFEM_Q_OPERATOR_F16, but  */
                              /* read back from the per-warp streams the kernel consumes (slot order,  */
                              /* descriptors, row table): every kept block exactly once                */
#define NPFEM_Q_STREAM_SHAPE 14 /* int32 [10]: warps, slots per warp, three-product slots of row slots  */
                              /* 0..3, one-product slots of row slots 0..3                             */
#define NPFEM_Q_STREAM_VAL 15  /* int32 [warps][slots][32 lanes][4]: the raw stream words (mma B         */
                              /* fragments: fp16 pairs) exactly as the kernel loads them               */
#define NPFEM_Q_STREAM_DESC 16 /* int32 [warps][32 lanes][4]: slot descriptors as the kernel loads them   */
#define NPFEM_Q_STREAM_ROWS 17 /* int32 [4][32]: output block row of (row slot, warp), 255 = none         */
#define NPFEM_Q_ROW_SCALE 18   /* double [n_verts]: 2^-k of each operator row's scaling, INTERNAL order   */
int npfem_plan_query(npfem_plan p, int what, void* dst, int dst_elems);

#ifdef __cplusplus
}
#endif
#endif /* NPFEM_H_ */
