/*
 * npfem_oracle.c -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * Plain, slow, fp64 CPU implementation of the npFEM nodal projective-FEM time step for closed
 * triangular surface meshes (red blood cells, platelets).  It is the parity oracle for the CUDA
 * library in paper_2011_04332_b200/ and shares no code with it.  Only tests/, bench.py's
 * cpu_baseline / --impl reference legs and __graft_entry__.smoke() may load it.
 *
 * What it follows
 * ---------------
 *  - PAPER.md:56-60 (Introduction, eq. 2): elastodynamics, Newton's 2nd law per body.
 *  - PAPER.md:66: "mass-lumped linear FE solver" on triangular surface meshes (:70), implicit.
 *  - PAPER.md:90-95: derived from ShapeOp / projective dynamics [3], time stepping after Liu et
 *    al. [11]; with no L-BFGS history and unit step length that scheme is the classic alternating
 *    local/global sweep implemented here (reading A-1).
 *  - PAPER.md:181: the body's potential energy is a sum of per-element energies, each with a weight
 *    and parameters.
 *  - BASELINE.json north_star: local step = projection of every triangle's strain, bending hinge
 *    and area/volume constraint; global step = solve (M/h^2 + sum w A^T A) x = rhs.
 *  - PAPER.md:60 ("with minor modifications of equation (2), one can readily simulate a
 *    viscoelastic material"), :145, :183 (parameters Calpha, Cbeta): Rayleigh damping
 *    f_d = -(c_alpha M + c_beta L_el) v, integrated implicitly (reading A-20).
 *  - PAPER.md:181-183 ("a weight and various parameters"): strain-dependent
 *    strain weight (reading A-23) and a global-area term, one constraint per cell on the total
 *    surface area (reading A-24; ORACLE ONLY, the CUDA library rejects it); both off by default.
 * The paper prints none of the energies; every formula below is a READING listed in DESIGN.md
 * (A-1 ... A-24).  Agreement with the real npFEM code is
 * "parity unpinned"; what IS pinned (tests/test_oracle_pins.py) are invariants, closed forms,
 * library routines and brute force.
 *
 * Formulation: ABSOLUTE positions, rhs b = M/h^2 s + sum w A^T p, dense Cholesky of A_sys.
 * (The CUDA path uses a different algebra: cell-local coordinates and an increment form.)
 * No blocking, no fusion, no reordering: one function per sentence of the algorithm.
 * OpenMP is used over cells only (one cell per thread, as the paper's CPU branch maps one cell
 * per core).
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define ORACLE_OK 0
#define ORACLE_EINVAL -1
#define ORACLE_ENOMEM -2

typedef struct {
  double cell_mass;
  double k_strain, s_min, s_max;
  double k_area, a_min, a_max;
  double k_bend;
  double w_volume, v_min, v_max;
  double c_alpha, c_beta;
  double w_collision, d_collision;   /* collision weight per vertex, contact distance (reading A-22) */
  double strain_hardening;           /* beta >= 0: strain-dependent weight w_s (1 + beta d^2) (reading A-23) */
  double w_garea, ga_min, ga_max;    /* global-area term: weight, band on A/A0 of the whole surface (reading A-24) */
} oracle_material;

typedef struct oracle_cell {
  int n, T, H;
  int32_t *tris;   /* [T][3] */
  double *X;       /* rest positions [n][3] */
  oracle_material mat;
  double h;
  double *G;       /* [T][2][3]: F^T = G [x_a; x_b; x_c] */
  double *area;    /* [T] rest areas A_t */
  double *mass;    /* [n] lumped masses */
  int32_t *hinge;  /* [H][4] stencils (x0,x1,x2,x3) */
  double *K;       /* [H][4] cotangent rows */
  double *w_h;     /* [H] hinge weights */
  double *r_h;     /* [H] rest magnitudes ||sum K_i X_i|| */
  double V0;       /* rest volume */
  double *Lel;     /* dense elastic Laplacian sum_t (w_s+w_a) G^T G + sum_h w_h K^T K [n][n] */
  double *A;       /* dense A_sys [n][n] */
  double *L;       /* dense lower Cholesky factor of A_sys [n][n] */
  double *LT;      /* its transpose, so that the backward substitution also reads rows */
} oracle_cell;

/* ---------------------------------------------------------------- small vector helpers */
static void sub3(const double *a, const double *b, double *o) { o[0]=a[0]-b[0]; o[1]=a[1]-b[1]; o[2]=a[2]-b[2]; }
static double dot3(const double *a, const double *b) { return a[0]*b[0]+a[1]*b[1]+a[2]*b[2]; }
static void cross3(const double *a, const double *b, double *o) {
  o[0]=a[1]*b[2]-a[2]*b[1]; o[1]=a[2]*b[0]-a[0]*b[2]; o[2]=a[0]*b[1]-a[1]*b[0];
}
static double norm3(const double *a) { return sqrt(dot3(a,a)); }
static double clampd(double v, double lo, double hi) { return v < lo ? lo : (v > hi ? hi : v); }

/* ---------------------------------------------------------------- geometry of the whole cell */
/* V(x) = 1/6 sum_t x_a . (x_b x x_c)   (SURVEY.md 8(c) create step 4) */
double oracle_volume(int T, const int32_t *tris, const double *x) {
  double V = 0.0;
  for (int t = 0; t < T; ++t) {
    const double *a = x + 3*tris[3*t], *b = x + 3*tris[3*t+1], *c = x + 3*tris[3*t+2];
    double bc[3]; cross3(b, c, bc);
    V += dot3(a, bc);
  }
  return V / 6.0;
}

/* (grad V)_a += 1/6 x_b x x_c (cyclic) per triangle   (volume) */
void oracle_volume_grad(int n, int T, const int32_t *tris, const double *x, double *g) {
  memset(g, 0, sizeof(double) * 3 * (size_t)n);
  for (int t = 0; t < T; ++t) {
    int ia = tris[3*t], ib = tris[3*t+1], ic = tris[3*t+2];
    const double *a = x + 3*ia, *b = x + 3*ib, *c = x + 3*ic;
    double bc[3], ca[3], ab[3];
    cross3(b, c, bc); cross3(c, a, ca); cross3(a, b, ab);
    for (int k = 0; k < 3; ++k) {
      g[3*ia+k] += bc[k] / 6.0;
      g[3*ib+k] += ca[k] / 6.0;
      g[3*ic+k] += ab[k] / 6.0;
    }
  }
}

/* ---------------------------------------------------------------- 3x2 thin SVD (one-sided Jacobi)
 * F (row-major 3x2) = U diag(S) V^T with U 3x2 (row-major), S[0] >= S[1] >= 0, V 2x2 (row-major).
 * For two columns one Hestenes rotation orthogonalises them exactly; it is repeated until the
 * columns are orthogonal to rounding.  Pinned against LAPACK (numpy.linalg.svd) in the tests. */
void oracle_svd32(const double *F, double *U, double *S, double *V) {
  double a[3] = {F[0], F[2], F[4]}, b[3] = {F[1], F[3], F[5]};
  double v00 = 1, v01 = 0, v10 = 0, v11 = 1;          /* V = I */
  for (int sweep = 0; sweep < 30; ++sweep) {
    double alpha = dot3(a,a), beta = dot3(b,b), gamma = dot3(a,b);
    if (fabs(gamma) <= 1e-300 || fabs(gamma) <= 1e-17 * sqrt(alpha*beta)) break;
    double zeta = (beta - alpha) / (2.0 * gamma);
    double t = (zeta >= 0 ? 1.0 : -1.0) / (fabs(zeta) + sqrt(1.0 + zeta*zeta));
    double c = 1.0 / sqrt(1.0 + t*t), s = c * t;
    for (int k = 0; k < 3; ++k) {
      double ak = a[k], bk = b[k];
      a[k] = c*ak - s*bk;
      b[k] = s*ak + c*bk;
    }
    double n00 = c*v00 - s*v01, n01 = s*v00 + c*v01;
    double n10 = c*v10 - s*v11, n11 = s*v10 + c*v11;
    v00 = n00; v01 = n01; v10 = n10; v11 = n11;
  }
  double s0 = norm3(a), s1 = norm3(b);
  if (s1 > s0) {                                       /* sort descending: swap columns */
    double tmp;
    for (int k = 0; k < 3; ++k) { tmp = a[k]; a[k] = b[k]; b[k] = tmp; }
    tmp = v00; v00 = v01; v01 = tmp;
    tmp = v10; v10 = v11; v11 = tmp;
    tmp = s0; s0 = s1; s1 = tmp;
  }
  double u0[3] = {0,0,0}, u1[3] = {0,0,0};
  if (s0 > 0) { for (int k = 0; k < 3; ++k) u0[k] = a[k] / s0; } else { u0[0] = 1; }
  if (s1 > 1e-300 && s1 > 1e-14 * s0) {
    for (int k = 0; k < 3; ++k) u1[k] = b[k] / s1;
  } else {
    /* collapsed triangle (A-9: several results are correct): any unit vector orthogonal to u0 */
    double e[3] = {0,0,0};
    int m = 0; if (fabs(u0[1]) < fabs(u0[m])) m = 1; if (fabs(u0[2]) < fabs(u0[m])) m = 2;
    e[m] = 1.0;
    double d = dot3(e, u0);
    for (int k = 0; k < 3; ++k) u1[k] = e[k] - d*u0[k];
    double nn = norm3(u1);
    for (int k = 0; k < 3; ++k) u1[k] /= nn;
  }
  for (int k = 0; k < 3; ++k) { U[2*k] = u0[k]; U[2*k+1] = u1[k]; }
  S[0] = s0; S[1] = s1;
  V[0] = v00; V[1] = v01; V[2] = v10; V[3] = v11;
}

/* P = U diag(d) V^T, row-major 3x2 */
static void compose32(const double *U, const double *d, const double *V, double *P) {
  for (int i = 0; i < 3; ++i)
    for (int j = 0; j < 2; ++j)
      P[2*i+j] = U[2*i]*d[0]*V[2*j] + U[2*i+1]*d[1]*V[2*j+1];
}

/* ---------------------------------------------------------------- local projections
 * strain: P_s = U diag(clamp(sigma_i,[s_min,s_max])) V^T */
void oracle_project_strain(const double *F, double s_min, double s_max, double *P) {
  double U[6], S[2], V[4], d[2];
  oracle_svd32(F, U, S, V);
  d[0] = clampd(S[0], s_min, s_max);
  d[1] = clampd(S[1], s_min, s_max);
  compose32(U, d, V, P);
}

/* Strain-dependent weight (NEXT-4, reading A-23; "every elemental potential energy
 * ... has a weight and various parameters", :183 "one can make the material stiffer or softer"):
 * with d_i = clamp(sigma_i) - sigma_i the strain energy density per singular value becomes
 *   psi(d) = 1/2 w_s (d^2 + 1/2 beta d^4),   psi'(d) = w_s d (1 + beta d^2),
 * i.e. the weight grows with the strain, w_s (1 + beta d^2) (hardening).  Following the
 * quasi-Newton view of projective dynamics (Liu et al.), the local step hands the global step the
 * EFFECTIVE target  P_eff = F + U diag(d_i (1 + beta d_i^2)) V^T,  so that w_s G^T (P_eff - F)
 * is the exact elastic force -dPsi/dx, while the system matrix keeps the constant weight w_s. */
void oracle_project_strain_hardening(const double *F, double s_min, double s_max, double beta, double *P) {
  double U[6], S[2], V[4], d[2];
  oracle_svd32(F, U, S, V);
  for (int i = 0; i < 2; ++i) {
    double di = clampd(S[i], s_min, s_max) - S[i];
    d[i] = S[i] + di * (1.0 + beta * di * di);
  }
  compose32(U, d, V, P);
}
/* strain energy of one triangle per unit weight: 1/2 sum_i (d_i^2 + 1/2 beta d_i^4) */
double oracle_strain_energy_density(const double *F, double s_min, double s_max, double beta) {
  double U[6], S[2], V[4], e = 0;
  oracle_svd32(F, U, S, V);
  for (int i = 0; i < 2; ++i) {
    double di = clampd(S[i], s_min, s_max) - S[i];
    e += 0.5 * (di*di + 0.5 * beta * di*di*di*di);
  }
  return e;
}

/* Closest point (o[0],o[1]) of the hyperbola branch {s1*s2 = a, s > 0} to (sg1,sg2), sg1 >= sg2.
 * Parametrise s = (q e^t, q e^-t), q = sqrt(a); phi(t) = (q e^t - sg1)^2 + (q e^-t - sg2)^2.
 * phi(t) <= phi(-t) for t >= 0 when sg1 >= sg2, so the global minimiser has t >= 0; there
 * phi'(0) = -2q(sg1-sg2) <= 0, phi' > 0 beyond t_hi, and phi' has a single sign change on
 * t >= 0 (the other normals from an interior point land on t < 0).  The root of phi' is found by
 * bracketed Newton (bisection whenever Newton leaves the bracket) to 1e-15.  The tests pin the
 * result against a brute-force scan of the whole branch (both signs of t).
 * (A-10: a tie sg1 == sg2 > 2q has two mirror minimisers; either is correct.) */
static double hyp_dphi(double t, double q, double s1, double s2) {
  double e = exp(t), ei = exp(-t);
  return e*(q*e - s1) - ei*(q*ei - s2);        /* phi'(t) / (2q) */
}
static double hyp_ddphi(double t, double q, double s1, double s2) {
  double e = exp(t), ei = exp(-t);
  return 2*q*e*e - s1*e + 2*q*ei*ei - s2*ei;   /* phi''(t) / (2q) */
}
void oracle_closest_on_hyperbola(double sg1, double sg2, double a, double *o) {
  double q = sqrt(a);
  double lo = 0.0, hi = log((sg1 > q ? sg1 : q) / q) + 1.0;   /* phi'(hi) > 0 */
  double t;
  if (hyp_dphi(lo, q, sg1, sg2) >= 0.0) {
    t = lo;                                     /* sg1 == sg2 <= 2q: minimiser at t = 0 ... */
    if (sg1 == sg2 && sg1 > 2.0*q) {            /* ... unless t = 0 is the local maximum (A-10) */
      double e = (sg1 + sqrt(sg1*sg1 - 4.0*q*q)) / (2.0*q);
      t = log(e);
    }
  } else {
    t = 0.5 * log((sg1 > 0 && sg2 > 0) ? sg1 / sg2 : 1.0);     /* same-ratio point as a start */
    if (!(t > lo && t < hi)) t = 0.5 * (lo + hi);
    for (int it = 0; it < 200; ++it) {
      double f = hyp_dphi(t, q, sg1, sg2);
      if (f == 0.0) break;
      if (f < 0.0) lo = t; else hi = t;
      double df = hyp_ddphi(t, q, sg1, sg2);
      double tn = (df > 0.0) ? t - f / df : lo - 1.0;
      if (!(tn > lo && tn < hi)) tn = 0.5 * (lo + hi);
      double step = fabs(tn - t);
      t = tn;
      if (step <= 1e-15 * (1.0 + fabs(t))) break;
    }
  }
  o[0] = q * exp(t); o[1] = q * exp(-t);
}

/* area: a* = clamp(s1 s2,[a_min,a_max]); P_a = F if s1 s2 == a*, else U diag(s') V^T with s' the
 * closest point of {s1 s2 = a*} to (sigma1, sigma2) */
void oracle_project_area(const double *F, double a_min, double a_max, double *P) {
  double U[6], S[2], V[4], d[2];
  oracle_svd32(F, U, S, V);
  double prod = S[0] * S[1];
  double astar = clampd(prod, a_min, a_max);
  if (prod == astar) { memcpy(P, F, 6 * sizeof(double)); return; }
  oracle_closest_on_hyperbola(S[0], S[1], astar, d);
  compose32(U, d, V, P);
}

/* bending: P_b = r k/||k||; if ||k|| < 1e-30, P_b = k (no force) */
void oracle_project_bend(const double *k, double r, double *P) {
  double nk = norm3(k);
  if (nk < 1e-30) { P[0] = k[0]; P[1] = k[1]; P[2] = k[2]; return; }
  for (int i = 0; i < 3; ++i) P[i] = r * k[i] / nk;
}

/* volume: P_v = configuration closest to x (Euclidean over all 3n coordinates) with V(P_v) = V*,
 * by D <- ((g.D - C)/(g.g)) g, C = V(x+D) - V*, g = grad V(x+D), from D = 0
 * until |C| < 1e-14 V0 and D has stopped moving
 * V and grad V of a CLOSED surface are translation invariant (create checks closedness), so they
 * are evaluated in coordinates translated by -x[vertex 0]: same numbers in exact arithmetic,
 * no 1e6-sized cancelling terms for a cell that sits 100 um from the origin.
 * returns the number of iterations used. */
double oracle_volume_closed(int n, int T, const int32_t *tris, const double *x) {
  double *y = (double*)malloc(sizeof(double) * 3 * (size_t)n);
  for (int v = 0; v < n; ++v) for (int d = 0; d < 3; ++d) y[3*v+d] = x[3*v+d] - x[d];
  double V = oracle_volume(T, tris, y);
  free(y);
  return V;
}

int oracle_project_volume(int n, int T, const int32_t *tris, const double *x, double Vstar,
                          double V0, double *P) {
  size_t m = 3 * (size_t)n;
  double *D = (double*)calloc(m, sizeof(double));
  double *g = (double*)malloc(m * sizeof(double));
  double *y = (double*)malloc(m * sizeof(double));
  int it = 0;
  for (int v = 0; v < n; ++v) for (int d = 0; d < 3; ++d) y[3*v+d] = x[3*v+d] - x[d];
  if (oracle_volume(T, tris, y) != Vstar) {
    for (it = 1; it <= 100; ++it) {
      double C = oracle_volume(T, tris, y) - Vstar;
      oracle_volume_grad(n, T, tris, y, g);
      double gD = 0, gg = 0;
      for (size_t i = 0; i < m; ++i) { gD += g[i]*D[i]; gg += g[i]*g[i]; }
      double lam = (gD - C) / gg;
      double move = 0, size = 0;
      for (size_t i = 0; i < m; ++i) {
        double Dn = lam * g[i];
        double y0 = y[i] - D[i];                        /* translated x */
        move += (Dn - D[i]) * (Dn - D[i]); size += y0*y0;
        D[i] = Dn; y[i] = y0 + Dn;
      }
      if (fabs(C) < 1e-14 * fabs(V0) && sqrt(move) <= 1e-15 * sqrt(size)) break;
    }
  }
  for (size_t i = 0; i < m; ++i) P[i] = x[i] + D[i];
  free(D); free(g); free(y);
  return it;
}

/* ---------------------------------------------------------------- create (per cell type) */
static double cot_at(const double *p, const double *q, const double *r) {
  double u[3], v[3], c[3]; sub3(q, p, u); sub3(r, p, v); cross3(u, v, c);
  return dot3(u, v) / norm3(c);
}

/* dense Cholesky A = L L^T (lower), returns 0 on success */
static int chol_dense(int n, const double *A, double *L) {
  memset(L, 0, sizeof(double) * (size_t)n * n);
  for (int j = 0; j < n; ++j) {
    double d = A[(size_t)j*n + j];
    for (int k = 0; k < j; ++k) d -= L[(size_t)j*n + k] * L[(size_t)j*n + k];
    if (!(d > 0.0)) return -1;
    d = sqrt(d);
    L[(size_t)j*n + j] = d;
    for (int i = j + 1; i < n; ++i) {
      double s = A[(size_t)i*n + j];
      for (int k = 0; k < j; ++k) s -= L[(size_t)i*n + k] * L[(size_t)j*n + k];
      L[(size_t)i*n + j] = s / d;
    }
  }
  return 0;
}

void oracle_destroy(oracle_cell *c) {
  if (!c) return;
  free(c->tris); free(c->X); free(c->G); free(c->area); free(c->mass); free(c->hinge);
  free(c->K); free(c->w_h); free(c->r_h); free(c->Lel); free(c->A); free(c->L); free(c->LT); free(c);
}

int oracle_create(int n, int T, const int32_t *tris, const double *X, const oracle_material *mat,
                  double h, oracle_cell **out) {
  if (!out) return ORACLE_EINVAL;
  *out = NULL;
  if (n < 4 || T < 4 || !tris || !X || !mat || !(h > 0)) return ORACLE_EINVAL;
  if (mat->s_min > mat->s_max || mat->a_min > mat->a_max || mat->v_min > mat->v_max) return ORACLE_EINVAL;
  if (mat->c_alpha < 0.0 || mat->c_beta < 0.0) return ORACLE_EINVAL;
  if (mat->w_collision < 0.0 || mat->d_collision < 0.0 || mat->strain_hardening < 0.0) return ORACLE_EINVAL;
  if (mat->w_garea < 0.0 || (mat->w_garea > 0.0 && mat->ga_min > mat->ga_max)) return ORACLE_EINVAL;
  if (!(mat->cell_mass > 0)) return ORACLE_EINVAL;
  for (int i = 0; i < 3*T; ++i) if (tris[i] < 0 || tris[i] >= n) return ORACLE_EINVAL;
  if ((3*T) % 2) return ORACLE_EINVAL;
  int H = 3*T/2;

  oracle_cell *c = (oracle_cell*)calloc(1, sizeof(oracle_cell));
  if (!c) return ORACLE_ENOMEM;
  c->n = n; c->T = T; c->H = H; c->mat = *mat; c->h = h;
  c->tris = (int32_t*)malloc(sizeof(int32_t)*3*T);
  c->X = (double*)malloc(sizeof(double)*3*n);
  c->G = (double*)malloc(sizeof(double)*6*T);
  c->area = (double*)malloc(sizeof(double)*T);
  c->mass = (double*)calloc(n, sizeof(double));
  c->hinge = (int32_t*)malloc(sizeof(int32_t)*4*H);
  c->K = (double*)malloc(sizeof(double)*4*H);
  c->w_h = (double*)malloc(sizeof(double)*H);
  c->r_h = (double*)malloc(sizeof(double)*H);
  c->Lel = (double*)calloc((size_t)n*n, sizeof(double));
  c->A = (double*)calloc((size_t)n*n, sizeof(double));
  c->L = (double*)malloc(sizeof(double)*(size_t)n*n);
  c->LT = (double*)malloc(sizeof(double)*(size_t)n*n);
  memcpy(c->tris, tris, sizeof(int32_t)*3*T);
  memcpy(c->X, X, sizeof(double)*3*n);

  /* A-14: closed, consistently oriented 2-manifold: every directed edge exactly once and its
   * reverse exactly once.  opp[u*n+v] = vertex opposite directed edge u->v, or -1. */
  int32_t *opp = (int32_t*)malloc(sizeof(int32_t)*(size_t)n*n);
  for (size_t i = 0; i < (size_t)n*n; ++i) opp[i] = -1;
  int bad = 0;
  for (int t = 0; t < T && !bad; ++t) {
    for (int e = 0; e < 3; ++e) {
      int u = tris[3*t+e], v = tris[3*t+(e+1)%3], w = tris[3*t+(e+2)%3];
      if (u == v || opp[(size_t)u*n+v] != -1) { bad = 1; break; }
      opp[(size_t)u*n+v] = w;
    }
  }
  for (int t = 0; t < T && !bad; ++t)
    for (int e = 0; e < 3; ++e) {
      int u = tris[3*t+e], v = tris[3*t+(e+1)%3];
      if (opp[(size_t)v*n+u] == -1) { bad = 1; break; }
    }
  if (bad) { free(opp); oracle_destroy(c); return ORACLE_EINVAL; }

  /* step 1: per-triangle rest frame, D_m, rest area, G_t = D_m^-T [[-1,1,0],[-1,0,1]] */
  double total_area = 0.0;
  for (int t = 0; t < T; ++t) {
    const double *Xa = X + 3*tris[3*t], *Xb = X + 3*tris[3*t+1], *Xc = X + 3*tris[3*t+2];
    double e1[3], e2[3], nrm[3], t1[3], t2[3];
    sub3(Xb, Xa, e1); sub3(Xc, Xa, e2); cross3(e1, e2, nrm);
    double nn = norm3(nrm), l1 = norm3(e1);
    if (!(nn > 0) || !(l1 > 0)) { free(opp); oracle_destroy(c); return ORACLE_EINVAL; }
    for (int k = 0; k < 3; ++k) { nrm[k] /= nn; t1[k] = e1[k] / l1; }
    cross3(nrm, t1, t2);
    double d00 = dot3(e1, t1), d01 = dot3(e2, t1), d11 = dot3(e2, t2);   /* D_m = [[d00,d01],[0,d11]] */
    c->area[t] = 0.5 * nn;
    total_area += c->area[t];
    /* D_m^-1 = [[1/d00, -d01/(d00 d11)],[0, 1/d11]];  D_m^-T = its transpose */
    double i00 = 1.0/d00, i01 = -d01/(d00*d11), i11 = 1.0/d11;
    double DmInvT[2][2] = {{i00, 0.0}, {i01, i11}};
    double S[2][3] = {{-1, 1, 0}, {-1, 0, 1}};
    for (int a = 0; a < 2; ++a)
      for (int v = 0; v < 3; ++v)
        c->G[6*t + 3*a + v] = DmInvT[a][0]*S[0][v] + DmInvT[a][1]*S[1][v];
  }
  /* step 2: lumped masses m_v = cell_mass a_v / sum a_v, a_v = 1/3 sum_{t contains v} A_t   (A-4) */
  for (int t = 0; t < T; ++t)
    for (int e = 0; e < 3; ++e) c->mass[tris[3*t+e]] += c->area[t] / 3.0;
  for (int v = 0; v < n; ++v) c->mass[v] = mat->cell_mass * c->mass[v] / total_area;

  /* step 3: hinges, one per undirected edge in increasing (min,max) order */
  int hcount = 0;
  for (int u = 0; u < n; ++u)
    for (int v = u + 1; v < n; ++v) {
      if (opp[(size_t)u*n+v] == -1) continue;
      int x2 = opp[(size_t)u*n+v], x3 = opp[(size_t)v*n+u];
      if (hcount >= H) { free(opp); oracle_destroy(c); return ORACLE_EINVAL; }
      int32_t *st = c->hinge + 4*hcount;
      st[0] = u; st[1] = v; st[2] = x2; st[3] = x3;
      const double *X0 = X+3*u, *X1 = X+3*v, *X2 = X+3*x2, *X3 = X+3*x3;
      double c01 = cot_at(X0, X1, X2), c02 = cot_at(X0, X1, X3);
      double c03 = cot_at(X1, X0, X2), c04 = cot_at(X1, X0, X3);
      double *K = c->K + 4*hcount;
      K[0] = c03 + c04; K[1] = c01 + c02; K[2] = -c01 - c03; K[3] = -c02 - c04;
      double a[3], b[3], cr[3];
      sub3(X1, X0, a); sub3(X2, X0, b); cross3(a, b, cr); double A0 = 0.5*norm3(cr);
      sub3(X3, X0, b); cross3(a, b, cr); double A1 = 0.5*norm3(cr);
      c->w_h[hcount] = mat->k_bend * 3.0 / (A0 + A1);
      double kv[3] = {0,0,0};
      for (int i = 0; i < 4; ++i) for (int k = 0; k < 3; ++k) kv[k] += K[i] * X[3*st[i]+k];
      c->r_h[hcount] = norm3(kv);
      ++hcount;
    }
  free(opp);
  if (hcount != H) { oracle_destroy(c); return ORACLE_EINVAL; }

  /* step 4: rest volume */
  c->V0 = oracle_volume(T, tris, X);
  if (!(c->V0 > 0)) { oracle_destroy(c); return ORACLE_EINVAL; }

  /* step 5: L_el = sum_t (w_s+w_a) G^T G + sum_h w_h K^T K;
   *         A_sys = (1/h^2 + c_alpha/h) diag(m) + (1 + c_beta/h) L_el + (w_volume + w_collision + w_garea) I
   * (c_alpha = c_beta = 0: the undamped system of SURVEY.md 8(c); otherwise reading A-20: the
   * Rayleigh damping force -(c_alpha M + c_beta L_el)(x - x_n)/h of implicit Euler moves
   * (c_alpha M + c_beta L_el)/h to the left-hand side) */
  for (int t = 0; t < T; ++t) {
    double w = (mat->k_strain + mat->k_area) * c->area[t];
    const double *G = c->G + 6*t;
    for (int p = 0; p < 3; ++p)
      for (int q = 0; q < 3; ++q)
        c->Lel[(size_t)tris[3*t+p]*n + tris[3*t+q]] += w * (G[p]*G[q] + G[3+p]*G[3+q]);
  }
  for (int hh = 0; hh < H; ++hh) {
    const int32_t *st = c->hinge + 4*hh; const double *K = c->K + 4*hh;
    for (int p = 0; p < 4; ++p)
      for (int q = 0; q < 4; ++q)
        c->Lel[(size_t)st[p]*n + st[q]] += c->w_h[hh] * K[p] * K[q];
  }
  for (size_t i = 0; i < (size_t)n*n; ++i) c->A[i] = (1.0 + mat->c_beta / h) * c->Lel[i];
  for (int v = 0; v < n; ++v)
    c->A[(size_t)v*n+v] += c->mass[v] * (1.0/(h*h) + mat->c_alpha / h) + mat->w_volume + mat->w_collision + mat->w_garea;
  if (chol_dense(n, c->A, c->L) != 0) { oracle_destroy(c); return ORACLE_EINVAL; }
  for (int i = 0; i < n; ++i) for (int j = 0; j < n; ++j) c->LT[(size_t)j*n+i] = c->L[(size_t)i*n+j];
  *out = c;
  return ORACLE_OK;
}

/* getters for the tests */
int oracle_n_hinges(const oracle_cell *c) { return c->H; }
double oracle_rest_volume(const oracle_cell *c) { return c->V0; }
void oracle_get_hinges(const oracle_cell *c, int32_t *o) { memcpy(o, c->hinge, sizeof(int32_t)*4*c->H); }
void oracle_get_K(const oracle_cell *c, double *o) { memcpy(o, c->K, sizeof(double)*4*c->H); }
void oracle_get_hinge_weights(const oracle_cell *c, double *w, double *r) {
  memcpy(w, c->w_h, sizeof(double)*c->H); memcpy(r, c->r_h, sizeof(double)*c->H);
}
void oracle_get_masses(const oracle_cell *c, double *o) { memcpy(o, c->mass, sizeof(double)*c->n); }
void oracle_get_areas(const oracle_cell *c, double *o) { memcpy(o, c->area, sizeof(double)*c->T); }
void oracle_get_G(const oracle_cell *c, double *o) { memcpy(o, c->G, sizeof(double)*6*c->T); }
void oracle_get_system(const oracle_cell *c, double *o) { memcpy(o, c->A, sizeof(double)*(size_t)c->n*c->n); }
void oracle_get_elastic_laplacian(const oracle_cell *c, double *o) { memcpy(o, c->Lel, sizeof(double)*(size_t)c->n*c->n); }

/* ---------------------------------------------------------------- the step, piece by piece */
/* F_t (row-major 3x2):  F^T = G [x_a; x_b; x_c] */
void oracle_deformation_gradient(const oracle_cell *c, int t, const double *x, double *F) {
  const double *G = c->G + 6*t; const int32_t *tr = c->tris + 3*t;
  for (int i = 0; i < 3; ++i)
    for (int a = 0; a < 2; ++a) {
      double s = 0;
      for (int v = 0; v < 3; ++v) s += G[3*a+v] * x[3*tr[v]+i];
      F[2*i+a] = s;
    }
}

static void hinge_vector(const oracle_cell *c, int hh, const double *x, double *k) {
  const int32_t *st = c->hinge + 4*hh; const double *K = c->K + 4*hh;
  k[0] = k[1] = k[2] = 0;
  for (int i = 0; i < 4; ++i) for (int d = 0; d < 3; ++d) k[d] += K[i] * x[3*st[i]+d];
}

/* local step: all projections at x.  Ps, Pa [T][6]; Pb [H][3]; Pv [n][3] */
void oracle_local(const oracle_cell *c, const double *x, double *Ps, double *Pa, double *Pb, double *Pv) {
  const oracle_material *m = &c->mat;
  for (int t = 0; t < c->T; ++t) {
    double F[6];
    oracle_deformation_gradient(c, t, x, F);
    if (m->strain_hardening != 0.0) oracle_project_strain_hardening(F, m->s_min, m->s_max, m->strain_hardening, Ps + 6*t);
    else oracle_project_strain(F, m->s_min, m->s_max, Ps + 6*t);
    oracle_project_area(F, m->a_min, m->a_max, Pa + 6*t);
  }
  for (int hh = 0; hh < c->H; ++hh) {
    double k[3];
    hinge_vector(c, hh, x, k);
    oracle_project_bend(k, c->r_h[hh], Pb + 3*hh);
  }
  double V = oracle_volume_closed(c->n, c->T, c->tris, x);
  double Vstar = clampd(V, m->v_min * c->V0, m->v_max * c->V0);
  oracle_project_volume(c->n, c->T, c->tris, x, Vstar, c->V0, Pv);
}

/* b = diag(m)/h^2 s + sum_t G^T (w_s Ps^T + w_a Pa^T) + sum_h w_h K^T Pb + w_volume Pv */
void oracle_rhs(const oracle_cell *c, const double *s, const double *Ps, const double *Pa,
                const double *Pb, const double *Pv, double *b) {
  const oracle_material *m = &c->mat;
  double ih2 = 1.0 / (c->h * c->h);
  for (int v = 0; v < c->n; ++v)
    for (int d = 0; d < 3; ++d)
      b[3*v+d] = c->mass[v] * ih2 * s[3*v+d] + m->w_volume * Pv[3*v+d];
  for (int t = 0; t < c->T; ++t) {
    double ws = m->k_strain * c->area[t], wa = m->k_area * c->area[t];
    const double *G = c->G + 6*t; const int32_t *tr = c->tris + 3*t;
    for (int v = 0; v < 3; ++v)
      for (int d = 0; d < 3; ++d)
        for (int a = 0; a < 2; ++a)
          b[3*tr[v]+d] += G[3*a+v] * (ws * Ps[6*t + 2*d + a] + wa * Pa[6*t + 2*d + a]);
  }
  for (int hh = 0; hh < c->H; ++hh) {
    const int32_t *st = c->hinge + 4*hh; const double *K = c->K + 4*hh;
    for (int i = 0; i < 4; ++i)
      for (int d = 0; d < 3; ++d)
        b[3*st[i]+d] += c->w_h[hh] * K[i] * Pb[3*hh+d];
  }
}

/* global step: x = A_sys^-1 b by forward/backward substitution with the dense factor (3 rhs) */
void oracle_solve(const oracle_cell *c, const double *b, double *x) {
  int n = c->n; const double *L = c->L, *LT = c->LT;
  for (int d = 0; d < 3; ++d) {
    for (int i = 0; i < n; ++i) {                       /* L y = b */
      double s = b[3*i+d];
      for (int k = 0; k < i; ++k) s -= L[(size_t)i*n+k] * x[3*k+d];
      x[3*i+d] = s / L[(size_t)i*n+i];
    }
    for (int i = n - 1; i >= 0; --i) {                  /* L^T x = y */
      double s = x[3*i+d];
      for (int k = i + 1; k < n; ++k) s -= LT[(size_t)i*n+k] * x[3*k+d];
      x[3*i+d] = s / L[(size_t)i*n+i];
    }
  }
}

/* E(x;p) = 1/2 ||x-s||^2_M / h^2 + sum 1/2 w_s ||F-Ps||^2 + sum 1/2 w_a ||F-Pa||^2
 *        + sum 1/2 w_h ||k-Pb||^2 + 1/2 w_volume ||x-Pv||^2       (pin P-3)
 * parts[5] receives the five terms if not NULL. */
double oracle_energy(const oracle_cell *c, const double *x, const double *s, const double *Ps,
                     const double *Pa, const double *Pb, const double *Pv, double *parts) {
  const oracle_material *m = &c->mat;
  double e[5] = {0,0,0,0,0};
  double ih2 = 1.0 / (c->h * c->h);
  for (int v = 0; v < c->n; ++v)
    for (int d = 0; d < 3; ++d) {
      double u = x[3*v+d] - s[3*v+d], q = x[3*v+d] - Pv[3*v+d];
      e[0] += 0.5 * c->mass[v] * ih2 * u*u;
      e[4] += 0.5 * m->w_volume * q*q;
    }
  for (int t = 0; t < c->T; ++t) {
    double F[6]; oracle_deformation_gradient(c, t, x, F);
    double ds = 0, da = 0;
    for (int k = 0; k < 6; ++k) {
      ds += (F[k]-Ps[6*t+k])*(F[k]-Ps[6*t+k]);
      da += (F[k]-Pa[6*t+k])*(F[k]-Pa[6*t+k]);
    }
    if (m->strain_hardening != 0.0)      /* Ps holds the effective targets: take the energy from F itself */
      e[1] += m->k_strain * c->area[t] * oracle_strain_energy_density(F, m->s_min, m->s_max, m->strain_hardening);
    else
      e[1] += 0.5 * m->k_strain * c->area[t] * ds;
    e[2] += 0.5 * m->k_area * c->area[t] * da;
  }
  for (int hh = 0; hh < c->H; ++hh) {
    double k[3]; hinge_vector(c, hh, x, k);
    double db = 0;
    for (int d = 0; d < 3; ++d) db += (k[d]-Pb[3*hh+d])*(k[d]-Pb[3*hh+d]);
    e[3] += 0.5 * c->w_h[hh] * db;
  }
  if (parts) memcpy(parts, e, sizeof(e));
  return e[0] + e[1] + e[2] + e[3] + e[4];
}

double oracle_garea_local(const oracle_cell *c, const double *x, double *Pg);

/* internal force f_int(x) = sum w A^T (p(x) - A x)   (pins P-2, P-8) */
void oracle_fint(const oracle_cell *c, const double *x, double *f) {
  int n = c->n; const oracle_material *m = &c->mat;
  double *Ps = (double*)malloc(sizeof(double)*6*c->T), *Pa = (double*)malloc(sizeof(double)*6*c->T);
  double *Pb = (double*)malloc(sizeof(double)*3*c->H), *Pv = (double*)malloc(sizeof(double)*3*n);
  double *zero = (double*)calloc(3*(size_t)n, sizeof(double));
  oracle_local(c, x, Ps, Pa, Pb, Pv);
  oracle_rhs(c, zero, Ps, Pa, Pb, Pv, f);               /* sum w A^T p */
  /* minus (sum w A^T A) x = (L_el + w_volume I) x */
  for (int i = 0; i < n; ++i)
    for (int d = 0; d < 3; ++d) {
      double s = m->w_volume * x[3*i+d];
      for (int j = 0; j < n; ++j) s += c->Lel[(size_t)i*n+j] * x[3*j+d];
      f[3*i+d] -= s;
    }
  if (m->w_garea > 0.0) {                                /* global-area term (A-24): w_garea (P_g - x) */
    oracle_garea_local(c, x, zero);
    for (size_t i = 0; i < 3*(size_t)n; ++i) f[i] += m->w_garea * (zero[i] - x[i]);
  }
  free(Ps); free(Pa); free(Pb); free(Pv); free(zero);
}

void oracle_damping_rhs(const oracle_cell *c, const double *xn, double *b);
double oracle_dissipation(const oracle_cell *c, const double *x, const double *xn);

/* ---------------------------------------------------------------- global-area term (NEXT-4, reading A-24)
 * every elemental potential has "a weight and various parameters"; SURVEY.md 8(f)
 * NEXT-4 names "a global-area term".  Reading: one constraint per cell on the TOTAL surface area
 * A(x) = sum_t 1/2 |(x_b - x_a) x (x_c - x_a)|, band [ga_min, ga_max] A0 (A0 = rest total area);
 * P_g = the configuration closest to x (plain Euclidean norm over all 3n coordinates) with
 * A(P_g) = A*; energy 1/2 w_garea ||x - P_g||^2 with selection matrix I, so w_garea sits on the
 * diagonal of A_sys.  Unlike the volume, the area's Hessian (a cotangent Laplacian, entries of
 * order 1) makes the fixed-point iteration D <- ((g.D - C)/(g.g)) g diverge already at a 10 %
 * violation, so the closest point is found by Newton's method on the KKT system
 *     P - x - lambda grad A(P) = 0,   A(P) = A*,
 * Jacobian [[I - lambda H(P), -g], [g^T, 0]], H = Hessian of A, dense LU, step halving on the
 * residual norm.  grad A: per triangle with unit normal nh, dA/dx_a = 1/2 nh x (x_c - x_b) (cyclic). */
double oracle_area_total(int T, const int32_t *tris, const double *x) {
  double A = 0.0;
  for (int t = 0; t < T; ++t) {
    const double *a = x + 3*tris[3*t], *b = x + 3*tris[3*t+1], *c = x + 3*tris[3*t+2];
    double e1[3] = {b[0]-a[0], b[1]-a[1], b[2]-a[2]}, e2[3] = {c[0]-a[0], c[1]-a[1], c[2]-a[2]}, nn[3];
    cross3(e1, e2, nn);
    A += 0.5 * sqrt(dot3(nn, nn));
  }
  return A;
}
void oracle_area_grad(int n, int T, const int32_t *tris, const double *x, double *g) {
  memset(g, 0, sizeof(double) * 3 * (size_t)n);
  for (int t = 0; t < T; ++t) {
    int id[3] = {tris[3*t], tris[3*t+1], tris[3*t+2]};
    const double *a = x + 3*id[0], *b = x + 3*id[1], *c = x + 3*id[2];
    double e1[3] = {b[0]-a[0], b[1]-a[1], b[2]-a[2]}, e2[3] = {c[0]-a[0], c[1]-a[1], c[2]-a[2]}, nn[3];
    cross3(e1, e2, nn);
    double len = sqrt(dot3(nn, nn));
    if (!(len > 0.0)) continue;                          /* collapsed triangle: no contribution */
    for (int k = 0; k < 3; ++k) nn[k] /= len;
    for (int v = 0; v < 3; ++v) {                         /* opposite edge of vertex v: x_{v+2} - x_{v+1} */
      const double *p = x + 3*id[(v+1)%3], *q = x + 3*id[(v+2)%3];
      double opp[3] = {q[0]-p[0], q[1]-p[1], q[2]-p[2]}, gv[3];
      cross3(nn, opp, gv);
      for (int k = 0; k < 3; ++k) g[3*id[v]+k] += 0.5 * gv[k];
    }
  }
}
/* Hessian of the total area, dense [3n][3n].  Per triangle with u = b - a, v = c - a, n = u x v:
 *   d n = J delta, J = [ -(e_k x v) - (u x e_k) | e_k x v | u x e_k ]  (3 x 9, columns a, b, c),
 *   d^2 A = [ |J delta|^2 - (nh . J delta)^2 ] / (2 |n|) + nh . (du x dv),
 * the last term being the quadratic form of 1/2 (X + X^T), X = S_v^T [nh]_x S_u, S_u = [-I I 0],
 * S_v = [-I 0 I]. */
void oracle_area_hessian(int n, int T, const int32_t *tris, const double *x, double *H) {
  size_t m = 3 * (size_t)n;
  memset(H, 0, sizeof(double) * m * m);
  for (int t = 0; t < T; ++t) {
    int id[3] = {tris[3*t], tris[3*t+1], tris[3*t+2]};
    const double *a = x + 3*id[0], *b = x + 3*id[1], *c = x + 3*id[2];
    double u[3] = {b[0]-a[0], b[1]-a[1], b[2]-a[2]}, v[3] = {c[0]-a[0], c[1]-a[1], c[2]-a[2]}, nn[3];
    cross3(u, v, nn);
    double len = sqrt(dot3(nn, nn));
    if (!(len > 0.0)) continue;
    double nh[3] = {nn[0]/len, nn[1]/len, nn[2]/len};
    double J[3][9], Jn[9];
    for (int k = 0; k < 3; ++k) {
      double e[3] = {0, 0, 0}, ev[3], ue[3];
      e[k] = 1.0;
      cross3(e, v, ev); cross3(u, e, ue);
      for (int r = 0; r < 3; ++r) { J[r][k] = -ev[r] - ue[r]; J[r][3+k] = ev[r]; J[r][6+k] = ue[r]; }
    }
    for (int q = 0; q < 9; ++q) Jn[q] = nh[0]*J[0][q] + nh[1]*J[1][q] + nh[2]*J[2][q];
    /* [nh]_x y = nh x y */
    double N[3][3] = {{0, -nh[2], nh[1]}, {nh[2], 0, -nh[0]}, {-nh[1], nh[0], 0}};
    double Su[3][9] = {{0}}, Sv[3][9] = {{0}};
    for (int k = 0; k < 3; ++k) { Su[k][k] = -1; Su[k][3+k] = 1; Sv[k][k] = -1; Sv[k][6+k] = 1; }
    for (int p = 0; p < 9; ++p)
      for (int q = 0; q < 9; ++q) {
        double jj = J[0][p]*J[0][q] + J[1][p]*J[1][q] + J[2][p]*J[2][q];
        double h = (jj - Jn[p]*Jn[q]) / (2.0 * len);
        double X = 0, Xt = 0;                            /* X[p][q] = sum_rs Sv[r][p] N[r][s] Su[s][q] */
        for (int r = 0; r < 3; ++r)
          for (int ss = 0; ss < 3; ++ss) { X += Sv[r][p]*N[r][ss]*Su[ss][q]; Xt += Sv[r][q]*N[r][ss]*Su[ss][p]; }
        h += 0.5 * (X + Xt);
        H[(3*(size_t)id[p/3] + p%3) * m + 3*(size_t)id[q/3] + q%3] += h;
      }
  }
}
/* dense LU with partial pivoting: solves M y = rhs in place (M [m][m] is destroyed); 0 on success */
static int lu_solve(int m, double *M, double *rhs) {
  for (int k = 0; k < m; ++k) {
    int piv = k; double best = fabs(M[(size_t)k*m+k]);
    for (int i = k+1; i < m; ++i) if (fabs(M[(size_t)i*m+k]) > best) { best = fabs(M[(size_t)i*m+k]); piv = i; }
    if (!(best > 0.0)) return -1;
    if (piv != k) {
      for (int j = 0; j < m; ++j) { double tmp = M[(size_t)k*m+j]; M[(size_t)k*m+j] = M[(size_t)piv*m+j]; M[(size_t)piv*m+j] = tmp; }
      double tmp = rhs[k]; rhs[k] = rhs[piv]; rhs[piv] = tmp;
    }
    for (int i = k+1; i < m; ++i) {
      double f = M[(size_t)i*m+k] / M[(size_t)k*m+k];
      if (f == 0.0) continue;
      for (int j = k+1; j < m; ++j) M[(size_t)i*m+j] -= f * M[(size_t)k*m+j];
      rhs[i] -= f * rhs[k];
    }
  }
  for (int i = m-1; i >= 0; --i) {
    double s = rhs[i];
    for (int j = i+1; j < m; ++j) s -= M[(size_t)i*m+j] * rhs[j];
    rhs[i] = s / M[(size_t)i*m+i];
  }
  return 0;
}
/* closest configuration with total area Astar; returns the Newton iterations used (-1: no convergence) */
int oracle_project_garea(int n, int T, const int32_t *tris, const double *x, double Astar, double A0,
                         double *P) {
  size_t m = 3 * (size_t)n; int mm = (int)m + 1;
  memcpy(P, x, m * sizeof(double));
  if (oracle_area_total(T, tris, x) == Astar) return 0;
  double *g = (double*)malloc(m * sizeof(double)), *H = (double*)malloc(m * m * sizeof(double));
  double *K = (double*)malloc((size_t)mm * mm * sizeof(double)), *rhs = (double*)malloc(mm * sizeof(double));
  double *Pt = (double*)malloc(m * sizeof(double));
  double lam = 0.0, scale = 0.0;
  for (size_t i = 0; i < m; ++i) { double x0 = x[i] - x[i % 3]; scale += x0*x0; }
  scale = sqrt(scale);                                   /* size of the cell, not its distance from the origin */
  int it, ok = -1;
  for (it = 1; it <= 60; ++it) {
    oracle_area_grad(n, T, tris, P, g);
    double C = oracle_area_total(T, tris, P) - Astar, r1n = 0;
    for (size_t i = 0; i < m; ++i) { rhs[i] = -(P[i] - x[i] - lam * g[i]); r1n += rhs[i]*rhs[i]; }
    rhs[m] = -C;
    double res = sqrt(r1n) / scale + fabs(C) / fabs(A0);
    if (res < 1e-14) { ok = it - 1; break; }
    oracle_area_hessian(n, T, tris, P, H);
    for (size_t i = 0; i < m; ++i) {
      for (size_t j = 0; j < m; ++j) K[i*mm+j] = (i == j ? 1.0 : 0.0) - lam * H[i*m+j];
      K[i*mm+m] = -g[i];
      K[m*mm+i] = g[i];
    }
    K[m*mm+m] = 0.0;
    if (lu_solve(mm, K, rhs) != 0) break;
    double step = 1.0;                                   /* halve the step while the residual grows */
    for (int ls = 0; ls < 30; ++ls, step *= 0.5) {
      for (size_t i = 0; i < m; ++i) Pt[i] = P[i] + step * rhs[i];
      double lt = lam + step * rhs[m];
      oracle_area_grad(n, T, tris, Pt, g);
      double Ct = oracle_area_total(T, tris, Pt) - Astar, rn = 0;
      for (size_t i = 0; i < m; ++i) { double q = Pt[i] - x[i] - lt * g[i]; rn += q*q; }
      if (sqrt(rn) / scale + fabs(Ct) / fabs(A0) < res || ls == 29) { memcpy(P, Pt, m * sizeof(double)); lam = lt; break; }
    }
  }
  free(g); free(H); free(K); free(rhs); free(Pt);
  return ok;
}
double oracle_rest_area(const oracle_cell *c) { double A = 0; for (int t = 0; t < c->T; ++t) A += c->area[t]; return A; }
/* P_g [n][3] at x; returns the energy 1/2 w_garea ||x - P_g||^2 (0 and P_g = x when the weight is 0) */
double oracle_garea_local(const oracle_cell *c, const double *x, double *Pg) {
  size_t m3 = 3*(size_t)c->n;
  if (!(c->mat.w_garea > 0.0)) { memcpy(Pg, x, sizeof(double)*m3); return 0.0; }
  double A0 = oracle_rest_area(c);
  double A = oracle_area_total(c->T, c->tris, x);
  double Astar = clampd(A, c->mat.ga_min * A0, c->mat.ga_max * A0);
  oracle_project_garea(c->n, c->T, c->tris, x, Astar, A0, Pg);
  double e = 0;
  for (size_t i = 0; i < m3; ++i) e += (x[i]-Pg[i])*(x[i]-Pg[i]);
  return 0.5 * c->mat.w_garea * e;
}

/* ---------------------------------------------------------------- collisions (NEXT-3, reading A-22)
 * the coupling hands "external forces & colliding neighbours" to the solid solver;
 * :145 "collision forces intensity (collisions_weight parameter)".  Reading: per vertex at most one
 * colliding neighbour per step, given as a point q on the other body and that body's outward unit
 * normal nrm at q (nrm = 0: no neighbour).  The vertex must stay on the outer side of the plane,
 * at least d_collision away:  (x_v - q).nrm >= d.  Projection (closest point of that half space):
 *   t = d - (x_v - q).nrm;   p = x_v + max(t, 0) nrm.
 * Energy 1/2 w_collision ||x_v - p||^2 with selection matrix I, so w_collision sits on the diagonal
 * of A_sys for EVERY vertex (inactive vertices project onto themselves and feel no force), which
 * keeps the system matrix constant while contacts come and go. */
void oracle_project_collision(const double *x, const double *q, const double *nrm, double d, double *p) {
  double t = d - ((x[0]-q[0])*nrm[0] + (x[1]-q[1])*nrm[1] + (x[2]-q[2])*nrm[2]);
  if (!(t > 0.0) || (nrm[0] == 0.0 && nrm[1] == 0.0 && nrm[2] == 0.0)) t = 0.0;
  p[0] = x[0] + t*nrm[0]; p[1] = x[1] + t*nrm[1]; p[2] = x[2] + t*nrm[2];
}
/* all vertices: Pc [n][3]; returns the collision energy 1/2 w_c sum ||x - Pc||^2 */
double oracle_collision_local(const oracle_cell *c, const double *x, const double *q, const double *nrm,
                              double *Pc) {
  double e = 0;
  for (int v = 0; v < c->n; ++v) {
    oracle_project_collision(x + 3*v, q + 3*v, nrm + 3*v, c->mat.d_collision, Pc + 3*v);
    for (int d = 0; d < 3; ++d) e += (x[3*v+d]-Pc[3*v+d])*(x[3*v+d]-Pc[3*v+d]);
  }
  return 0.5 * c->mat.w_collision * e;
}

/* One time step of ONE cell with colliding neighbours (q, nrm: [n][3], held fixed over the step):
 * the local/global sweeps of oracle_step_cell with the collision projections added to the rhs.
 * energies [2*n_iters] as in oracle_step_cell (collision energy included). */
void oracle_step_cell_collide(const oracle_cell *c, double *pos, double *vel, const double *fext,
                              const double *q, const double *nrm, int n_iters, double *iterates,
                              double *energies) {
  int n = c->n; size_t m3 = 3*(size_t)n; double h = c->h, wc = c->mat.w_collision, wg = c->mat.w_garea;
  double *s = (double*)malloc(sizeof(double)*m3), *x = (double*)malloc(sizeof(double)*m3);
  double *b = (double*)malloc(sizeof(double)*m3), *Pc = (double*)malloc(sizeof(double)*m3);
  double *Pg = wg > 0.0 ? (double*)malloc(sizeof(double)*m3) : NULL;   /* global-area term (A-24), off by default */
  double *Ps = (double*)malloc(sizeof(double)*6*c->T), *Pa = (double*)malloc(sizeof(double)*6*c->T);
  double *Pb = (double*)malloc(sizeof(double)*3*c->H), *Pv = (double*)malloc(sizeof(double)*m3);
  for (int v = 0; v < n; ++v)
    for (int d = 0; d < 3; ++d)
      s[3*v+d] = pos[3*v+d] + h * vel[3*v+d] + h*h * fext[3*v+d] / c->mass[v];
  memcpy(x, s, sizeof(double)*m3);
  if (iterates) memcpy(iterates, x, sizeof(double)*m3);
  for (int k = 0; k < n_iters; ++k) {
    oracle_local(c, x, Ps, Pa, Pb, Pv);
    double ec = oracle_collision_local(c, x, q, nrm, Pc);
    double eg = Pg ? oracle_garea_local(c, x, Pg) : 0.0;
    if (energies) energies[2*k] = oracle_energy(c, x, s, Ps, Pa, Pb, Pv, NULL) + oracle_dissipation(c, x, pos) + ec + eg;
    oracle_rhs(c, s, Ps, Pa, Pb, Pv, b);
    oracle_damping_rhs(c, pos, b);
    for (size_t i = 0; i < m3; ++i) b[i] += wc * Pc[i];
    if (Pg) for (size_t i = 0; i < m3; ++i) b[i] += wg * Pg[i];
    oracle_solve(c, b, x);
    if (energies) {
      double e2 = 0, e3 = 0;
      for (size_t i = 0; i < m3; ++i) e2 += (x[i]-Pc[i])*(x[i]-Pc[i]);
      if (Pg) for (size_t i = 0; i < m3; ++i) e3 += (x[i]-Pg[i])*(x[i]-Pg[i]);
      energies[2*k+1] = oracle_energy(c, x, s, Ps, Pa, Pb, Pv, NULL) + oracle_dissipation(c, x, pos) + 0.5*wc*e2 + 0.5*wg*e3;
    }
    if (iterates) memcpy(iterates + (size_t)(k+1)*m3, x, sizeof(double)*m3);
  }
  for (size_t i = 0; i < m3; ++i) { vel[i] = (x[i] - pos[i]) / h; pos[i] = x[i]; }
  free(s); free(x); free(b); free(Pc); free(Pg); free(Ps); free(Pa); free(Pb); free(Pv);
}
void oracle_step_collide(const oracle_cell *c, int n_cells, double *pos, double *vel, const double *fext,
                         const double *q, const double *nrm, int n_iters) {
  size_t stride = 3*(size_t)c->n;
#pragma omp parallel for schedule(dynamic, 1)
  for (int i = 0; i < n_cells; ++i)
    oracle_step_cell_collide(c, pos + i*stride, vel + i*stride, fext + i*stride, q + i*stride,
                             nrm + i*stride, n_iters, NULL, NULL);
}

/* area per surface vertex at the current configuration (consumed by the IBM):
 * a_v = 1/3 sum over the triangles around v of their area */
void oracle_vertex_areas(const oracle_cell *c, const double *x, double *a) {
  for (int v = 0; v < c->n; ++v) a[v] = 0.0;
  for (int t = 0; t < c->T; ++t) {
    const int32_t *tr = c->tris + 3*t;
    double e1[3], e2[3], cr[3];
    sub3(x + 3*tr[1], x + 3*tr[0], e1); sub3(x + 3*tr[2], x + 3*tr[0], e2); cross3(e1, e2, cr);
    double A = 0.5 * norm3(cr);
    for (int e = 0; e < 3; ++e) a[tr[e]] += A / 3.0;
  }
}

/* Rayleigh damping, implicit (reading A-20): C = c_alpha M + c_beta L_el, f_d = -C (x - x_n)/h.
 * b += (C/h) x_n  (the other half, (C/h) x, sits in A_sys). */
void oracle_damping_rhs(const oracle_cell *c, const double *xn, double *b) {
  int n = c->n; double ca = c->mat.c_alpha / c->h, cb = c->mat.c_beta / c->h;
  if (ca == 0.0 && cb == 0.0) return;
  for (int i = 0; i < n; ++i)
    for (int d = 0; d < 3; ++d) {
      double s = ca * c->mass[i] * xn[3*i+d];
      if (cb != 0.0) {
        double l = 0;
        for (int j = 0; j < n; ++j) l += c->Lel[(size_t)i*n+j] * xn[3*j+d];
        s += cb * l;
      }
      b[3*i+d] += s;
    }
}
/* dissipation potential of the step, 1/(2h) (x - x_n)^T C (x - x_n): the term the damping adds to
 * the implicit-Euler objective (its gradient is C (x - x_n)/h = -f_d) */
double oracle_dissipation(const oracle_cell *c, const double *x, const double *xn) {
  int n = c->n; double ca = c->mat.c_alpha, cb = c->mat.c_beta, e = 0;
  if (ca == 0.0 && cb == 0.0) return 0.0;
  for (int d = 0; d < 3; ++d)
    for (int i = 0; i < n; ++i) {
      double ui = x[3*i+d] - xn[3*i+d], l = 0;
      if (cb != 0.0) for (int j = 0; j < n; ++j) l += c->Lel[(size_t)i*n+j] * (x[3*j+d] - xn[3*j+d]);
      e += ui * (ca * c->mass[i] * ui + cb * l);
    }
  return 0.5 * e / c->h;
}

/* One time step of ONE cell (SURVEY.md 8(c) "Step"):
 *   s = x_n + h v_n + h^2 f/m;  x^0 = s;
 *   repeat n_iters: local projections at x^k, b (+ (C/h) x_n with damping, A-20), x^{k+1} = A_sys^-1 b;
 *   x_{n+1} = x^{n_iters};  v_{n+1} = (x_{n+1} - x_n)/h.
 * Optional outputs: iterates [(n_iters+1)][n][3] (x^0 ... x^{n_iters}) and
 * energies [2*n_iters]: E(x^k;p^k) after each local step, E(x^{k+1};p^k) after each global step. */
void oracle_step_cell(const oracle_cell *c, double *pos, double *vel, const double *fext,
                      int n_iters, double *iterates, double *energies) {
  int n = c->n; size_t m3 = 3*(size_t)n; double h = c->h, wg = c->mat.w_garea;
  double *s = (double*)malloc(sizeof(double)*m3), *x = (double*)malloc(sizeof(double)*m3);
  double *b = (double*)malloc(sizeof(double)*m3);
  double *Ps = (double*)malloc(sizeof(double)*6*c->T), *Pa = (double*)malloc(sizeof(double)*6*c->T);
  double *Pb = (double*)malloc(sizeof(double)*3*c->H), *Pv = (double*)malloc(sizeof(double)*m3);
  double *Pg = wg > 0.0 ? (double*)malloc(sizeof(double)*m3) : NULL;   /* global-area term (A-24), off by default */
  for (int v = 0; v < n; ++v)
    for (int d = 0; d < 3; ++d)
      s[3*v+d] = pos[3*v+d] + h * vel[3*v+d] + h*h * fext[3*v+d] / c->mass[v];
  memcpy(x, s, sizeof(double)*m3);
  if (iterates) memcpy(iterates, x, sizeof(double)*m3);
  for (int k = 0; k < n_iters; ++k) {
    oracle_local(c, x, Ps, Pa, Pb, Pv);
    if (!Pg) {                                             /* the path of the five configs, untouched */
      if (energies) energies[2*k] = oracle_energy(c, x, s, Ps, Pa, Pb, Pv, NULL) + oracle_dissipation(c, x, pos);
      oracle_rhs(c, s, Ps, Pa, Pb, Pv, b);
      oracle_damping_rhs(c, pos, b);
      oracle_solve(c, b, x);
      if (energies) energies[2*k+1] = oracle_energy(c, x, s, Ps, Pa, Pb, Pv, NULL) + oracle_dissipation(c, x, pos);
    } else {
      double eg = oracle_garea_local(c, x, Pg), e3 = 0;
      if (energies) energies[2*k] = oracle_energy(c, x, s, Ps, Pa, Pb, Pv, NULL) + oracle_dissipation(c, x, pos) + eg;
      oracle_rhs(c, s, Ps, Pa, Pb, Pv, b);
      oracle_damping_rhs(c, pos, b);
      for (size_t i = 0; i < m3; ++i) b[i] += wg * Pg[i];
      oracle_solve(c, b, x);
      for (size_t i = 0; i < m3; ++i) e3 += (x[i]-Pg[i])*(x[i]-Pg[i]);
      if (energies) energies[2*k+1] = oracle_energy(c, x, s, Ps, Pa, Pb, Pv, NULL) + oracle_dissipation(c, x, pos) + 0.5*wg*e3;
    }
    if (iterates) memcpy(iterates + (size_t)(k+1)*m3, x, sizeof(double)*m3);
  }
  for (size_t i = 0; i < m3; ++i) { vel[i] = (x[i] - pos[i]) / h; pos[i] = x[i]; }
  free(s); free(x); free(b); free(Ps); free(Pa); free(Pb); free(Pv); free(Pg);
}

/* ---------------------------------------------------------------- converged solve (NEXT-1)
 * "Our approach follows the redesigned projective dynamics approach as described
 * in Liu et al. [11] ... we provide a converged solution"; :133 "unconditional stability for
 * arbitrary time steps".  Reading A-21: the step minimises the implicit-Euler objective
 *   g(x) = 1/2 ||x - s||^2_M / h^2 + E_el(x) [+ 1/(2h) (x - x_n)^T C (x - x_n)],
 *   E_el(x) = sum_t 1/2 w_s dist^2(F_t, strain set) + 1/2 w_a dist^2(F_t, area set)
 *           + sum_h 1/2 w_h dist^2(k_h, sphere r_h) + 1/2 w_volume dist^2(x, {V = V*}),
 * whose gradient is  grad g(x) = M (x - s)/h^2 - f_int(x) [+ C (x - x_n)/h]  (the projections
 * are closest points, so their derivatives drop out), by L-BFGS with the constant, prefactored
 * A_sys as initial Hessian (two-loop recursion over the last `history` pairs), a backtracking
 * (halving) line search on g with the Armijo constant 1e-4, and the stop criterion
 *   res(x) = max_v || (h^2/m_v) grad g(x)_v ||_inf <= tol
 * (a length: the displacement the unbalanced force would cause in one free step).
 * history = 0 and line_search = 0 is the plain local/global sweep (pin P-8). */

/* g(x) and its gradient; work arrays are allocated by the caller (Ps,Pa [T][6], Pb [H][3], Pv [n][3]) */
double oracle_objective(const oracle_cell *c, const double *x, const double *s, const double *xn,
                        double *grad) {
  int n = c->n; size_t m3 = 3*(size_t)n; double ih2 = 1.0 / (c->h * c->h);
  double *Ps = (double*)malloc(sizeof(double)*6*c->T), *Pa = (double*)malloc(sizeof(double)*6*c->T);
  double *Pb = (double*)malloc(sizeof(double)*3*c->H), *Pv = (double*)malloc(sizeof(double)*m3);
  oracle_local(c, x, Ps, Pa, Pb, Pv);
  double gval = oracle_energy(c, x, s, Ps, Pa, Pb, Pv, NULL) + oracle_dissipation(c, x, xn);
  if (c->mat.w_garea > 0.0) gval += oracle_garea_local(c, x, Pv);   /* Pv is free again: global-area energy (A-24) */
  if (grad) {
    double *f = (double*)malloc(sizeof(double)*m3), *dmp = (double*)calloc(m3, sizeof(double));
    oracle_fint(c, x, f);
    /* C (x - x_n)/h = (C/h) x - (C/h) x_n, with oracle_damping_rhs(v) = (C/h) v */
    double *tmp = (double*)calloc(m3, sizeof(double));
    oracle_damping_rhs(c, x, dmp); oracle_damping_rhs(c, xn, tmp);
    for (int v = 0; v < n; ++v)
      for (int d = 0; d < 3; ++d)
        grad[3*v+d] = c->mass[v] * ih2 * (x[3*v+d] - s[3*v+d]) - f[3*v+d] + dmp[3*v+d] - tmp[3*v+d];
    free(f); free(dmp); free(tmp);
  }
  free(Ps); free(Pa); free(Pb); free(Pv);
  return gval;
}

static double residual_length(const oracle_cell *c, const double *grad) {
  double r = 0, h2 = c->h * c->h;
  for (int v = 0; v < c->n; ++v)
    for (int d = 0; d < 3; ++d) { double q = fabs(grad[3*v+d]) * h2 / c->mass[v]; if (q > r) r = q; }
  return r;
}
static double dotn(const double *a, const double *b, size_t m) { double s = 0; for (size_t i = 0; i < m; ++i) s += a[i]*b[i]; return s; }

/* One converged time step of ONE cell.  Returns the number of iterations taken.
 * Optional traces: gtrace[max_iters+1] objective after each accepted iterate (gtrace[0] = g(s)),
 * rtrace[max_iters+1] residual lengths, iterates [(max_iters+1)][n][3]. */
int oracle_step_cell_converged(const oracle_cell *c, double *pos, double *vel, const double *fext,
                               double tol, int max_iters, int history, int line_search,
                               double *gtrace, double *rtrace, double *iterates) {
  int n = c->n; size_t m3 = 3*(size_t)n; double h = c->h;
  if (history < 0) history = 0;
  double *s = (double*)malloc(sizeof(double)*m3), *x = (double*)malloc(sizeof(double)*m3);
  double *grad = (double*)malloc(sizeof(double)*m3), *gnew = (double*)malloc(sizeof(double)*m3);
  double *q = (double*)malloc(sizeof(double)*m3), *r = (double*)malloc(sizeof(double)*m3);
  double *xt = (double*)malloc(sizeof(double)*m3);
  double *S = (double*)malloc(sizeof(double)*m3*(size_t)(history ? history : 1));
  double *Y = (double*)malloc(sizeof(double)*m3*(size_t)(history ? history : 1));
  double *rho = (double*)malloc(sizeof(double)*(size_t)(history ? history : 1));
  double *alpha = (double*)malloc(sizeof(double)*(size_t)(history ? history : 1));
  for (int v = 0; v < n; ++v)
    for (int d = 0; d < 3; ++d)
      s[3*v+d] = pos[3*v+d] + h * vel[3*v+d] + h*h * fext[3*v+d] / c->mass[v];
  memcpy(x, s, sizeof(double)*m3);
  double gval = oracle_objective(c, x, s, pos, grad);
  int npairs = 0, k = 0;
  if (gtrace) gtrace[0] = gval;
  if (rtrace) rtrace[0] = residual_length(c, grad);
  if (iterates) memcpy(iterates, x, sizeof(double)*m3);
  while (k < max_iters && residual_length(c, grad) > tol) {
    /* two-loop recursion; pair j of age a (0 = newest) sits in slot (k-1-a) % history */
    memcpy(q, grad, sizeof(double)*m3);
    for (int a = 0; a < npairs; ++a) {
      int j = (k - 1 - a) % history;
      alpha[j] = rho[j] * dotn(S + j*m3, q, m3);
      for (size_t i = 0; i < m3; ++i) q[i] -= alpha[j] * Y[j*m3 + i];
    }
    oracle_solve(c, q, r);                                   /* r = A_sys^-1 q */
    for (int a = npairs - 1; a >= 0; --a) {
      int j = (k - 1 - a) % history;
      double beta = rho[j] * dotn(Y + j*m3, r, m3);
      for (size_t i = 0; i < m3; ++i) r[i] += S[j*m3 + i] * (alpha[j] - beta);
    }
    /* direction p = -r.  The distance energies are only piecewise smooth, so a quasi-Newton
     * direction can fail to descend: then the history is dropped and p = -A_sys^-1 grad g, which
     * always descends (A_sys is SPD). */
    double slope = -dotn(grad, r, m3), step = 1.0, gtry;
    if (npairs > 0 && !(slope < 0.0)) {
      npairs = 0;
      oracle_solve(c, grad, r);
      slope = -dotn(grad, r, m3);
    }
    for (;;) {
      for (size_t i = 0; i < m3; ++i) xt[i] = x[i] - step * r[i];
      gtry = oracle_objective(c, xt, s, pos, gnew);
      /* sufficient decrease, up to the rounding of g itself (near convergence the decrease is
       * below fp64 resolution of g and an exact test would reject every step) */
      if (!line_search || gtry <= gval + 1e-4 * step * slope + 8.0 * 2.220446049250313e-16 * fabs(gval) || step < 1e-6) break;
      step *= 0.5;
    }
    if (history > 0) {
      int j = k % history;
      double sy = 0;
      for (size_t i = 0; i < m3; ++i) { S[j*m3+i] = xt[i] - x[i]; Y[j*m3+i] = gnew[i] - grad[i]; sy += S[j*m3+i]*Y[j*m3+i]; }
      if (sy > 1e-300) { rho[j] = 1.0 / sy; if (npairs < history) ++npairs; }
      else npairs = 0;                                       /* curvature condition failed: restart */
    }
    memcpy(x, xt, sizeof(double)*m3); memcpy(grad, gnew, sizeof(double)*m3); gval = gtry;
    ++k;
    if (gtrace) gtrace[k] = gval;
    if (rtrace) rtrace[k] = residual_length(c, grad);
    if (iterates) memcpy(iterates + (size_t)k*m3, x, sizeof(double)*m3);
  }
  for (size_t i = 0; i < m3; ++i) { vel[i] = (x[i] - pos[i]) / h; pos[i] = x[i]; }
  free(s); free(x); free(grad); free(gnew); free(q); free(r); free(xt); free(S); free(Y); free(rho); free(alpha);
  return k;
}

/* All cells, OpenMP over cells; iters_out[n_cells] receives the iterations each cell took. */
void oracle_step_converged(const oracle_cell *c, int n_cells, double *pos, double *vel,
                           const double *fext, double tol, int max_iters, int history,
                           int32_t *iters_out) {
  size_t stride = 3*(size_t)c->n;
#pragma omp parallel for schedule(dynamic, 1)
  for (int i = 0; i < n_cells; ++i) {
    int it = oracle_step_cell_converged(c, pos + i*stride, vel + i*stride, fext + i*stride, tol,
                                        max_iters, history, 1, NULL, NULL, NULL);
    if (iters_out) iters_out[i] = it;
  }
}

/* All cells of one type, [n_cells][n][3] fp64 arrays, OpenMP over cells only. */
void oracle_step(const oracle_cell *c, int n_cells, double *pos, double *vel, const double *fext,
                 int n_iters) {
  size_t stride = 3*(size_t)c->n;
#pragma omp parallel for schedule(dynamic, 1)
  for (int i = 0; i < n_cells; ++i)
    oracle_step_cell(c, pos + i*stride, vel + i*stride, fext + i*stride, n_iters, NULL, NULL);
}

int oracle_num_threads(void) {
#ifdef _OPENMP
  return omp_get_max_threads();
#else
  return 1;
#endif
}
