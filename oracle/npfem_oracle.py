"""ctypes front end of the fp64 CPU oracle (oracle/npfem_oracle.c).

TEST INFRASTRUCTURE, NOT THE PRODUCT: only tests/, bench.py's cpu_baseline / --impl reference legs
and __graft_entry__.smoke() may import this module.  It shares no code with, and never imports,
paper_2011_04332_b200.  All arithmetic happens in the C file; this module only marshals arrays.
Algorithm and citations: see the header of npfem_oracle.c and DESIGN.md.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

from . import build as _build

MATERIAL_FIELDS = ("cell_mass", "k_strain", "s_min", "s_max", "k_area", "a_min", "a_max",
                   "k_bend", "w_volume", "v_min", "v_max", "c_alpha", "c_beta", "w_collision",
                   "d_collision", "strain_hardening", "w_garea", "ga_min", "ga_max")


class _Material(C.Structure):
    _fields_ = [(f, C.c_double) for f in MATERIAL_FIELDS]


_lib = None
_dp = C.POINTER(C.c_double)
_ip = C.POINTER(C.c_int32)


def lib():
    global _lib
    if _lib is None:
        path = _build.build()
        L = C.CDLL(path)
        L.oracle_create.restype = C.c_int
        L.oracle_create.argtypes = [C.c_int, C.c_int, _ip, _dp, C.POINTER(_Material), C.c_double,
                                    C.POINTER(C.c_void_p)]
        L.oracle_destroy.argtypes = [C.c_void_p]
        L.oracle_n_hinges.restype = C.c_int
        L.oracle_n_hinges.argtypes = [C.c_void_p]
        L.oracle_rest_volume.restype = C.c_double
        L.oracle_rest_volume.argtypes = [C.c_void_p]
        for name in ("oracle_get_hinges",):
            getattr(L, name).argtypes = [C.c_void_p, _ip]
        for name in ("oracle_get_K", "oracle_get_masses", "oracle_get_areas", "oracle_get_G",
                     "oracle_get_system", "oracle_get_elastic_laplacian"):
            getattr(L, name).argtypes = [C.c_void_p, _dp]
        L.oracle_get_hinge_weights.argtypes = [C.c_void_p, _dp, _dp]
        L.oracle_svd32.argtypes = [_dp, _dp, _dp, _dp]
        L.oracle_project_strain.argtypes = [_dp, C.c_double, C.c_double, _dp]
        L.oracle_project_area.argtypes = [_dp, C.c_double, C.c_double, _dp]
        L.oracle_closest_on_hyperbola.argtypes = [C.c_double, C.c_double, C.c_double, _dp]
        L.oracle_project_bend.argtypes = [_dp, C.c_double, _dp]
        L.oracle_volume.restype = C.c_double
        L.oracle_volume.argtypes = [C.c_int, _ip, _dp]
        L.oracle_volume_closed.restype = C.c_double
        L.oracle_volume_closed.argtypes = [C.c_int, C.c_int, _ip, _dp]
        L.oracle_volume_grad.argtypes = [C.c_int, C.c_int, _ip, _dp, _dp]
        L.oracle_project_volume.restype = C.c_int
        L.oracle_project_volume.argtypes = [C.c_int, C.c_int, _ip, _dp, C.c_double, C.c_double, _dp]
        L.oracle_area_total.restype = C.c_double
        L.oracle_area_total.argtypes = [C.c_int, _ip, _dp]
        L.oracle_area_grad.argtypes = [C.c_int, C.c_int, _ip, _dp, _dp]
        L.oracle_area_hessian.argtypes = [C.c_int, C.c_int, _ip, _dp, _dp]
        L.oracle_project_garea.restype = C.c_int
        L.oracle_project_garea.argtypes = [C.c_int, C.c_int, _ip, _dp, C.c_double, C.c_double, _dp]
        L.oracle_rest_area.restype = C.c_double
        L.oracle_rest_area.argtypes = [C.c_void_p]
        L.oracle_garea_local.restype = C.c_double
        L.oracle_garea_local.argtypes = [C.c_void_p, _dp, _dp]
        L.oracle_deformation_gradient.argtypes = [C.c_void_p, C.c_int, _dp, _dp]
        L.oracle_local.argtypes = [C.c_void_p, _dp, _dp, _dp, _dp, _dp]
        L.oracle_rhs.argtypes = [C.c_void_p, _dp, _dp, _dp, _dp, _dp, _dp]
        L.oracle_solve.argtypes = [C.c_void_p, _dp, _dp]
        L.oracle_energy.restype = C.c_double
        L.oracle_energy.argtypes = [C.c_void_p, _dp, _dp, _dp, _dp, _dp, _dp, _dp]
        L.oracle_fint.argtypes = [C.c_void_p, _dp, _dp]
        L.oracle_project_collision.argtypes = [_dp, _dp, _dp, C.c_double, _dp]
        L.oracle_step_cell_collide.argtypes = [C.c_void_p, _dp, _dp, _dp, _dp, _dp, C.c_int, _dp, _dp]
        L.oracle_step_collide.argtypes = [C.c_void_p, C.c_int, _dp, _dp, _dp, _dp, _dp, C.c_int]
        L.oracle_vertex_areas.argtypes = [C.c_void_p, _dp, _dp]
        L.oracle_damping_rhs.argtypes = [C.c_void_p, _dp, _dp]
        L.oracle_dissipation.restype = C.c_double
        L.oracle_dissipation.argtypes = [C.c_void_p, _dp, _dp]
        L.oracle_step_cell.argtypes = [C.c_void_p, _dp, _dp, _dp, C.c_int, _dp, _dp]
        L.oracle_objective.restype = C.c_double
        L.oracle_objective.argtypes = [C.c_void_p, _dp, _dp, _dp, _dp]
        L.oracle_step_cell_converged.restype = C.c_int
        L.oracle_step_cell_converged.argtypes = [C.c_void_p, _dp, _dp, _dp, C.c_double, C.c_int,
                                                 C.c_int, C.c_int, _dp, _dp, _dp]
        L.oracle_step_converged.argtypes = [C.c_void_p, C.c_int, _dp, _dp, _dp, C.c_double, C.c_int,
                                            C.c_int, _ip]
        L.oracle_step.argtypes = [C.c_void_p, C.c_int, _dp, _dp, _dp, C.c_int]
        L.oracle_num_threads.restype = C.c_int
        _lib = L
    return _lib


def _d(a):
    return a.ctypes.data_as(_dp)


def _i(a):
    return a.ctypes.data_as(_ip)


def _f64(a, shape=None):
    a = np.ascontiguousarray(a, dtype=np.float64)
    if shape is not None:
        a = a.reshape(shape)
    return a


def num_threads() -> int:
    return int(lib().oracle_num_threads())


# ------------------------------------------------------------------ stand-alone projections
def svd32(F):
    F = _f64(F, (3, 2))
    U, S, V = np.empty((3, 2)), np.empty(2), np.empty((2, 2))
    lib().oracle_svd32(_d(F), _d(U), _d(S), _d(V))
    return U, S, V


def project_strain(F, s_min, s_max):
    F = _f64(F, (3, 2)); P = np.empty((3, 2))
    lib().oracle_project_strain(_d(F), float(s_min), float(s_max), _d(P))
    return P


def project_area(F, a_min, a_max):
    F = _f64(F, (3, 2)); P = np.empty((3, 2))
    lib().oracle_project_area(_d(F), float(a_min), float(a_max), _d(P))
    return P


def closest_on_hyperbola(s1, s2, a):
    o = np.empty(2)
    lib().oracle_closest_on_hyperbola(float(s1), float(s2), float(a), _d(o))
    return o


def project_bend(k, r):
    k = _f64(k, (3,)); P = np.empty(3)
    lib().oracle_project_bend(_d(k), float(r), _d(P))
    return P


def project_collision(x, q, nrm, d):
    x, q, nrm = _f64(x, (3,)), _f64(q, (3,)), _f64(nrm, (3,)); p = np.empty(3)
    lib().oracle_project_collision(_d(x), _d(q), _d(nrm), float(d), _d(p))
    return p


def volume(tris, x):
    tris = np.ascontiguousarray(tris, dtype=np.int32); x = _f64(x)
    return float(lib().oracle_volume(tris.shape[0], _i(tris), _d(x)))


def volume_grad(tris, x):
    tris = np.ascontiguousarray(tris, dtype=np.int32); x = _f64(x)
    g = np.empty_like(x)
    lib().oracle_volume_grad(x.shape[0], tris.shape[0], _i(tris), _d(x), _d(g))
    return g


def project_volume(tris, x, v_star, v0):
    tris = np.ascontiguousarray(tris, dtype=np.int32); x = _f64(x)
    P = np.empty_like(x)
    its = lib().oracle_project_volume(x.shape[0], tris.shape[0], _i(tris), _d(x), float(v_star),
                                      float(v0), _d(P))
    return P, int(its)


def area_total(tris, x):
    """Total surface area (global-area term, reading A-24)."""
    tris = np.ascontiguousarray(tris, dtype=np.int32); x = _f64(x)
    return float(lib().oracle_area_total(tris.shape[0], _i(tris), _d(x)))


def area_grad(tris, x):
    tris = np.ascontiguousarray(tris, dtype=np.int32); x = _f64(x)
    g = np.empty_like(x)
    lib().oracle_area_grad(x.shape[0], tris.shape[0], _i(tris), _d(x), _d(g))
    return g


def area_hessian(tris, x):
    tris = np.ascontiguousarray(tris, dtype=np.int32); x = _f64(x)
    H = np.empty((3 * x.shape[0], 3 * x.shape[0]))
    lib().oracle_area_hessian(x.shape[0], tris.shape[0], _i(tris), _d(x), _d(H))
    return H


def project_garea(tris, x, a_star, a0):
    """Closest configuration with total area a_star (Newton on the KKT system); (P, iterations)."""
    tris = np.ascontiguousarray(tris, dtype=np.int32); x = _f64(x)
    P = np.empty_like(x)
    its = lib().oracle_project_garea(x.shape[0], tris.shape[0], _i(tris), _d(x), float(a_star),
                                     float(a0), _d(P))
    return P, int(its)


# ------------------------------------------------------------------ one cell type
class OracleCell:
    """One cell TYPE: topology + rest shape + material + dt (SURVEY.md 8(c) "Create")."""

    def __init__(self, tris, rest_xyz, material: dict, dt: float):
        self.tris = np.ascontiguousarray(tris, dtype=np.int32)
        self.rest = _f64(rest_xyz)
        self.n = self.rest.shape[0]
        self.T = self.tris.shape[0]
        self.dt = float(dt)
        self.material = dict(material)
        m = _Material(**{k: float(material.get(k, 0.0)) for k in MATERIAL_FIELDS})
        h = C.c_void_p()
        rc = lib().oracle_create(self.n, self.T, _i(self.tris), _d(self.rest), C.byref(m),
                                 self.dt, C.byref(h))
        if rc != 0:
            raise ValueError(f"oracle_create failed with code {rc}")
        self._h = h
        self.H = int(lib().oracle_n_hinges(h))

    def __del__(self):
        h = getattr(self, "_h", None)
        if h is not None and _lib is not None:
            _lib.oracle_destroy(h)
            self._h = None

    # ---- create-time data
    @property
    def rest_volume(self):
        return float(lib().oracle_rest_volume(self._h))

    def hinges(self):
        o = np.empty((self.H, 4), dtype=np.int32); lib().oracle_get_hinges(self._h, _i(o)); return o

    def hinge_rows(self):
        o = np.empty((self.H, 4)); lib().oracle_get_K(self._h, _d(o)); return o

    def hinge_weights(self):
        w, r = np.empty(self.H), np.empty(self.H)
        lib().oracle_get_hinge_weights(self._h, _d(w), _d(r)); return w, r

    def masses(self):
        o = np.empty(self.n); lib().oracle_get_masses(self._h, _d(o)); return o

    def areas(self):
        o = np.empty(self.T); lib().oracle_get_areas(self._h, _d(o)); return o

    def G(self):
        o = np.empty((self.T, 2, 3)); lib().oracle_get_G(self._h, _d(o)); return o

    def system_matrix(self):
        o = np.empty((self.n, self.n)); lib().oracle_get_system(self._h, _d(o)); return o

    def elastic_laplacian(self):
        """L_el = sum_t (w_s+w_a) G^T G + sum_h w_h K^T K (the stiffness the c_beta damping uses)."""
        o = np.empty((self.n, self.n)); lib().oracle_get_elastic_laplacian(self._h, _d(o)); return o

    # ---- pieces of the step
    def deformation_gradient(self, t, x):
        x = _f64(x); F = np.empty((3, 2))
        lib().oracle_deformation_gradient(self._h, int(t), _d(x), _d(F)); return F

    def local(self, x):
        x = _f64(x)
        Ps, Pa = np.empty((self.T, 3, 2)), np.empty((self.T, 3, 2))
        Pb, Pv = np.empty((self.H, 3)), np.empty((self.n, 3))
        lib().oracle_local(self._h, _d(x), _d(Ps), _d(Pa), _d(Pb), _d(Pv))
        return Ps, Pa, Pb, Pv

    def rhs(self, s, proj):
        s = _f64(s); b = np.empty((self.n, 3))
        Ps, Pa, Pb, Pv = (_f64(p) for p in proj)
        lib().oracle_rhs(self._h, _d(s), _d(Ps), _d(Pa), _d(Pb), _d(Pv), _d(b)); return b

    def solve(self, b):
        b = _f64(b); x = np.empty((self.n, 3))
        lib().oracle_solve(self._h, _d(b), _d(x)); return x

    def energy(self, x, s, proj, parts=False):
        x, s = _f64(x), _f64(s)
        Ps, Pa, Pb, Pv = (_f64(p) for p in proj)
        e = np.empty(5)
        tot = float(lib().oracle_energy(self._h, _d(x), _d(s), _d(Ps), _d(Pa), _d(Pb), _d(Pv), _d(e)))
        return (tot, e) if parts else tot

    def fint(self, x):
        x = _f64(x); f = np.empty((self.n, 3))
        lib().oracle_fint(self._h, _d(x), _d(f)); return f

    def damping_rhs(self, xn):
        """(C/h) x_n with C = c_alpha M + c_beta L_el: what the damping adds to the rhs (A-20)."""
        xn = _f64(xn); b = np.zeros((self.n, 3))
        lib().oracle_damping_rhs(self._h, _d(xn), _d(b)); return b

    def dissipation(self, x, xn):
        x, xn = _f64(x), _f64(xn)
        return float(lib().oracle_dissipation(self._h, _d(x), _d(xn)))

    # ---- whole steps
    def step_cell(self, pos, vel, fext, n_iters, trace=False):
        """One step of one cell. Returns (pos, vel[, iterates, energies]); inputs are not modified."""
        pos, vel, fext = _f64(pos).copy(), _f64(vel).copy(), _f64(fext)
        if trace:
            its = np.empty((n_iters + 1, self.n, 3)); en = np.empty(2 * n_iters)
            lib().oracle_step_cell(self._h, _d(pos), _d(vel), _d(fext), int(n_iters), _d(its), _d(en))
            return pos, vel, its, en
        lib().oracle_step_cell(self._h, _d(pos), _d(vel), _d(fext), int(n_iters), None, None)
        return pos, vel

    # ---- collisions and area per vertex (NEXT-3, reading A-22)
    def step_cell_collide(self, pos, vel, fext, q, nrm, n_iters, trace=False):
        pos, vel, fext = _f64(pos).copy(), _f64(vel).copy(), _f64(fext)
        q, nrm = _f64(q), _f64(nrm)
        if trace:
            its = np.empty((n_iters + 1, self.n, 3)); en = np.empty(2 * n_iters)
            lib().oracle_step_cell_collide(self._h, _d(pos), _d(vel), _d(fext), _d(q), _d(nrm),
                                           int(n_iters), _d(its), _d(en))
            return pos, vel, its, en
        lib().oracle_step_cell_collide(self._h, _d(pos), _d(vel), _d(fext), _d(q), _d(nrm),
                                       int(n_iters), None, None)
        return pos, vel

    def step_collide(self, pos, vel, fext, q, nrm, n_iters):
        pos = np.array(pos, dtype=np.float64, order="C", copy=True)
        vel = np.array(vel, dtype=np.float64, order="C", copy=True)
        fext, q, nrm = _f64(fext), _f64(q), _f64(nrm)
        lib().oracle_step_collide(self._h, pos.shape[0], _d(pos), _d(vel), _d(fext), _d(q), _d(nrm),
                                  int(n_iters))
        return pos, vel

    def rest_area(self):
        return float(lib().oracle_rest_area(self._h))

    def garea_local(self, x):
        """(P_g, energy) of the global-area term at x (reading A-24); P_g = x, 0 when w_garea = 0."""
        x = _f64(x); P = np.empty_like(x)
        e = float(lib().oracle_garea_local(self._h, _d(x), _d(P)))
        return P, e

    def vertex_areas(self, x):
        x = _f64(x); a = np.empty(self.n)
        lib().oracle_vertex_areas(self._h, _d(x), _d(a)); return a

    # ---- converged solve (NEXT-1, reading A-21)
    def objective(self, x, s, xn, grad=False):
        """g(x) of the implicit-Euler step [and its gradient]."""
        x, s, xn = _f64(x), _f64(s), _f64(xn)
        if grad:
            gr = np.empty((self.n, 3))
            return float(lib().oracle_objective(self._h, _d(x), _d(s), _d(xn), _d(gr))), gr
        return float(lib().oracle_objective(self._h, _d(x), _d(s), _d(xn), None))

    def step_cell_converged(self, pos, vel, fext, tol, max_iters=200, history=5, line_search=True,
                            trace=False):
        """One converged step of one cell: L-BFGS seeded with A_sys^-1 + backtracking line search.
        Returns (pos, vel, iters[, g_trace, res_trace, iterates])."""
        pos, vel, fext = _f64(pos).copy(), _f64(vel).copy(), _f64(fext)
        if trace:
            gt, rt = np.full(max_iters + 1, np.nan), np.full(max_iters + 1, np.nan)
            its = np.full((max_iters + 1, self.n, 3), np.nan)
            k = lib().oracle_step_cell_converged(self._h, _d(pos), _d(vel), _d(fext), float(tol),
                                                 int(max_iters), int(history), int(line_search),
                                                 _d(gt), _d(rt), _d(its))
            return pos, vel, int(k), gt[: k + 1], rt[: k + 1], its[: k + 1]
        k = lib().oracle_step_cell_converged(self._h, _d(pos), _d(vel), _d(fext), float(tol),
                                             int(max_iters), int(history), int(line_search),
                                             None, None, None)
        return pos, vel, int(k)

    def step_converged(self, pos, vel, fext, tol, max_iters=200, history=5):
        """One converged step of N cells [N,n,3]; returns (pos, vel, iters[N])."""
        pos = np.array(pos, dtype=np.float64, order="C", copy=True)
        vel = np.array(vel, dtype=np.float64, order="C", copy=True)
        fext = _f64(fext)
        its = np.zeros(pos.shape[0], dtype=np.int32)
        lib().oracle_step_converged(self._h, pos.shape[0], _d(pos), _d(vel), _d(fext), float(tol),
                                    int(max_iters), int(history), _i(its))
        return pos, vel, its

    def step(self, pos, vel, fext, n_iters):
        """One step of N cells, arrays [N,n,3]; fp32 inputs are promoted to fp64. Returns (pos, vel) fp64."""
        pos = np.array(pos, dtype=np.float64, order="C", copy=True)
        vel = np.array(vel, dtype=np.float64, order="C", copy=True)
        fext = _f64(fext)
        assert pos.shape == vel.shape == fext.shape and pos.shape[1:] == (self.n, 3)
        lib().oracle_step(self._h, pos.shape[0], _d(pos), _d(vel), _d(fext), int(n_iters))
        return pos, vel
