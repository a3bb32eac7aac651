"""Pins of the fp64 CPU oracle against things OTHER than itself (no GPU needed).

The paper prints no worked example (PAPER.md has no numeric vector or table for the solid solver),
so every pin is an invariant, a closed form, a library routine (LAPACK SVD, scipy optimisers),
finite differences or brute force on tiny inputs -- SURVEY.md 8(c) pins P-1 ... P-12 plus extras.
Each is chosen so that a plausible mistake in the oracle (dropped term, wrong sign or index,
transposed operand) fails at least one of them.
"""
import numpy as np
import pytest
from scipy import optimize

import workloads as W
from oracle import npfem_oracle as O

DT = 0.1


def make_cell(kind="rbc", level=2, **over):
    rest, tris = W.rest_shape(kind, level)
    mat = W.default_material(rest, tris, **over)
    return O.OracleCell(tris, rest, mat, DT), rest, tris, mat


def random_rotation(rng):
    q = rng.standard_normal(4)
    q /= np.linalg.norm(q)
    return W.quat_to_rot(q[None])[0]


# ----------------------------------------------------------------------------- SVD / projections
def test_svd32_matches_lapack():
    rng = np.random.default_rng(1)
    for _ in range(200):
        F = rng.standard_normal((3, 2)) * rng.uniform(0.1, 3.0)
        U, S, V = O.svd32(F)
        s_ref = np.linalg.svd(F, compute_uv=False)
        assert np.allclose(S, s_ref, rtol=1e-13, atol=1e-14)
        assert np.allclose(U @ np.diag(S) @ V.T, F, atol=1e-13)
        assert np.allclose(U.T @ U, np.eye(2), atol=1e-13)
        assert np.allclose(V.T @ V, np.eye(2), atol=1e-13)
        assert S[0] >= S[1] >= 0


def _strain_ref(F, lo, hi):
    U, S, Vt = np.linalg.svd(F, full_matrices=False)
    return U @ np.diag(np.clip(S, lo, hi)) @ Vt


def test_strain_projection_matches_lapack_formula():
    rng = np.random.default_rng(2)
    for lo, hi in [(1.0, 1.0), (0.8, 1.3), (0.0, 0.5)]:
        for _ in range(50):
            F = rng.standard_normal((3, 2))
            assert np.allclose(O.project_strain(F, lo, hi), _strain_ref(F, lo, hi), atol=1e-12)


def _param_P(z):
    """3x2 matrix U diag(d) V^T from 6 free parameters (3 Euler angles, 1 angle, 2 values)."""
    a, b, c, th, d0, d1 = z
    Rz = lambda t: np.array([[np.cos(t), -np.sin(t), 0], [np.sin(t), np.cos(t), 0], [0, 0, 1]])
    Ry = lambda t: np.array([[np.cos(t), 0, np.sin(t)], [0, 1, 0], [-np.sin(t), 0, np.cos(t)]])
    R = Rz(a) @ Ry(b) @ Rz(c)
    V = np.array([[np.cos(th), -np.sin(th)], [np.sin(th), np.cos(th)]])
    return R[:, :2], np.array([d0, d1]), V


def test_strain_projection_vs_brute_force():
    """P-5: minimise ||F-P|| over {P : singular values in [lo,hi]} with a generic optimiser."""
    rng = np.random.default_rng(3)
    for lo, hi in [(1.0, 1.0), (0.8, 1.3)]:
        for _ in range(6):
            F = rng.standard_normal((3, 2)) * 1.2
            P = O.project_strain(F, lo, hi)
            d_or = np.linalg.norm(F - P)
            sv = np.linalg.svd(P, compute_uv=False)
            assert np.all(sv >= lo - 1e-12) and np.all(sv <= hi + 1e-12)

            def obj(z):
                U, d, V = _param_P(z)
                d = lo + (hi - lo) * (0.5 + 0.5 * np.sin(d))      # smooth map onto the band
                return np.sum((F - U @ np.diag(d) @ V.T) ** 2)

            best = np.inf
            for _ in range(24):
                z0 = rng.uniform(-np.pi, np.pi, 6)
                r = optimize.minimize(obj, z0, method="BFGS", options=dict(gtol=1e-12))
                best = min(best, np.sqrt(r.fun))
            assert d_or <= best + 1e-9          # the oracle is never worse than brute force
            assert best <= d_or + 1e-5          # and brute force finds (about) the same distance


def _hyperbola_brute(s1, s2, a):
    q = np.sqrt(a)
    t = np.linspace(-4.0, 4.0, 400001)          # BOTH signs of t: the whole branch
    d2 = (q * np.exp(t) - s1) ** 2 + (q * np.exp(-t) - s2) ** 2
    i = int(np.argmin(d2))
    lo, hi = t[max(i - 1, 0)], t[min(i + 1, len(t) - 1)]
    r = optimize.minimize_scalar(lambda u: (q * np.exp(u) - s1) ** 2 + (q * np.exp(-u) - s2) ** 2,
                                 bounds=(lo, hi), method="bounded", options=dict(xatol=1e-14))
    return np.array([q * np.exp(r.x), q * np.exp(-r.x)]), r.fun


def test_hyperbola_closest_point_vs_scan():
    """P-5 (area): 1-D brute-force scan over the hyperbola s1 s2 = a in sigma space."""
    rng = np.random.default_rng(4)
    cases = [(1.0, 1.0, 1.0), (1.00001, 0.99998, 1.0), (3.0, 2.9, 1.0), (0.3, 0.2, 1.0),
             (4.0, 0.2, 1.0), (2.5, 2.4999, 0.7), (5.0, 4.0, 1.3)]
    cases += [tuple(sorted(rng.uniform(0.2, 4.0, 2), reverse=True)) + (rng.uniform(0.5, 1.5),)
              for _ in range(150)]
    for s1, s2, a in cases:
        o = O.closest_on_hyperbola(s1, s2, a)
        assert abs(o[0] * o[1] - a) < 1e-12 * max(1.0, a)
        ref, d2ref = _hyperbola_brute(s1, s2, a)
        d2 = (o[0] - s1) ** 2 + (o[1] - s2) ** 2
        assert d2 <= d2ref + 1e-12, (s1, s2, a)
        assert np.allclose(o, ref, atol=2e-6), (s1, s2, a)


def test_area_projection_matrix_brute_force():
    """P-5 (area), in matrix space: min ||F-P|| s.t. sigma1(P) sigma2(P) = a."""
    rng = np.random.default_rng(5)
    for _ in range(4):
        F = rng.standard_normal((3, 2)) * 1.1
        a = 1.0
        P = O.project_area(F, a, a)
        sv = np.linalg.svd(P, compute_uv=False)
        assert abs(sv[0] * sv[1] - a) < 1e-11
        d_or = np.linalg.norm(F - P)

        def obj(z):
            U, _, V = _param_P(np.concatenate([z[:4], [1, 1]]))
            d = np.array([np.sqrt(a) * np.exp(z[4]), np.sqrt(a) * np.exp(-z[4])])
            return np.sum((F - U @ np.diag(d) @ V.T) ** 2)

        best = np.inf
        for _ in range(24):
            z0 = np.concatenate([rng.uniform(-np.pi, np.pi, 4), rng.uniform(-1, 1, 1)])
            r = optimize.minimize(obj, z0, method="BFGS", options=dict(gtol=1e-12))
            best = min(best, np.sqrt(r.fun))
        assert d_or <= best + 1e-9
        assert best <= d_or + 1e-5


def test_area_projection_inside_band_is_identity():
    F = np.array([[1.1, 0.0], [0.0, 0.95], [0.0, 0.0]])
    assert np.array_equal(O.project_area(F, 0.9, 1.2), F)
    P = O.project_area(F, 1.2, 1.3)               # below the band: pushed to a = 1.2
    sv = np.linalg.svd(P, compute_uv=False)
    assert abs(sv[0] * sv[1] - 1.2) < 1e-12


def test_bend_projection_is_radial_projection_onto_sphere():
    rng = np.random.default_rng(6)
    for _ in range(20):
        k = rng.standard_normal(3)
        r = rng.uniform(0.1, 2.0)
        P = O.project_bend(k, r)
        assert abs(np.linalg.norm(P) - r) < 1e-14
        # brute force: no point of the sphere is closer
        u = rng.standard_normal((20000, 3))
        u *= r / np.linalg.norm(u, axis=1, keepdims=True)
        assert np.linalg.norm(P - k) <= np.linalg.norm(u - k, axis=1).min() + 1e-12
    assert np.array_equal(O.project_bend(np.zeros(3), 1.0), np.zeros(3))     # ||k|| < 1e-30: P = k
    assert np.allclose(O.project_bend(np.array([0, 0, 2.0]), 0.0), 0.0)      # flat rest hinge


TET_V = np.array([[0, 0, 0], [1, 0, 0], [0, 1, 0], [0, 0, 1]], dtype=np.float64)
TET_T = np.array([[0, 2, 1], [0, 1, 3], [0, 3, 2], [1, 2, 3]], dtype=np.int32)
OCT_V = np.array([[1, 0, 0], [-1, 0, 0], [0, 1, 0], [0, -1, 0], [0, 0, 1], [0, 0, -1]], dtype=np.float64)
OCT_T = np.array([[0, 2, 4], [2, 1, 4], [1, 3, 4], [3, 0, 4], [2, 0, 5], [1, 2, 5], [3, 1, 5], [0, 3, 5]],
                 dtype=np.int32)


def test_volume_textbook_values_and_gradient():
    assert abs(O.volume(TET_T, TET_V) - 1.0 / 6.0) < 1e-15
    assert abs(O.volume(OCT_T, OCT_V) - 4.0 / 3.0) < 1e-15
    v, t = W.icosphere(3)
    assert abs(O.volume(t, v) - 4 * np.pi / 3) < 0.02 * 4 * np.pi / 3     # inscribed polyhedron
    assert O.volume(t, v) < 4 * np.pi / 3
    # translation invariance of V for a closed surface
    assert abs(O.volume(t, v + np.array([50.0, -20.0, 7.0])) - O.volume(t, v)) < 1e-9
    # gradient vs central finite differences
    rng = np.random.default_rng(7)
    x = OCT_V + 0.1 * rng.standard_normal(OCT_V.shape)
    g = O.volume_grad(OCT_T, x)
    for i in range(6):
        for d in range(3):
            e = np.zeros_like(x); e[i, d] = 1e-6
            fd = (O.volume(OCT_T, x + e) - O.volume(OCT_T, x - e)) / 2e-6
            assert abs(fd - g[i, d]) < 1e-9
    assert np.allclose(g.sum(axis=0), 0, atol=1e-14)          # sum grad V = 0 (translation)


@pytest.mark.parametrize("verts,tris", [(TET_V, TET_T), (OCT_V, OCT_T)])
def test_volume_projection_vs_slsqp(verts, tris):
    """P-5 (volume): constrained minimiser on a tetrahedron / octahedron (12-18 unknowns)."""
    rng = np.random.default_rng(8)
    v0 = O.volume(tris, verts)
    for scale in (0.85, 1.05, 1.2):
        x = verts * scale + 0.05 * rng.standard_normal(verts.shape) + np.array([3.0, -2.0, 1.0])
        P, its = O.project_volume(tris, x, v0, v0)
        assert abs(O.volume(tris, P - P[0]) - v0) < 1e-13
        cons = dict(type="eq", fun=lambda z: O.volume(tris, z.reshape(-1, 3) - x[0]) - v0)
        r = optimize.minimize(lambda z: 0.5 * np.sum((z - x.ravel()) ** 2), x.ravel(),
                              jac=lambda z: z - x.ravel(), constraints=[cons], method="SLSQP",
                              options=dict(ftol=1e-16, maxiter=500))
        d_or, d_ref = np.linalg.norm(P - x), np.sqrt(2 * r.fun)
        assert abs(d_or - d_ref) < 1e-7 * max(d_ref, 1e-3)
        assert np.abs(P.ravel() - r.x).max() < 1e-6


# ----------------------------------------------------------------------------- create-time data
def test_P9_hinge_rows_vanish_on_constants_and_on_flat_hinges():
    """P-9: sum_i K_i = 0 for every hinge, and sum_i K_i X_i = 0 for a flat hinge.

    The cotangents only depend on the interior angles of the two triangles, so unfolding a hinge
    of the icosahedron into its edge-plane keeps its row K and must give a zero hinge vector.
    """
    c, rest, tris, _ = make_cell("rbc", 2)
    assert np.abs(c.hinge_rows().sum(axis=1)).max() < 1e-12
    v, t = W.icosphere(0)
    c0 = O.OracleCell(t, v, W.default_material(v, t), DT)
    st0, K0 = c0.hinges(), c0.hinge_rows()
    rng = np.random.default_rng(9)
    for h in range(c0.H):
        x0, x1, x2, x3 = (v[i] for i in st0[h])
        e = x1 - x0
        n = np.cross(e, rng.standard_normal(3)); n /= np.linalg.norm(n)

        def unfold(p):
            along = np.dot(p - x0, e) / np.dot(e, e)
            return along, np.linalg.norm((p - x0) - along * e)

        a2, h2 = unfold(x2); a3, h3 = unfold(x3)
        y2 = x0 + a2 * e + h2 * n                  # congruent triangles, now coplanar
        y3 = x0 + a3 * e - h3 * n
        k = K0[h, 0] * x0 + K0[h, 1] * x1 + K0[h, 2] * y2 + K0[h, 3] * y3
        assert np.linalg.norm(k) < 1e-12
        k_folded = K0[h, 0] * x0 + K0[h, 1] * x1 + K0[h, 2] * x2 + K0[h, 3] * x3
        assert np.linalg.norm(k_folded) > 0.1      # the folded hinge is NOT in the null space


def test_hinge_enumeration_and_stencil_orientation():
    c, rest, tris, _ = make_cell("plt", 1)
    st = c.hinges()
    assert st.shape == (120, 4)
    assert np.all(st[:, 0] < st[:, 1])
    keys = st[:, 0].astype(np.int64) * 1000 + st[:, 1]
    assert np.all(np.diff(keys) > 0)                  # increasing (min,max) order, unique
    tri_set = {tuple(np.roll(t, k)) for t in tris.tolist() for k in range(3)}
    for u, v, a, b in st.tolist():
        assert (u, v, a) in tri_set                   # x2 opposite the directed edge u->v
        assert (v, u, b) in tri_set                   # x3 opposite v->u


def test_helfrich_sphere_energy_is_8pi():
    """P-10: unit icosphere, r_h := 0, k_bend = 1: sum 1/2 w_h ||K x||^2 ~ 8 pi (+1.5 %)."""
    for level in (2, 3):
        v, t = W.icosphere(level)
        c = O.OracleCell(t, v, W.default_material(v, t, k_bend=1.0), DT)
        st, K = c.hinges(), c.hinge_rows()
        w, _ = c.hinge_weights()
        kv = np.einsum("hi,hid->hd", K, v[st])
        e = 0.5 * np.sum(w * np.sum(kv * kv, axis=1))
        assert abs(e / (8 * np.pi) - 1.0) < 0.03


def test_masses_lumped_by_area_share():
    c, rest, tris, mat = make_cell("rbc", 2)
    m = c.masses()
    assert abs(m.sum() - mat["cell_mass"]) < 1e-12 * mat["cell_mass"]
    areas = c.areas()
    a, b, cc = rest[tris[:, 0]], rest[tris[:, 1]], rest[tris[:, 2]]
    assert np.allclose(areas, 0.5 * np.linalg.norm(np.cross(b - a, cc - a), axis=1), rtol=1e-13)
    av = np.zeros(len(rest)); np.add.at(av, tris.ravel(), np.repeat(areas / 3, 3))
    assert np.allclose(m, mat["cell_mass"] * av / av.sum(), rtol=1e-13)


def test_deformation_gradient_of_affine_maps():
    """F(X) is an isometry; for x = M X + t, F_t = M F_t(X) (linear elements reproduce affine maps)."""
    c, rest, tris, _ = make_cell("rbc", 2)
    rng = np.random.default_rng(10)
    M = np.eye(3) + 0.3 * rng.standard_normal((3, 3))
    x = rest @ M.T + np.array([5.0, -3.0, 2.0])
    for t in rng.integers(0, len(tris), 25):
        F0 = c.deformation_gradient(t, rest)
        assert np.allclose(F0.T @ F0, np.eye(2), atol=1e-12)
        assert np.allclose(c.deformation_gradient(t, x), M @ F0, atol=1e-12)


def test_system_matrix_properties():
    """A_sys symmetric; (A_sys - M/h^2 - w_v I) 1 = 0; quadratic form equals the energy with p = 0."""
    c, rest, tris, mat = make_cell("rbc", 2)
    A = c.system_matrix()
    assert np.abs(A - A.T).max() < 1e-12
    m = c.masses()
    Lel = A - np.diag(m / DT ** 2) - mat["w_volume"] * np.eye(len(m))
    assert np.abs(Lel @ np.ones(len(m))).max() < 1e-11
    assert np.linalg.eigvalsh(Lel).min() > -1e-10
    rng = np.random.default_rng(11)
    x = rng.standard_normal(rest.shape)
    zero = (np.zeros((c.T, 3, 2)), np.zeros((c.T, 3, 2)), np.zeros((c.H, 3)), x.copy())
    _, parts = c.energy(x, x, zero, parts=True)       # s = x, Pv = x: only elastic terms, p = 0
    quad = 0.5 * np.einsum("id,ij,jd->", x, Lel, x)
    assert abs(parts[1] + parts[2] + parts[3] - quad) < 1e-10 * abs(quad)
    # solve really inverts A_sys
    b = rng.standard_normal(rest.shape)
    assert np.abs(A @ c.solve(b) - b).max() < 1e-12


def test_create_rejects_bad_meshes():
    rest, tris = W.rest_shape("plt", 1)
    mat = W.default_material(rest, tris)
    with pytest.raises(ValueError):
        O.OracleCell(tris[:-1], rest, mat, DT)                    # open mesh
    flipped = tris.copy(); flipped[3] = flipped[3][[0, 2, 1]]
    with pytest.raises(ValueError):
        O.OracleCell(flipped, rest, mat, DT)                      # inconsistent orientation
    with pytest.raises(ValueError):
        O.OracleCell(tris[:, [0, 2, 1]], rest, mat, DT)           # inside-out: V0 <= 0
    with pytest.raises(ValueError):
        O.OracleCell(tris, rest, dict(mat, c_alpha=-0.1), DT)     # negative damping
    with pytest.raises(ValueError):
        O.OracleCell(tris, rest, dict(mat, s_min=1.2, s_max=1.0), DT)


# ----------------------------------------------------------------------------- the step
def test_P1_rest_shape_is_a_fixed_point():
    c, rest, _, _ = make_cell("rbc", 2)
    z = np.zeros_like(rest)
    x, v = c.step_cell(rest, z, z, 10)
    assert np.abs(x - rest).max() < 1e-13
    assert np.abs(v).max() < 1e-12


def test_P2_rigid_motion_gives_zero_internal_force_and_momentum_balance():
    c, rest, _, _ = make_cell("rbc", 2)
    rng = np.random.default_rng(12)
    R = random_rotation(rng)
    x = rest @ R.T + np.array([40.0, -12.0, 7.0])
    assert np.abs(c.fint(x)).max() < 1e-10         # vs |f| ~ 0.1 for a 5 % perturbation below
    y = x + 0.05 * rng.standard_normal(x.shape)        # any state
    f = c.fint(y)
    assert np.abs(f).max() > 1e-4
    assert np.abs(f.sum(axis=0)).max() < 1e-9 * np.abs(f).max()          # linear momentum
    assert np.abs(np.cross(y, f).sum(axis=0)).max() < 1e-9 * np.abs(np.cross(y, f)).max()   # angular


def test_fint_is_minus_gradient_of_the_distance_energy():
    """Finite differences of E_el(x) = sum 1/2 w dist(Ax, C)^2 reproduce f_int (sign, transposes)."""
    c, rest, _, _ = make_cell("plt", 1, w_volume=0.5)
    rng = np.random.default_rng(13)
    x = rest * 1.05 + 0.03 * rng.standard_normal(rest.shape)
    f = c.fint(x)

    def e_el(y):
        _, parts = c.energy(y, y, c.local(y), parts=True)
        return parts[1] + parts[2] + parts[3] + parts[4]

    for i, d in [(0, 0), (5, 1), (17, 2), (30, 0), (41, 2)]:
        e = np.zeros_like(x); e[i, d] = 1e-6
        fd = -(e_el(x + e) - e_el(x - e)) / 2e-6
        assert abs(fd - f[i, d]) < 2e-7 * max(1.0, abs(f[i, d]) / 1e-3)


def test_P3_energy_is_monotone_over_local_global_half_steps():
    c, rest, _, _ = make_cell("rbc", 2)
    rng = np.random.default_rng(14)
    pos = rest + np.array([10.0, 20.0, 30.0])
    vel = 1e-3 * rng.standard_normal(rest.shape)
    pull = W.cap_pull_forces(rest, np.eye(3)[None], 20e-3)[0].astype(np.float64)
    for step in range(8):
        pos, vel, _, en = c.step_cell(pos, vel, pull, 12, trace=True)
        assert np.all(np.diff(en) <= 1e-10 * np.abs(en[:-1])), (step, np.diff(en).max())  # rounding floor of E at 30 um offsets


def test_P4_free_cell_follows_closed_form_trajectory():
    rest, tris = W.rest_shape("plt", 1)
    mat = W.default_material(rest, tris, k_strain=0, k_area=0, k_bend=0, w_volume=0)
    c = O.OracleCell(tris, rest, mat, DT)
    rng = np.random.default_rng(15)
    f = 1e-3 * rng.standard_normal(rest.shape)
    v0 = 1e-2 * rng.standard_normal(rest.shape)
    m = c.masses()[:, None]
    x, v = rest.copy(), v0.copy()
    N = 7
    for _ in range(N):
        x, v = c.step_cell(x, v, f, 3)
    assert np.abs(x - (rest + N * DT * v0 + DT ** 2 * (f / m) * N * (N + 1) / 2)).max() < 1e-13
    assert np.abs(v - (v0 + N * DT * f / m)).max() < 1e-13


def test_P6_uniform_scaling_closed_forms():
    c, rest, _, mat = make_cell("rbc", 2)
    a_tot = c.areas().sum()
    w, r = c.hinge_weights()
    for s in (0.9, 1.1, 1.5):
        x = rest * s
        proj = c.local(x)
        _, parts = c.energy(x, x, proj, parts=True)
        assert abs(parts[1] - mat["k_strain"] * a_tot * (s - 1) ** 2) < 1e-10
        assert abs(parts[2] - mat["k_area"] * a_tot * (s - 1) ** 2) < 1e-10
        assert abs(parts[3] - (s - 1) ** 2 * np.sum(0.5 * w * r * r)) < 1e-12
        assert abs(O.volume(c.tris, proj[3]) - c.rest_volume) < 1e-11


def test_P7_centre_of_mass_follows_rigid_body_closed_form():
    rng = np.random.default_rng(16)
    for wv, sweeps, tol in [(0.0, 1, 1e-13), (0.5, 1, 1e-5), (0.5, 4, 1e-8)]:
        c, rest, _, _ = make_cell("rbc", 2, w_volume=wv)
        m = c.masses()[:, None]
        x = rest * 1.02 + 0.01 * rng.standard_normal(rest.shape)
        v = 1e-3 * rng.standard_normal(rest.shape)
        f = 1e-3 * rng.standard_normal(rest.shape)
        x1, _ = c.step_cell(x, v, f, sweeps)
        cm0 = (m * x).sum(0) / m.sum()
        cm_pred = cm0 + DT * (m * v).sum(0) / m.sum() + DT ** 2 * f.sum(0) / m.sum()
        assert np.abs((m * x1).sum(0) / m.sum() - cm_pred).max() < tol


def test_P8_global_update_is_quasi_newton_step():
    """x^{k+1} = x^k - A_sys^-1 [ M (x^k - s)/h^2 - f_int(x^k) ]  (ties PAPER.md:94 to local/global)."""
    c, rest, _, _ = make_cell("rbc", 2)
    rng = np.random.default_rng(17)
    x0 = rest + 0.01 * rng.standard_normal(rest.shape)
    f = 5e-3 * rng.standard_normal(rest.shape)
    m = c.masses()[:, None]
    _, _, its, _ = c.step_cell(x0, np.zeros_like(x0), f, 3, trace=True)
    s = its[0]
    for k in range(3):
        grad = m * (its[k] - s) / DT ** 2 - c.fint(its[k])
        pred = its[k] - c.solve(grad)
        assert np.abs(pred - its[k + 1]).max() < 1e-13


def test_P12_iteration_contraction_regression_guard():
    c, rest, _, _ = make_cell("rbc", 3)
    f = W.gaussian_forces(rest.shape, 1e-3, seed=99).astype(np.float64)
    z = np.zeros_like(rest)
    _, _, its, _ = c.step_cell(rest, z, f, 40, trace=True)
    dist = [np.abs(its[k] - its[-1]).max() for k in (1, 2, 3, 4)]
    expect = [1.3e-5, 3.2e-6, 8.0e-7, 2.9e-7]              # SURVEY.md P-12 (order of magnitude)
    for d, e in zip(dist, expect):
        assert e / 4 < d < e * 4, (dist, expect)
    assert all(dist[i + 1] < dist[i] for i in range(3))


def test_step_many_cells_matches_single_cell_calls():
    c, rest, _, _ = make_cell("plt", 1)
    rng = np.random.default_rng(18)
    pos = np.stack([rest + rng.uniform(0, 50, 3) for _ in range(5)])
    vel = 1e-3 * rng.standard_normal(pos.shape)
    f = 1e-3 * rng.standard_normal(pos.shape)
    p, v = c.step(pos, vel, f, 4)
    for i in range(5):
        pi, vi = c.step_cell(pos[i], vel[i], f[i], 4)
        assert np.array_equal(p[i], pi) and np.array_equal(v[i], vi)


def test_oracle_reproduces_its_committed_config1_result():
    """Regression guard of the oracle's own arithmetic: tests/golden/config1_oracle.txt was written
    by tests/golden/make_golden.py from the oracle alone (the paper prints no value to cite).  A
    change to the oracle that moves these numbers must name the passage or DESIGN.md reading that
    justifies it and regenerate the file."""
    import os
    path = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden", "config1_oracle.txt")
    ref = np.loadtxt(path)
    w = W.make_config(1)
    g = w.groups[0]
    oc = O.OracleCell(g.tris, g.rest, g.material, w.dt)
    pos, vel = oc.step(g.pos0, g.vel0, w.forces(0, 0), w.n_iters)
    disp = pos[0] - g.pos0[0].astype(np.float64)
    assert ref.shape == (g.rest.shape[0], 6)
    scale = np.abs(ref[:, :3]).max()
    assert np.abs(disp - ref[:, :3]).max() <= 1e-9 * scale      # fp64 summation-order slack
    assert np.abs(vel[0] - ref[:, 3:]).max() <= 1e-9 * np.abs(ref[:, 3:]).max()


# ----------------------------------------------------------------------------- damping (A-20)
def test_P13_free_cell_with_mass_proportional_damping_decays_at_the_implicit_euler_rate():
    """No elasticity, c_alpha > 0: M (v' - v)/h = f - c_alpha M v'  =>  v' = r (v + h f/m),
    r = 1/(1 + h c_alpha).  After N steps (geometric series):
        v_N = r^N v_0 + (h f/m) r (1 - r^N)/(1 - r),   x_N = x_0 + h sum_{k=1..N} v_k."""
    rest, tris = W.rest_shape("plt", 1)
    ca = 0.7
    mat = W.default_material(rest, tris, k_strain=0, k_area=0, k_bend=0, w_volume=0, c_alpha=ca)
    c = O.OracleCell(tris, rest, mat, DT)
    rng = np.random.default_rng(31)
    f = 1e-3 * rng.standard_normal(rest.shape)
    v0 = 1e-2 * rng.standard_normal(rest.shape)
    a = DT * f / c.masses()[:, None]
    r = 1.0 / (1.0 + DT * ca)
    x, v = rest.copy(), v0.copy()
    N = 9
    for _ in range(N):
        x, v = c.step_cell(x, v, f, 2)
    vN = r ** N * v0 + a * r * (1 - r ** N) / (1 - r)
    # sum_{k=1..N} v_k with v_k = r^k v0 + a r (1 - r^k)/(1 - r)
    geo = r * (1 - r ** N) / (1 - r)
    xN = rest + DT * (geo * v0 + a * r / (1 - r) * (N - geo))
    assert np.abs(v - vN).max() < 1e-12 and np.abs(x - xN).max() < 1e-13   # v = (x' - x)/h: rounding / h
    assert np.abs(vN).max() < np.abs(v0 + N * a).max()              # and it does damp


def test_P14_stiffness_proportional_damping_leaves_rigid_translation_alone():
    """L_el has zero row sums (it only sees differences), so c_beta does not act on a uniform
    velocity: the rest shape drifting at constant velocity stays rigid and keeps its velocity."""
    c, rest, _, _ = make_cell("rbc", 2, c_beta=0.5)
    L = c.elastic_laplacian()
    assert np.abs(L - L.T).max() < 1e-12 and np.abs(L.sum(axis=1)).max() < 1e-10
    assert np.linalg.eigvalsh(L).min() > -1e-10
    v0 = np.tile(np.array([3e-3, -1e-3, 2e-3]), (rest.shape[0], 1))
    x, v = rest.copy(), v0.copy()
    for _ in range(5):
        x, v = c.step_cell(x, v, np.zeros_like(rest), 4)
    assert np.abs(x - (rest + 5 * DT * v0)).max() < 1e-12 and np.abs(v - v0).max() < 1e-11
    # while a deformation rate IS damped: stretch velocity field, compare against c_beta = 0
    c0, _, _, _ = make_cell("rbc", 2)
    vs = 1e-2 * np.random.default_rng(34).standard_normal(rest.shape)     # vertex-wise noise: all deformation
    _, v_damped = c.step_cell(rest, vs, np.zeros_like(rest), 20)
    _, v_free = c0.step_cell(rest, vs, np.zeros_like(rest), 20)
    assert np.linalg.norm(v_damped) < 0.9 * np.linalg.norm(v_free)


def test_P15_damped_global_update_is_quasi_newton_step_on_the_damped_objective():
    """g(x) = 1/2 ||x-s||^2_M/h^2 + E_el(x) + 1/(2h) (x-x_n)^T C (x-x_n), C = c_alpha M + c_beta L_el;
    one sweep = x - A_sys^-1 grad g(x), with A_sys = (1/h^2 + c_alpha/h) M + (1 + c_beta/h) L_el + w_vol I.
    C is rebuilt here from the masses and the elastic Laplacian; the dissipation term is checked
    against its own finite differences."""
    c, rest, _, mat = make_cell("rbc", 2, c_alpha=0.3, c_beta=0.05)
    rng = np.random.default_rng(32)
    xn = rest + 0.01 * rng.standard_normal(rest.shape)
    vn = 1e-2 * rng.standard_normal(rest.shape)
    f = 5e-3 * rng.standard_normal(rest.shape)
    m = c.masses()[:, None]
    Cmat = 0.3 * np.diag(c.masses()) + 0.05 * c.elastic_laplacian()
    A = c.system_matrix()
    A_expect = np.diag(c.masses()) / DT ** 2 + c.elastic_laplacian() + mat["w_volume"] * np.eye(rest.shape[0]) + Cmat / DT
    assert np.abs(A - A_expect).max() < 1e-10 * np.abs(A).max()
    _, _, its, en = c.step_cell(xn, vn, f, 4, trace=True)
    s = its[0]
    assert np.abs(s - (xn + DT * vn + DT ** 2 * f / m)).max() < 1e-14
    for k in range(4):
        grad = m * (its[k] - s) / DT ** 2 - c.fint(its[k]) + Cmat @ (its[k] - xn) / DT
        pred = its[k] - c.solve(grad)
        assert np.abs(pred - its[k + 1]).max() < 1e-12
    assert (np.diff(en) <= 1e-12 * np.abs(en[:-1])).all()            # damped objective is monotone too
    # dissipation potential: value and gradient
    x = its[2]
    assert c.dissipation(x, xn) == pytest.approx(0.5 * np.sum((x - xn) * (Cmat @ (x - xn))) / DT, rel=1e-12)
    eps = 1e-6
    e = np.zeros_like(x); e[5, 1] = eps
    fd = (c.dissipation(x + e, xn) - c.dissipation(x - e, xn)) / (2 * eps)
    assert fd == pytest.approx((Cmat @ (x - xn) / DT)[5, 1], rel=1e-6)
    assert np.abs(c.damping_rhs(xn) - Cmat @ xn / DT).max() < 1e-12 * np.abs(Cmat @ xn / DT).max()


def test_P16_damping_dissipates_mechanical_energy():
    """Free vibration from a stretched state: kinetic + elastic energy after 30 steps is lower
    with viscoelastic damping than without, for c_alpha alone, c_beta alone and both."""
    rest, tris = W.rest_shape("rbc", 2)
    z = np.zeros_like(rest)

    def mech_energy(cell, x, v):
        proj = cell.local(x)
        _, parts = cell.energy(x, x, proj, parts=True)               # s = x: no inertial term
        return 0.5 * np.sum(cell.masses()[:, None] * v * v) + parts[1:].sum()

    out = {}
    for key, over in (("none", {}), ("alpha", dict(c_alpha=0.5)), ("beta", dict(c_beta=0.05)),
                      ("both", dict(c_alpha=0.5, c_beta=0.05))):
        cell = O.OracleCell(tris, rest, W.default_material(rest, tris, **over), DT)
        x, v = rest * 1.05, z.copy()
        for _ in range(30):
            x, v = cell.step_cell(x, v, z, 10)
        out[key] = mech_energy(cell, x, v)
    assert out["alpha"] < out["none"] and out["beta"] < out["none"]
    assert out["both"] < min(out["alpha"], out["beta"])


# ----------------------------------------------------------------------------- converged solve (A-21)
def _residual_length(cell, x, s, xn, dt):
    _, gr = cell.objective(x, s, xn, grad=True)
    return np.abs(gr * dt ** 2 / cell.masses()[:, None]).max()


def test_P17_no_history_unit_step_is_the_plain_local_global_sweep():
    """PAPER.md:94 via P-8: with no L-BFGS history and no line search the converged-solve driver
    walks exactly the iterates of the fixed-count step."""
    c, rest, _, _ = make_cell("rbc", 2)
    rng = np.random.default_rng(41)
    x0 = rest + 0.01 * rng.standard_normal(rest.shape)
    v0 = 1e-3 * rng.standard_normal(rest.shape)
    f = 5e-3 * rng.standard_normal(rest.shape)
    K = 6
    _, _, its_plain, _ = c.step_cell(x0, v0, f, K, trace=True)
    x, v, k, gt, rt, its = c.step_cell_converged(x0, v0, f, 0.0, K, history=0, line_search=False, trace=True)
    assert k == K and np.abs(its - its_plain).max() < 1e-13
    xp, vp = c.step_cell(x0, v0, f, K)
    assert np.abs(x - xp).max() < 1e-13 and np.abs(v - vp).max() < 1e-11


@pytest.mark.parametrize("damp", [{}, dict(c_alpha=0.3, c_beta=0.05)])
def test_P18_objective_gradient_matches_finite_differences(damp):
    """grad g = M (x-s)/h^2 - f_int(x) [+ C (x-x_n)/h]: the projections are closest points, so
    their derivatives drop out (envelope).  Central differences of g on random coordinates."""
    c, rest, _, _ = make_cell("plt", 1, s_min=0.9, s_max=1.1, a_min=0.95, a_max=1.05, **damp)
    rng = np.random.default_rng(42)
    xn = rest + 0.02 * rng.standard_normal(rest.shape)
    s = xn + 0.01 * rng.standard_normal(rest.shape)
    x = xn + 0.03 * rng.standard_normal(rest.shape)
    g0, gr = c.objective(x, s, xn, grad=True)
    assert g0 > 0
    eps = 1e-6
    for _ in range(12):
        i, d = rng.integers(rest.shape[0]), rng.integers(3)
        e = np.zeros_like(x); e[i, d] = eps
        fd = (c.objective(x + e, s, xn) - c.objective(x - e, s, xn)) / (2 * eps)
        assert fd == pytest.approx(gr[i, d], rel=2e-5, abs=1e-9)


@pytest.mark.parametrize("dt", [0.1, 1.0, 10.0])
def test_P19_objective_decreases_at_every_accepted_step(dt):
    rest, tris = W.rest_shape("rbc", 2)
    c = O.OracleCell(tris, rest, W.default_material(rest, tris), dt)
    rng = np.random.default_rng(43)
    f = 1e-3 * rng.standard_normal(rest.shape)
    x, v, k, gt, rt, _ = c.step_cell_converged(rest * 1.03, np.zeros_like(rest), f, 1e-9, 400, 3, True, trace=True)
    assert k >= 3
    assert (np.diff(gt) <= 1e-12 * np.abs(gt[:-1])).all()
    assert rt[-1] < 1e-3 * rt[0]


def test_P20_converged_state_is_the_limit_of_plain_sweeps():
    c, rest, _, _ = make_cell("rbc", 2)
    rng = np.random.default_rng(44)
    x0 = rest + 0.01 * rng.standard_normal(rest.shape)
    f = 5e-3 * rng.standard_normal(rest.shape)
    z = np.zeros_like(rest)
    x_lim, _ = c.step_cell(x0, z, f, 250)
    x, v, k = c.step_cell_converged(x0, z, f, 1e-12, 200, history=5)
    assert k < 60
    assert np.abs(x - x_lim).max() < 1e-10
    s = x0 + DT ** 2 * f / c.masses()[:, None]
    assert _residual_length(c, x, s, x0, DT) <= 1e-12


@pytest.mark.parametrize("scale", [10, 100])
def test_P21_large_time_steps_converge_where_20_fixed_sweeps_do_not(scale):
    """PAPER.md:133 "unconditional stability for arbitrary time steps": at dt x 10 and x 100 the
    inertial diagonal no longer dominates, 20 plain sweeps leave a large unbalanced force, the
    quasi-Newton iteration with line search still reaches the tolerance."""
    dt = DT * scale
    rest, tris = W.rest_shape("rbc", 2)
    c = O.OracleCell(tris, rest, W.default_material(rest, tris), dt)
    rng = np.random.default_rng(45)
    f = 1e-3 * rng.standard_normal(rest.shape)
    z = np.zeros_like(rest)
    x0 = rest * 1.02
    s = x0 + dt ** 2 * f / c.masses()[:, None]
    tol = 1e-7
    x20, _ = c.step_cell(x0, z, f, 20)
    x, v, k = c.step_cell_converged(x0, z, f, tol, 3000, history=5)
    r20, rc = _residual_length(c, x20, s, x0, dt), _residual_length(c, x, s, x0, dt)
    assert rc <= tol and r20 > 100 * tol
    # and the history pays: far fewer iterations than the same driver without it
    _, _, k0 = c.step_cell_converged(x0, z, f, tol, 3000, history=0)
    assert k < 0.5 * k0


# ----------------------------------------------------------------------------- collisions, areas (A-22)
def test_P22_collision_projection_is_the_closest_point_of_the_half_space():
    rng = np.random.default_rng(51)
    for _ in range(40):
        x, q = rng.standard_normal(3), rng.standard_normal(3)
        nrm = rng.standard_normal(3); nrm /= np.linalg.norm(nrm)
        d = rng.uniform(0.0, 0.5)
        p = O.project_collision(x, q, nrm, d)
        assert (p - q) @ nrm >= d - 1e-12                               # feasible
        if (x - q) @ nrm >= d:
            assert np.array_equal(p, x)                                 # inactive: no force
        # brute force: no feasible sample is closer
        cand = x + rng.standard_normal((4000, 3)) * (np.linalg.norm(p - x) + 0.1)
        feas = cand[(cand - q) @ nrm >= d]
        if len(feas):
            assert np.linalg.norm(p - x) <= np.linalg.norm(feas - x, axis=1).min() + 1e-12
    assert np.array_equal(O.project_collision(np.ones(3), np.zeros(3), np.zeros(3), 0.3), np.ones(3))


def test_P23_free_cell_pressed_against_a_wall_settles_at_the_closed_form_penetration():
    """No elasticity, constant force f on every vertex towards a wall (every vertex has the wall as
    colliding neighbour): static equilibrium w_c (d - gap) = |f|  =>  gap = d - |f|/w_c."""
    rest, tris = W.rest_shape("plt", 1)
    wc, d, fmag = 2.0, 0.05, 1e-2
    mat = W.default_material(rest, tris, k_strain=0, k_area=0, k_bend=0, w_volume=0, c_alpha=2.0,
                             w_collision=wc, d_collision=d)
    c = O.OracleCell(tris, rest, mat, DT)
    n = rest.shape[0]
    nrm = np.tile([0.0, 0.0, 1.0], (n, 1))                               # wall z = 0, outward normal +z
    q = np.zeros((n, 3))
    f = np.tile([0.0, 0.0, -fmag], (n, 1))
    x = rest + np.array([0.0, 0.0, 0.5 - rest[:, 2].min()])              # lowest vertex 0.5 above the wall
    v = np.zeros_like(x)
    for _ in range(4000):
        x, v = c.step_cell_collide(x, v, f, q, nrm, 3)
    assert np.abs(v).max() < 1e-9
    assert np.abs(x[:, 2] - (d - fmag / wc)).max() < 1e-8                # every vertex: same gap (no elasticity)


def test_P24_collide_step_identities():
    """(i) no active neighbour: identical to the plain step although w_c sits on the diagonal;
    (ii) one sweep = x - A_sys^-1 grad of the objective with the collision energy
    (iii) the objective is monotone over the local/global half steps (P-3 with collisions)."""
    c, rest, _, mat = make_cell("rbc", 2, w_collision=1.5, d_collision=0.02)
    c0, _, _, _ = make_cell("rbc", 2)
    rng = np.random.default_rng(52)
    x0 = rest + 0.01 * rng.standard_normal(rest.shape)
    v0 = 1e-3 * rng.standard_normal(rest.shape)
    f = 5e-3 * rng.standard_normal(rest.shape)
    n = rest.shape[0]
    zero = np.zeros_like(rest)
    xa, va = c.step_cell_collide(x0, v0, f, zero, zero, 5)
    xb, vb = c0.step_cell(x0, v0, f, 5)
    assert np.abs(xa - xb).max() < 1e-6        # same fixed point, different (both contracting) iterations
    xa, _ = c.step_cell_collide(x0, v0, f, zero, zero, 60)
    xb, _ = c0.step_cell(x0, v0, f, 60)
    assert np.abs(xa - xb).max() < 1e-12
    # a plane cutting through the cell: about half of the vertices active
    nrm = np.tile([1.0, 0.0, 0.0], (n, 1)); q = np.tile([0.5, 0.0, 0.0], (n, 1))
    _, _, its, en = c.step_cell_collide(x0, v0, f, q, nrm, 6, trace=True)
    assert (np.diff(en) <= 1e-12 * np.abs(en[:-1])).all()
    m = c.masses()[:, None]
    s = its[0]
    A = c.system_matrix()
    assert np.allclose(np.diag(A) - np.diag(c0.system_matrix()), 1.5)
    for k in range(6):
        Pc = np.array([O.project_collision(its[k][i], q[i], nrm[i], 0.02) for i in range(n)])
        active = ((its[k] - q) * nrm).sum(axis=1) < 0.02
        assert 0.2 * n < active.sum() < 0.8 * n or k > 0
        grad = m * (its[k] - s) / DT ** 2 - c.fint(its[k]) + 1.5 * (its[k] - Pc)
        pred = its[k] - c.solve(grad)
        assert np.abs(pred - its[k + 1]).max() < 1e-12


def test_P25_vertex_areas():
    """a_v = 1/3 of the areas of the triangles around v: sums to the surface area (unit icosphere
    -> 4 pi from below), equals the lumped-mass share at rest, scales with the square of a scaling."""
    c, rest, tris, mat = make_cell("rbc", 3)
    a = c.vertex_areas(rest)
    assert a.sum() == pytest.approx(c.areas().sum(), rel=1e-13)
    assert np.allclose(a / a.sum(), c.masses() / c.masses().sum(), rtol=1e-12)
    assert np.allclose(c.vertex_areas(1.7 * rest), 1.7 ** 2 * a, rtol=1e-12)
    sph, st = W.mesh.icosphere(3)
    cs = O.OracleCell(st, sph, W.default_material(sph, st), DT)
    assert 0.98 * 4 * np.pi < cs.vertex_areas(sph).sum() < 4 * np.pi


# ----------------------------------------------------------------------------- strain-dependent weight (A-23)
def test_P26_strain_hardening_energy_force_and_fixed_point():
    """psi(d) = 1/2 w_s (d^2 + 1/2 beta d^4): (i) closed form under uniform scaling,
    E_strain = k_strain A_tot ((s-1)^2 + 1/2 beta (s-1)^4); (ii) f_int = -grad E by central
    differences (the effective targets carry psi'); (iii) the rest shape is still a fixed point and
    beta = 0 is the plain strain term; (iv) hardening stiffens: smaller stretch under the same pull."""
    beta = 40.0
    c, rest, tris, mat = make_cell("rbc", 2, strain_hardening=beta)
    c0, _, _, _ = make_cell("rbc", 2)
    a_tot = c.areas().sum()
    for sc in (0.9, 1.1, 1.3):
        x = rest * sc
        _, parts = c.energy(x, x, c.local(x), parts=True)
        assert parts[1] == pytest.approx(mat["k_strain"] * a_tot * ((sc - 1) ** 2 + 0.5 * beta * (sc - 1) ** 4), rel=1e-9)
    rng = np.random.default_rng(61)
    x = rest * 1.08 + 0.02 * rng.standard_normal(rest.shape)
    f = c.fint(x)

    def E(y):
        _, parts = c.energy(y, y, c.local(y), parts=True)
        return parts[1:].sum()

    eps = 1e-6
    for _ in range(10):
        i, d = rng.integers(rest.shape[0]), rng.integers(3)
        e = np.zeros_like(x); e[i, d] = eps
        assert -(E(x + e) - E(x - e)) / (2 * eps) == pytest.approx(f[i, d], rel=2e-5, abs=1e-9)
    assert np.abs(f - c0.fint(x)).max() > 1e-3 * np.abs(f).max()         # and it differs from beta = 0
    z = np.zeros_like(rest)
    xr, vr = c.step_cell(rest, z, z, 10)
    assert np.abs(xr - rest).max() < 1e-13
    pull = W.cap_pull_forces(rest, np.eye(3)[None], 40e-3)[0].astype(np.float64)
    xs, vs, xh, vh = rest.copy(), z.copy(), rest.copy(), z.copy()
    for _ in range(150):
        xs, vs = c0.step_cell(xs, vs, pull, 10)
        xh, vh = c.step_cell(xh, vh, pull, 10)
    assert np.ptp(xh[:, 0]) < np.ptp(xs[:, 0]) - 1e-3


# ----------------------------------------------------------------------------- global-area term (A-24)
def test_P27_total_area_gradient_hessian_and_projection():
    """Global-area term, geometry: (i) textbook areas (octahedron 4 sqrt 3, icosphere -> 4 pi from
    below, translation invariance, scaling by s^2); (ii) grad A against central differences, with
    sum_v grad_v A = 0 (translation) and sum_v x_v . grad_v A = 2 A (degree-2 homogeneity);
    (iii) the Hessian against central differences of the gradient, symmetric, H x = grad A
    (homogeneity again); (iv) the projection lands on A = A*, satisfies the KKT condition
    P - x parallel to grad A(P), and is the closest such configuration: against SLSQP on the
    perturbed tetrahedron / octahedron; (v) it converges where the volume's fixed-point iteration
    does not (perturbed RBC-2 at a 12 % area excess)."""
    assert O.area_total(OCT_T, OCT_V) == pytest.approx(4 * np.sqrt(3.0), rel=1e-14)
    v, t = W.icosphere(3)
    a = O.area_total(t, v)
    assert 0.97 * 4 * np.pi < a < 4 * np.pi
    assert O.area_total(t, v + np.array([50.0, -20.0, 7.0])) == pytest.approx(a, rel=1e-12)
    assert O.area_total(t, 1.7 * v) == pytest.approx(1.7 ** 2 * a, rel=1e-13)
    rng = np.random.default_rng(71)
    x = OCT_V + 0.1 * rng.standard_normal(OCT_V.shape) + np.array([2.0, 1.0, -3.0])
    g = O.area_grad(OCT_T, x)
    H = O.area_hessian(OCT_T, x)
    for i in range(6):
        for d in range(3):
            e = np.zeros_like(x); e[i, d] = 1e-6
            fd = (O.area_total(OCT_T, x + e) - O.area_total(OCT_T, x - e)) / 2e-6
            assert abs(fd - g[i, d]) < 1e-9
            fdg = (O.area_grad(OCT_T, x + e) - O.area_grad(OCT_T, x - e)).ravel() / 2e-6
            assert np.abs(fdg - H[:, 3 * i + d]).max() < 1e-8
    assert np.allclose(g.sum(axis=0), 0, atol=1e-14)
    xc = x - x.mean(axis=0)
    assert np.sum(xc * g) == pytest.approx(2 * O.area_total(OCT_T, x), rel=1e-12)
    assert np.abs(H - H.T).max() < 1e-14
    assert np.abs(H @ x.ravel() - g.ravel()).max() < 1e-12               # grad A is degree-1 homogeneous
    for verts, tris in ((TET_V, TET_T), (OCT_V, OCT_T)):
        a0 = O.area_total(tris, verts)
        for scale in (0.85, 1.05, 1.2):
            x = verts * scale + 0.05 * rng.standard_normal(verts.shape) + np.array([3.0, -2.0, 1.0])
            P, its = O.project_garea(tris, x, a0, a0)
            assert 0 < its < 30
            assert abs(O.area_total(tris, P) - a0) < 1e-13 * a0
            gP, D = O.area_grad(tris, P).ravel(), (P - x).ravel()
            assert np.abs(D - (D @ gP) / (gP @ gP) * gP).max() < 1e-12
            cons = dict(type="eq", fun=lambda z: O.area_total(tris, z.reshape(-1, 3)) - a0,
                        jac=lambda z: O.area_grad(tris, z.reshape(-1, 3)).ravel())
            r = optimize.minimize(lambda z: 0.5 * np.sum((z - x.ravel()) ** 2), x.ravel(),
                                  jac=lambda z: z - x.ravel(), constraints=[cons], method="SLSQP",
                                  options=dict(ftol=1e-16, maxiter=500))
            d_or, d_ref = np.linalg.norm(P - x), np.sqrt(2 * r.fun)
            assert abs(d_or - d_ref) < 1e-7 * max(d_ref, 1e-3)
            assert np.abs(P.ravel() - r.x).max() < 1e-6
    rest, tris = W.rest_shape("rbc", 2)
    x = rest * 1.06 + 0.02 * rng.standard_normal(rest.shape) + np.array([80.0, -30.0, 10.0])
    a0 = O.area_total(tris, rest)
    assert O.area_total(tris, x) > 1.1 * a0
    P, its = O.project_garea(tris, x, a0, a0)
    assert 0 < its < 15 and abs(O.area_total(tris, P) - a0) < 1e-12 * a0
    gP, D = O.area_grad(tris, P).ravel(), (P - x).ravel()
    assert np.abs(D - (D @ gP) / (gP @ gP) * gP).max() < 1e-12


def test_P28_global_area_term_in_the_step():
    """Global-area term in the solver (reading A-24): (i) closed form on the vertex-transitive
    icosahedron scaled by s: the closest configuration with the rest area is the rest shape itself,
    E = 1/2 w n R^2 (s-1)^2; (ii) w_garea sits on the diagonal of A_sys; (iii) f_int = -grad E by
    central differences with the term on; (iv) the rest shape stays a fixed point; (v) the energy is
    monotone over local/global half steps and the quasi-Newton identity (P-8) holds with the term;
    (vi) the term does what it is for: under an inflating load the total area stays closer to A0;
    (vii) weight 0 leaves everything bit-identical; negative weight and an inverted band are rejected."""
    w = 0.8
    v0, t0 = W.icosphere(0)
    mat0 = W.default_material(v0, t0, w_garea=w, ga_min=1.0, ga_max=1.0)
    ico = O.OracleCell(t0, v0, mat0, DT)
    for sc in (0.9, 1.15):
        P, e = ico.garea_local(sc * v0)
        assert np.abs(P - v0).max() < 1e-12
        assert e == pytest.approx(0.5 * w * 12 * (sc - 1) ** 2, rel=1e-12)
    c, rest, tris, mat = make_cell("rbc", 2, w_garea=w, ga_min=1.0, ga_max=1.0)
    c0, _, _, _ = make_cell("rbc", 2)
    assert np.allclose(c.system_matrix() - c0.system_matrix(), w * np.eye(rest.shape[0]), atol=1e-12)
    assert c.rest_area() == pytest.approx(O.area_total(tris, rest), rel=1e-13)
    rng = np.random.default_rng(72)
    x = rest * 1.06 + 0.02 * rng.standard_normal(rest.shape)
    f = c.fint(x)

    def E(y):
        _, parts = c.energy(y, y, c.local(y), parts=True)
        return parts[1:].sum() + c.garea_local(y)[1]

    for _ in range(10):
        i, d = rng.integers(rest.shape[0]), rng.integers(3)
        e = np.zeros_like(x); e[i, d] = 1e-6
        assert -(E(x + e) - E(x - e)) / 2e-6 == pytest.approx(f[i, d], rel=2e-5, abs=1e-9)
    assert np.abs(f - c0.fint(x)).max() > 1e-3 * np.abs(f).max()
    z = np.zeros_like(rest)
    xr, vr = c.step_cell(rest, z, z, 10)
    assert np.abs(xr - rest).max() < 1e-13
    vel = 1e-3 * rng.standard_normal(rest.shape)
    fext = 5e-3 * rng.standard_normal(rest.shape)
    xs, vs, its, en = c.step_cell(x, vel, fext, 8, trace=True)
    assert (np.diff(en) <= 1e-12 * np.abs(en[:-1])).all()
    m = c.masses()[:, None]
    s = x + DT * vel + DT * DT * fext / m
    assert np.abs(its[0] - s).max() < 1e-15
    grad = -c.fint(s)                                                     # x^0 = s: the inertia term vanishes
    assert np.abs(its[1] - (s - np.linalg.solve(c.system_matrix(), grad))).max() < 1e-12
    g_obj, g_grad = c.objective(x, s, x, grad=True)                       # converged-solve objective carries the term
    for _ in range(4):
        i, d = rng.integers(rest.shape[0]), rng.integers(3)
        e = np.zeros_like(x); e[i, d] = 1e-6
        fd = (c.objective(x + e, s, x) - c.objective(x - e, s, x)) / 2e-6
        assert fd == pytest.approx(g_grad[i, d], rel=2e-5, abs=1e-8)
    nrm = rest / np.linalg.norm(rest, axis=1, keepdims=True)
    load = 2e-2 * nrm
    xa, va, xb, vb = rest.copy(), z.copy(), rest.copy(), z.copy()
    strong, _, _, _ = make_cell("rbc", 2, w_garea=20.0, ga_min=1.0, ga_max=1.0)
    for _ in range(40):
        xa, va = c0.step_cell(xa, va, load, 10)
        xb, vb = strong.step_cell(xb, vb, load, 10)
    a0 = c0.rest_area()
    assert abs(O.area_total(tris, xb) - a0) < 0.7 * abs(O.area_total(tris, xa) - a0)
    off, _, _, _ = make_cell("rbc", 2, w_garea=0.0, ga_min=1.0, ga_max=1.0)
    pa, va2 = off.step_cell(x, vel, fext, 6)
    pb, vb2 = c0.step_cell(x, vel, fext, 6)
    assert np.array_equal(pa, pb) and np.array_equal(va2, vb2)
    with pytest.raises(Exception):
        make_cell("rbc", 2, w_garea=-1.0)
    with pytest.raises(Exception):
        make_cell("rbc", 2, w_garea=1.0, ga_min=1.2, ga_max=0.9)
