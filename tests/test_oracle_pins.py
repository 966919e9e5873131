"""Pins of the CPU oracle to things other than itself (SURVEY.md §8(c) "What pins the oracle").

Every expected value here comes from brute-force quadrature of the paper's defining integrals
(P:121), from a closed form / invariant the mathematics fixes, from a physical
constant, or from a library routine (numpy.linalg) — never from oracle/ or the CUDA path.
"""
import os

import numpy as np
import pytest

from workloads import configs as W

GOLD = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden")
RECT, TRI, WIRE = 0, 1, 2
PI = np.pi


def local_elem(kind, a, b):
    """Element in the local frame of P:119: XZ plane from the origin, normal +Y (wires on X)."""
    return dict(kind=kind, v0=[0, 0, 0], e1=[a, 0, 0], e2=[0, 0, b if kind != WIRE else 0.0])


def infl(orc, kind, a, b, P, mode="ld", radius=0.0):
    e = local_elem(kind, a, b)
    return orc.influence(e["kind"], e["v0"], e["e1"], e["e2"], P, radius=radius, mode=mode)


# ---------------------------------------------------------------------------------------------
# 1. brute-force quadrature of the defining integrals (stored pins, mpmath 30 digits)
# ---------------------------------------------------------------------------------------------
def _gold_cases():
    out = []
    with open(os.path.join(GOLD, "quadrature_pins.txt")) as fh:
        for line in fh:
            if line.startswith("#") or not line.strip():
                continue
            t = line.split()
            out.append((t[0], float(t[1]), float(t[2]), [float(x) for x in t[3:6]], np.array([float(x) for x in t[6:10]])))
    return out


@pytest.mark.parametrize("mode,tol", [("ld", 2e-14), ("f64", 5e-12)])
def test_quadrature_pins(orc, mode, tol):
    cases = _gold_cases()
    assert len(cases) >= 15
    for kind, a, b, P, want in cases:
        k = {"rect": RECT, "tri": TRI, "wire": WIRE}[kind]
        if k == WIRE:
            r = 1e-3
            got = infl(orc, k, a, b, P, mode, radius=r) / (2 * PI * r)      # S24: lambda = 2 pi r_w sigma
        else:
            got = infl(orc, k, a, b, P, mode)
        scale = max(abs(want[0]), np.linalg.norm(want[1:]))
        assert np.max(np.abs(got - want)) <= tol * scale, (kind, a, b, P, got, want)


# ---------------------------------------------------------------------------------------------
# 2. independent tensor Gauss-Legendre quadrature (numpy) at random non-singular points, random
#    orientation in space: pins the local-frame convention and the rotation of E' to global
# ---------------------------------------------------------------------------------------------
def _gl_quadrature(kind, v0, e1, e2, P, n=96):
    x, w = np.polynomial.legendre.leggauss(n)
    s = 0.5 * (x + 1.0)
    ws = 0.5 * w
    if kind == WIRE:
        src = v0[:, None] + e1[:, None] * s[None, :]
        wt = ws * np.linalg.norm(e1)
    else:
        S, T = np.meshgrid(s, s, indexing="ij")
        WS, WT = np.meshgrid(ws, ws, indexing="ij")
        if kind == TRI:                     # collapsed map: z runs to (1 - s) of the second leg
            T = T * (1.0 - S)
            WT = WT * (1.0 - S)
        src = v0[:, None] + e1[:, None] * S.ravel()[None, :] + e2[:, None] * T.ravel()[None, :]
        wt = (WS * WT).ravel() * np.linalg.norm(np.cross(e1, e2))
    d = P[:, None] - src
    r = np.linalg.norm(d, axis=0)
    return np.concatenate([[np.sum(wt / r)], (d / r ** 3) @ wt])


@pytest.mark.parametrize("kind", [RECT, TRI, WIRE])
def test_random_orientation_vs_gauss_legendre(orc, kind):
    pr = W.random_elements(24, seed=11 + kind, kinds=(kind,), size_mm=(0.3, 1.0))
    rs = np.random.RandomState(5 + kind)
    worst = 0.0
    for j in range(pr.n):
        v0, e1, e2 = pr.v0[:, j], pr.e1[:, j], pr.e2[:, j]
        L = max(np.linalg.norm(e1), np.linalg.norm(e2))
        c = v0 + 0.5 * e1 + (0.5 * e2 if kind != WIRE else 0)
        u = rs.normal(size=3)
        u /= np.linalg.norm(u)
        P = c + u * L * rs.uniform(1.2, 4.0)                # distance >= 0.2 L from the element
        want = _gl_quadrature(kind, v0, e1, e2, P)
        rad = 1e-6
        got = orc.influence(kind, v0, e1, e2, P, radius=rad, mode="ld")
        if kind == WIRE:
            got = got / (2 * PI * rad)
        scale = max(abs(want[0]), np.linalg.norm(want[1:]))
        worst = max(worst, np.max(np.abs(got - want)) / scale)
    assert worst < 1e-12, worst


# ---------------------------------------------------------------------------------------------
# 3. closed forms the mathematics fixes
# ---------------------------------------------------------------------------------------------
def test_rectangle_centre_closed_form(orc):
    # Phi' at the centre of an a x b rectangle = 2[a asinh(b/a) + b asinh(a/b)]; field vanishes (symmetry, S5)
    for a, b in [(2.0, 3.0), (1.0, 1.0), (0.01, 7.0)]:
        got = infl(orc, RECT, a, b, [a / 2, 0.0, b / 2])
        want = 2 * (a * np.arcsinh(b / a) + b * np.arcsinh(a / b))
        assert abs(got[0] - want) < 1e-14 * want
        assert np.max(np.abs(got[1:])) < 1e-14
    assert abs(infl(orc, RECT, 2.0, 3.0, [1.0, 0.0, 1.5])[0] - 8.5299235726509373) < 1e-13   # SURVEY value, a=2,b=3
    a = 1.7
    assert abs(infl(orc, RECT, a, a, [a / 2, 0, a / 2])[0] - 4 * a * np.log(1 + np.sqrt(2))) < 1e-14


def test_square_on_axis_closed_form(orc):
    # Phi' = 2a ln[(r+a/2)/(r-a/2)] - 4h atan(a^2/(4hr)),  E'_y = 4 atan(a^2/(4hr)),  r = sqrt(a^2/2+h^2)
    for a, h in [(1.0, 0.3), (2.5, 0.01), (1.0, 40.0)]:
        r = np.sqrt(a * a / 2 + h * h)
        phi = 2 * a * np.log((r + a / 2) / (r - a / 2)) - 4 * h * np.arctan(a * a / (4 * h * r))
        ey = 4 * np.arctan(a * a / (4 * h * r))
        for sgn in (+1, -1):
            got = infl(orc, RECT, a, a, [a / 2, sgn * h, a / 2])
            assert abs(got[0] - phi) < 2e-13 * phi
            assert abs(got[2] - sgn * ey) < 2e-13 * ey
            assert abs(got[1]) < 1e-13 and abs(got[3]) < 1e-13


def test_triangle_centroid_solid_angle_limit(orc):
    # just above the interior the element fills half of space: Omega -> 2 pi, E'_y -> +-2 pi
    for sgn in (+1, -1):
        got = infl(orc, TRI, 1.0, 1.0, [1 / 3, sgn * 1e-9, 1 / 3])
        assert abs(got[2] - sgn * 2 * PI) < 1e-7
    got = infl(orc, TRI, 1.0, 1.0, [1 / 3, 0.0, 1 / 3])
    assert got[2] == 0.0                                   # reading S5: principal value on the surface
    assert abs(got[1] - got[3]) < 1e-14                    # mirror symmetry of the isosceles right triangle


def test_wire_closed_form_midplane(orc):
    # mid-plane of a wire of length 2h: Phi' = 2 asinh(h/rho); E' radial = 2h/(rho sqrt(rho^2+h^2))
    h, rho, rw = 0.5, 0.2, 1e-3
    got = orc.influence(WIRE, [0, 0, -h], [0, 0, 2 * h], [0, 0, 0], [rho, 0, 0], radius=rw) / (2 * PI * rw)
    assert abs(got[0] - 2 * np.arcsinh(h / rho)) < 1e-14
    assert abs(got[1] - 2 * h / (rho * np.hypot(rho, h))) < 1e-13
    assert abs(got[2]) < 1e-15 and abs(got[3]) < 1e-15


def test_wire_survey_pin(orc):
    # SURVEY 8(c) pin (40-digit quadrature of the line integral during the survey; tests/golden holds the same point,
    # re-integrated by make_quadrature_pins.py): h = 0.5, rho = 0.2, Z = 0.35 from the centre along the axis:
    # Phi' = 2.84677535102197, E'_rho = 7.86708584166788, E'_z = 2.85480333137226 per unit line density
    h, rho, Z, rw = 0.5, 0.2, 0.35, 1e-3
    got = orc.influence(WIRE, [0, 0, -h], [0, 0, 2 * h], [0, 0, 0], [rho, 0, Z], radius=rw) / (2 * PI * rw)
    assert abs(got[0] - 2.84677535102197) < 2e-14 * 2.85 and abs(got[1] - 7.86708584166788) < 2e-14 * 7.87
    assert abs(got[3] - 2.85480333137226) < 2e-14 * 2.85 and abs(got[2]) < 1e-15
    gold = [c for c in _gold_cases() if c[0] == "wire" and c[3] == [0.85, 0.0, 0.2]]
    assert len(gold) == 1 and abs(gold[0][4][0] - 2.84677535102197) < 1e-14 and abs(gold[0][4][3] - 7.86708584166788) < 1e-14


# ---------------------------------------------------------------------------------------------
# 4. far-field limit Eq.(2) P:68 and E = -grad Phi P:75
# ---------------------------------------------------------------------------------------------
@pytest.mark.parametrize("kind", [RECT, TRI, WIRE])
def test_far_field_monopole(orc, kind):
    a, b = 1.0, 0.6
    area = {RECT: a * b, TRI: 0.5 * a * b, WIRE: a}[kind]
    cen = {RECT: np.array([a / 2, 0, b / 2]), TRI: np.array([a / 3, 0, b / 3]), WIRE: np.array([a / 2, 0, 0])}[kind]
    u = np.array([0.3, -0.5, 0.81]); u /= np.linalg.norm(u)
    prev = None
    for R in (50.0, 100.0, 200.0):
        rw = 1e-3
        got = infl(orc, kind, a, b, cen + R * u, radius=rw)
        if kind == WIRE:
            got = got / (2 * PI * rw)
        err = abs(got[0] * R / area - 1.0)
        assert err < 0.6 * (a / R) ** 2                      # O((L/r)^2): no dipole about the centroid
        assert np.linalg.norm(got[1:] * R * R / area - u) < 2 * (a / R) ** 2
        if prev is not None:
            assert err < 0.3 * prev                          # and it really falls off quadratically
        prev = err


@pytest.mark.parametrize("kind", [RECT, TRI, WIRE])
def test_field_is_minus_gradient(orc, kind):
    pr = W.random_elements(16, seed=40 + kind, kinds=(kind,), size_mm=(0.3, 1.0))
    rs = np.random.RandomState(17)
    for j in range(pr.n):
        v0, e1, e2 = pr.v0[:, j], pr.e1[:, j], pr.e2[:, j]
        L = max(np.linalg.norm(e1), np.linalg.norm(e2))
        P = v0 + 0.4 * e1 + 0.3 * e2 + rs.normal(size=3) * L * 0.7
        rad = pr.radius[j]
        if kind == WIRE:                                     # stay outside the wire surface
            P = P + 5 * rad * np.cross(e1 / np.linalg.norm(e1), [0.3, 0.5, 0.8])
        f = lambda Q: orc.influence(kind, v0, e1, e2, Q, radius=rad, mode="ld")
        E = f(P)[1:]
        h = 1e-5 * L
        G = np.array([(f(P + h * np.eye(3)[c])[0] - f(P - h * np.eye(3)[c])[0]) / (2 * h) for c in range(3)])
        assert np.linalg.norm(E + G) < 1e-7 * np.linalg.norm(E), (j, E, G)


# ---------------------------------------------------------------------------------------------
# 5. additivity and invariances
# ---------------------------------------------------------------------------------------------
def test_rectangle_is_two_right_triangles(orc):
    a, b = 1.0, 0.7
    for P in ([0.3, 0.25, 0.4], [0.9, -0.1, 0.1], [2.0, 0.0, -1.0], [0.5, 1e-4, 0.35]):
        r = orc.influence(RECT, [0, 0, 0], [a, 0, 0], [0, 0, b], P)
        t1 = orc.influence(TRI, [0, 0, 0], [a, 0, 0], [0, 0, b], P)
        # complementary triangle: right angle at (a,0,b), legs -e1 and -e2 (same normal: (-e2)x(-e1) = e2 x e1)
        t2 = orc.influence(TRI, [a, 0, b], [-a, 0, 0], [0, 0, -b], P)
        assert np.max(np.abs(r - t1 - t2)) < 2e-14 * max(1.0, np.max(np.abs(r)))
    assert abs(orc.influence(RECT, [0, 0, 0], [a, 0, 0], [0, 0, b], [0.3, 0.25, 0.4])[0] - 1.67956850898329) < 1e-13


def test_rectangle_is_four_subrectangles(orc):
    a, b, sx, sz = 1.3, 0.9, 0.45, 0.7
    for P in ([0.37, 0.21, -0.45], [0.45, 0.0, 0.7], [0.1, -0.02, 0.2]):
        whole = orc.influence(RECT, [0, 0, 0], [a, 0, 0], [0, 0, b], P)
        parts = sum(orc.influence(RECT, [x0, 0, z0], [dx, 0, 0], [0, 0, dz], P)
                    for x0, dx in ((0, sx), (sx, a - sx)) for z0, dz in ((0, sz), (sz, b - sz)))
        # at the shared corner (second point) the sub-rectangles' in-plane fields are log-singular (S6): Phi' only
        idx = [0, 2] if P[1] == 0.0 else [0, 1, 2, 3]
        assert np.max(np.abs(whole - parts)[idx]) < 3e-14 * max(1.0, np.max(np.abs(whole)))


def test_rotation_translation_invariance(orc):
    rs = np.random.RandomState(3)
    for kind in (RECT, TRI, WIRE):
        A, _ = np.linalg.qr(rs.normal(size=(3, 3)))
        if np.linalg.det(A) < 0:
            A[:, 0] = -A[:, 0]
        t = rs.normal(size=3)
        v0, e1, e2, P = np.array([0.1, 0.2, -0.3]), np.array([0.8, 0, 0]), np.array([0, 0, 0.5]), np.array([0.5, 0.3, 0.9])
        ref = orc.influence(kind, v0, e1, e2, P, radius=0.01)
        got = orc.influence(kind, A @ v0 + t, A @ e1, A @ e2, A @ P + t, radius=0.01)
        assert abs(got[0] - ref[0]) < 1e-14 * abs(ref[0])
        assert np.linalg.norm(got[1:] - A @ ref[1:]) < 1e-14 * np.linalg.norm(ref[1:])


def test_normal_convention_and_side(orc):
    # n = e2 x e1 / |..| (include/neb.h); E' points away from the element on both sides
    v0, e1, e2 = np.array([0, 0, 0.0]), np.array([0, 1.0, 0]), np.array([1.0, 0, 0])      # n = x cross y = +z
    up = orc.influence(RECT, v0, e1, e2, [0.5, 0.5, 0.2])
    dn = orc.influence(RECT, v0, e1, e2, [0.5, 0.5, -0.2])
    assert up[3] > 0 and dn[3] < 0 and abs(up[3] + dn[3]) < 1e-15 and abs(up[0] - dn[0]) < 1e-15


def test_gauss_law_closed_cube(orc):
    # sum over the faces of a closed cube of n_j.E'_j(P) = sum sgn(d_j) Omega_j = -4 pi inside, 0 outside
    pr = W.cube(n_side=2, m_points=1)
    nrm = pr.normals()
    for P, want in (([1e-3, -2e-3, 1.5e-3], -4 * PI), ([0.0, 0.0, 0.0], -4 * PI), ([9e-3, 1e-3, -2e-3], 0.0),
                    ([-6e-3, 7e-3, 8e-3], 0.0)):
        tot = 0.0
        for j in range(pr.n):
            o = orc.influence(RECT, pr.v0[:, j], pr.e1[:, j], pr.e2[:, j], P)
            tot += float(np.dot(nrm[:, j], o[1:]))
        assert abs(tot - want) < 1e-12, (P, tot)


def test_edge_and_corner_limits_are_finite(orc):
    # reading S6: on an edge / corner / edge extension nothing is inf or NaN and Phi' stays exact
    a, b = 1.0, 0.6
    on_edge = infl(orc, RECT, a, b, [0.4, 0.0, 0.0])
    corner = infl(orc, RECT, a, b, [0.0, 0.0, 0.0])
    ext = infl(orc, RECT, a, b, [1.7, 0.0, 0.0])
    for v in (on_edge, corner, ext):
        assert np.all(np.isfinite(v))
    # Phi' at a corner of an a x b rectangle: a asinh(b/a) + b asinh(a/b) (quarter of the centre value of 2a x 2b)
    assert abs(corner[0] - (a * np.arcsinh(b / a) + b * np.arcsinh(a / b))) < 1e-14
    # Phi' on an edge at abscissa s: two corner values
    s = 0.4
    want = sum(x * np.arcsinh(b / x) + b * np.arcsinh(x / b) for x in (s, a - s))
    assert abs(on_edge[0] - want) < 1e-14
    for v in (infl(orc, TRI, a, b, [0.5, 0.0, 0.3]), infl(orc, TRI, a, b, [0, 0, 0]), infl(orc, TRI, a, b, [0.3, 0, 0])):
        assert np.all(np.isfinite(v))


# ---------------------------------------------------------------------------------------------
# 6. point charges (Eq. 2, Alg. 2)
# ---------------------------------------------------------------------------------------------
def test_point_charge_coulomb_constant_and_skip(orc):
    # 1 C at 1 m: Phi = k_e = 8.9875517923e9 V (CODATA), |E| = k_e V/m, pointing away
    pts = np.array([[1.0, 0.0], [0.0, 0.0], [0.0, 0.0]])
    phi, E = orc.point_charges(pts, np.zeros((3, 1)), np.array([1.0]))
    assert abs(phi[0] / 8.9875517923e9 - 1) < 1e-10
    assert abs(E[0, 0] / 8.9875517923e9 - 1) < 1e-10 and E[1, 0] == 0 and E[2, 0] == 0
    assert phi[1] == 0 and np.all(E[:, 1] == 0)            # r = 0 contributes nothing (S11)


def test_point_charge_superposition_and_gradient(orc):
    rs = np.random.RandomState(0)
    pos, q = rs.normal(size=(3, 50)), rs.normal(size=50)
    P = np.array([[3.0], [-2.0], [1.5]])
    phi, E = orc.point_charges(P, pos, q)
    one = sum(orc.point_charges(P, pos[:, k:k + 1], q[k:k + 1])[0][0] for k in range(50))
    assert abs(phi[0] - one) < 1e-12 * abs(phi[0])
    h = 1e-5
    G = [(orc.point_charges(P + h * np.eye(3)[:, c:c + 1], pos, q)[0][0]
          - orc.point_charges(P - h * np.eye(3)[:, c:c + 1], pos, q)[0][0]) / (2 * h) for c in range(3)]
    assert np.linalg.norm(E[:, 0] + G) < 1e-8 * np.linalg.norm(E[:, 0])
    # far away the cloud is a monopole
    far = np.array([[4e3], [3e3], [0.0]])
    phi_f, _ = orc.point_charges(far, pos, q)
    assert abs(phi_f[0] - 8.9875517923e9 * q.sum() / 5e3) < 2e-3 * abs(phi_f[0])


# ---------------------------------------------------------------------------------------------
# 7. dense solve (Alg. 1; S13, S15, S16) against numpy.linalg
# ---------------------------------------------------------------------------------------------
@pytest.mark.parametrize("mode", ["ld", "f64"])
def test_lu_against_numpy(orc, mode):
    rs = np.random.RandomState(1)
    n = 200
    K = rs.normal(size=(n, n))
    K[np.arange(n), np.arange(n)] = 0.0                      # forces row exchanges
    K *= 10.0 ** rs.uniform(-6, 6, size=(n, 1))              # rows spanning 12 decades (S15)
    b = rs.normal(size=n) * np.abs(K).max(axis=1)
    x = orc.solve(K, b, mode=mode)
    want = np.linalg.solve(K / np.abs(K).max(axis=1, keepdims=True), b / np.abs(K).max(axis=1))
    assert np.max(np.abs(x - want)) < 1e-9 * np.max(np.abs(want))
    lu = orc.LU(K, mode=mode)
    b2 = rs.normal(size=n)
    x2 = lu.solve(b2)
    rowmax = np.abs(K).max(axis=1)
    assert np.max(np.abs(K @ x2 - b2) / rowmax) < 1e-12 * n * np.max(np.abs(x2))     # S16 residual, row-scaled
    with pytest.raises(np.linalg.LinAlgError):
        orc.solve(np.zeros((4, 4)), np.ones(4), mode=mode)


# ---------------------------------------------------------------------------------------------
# 8. whole pipeline on problems with known answers
# ---------------------------------------------------------------------------------------------
def _solve_dirichlet(orc, pr, mode="f64"):
    g = orc.Geometry(pr)
    K = orc.assemble(g, mode=mode)
    b = orc.rhs(g, mode=mode)
    return g, K, orc.solve(K, b, mode=mode)


def _areas(pr):
    a = np.linalg.norm(np.cross(pr.e1.T, pr.e2.T), axis=1)
    return np.where(pr.kind == TRI, 0.5 * a, a)


def test_c0_plate_charge_density_and_capacitance(orc):
    pr = W.plate()
    g, K, sig = _solve_dirichlet(orc, pr)
    n = 16
    S = sig.reshape(n, n)
    # the 8 symmetries of the square
    for T in (S.T, S[::-1], S[:, ::-1], S[::-1, ::-1].T):
        assert np.max(np.abs(T - S)) < 1e-12 * S.max()
    # edge peaking: monotone from centre to edge along a row, largest at the corners, smallest at the centre
    assert np.all(np.diff(S[n // 2, n // 2:]) > 0)
    assert S.max() == pytest.approx(S[0, 0]) and S.min() == pytest.approx(S[n // 2, n // 2])
    # capacitance of a square plate of side a: C/(4 pi eps0 a) = 0.3667896 (literature value, 7 digits);
    # uniform panels converge to it from below (16x16 gives 0.3593, 2 % low)
    a = pr.meta["side"]
    cap = np.sum(sig * _areas(pr)) / (4 * PI * orc.EPS0 * a)
    assert 0.355 < cap < 0.3668
    cap8 = np.sum(_solve_dirichlet(orc, W.plate(n_side=8))[2] * _areas(W.plate(n_side=8))) / (4 * PI * orc.EPS0 * a)
    assert cap8 < cap
    # boundary condition reproduced at the collocation points by the evaluation path (assembly/eval consistent)
    phi, _ = orc.evaluate(g, sig, g.colloc, mode="f64")
    assert np.max(np.abs(phi - 1.0)) < 1e-12
    # on-axis field: odd in z, no transverse component; potential even in z
    pts = np.array([[0, 0, 0, 0], [0, 0, 0, 0], [1e-3, -1e-3, 5e-3, -5e-3]], dtype=float)
    phi, E = orc.evaluate(g, sig, pts, mode="f64")
    assert abs(phi[0] - phi[1]) < 1e-13 and abs(E[2, 0] + E[2, 1]) < 1e-10 * abs(E[2, 0])
    assert np.max(np.abs(E[:2])) < 1e-9 * abs(E[2, 0])
    assert 0.5 < phi[2] < phi[0] < 1.0 and E[2, 0] > 0 and E[2, 1] < 0


def test_c1_cube_capacitance_sequence(orc):
    # unit-cube capacitance C/(4 pi eps0 a) = 0.66078 (literature, 5 digits); uniform-panel BEM converges from below
    caps = []
    for ns in (4, 6, 8, 12):
        pr = W.cube(n_side=ns, m_points=1)
        _, _, sig = _solve_dirichlet(orc, pr)
        caps.append(np.sum(sig * _areas(pr)) / (4 * PI * orc.EPS0 * pr.meta["side"]))
    assert np.all(np.diff(caps) > 0) and caps[-1] < 0.6608
    assert abs(caps[-1] - 0.6608) < 0.004
    # Richardson with error ~ 1/ns
    rich = (12 * caps[3] - 8 * caps[2]) / 4
    assert abs(rich - 0.6608) < 1.5e-3
    # inside a closed conductor Phi = V and E = 0 up to discretisation error
    pr = W.cube(n_side=8, m_points=1)
    g, _, sig = _solve_dirichlet(orc, pr)
    phi, E = orc.evaluate(g, sig, np.array([[1e-3], [-2e-3], [0.5e-3]]), mode="f64")
    assert abs(phi[0] - 1.0) < 2e-3
    e_surface = sig.mean() / orc.EPS0
    assert np.linalg.norm(E[:, 0]) < 2e-2 * e_surface


def test_two_plate_capacitor_uniform_field(orc):
    # stand-in for the paper's Case 1: between large plates the field tends to V/gap
    side, gap, ns = 10.0, 0.5, 20
    top, bot = W.plate(n_side=ns, side_mm=side, volt=+0.5, m_points=1), W.plate(n_side=ns, side_mm=side, volt=-0.5, m_points=1)
    top.v0[2] += gap / 2 * W.MM
    bot.v0[2] -= gap / 2 * W.MM
    pr = _concat(top, bot)
    g, _, sig = _solve_dirichlet(orc, pr)
    phi, E = orc.evaluate(g, sig, np.zeros((3, 1)), mode="f64")
    assert abs(phi[0]) < 1e-9
    assert abs(E[2, 0] / (-1.0 / (gap * W.MM)) - 1) < 5e-3


def _concat(*prs):
    cat = lambda k: np.concatenate([getattr(p, k) for p in prs], axis=-1)
    return W.Problem(name="+".join(p.name for p in prs), kind=cat("kind"), v0=cat("v0"), e1=cat("e1"), e2=cat("e2"),
                     radius=cat("radius"), bc_kind=cat("bc_kind"), bc_value=cat("bc_value"), eps_plus=cat("eps_plus"),
                     eps_minus=cat("eps_minus"))


def _sheet(ns, side_mm, z_mm, normal_sign, **bc):
    b = W._Builder()
    p = side_mm / ns
    ia, ib = W._grid_cells(ns, ns)
    b.rect_cells((-side_mm / 2, -side_mm / 2, z_mm), (p, 0, 0), (0, p, 0), ia, ib, (0, 0, normal_sign), **bc)
    return b.finish("sheet")


def test_point_charge_over_dielectric_half_space(orc):
    # dielectric rows only (reading S8 sign and lambda, S10 RHS): coplanar panels exert no normal field on each
    # other, so K is diagonal and sigma_i equals the textbook image-solution bound charge at every centroid:
    #   sigma_b(rho) = -(q / 2 pi) (eps_r - 1)/(eps_r + 1) d / (rho^2 + d^2)^(3/2)
    eps_r, d, q = 4.4, 0.7e-3, 3e-15
    pr = _sheet(10, 4.0, 0.0, +1, bc_kind=W.DIELECTRIC, bc_value=0.0, eps_plus=1.0, eps_minus=eps_r)
    g = orc.Geometry(pr)
    K = orc.assemble(g, mode="ld")
    off = K - np.diag(np.diag(K))
    assert np.max(np.abs(off)) == 0.0
    b = orc.rhs(g, np.array([[0.0], [0.0], [d]]), np.array([q]), mode="ld")
    sig = orc.solve(K, b, mode="ld")
    rho2 = g.colloc[0] ** 2 + g.colloc[1] ** 2
    want = -(q / (2 * PI)) * (eps_r - 1) / (eps_r + 1) * d / (rho2 + d * d) ** 1.5
    assert np.max(np.abs(sig - want)) < 1e-13 * np.max(np.abs(want))


def test_dielectric_slab_in_capacitor(orc):
    # plates +-0.5 V at z=+-0.5 mm, slab faces at z=+-0.2 mm, eps_r=4.4, all W x W with W=8 mm, 20x20 panels each.
    # central |E_z|: gas 1/(0.6+0.4/4.4) V/mm = 1.447368, slab 0.328947 (series capacitor), finite-size error ~1e-4
    ns, Wd = 20, 8.0
    pr = _concat(_sheet(ns, Wd, +0.5, -1, bc_kind=W.DIRICHLET, bc_value=+0.5),
                 _sheet(ns, Wd, -0.5, +1, bc_kind=W.DIRICHLET, bc_value=-0.5),
                 _sheet(ns, Wd, +0.2, +1, bc_kind=W.DIELECTRIC, bc_value=0.0, eps_plus=1.0, eps_minus=4.4),
                 _sheet(ns, Wd, -0.2, -1, bc_kind=W.DIELECTRIC, bc_value=0.0, eps_plus=1.0, eps_minus=4.4))
    g, _, sig = _solve_dirichlet(orc, pr)
    # keep off the panel centroids' singular normal-field jump: evaluate mid-gas and mid-slab on the axis
    _, E = orc.evaluate(g, sig, np.array([[0.0, 0.0], [0.0, 0.0], [0.35e-3, 0.0]]), mode="f64")
    assert abs(abs(E[2, 0]) * 1e-3 / 1.447368 - 1) < 5e-4
    assert abs(abs(E[2, 1]) * 1e-3 / 0.328947 - 1) < 5e-4
    assert E[2, 0] < 0 and E[2, 1] < 0                      # from the +0.5 V plate down to the -0.5 V plate


def test_image_copies_equal_explicit_replication(orc):
    # reading S12: summing shifted copies inside each coefficient == meshing the copies explicitly with shared sigma
    pr = W.random_elements(6, seed=9, kinds=(RECT, TRI), size_mm=(0.2, 0.5), box_mm=0.4, m_points=5)
    shifts = W.image_shifts(1, pitch_mm=1.0)
    pr.img_shift = shifts
    g = orc.Geometry(pr)
    sig = np.linspace(1.0, 2.0, pr.n) * 1e-6
    phi, E = orc.evaluate(g, sig, pr.points)
    reps = []
    for s in range(shifts.shape[1]):
        c = W.random_elements(6, seed=9, kinds=(RECT, TRI), size_mm=(0.2, 0.5), box_mm=0.4)
        c.v0 = c.v0 + shifts[:, s:s + 1]
        reps.append(c)
    big = _concat(*reps)
    phi2, E2 = orc.evaluate(orc.Geometry(big), np.tile(sig, shifts.shape[1]), pr.points)
    assert np.max(np.abs(phi - phi2)) < 1e-13 * np.max(np.abs(phi))
    assert np.max(np.abs(E - E2)) < 1e-13 * np.max(np.abs(E))
    K = orc.assemble(g)
    Kbig = orc.assemble(orc.Geometry(big))
    fold = sum(Kbig[:pr.n, s * pr.n:(s + 1) * pr.n] for s in range(shifts.shape[1]))
    assert np.max(np.abs(K - fold)) < 1e-13 * np.max(np.abs(K))


# ---------------------------------------------------------------------------------------------
# 8b. the principal-value rule of dielectric rows (readings S5/S8: the UNSHIFTED copy of element i gives no
#     field at its own collocation point, applied by index; "its image copies do contribute") on obliquely
#     oriented elements and with periodic copies.  None of the expected values below comes from the rule itself.
# ---------------------------------------------------------------------------------------------
def _rotation(seed):
    A, _ = np.linalg.qr(np.random.RandomState(seed).normal(size=(3, 3)))
    if np.linalg.det(A) < 0:
        A[:, 0] = -A[:, 0]
    return A


def _moved(pr, A, t):
    """The same problem rotated by A and translated by t (a rigid motion of every element)."""
    return W.Problem(name=pr.name + "_moved", kind=pr.kind.copy(), v0=A @ pr.v0 + t[:, None], e1=A @ pr.e1, e2=A @ pr.e2,
                     radius=pr.radius.copy(), bc_kind=pr.bc_kind.copy(), bc_value=pr.bc_value.copy(),
                     eps_plus=pr.eps_plus.copy(), eps_minus=pr.eps_minus.copy(),
                     img_shift=None if pr.img_shift is None else A @ pr.img_shift)


def _dielectric_cube(ns=3, eps_r=4.4):
    """Closed cube of side 1 mm, outward normals, every panel a dielectric row (eps_r inside, 1 outside); the top
    face's panels are split into right triangles so both flat kinds sit on dielectric rows."""
    b = W._Builder()
    h, p = 0.5, 1.0 / ns
    ax = np.eye(3)
    bc = dict(bc_kind=W.DIELECTRIC, bc_value=0.0, eps_plus=1.0, eps_minus=eps_r)
    ia, ib = W._grid_cells(ns, ns)
    for k in range(3):
        a, c = ax[(k + 1) % 3], ax[(k + 2) % 3]
        for s in (+1.0, -1.0):
            org = s * h * ax[k] - h * a - h * c
            if k == 2 and s > 0:
                for i, j in zip(ia, ib):
                    o = org + i * p * a + j * p * c
                    b.add(TRI, o, p * a, p * c, s * ax[k], **bc)
                    b.add(TRI, o + p * a + p * c, -p * a, -p * c, s * ax[k], **bc)
            else:
                b.rect_cells(org, p * a, p * c, ia, ib, s * ax[k], **bc)
    return b.finish("dielectric_cube")


def test_dielectric_self_term_on_oblique_elements(orc):
    # A matrix entry is a scalar of the geometry: a rigid motion of the whole problem leaves K unchanged.  On the
    # axis-aligned cube every centroid lies in its panel's plane EXACTLY (Y == 0, where sgn(0) Omega = 0 is the
    # formula's own value and the half-space pin above fixes the row); on the moved cube it lies there only up to
    # rounding, where a sign test on Y would add +-2 pi k_e — as large as the diagonal term k_e 2 pi / lambda.
    pr = _dielectric_cube()
    assert np.sum(pr.kind == TRI) == 18 and pr.n == 5 * 9 + 18
    Ka = orc.assemble(orc.Geometry(pr))
    rowmax = np.abs(Ka).max(axis=1, keepdims=True)
    lam = (1.0 - 4.4) / (1.0 + 4.4)
    # the self term contributes nothing: the diagonal is the analytic jump term alone (reading S8)
    assert np.max(np.abs(np.diag(Ka) * (2 * orc.EPS0 * lam) - 1.0)) < 1e-15
    for seed in (1, 2, 3):
        A, t = _rotation(seed), np.random.RandomState(seed).normal(size=3) * 1e-3
        Km = orc.assemble(orc.Geometry(_moved(pr, A, t)))
        assert np.max(np.abs(Km - Ka) / rowmax) < 1e-13, seed
        assert np.max(np.abs(np.diag(Km) * (2 * orc.EPS0 * lam) - 1.0)) < 1e-15, seed


def test_dielectric_flux_identity_on_closed_oblique_cube(orc):
    # Gauss's law for the field of panel j through the closed surface it is part of: the flux of E'_j is
    # 4 pi A_j x (1/2) (the source lies ON the surface: principal value), so with the centroid rule
    #   sum_i A_i n_i . E'_j(p_i)  ~  2 pi A_j   for every j,
    # up to the quadrature error of one point per panel: < 1 % for panels that do not touch an edge of the cube (a
    # panel at an edge sees its neighbour across the edge at a scale-invariant angle: 19 % / 31 % for rectangles /
    # triangles at any mesh, so those are only checked in the area-weighted total, which converges like 1/ns),
    # whereas a self term of +-2 pi (sign of a rounding error in Y) would change the i = j summand from 0 to
    # +-2 pi A_j: an error of 100 % on that panel.  Same on the axis-aligned and on obliquely moved cubes, and with
    # 3 x 3 periodic copies a pitch of 3 sides away (their flux through the closed surface is zero: sources outside).
    lam = (1.0 - 4.4) / (1.0 + 4.4)
    for ns, lim, lim_tot in ((4, 0.01, 0.10), (8, 0.005, 0.055)):
        pr = _dielectric_cube(ns)
        area = _areas(pr)
        second = np.sort(np.abs(pr.centroids()), axis=0)[1]          # distance to the nearest cube edge, via the centroid
        interior = second < (0.5 - 1.0 / ns) * W.MM
        assert interior.sum() >= 28 and np.any(interior & (pr.kind == TRI))
        for motion in (None, 5):
            for images in (False, True):
                q = pr if motion is None else _moved(pr, _rotation(motion), np.array([1e-3, -2e-3, 0.5e-3]))
                if images:
                    sh = W.image_shifts(1, pitch_mm=3.0)
                    q.img_shift = sh if motion is None else _rotation(motion) @ sh
                K = orc.assemble(orc.Geometry(q), mode="f64")
                F = (K - np.diag(np.full(pr.n, 1.0 / (2 * orc.EPS0 * lam)))) / orc.K_COULOMB     # n_i . E'_j(p_i)
                flux = area @ F
                assert np.max(np.abs(flux[interior] / (2 * PI * area[interior]) - 1.0)) < lim, (ns, motion, images)
                assert abs(flux.sum() / (2 * PI * area.sum()) - 1.0) < lim_tot, (ns, motion, images)
                q.img_shift = None


def test_dielectric_rows_with_image_copies_vs_quadrature(orc):
    # "its image copies do contribute" (S8): on a dielectric row the diagonal entry is the jump term plus the normal
    # field of the element's OWN shifted copies, and an off-diagonal entry sums all copies of the other element.
    # Expected values: tensor Gauss-Legendre quadrature of the defining integral P:131 (no oracle code); the copies
    # are a pitch (>= 1.7 element sizes) away, where 96^2 nodes are exact to rounding.
    pr = W.random_elements(5, seed=17, kinds=(RECT, TRI), size_mm=(0.2, 0.4), box_mm=0.3, dielectric_fraction=1.0)
    assert np.all(pr.bc_kind == W.DIELECTRIC)
    # a ONE-SIDED set of copies (x >= 0): in a set symmetric about the element the copies at +s and -s of a
    # centro-symmetric element (a rectangle) cancel at its centroid, and the check would be vacuous
    full = W.image_shifts(1, pitch_mm=0.7)
    shifts = np.ascontiguousarray(full[:, full[0] >= 0])
    assert shifts.shape[1] == 6 and np.all(shifts[:, 0] == 0)
    pr.img_shift = shifts
    g = orc.Geometry(pr)
    K = orc.assemble(g)
    nrm, col = pr.normals(), pr.centroids()
    lam = (pr.eps_plus - pr.eps_minus) / (pr.eps_plus + pr.eps_minus)
    for i in range(pr.n):
        own = sum(nrm[:, i] @ _gl_quadrature(pr.kind[i], pr.v0[:, i] + shifts[:, s], pr.e1[:, i], pr.e2[:, i], col[:, i])[1:]
                  for s in range(1, shifts.shape[1]))
        want = orc.K_COULOMB * own + 1.0 / (2 * orc.EPS0 * lam[i])
        assert abs(own) > 1e-3                                   # the copies really contribute (oblique elements, one-sided set)
        assert abs(K[i, i] - want) < 1e-12 * abs(want), i
    # off-diagonal entries between well separated elements (all nine copies by quadrature)
    done = 0
    for i in range(pr.n):
        for j in range(pr.n):
            L = max(np.linalg.norm(pr.e1[:, j]), np.linalg.norm(pr.e2[:, j]))
            if i == j or np.linalg.norm(col[:, i] - col[:, j]) < 1.5 * L:
                continue
            tot = sum(nrm[:, i] @ _gl_quadrature(pr.kind[j], pr.v0[:, j] + shifts[:, s], pr.e1[:, j], pr.e2[:, j], col[:, i], n=128)[1:]
                      for s in range(shifts.shape[1]))
            assert abs(K[i, j] - orc.K_COULOMB * tot) < 2e-10 * orc.K_COULOMB * abs(tot) + 1e-12 * np.abs(K[i]).max(), (i, j)
            done += 1
    assert done >= 4


def test_image_copies_equal_explicit_replication_dielectric_rows(orc):
    # reading S12 on dielectric rows: the field branch of the image sum == explicit copies of the mesh with shared
    # sigma; in the replicated mesh the copies of element i are ordinary OTHER elements (entries pinned above by
    # quadrature), so the fold's diagonal holds exactly what "its image copies do contribute" means.
    pr = W.random_elements(7, seed=23, kinds=(RECT, TRI), size_mm=(0.2, 0.5), box_mm=0.4, dielectric_fraction=0.6)
    assert 0 < np.sum(pr.bc_kind == W.DIELECTRIC) < pr.n
    full = W.image_shifts(1, pitch_mm=0.9)
    shifts = np.ascontiguousarray(full[:, full[0] >= 0])       # one-sided: a symmetric set cancels at a rectangle's centre
    pr.img_shift = shifts
    K = orc.assemble(orc.Geometry(pr))
    reps = []
    for s in range(shifts.shape[1]):
        c = W.random_elements(7, seed=23, kinds=(RECT, TRI), size_mm=(0.2, 0.5), box_mm=0.4, dielectric_fraction=0.6)
        c.v0 = c.v0 + shifts[:, s:s + 1]
        reps.append(c)
    Kbig = orc.assemble(orc.Geometry(_concat(*reps)))
    fold = sum(Kbig[:pr.n, s * pr.n:(s + 1) * pr.n] for s in range(shifts.shape[1]))
    assert np.max(np.abs(K - fold) / np.abs(K).max(axis=1, keepdims=True)) < 1e-13
    d = pr.bc_kind == W.DIELECTRIC
    copies_on_diag = np.diag(fold)[d] - np.diag(Kbig[:pr.n, :pr.n])[d]
    assert np.all(np.abs(copies_on_diag) > 1e-8 * np.abs(np.diag(K)[d]))    # not a vacuous check (tolerance above: 1e-13)


def test_rotated_dielectric_slab_in_capacitor(orc):
    # the series-capacitor pin above on an obliquely rotated geometry: same sigma (rigid motion), textbook fields
    ns, Wd = 12, 8.0
    pr = _concat(_sheet(ns, Wd, +0.5, -1, bc_kind=W.DIRICHLET, bc_value=+0.5),
                 _sheet(ns, Wd, -0.5, +1, bc_kind=W.DIRICHLET, bc_value=-0.5),
                 _sheet(ns, Wd, +0.2, +1, bc_kind=W.DIELECTRIC, bc_value=0.0, eps_plus=1.0, eps_minus=4.4),
                 _sheet(ns, Wd, -0.2, -1, bc_kind=W.DIELECTRIC, bc_value=0.0, eps_plus=1.0, eps_minus=4.4))
    A, t = _rotation(11), np.array([0.3e-3, 0.1e-3, -0.2e-3])
    _, _, sig0 = _solve_dirichlet(orc, pr)
    g, _, sig = _solve_dirichlet(orc, _moved(pr, A, t))
    assert np.max(np.abs(sig - sig0)) < 1e-10 * np.max(np.abs(sig0))
    pts = A @ np.array([[0.0, 0.0], [0.0, 0.0], [0.35e-3, 0.0]]) + t[:, None]
    _, E = orc.evaluate(g, sig, pts, mode="f64")
    Ez = A[:, 2] @ E                                            # component along the rotated z axis
    assert abs(abs(Ez[0]) * 1e-3 / 1.447368 - 1) < 2e-3 and abs(abs(Ez[1]) * 1e-3 / 0.328947 - 1) < 2e-3
    assert Ez[0] < 0 and Ez[1] < 0


def test_eval_abs_is_the_sum_of_term_magnitudes(orc):
    # orc_eval_abs (tolerance scale of the parity tests): rebuilt here term by term from single-element and
    # single-charge evaluations; equals |Phi| when all terms have one sign; >= |Phi|, |E| always.
    pr = W.random_elements(9, seed=41, m_points=7)
    pr.img_shift = W.image_shifts(1, pitch_mm=5.0)
    g = orc.Geometry(pr)
    rs = np.random.RandomState(2)
    sig = rs.normal(size=pr.n) * 1e-6
    pos, ch = rs.normal(size=(3, 4)) * 1e-3, rs.normal(size=4) * 1e-15
    sp, se = orc.evaluate_abs(g, sig, pr.points, pos, ch, mode="ld")
    wp, we = np.zeros(7), np.zeros(7)
    for j in range(pr.n):
        for s in range(9):
            for p in range(7):
                o = orc.influence(pr.kind[j], pr.v0[:, j] + pr.img_shift[:, s], pr.e1[:, j], pr.e2[:, j], pr.points[:, p],
                                  radius=pr.radius[j])
                wp[p] += orc.K_COULOMB * abs(sig[j]) * abs(o[0])
                we[p] += orc.K_COULOMB * abs(sig[j]) * np.linalg.norm(o[1:])
    for k in range(4):
        r = np.linalg.norm(pr.points - pos[:, k:k + 1], axis=0)
        wp += orc.K_COULOMB * abs(ch[k]) / r
        we += orc.K_COULOMB * abs(ch[k]) / r ** 2
    assert np.max(np.abs(sp / wp - 1)) < 1e-13 and np.max(np.abs(se / we - 1)) < 1e-13
    phi, E = orc.evaluate(g, sig, pr.points, pos, ch)
    for mode in ("ld", "f64"):                                         # the one-pass variant returns evaluate()'s own sums
        sp2, se2, phi2, E2 = orc.evaluate_abs(g, sig, pr.points, pos, ch, mode=mode, with_field=True)
        phi_m, E_m = orc.evaluate(g, sig, pr.points, pos, ch, mode=mode)
        assert np.array_equal(phi2, phi_m) and np.array_equal(E2, E_m)
        assert np.array_equal(sp2, orc.evaluate_abs(g, sig, pr.points, pos, ch, mode=mode)[0])
    assert np.all(sp >= np.abs(phi)) and np.all(se >= np.linalg.norm(E, axis=0) * (1 - 1e-15))
    phi1, _ = orc.evaluate(g, np.abs(sig), pr.points, pos, np.abs(ch))
    flat = np.abs(pr.kind) >= 0
    sp1, _ = orc.evaluate_abs(g, np.abs(sig), pr.points, pos, np.abs(ch), mode="ld")
    assert flat.all() and np.max(np.abs(sp1 / phi1 - 1)) < 1e-13        # Phi' > 0 for every element kind


def test_solve_library_equals_plain_lu(orc):
    # oracle.solve_library (numpy/LAPACK after the S15 row scaling) against the plain C elimination, on a mixed
    # Dirichlet/dielectric system (rows of 1e5 and 1e11) and on a matrix that forces row exchanges
    pr = W.thgem(d=10, n_plane=6, n_grid=2)
    g = orc.Geometry(pr)
    K, b = orc.assemble(g, mode="f64"), orc.rhs(g, mode="f64")
    x0, x1 = orc.solve(K, b, mode="ld"), orc.solve_library(K, b)
    assert np.max(np.abs(x0 - x1)) < 1e-11 * np.max(np.abs(x0))
    rs = np.random.RandomState(4)
    M = rs.normal(size=(150, 150))
    M[np.arange(150), np.arange(150)] = 0.0
    M *= 10.0 ** rs.uniform(-5, 5, size=(150, 1))
    v = rs.normal(size=150) * np.abs(M).max(axis=1)
    x0, x1 = orc.solve(M, v, mode="ld"), orc.solve_library(M, v)
    assert np.max(np.abs(x0 - x1)) < 1e-9 * np.max(np.abs(x0))


def test_solve_svd_minimum_norm_on_overlapping_panels(orc):
    """OptSVD (reading S31).  Pins of oracle.solve_svd to things other than itself:
    (i) on a non-singular system it gives what the plain C elimination gives (a different algorithm);
    (ii) with k panels listed twice the matrix has k pairs of equal columns (and rows): the LU path fails; the
        minimum-norm solution must share each doubled panel's charge EQUALLY between the two copies (for equal columns
        a, a the norm x1^2 + x2^2 at fixed x1 + x2 is least at x1 = x2) and reproduce the non-overlapping solution:
        sigma_a + sigma_a' = sigma_single, every other sigma unchanged;
    (iii) the Moore-Penrose conditions on a random rank-deficient matrix M = L R: the residual is orthogonal to the
        range (M^T (M x - v) = 0) and x is orthogonal to the null space of R, built independently by a QR of R^T."""
    pr = W.plate(n_side=10)
    g = orc.Geometry(pr)
    K, b = orc.assemble(g, mode="f64"), orc.rhs(g, mode="f64")
    s_lu = orc.solve(K, b, mode="ld")
    s_svd = orc.solve_svd(K, b)
    assert np.max(np.abs(s_svd - s_lu)) < 1e-10 * np.max(np.abs(s_lu))
    idx = np.array([0, 17, 44, 45, 99])
    pr2 = W.with_coincident_panels(pr, idx)
    g2 = orc.Geometry(pr2)
    K2, b2 = orc.assemble(g2, mode="f64"), orc.rhs(g2, mode="f64")
    assert np.array_equal(K2[:, idx], K2[:, pr.n:]) and np.array_equal(K2[idx, :], K2[pr.n:, :])
    with pytest.raises(np.linalg.LinAlgError):
        orc.solve(K2, b2, mode="ld")
    s2 = orc.solve_svd(K2, b2)
    scale = np.max(np.abs(s_lu))
    assert np.max(np.abs(s2[idx] - s2[pr.n:])) < 1e-9 * scale                      # equal split
    merged = s2[: pr.n].copy()
    merged[idx] += s2[pr.n:]
    assert np.max(np.abs(merged - s_lu)) < 1e-9 * scale                           # same physics as without the overlap
    phi1, E1 = orc.evaluate(g, s_lu, pr.points[:, :50])
    phi2, E2 = orc.evaluate(g2, s2, pr.points[:, :50])
    assert np.max(np.abs(phi2 - phi1)) < 1e-9 * np.max(np.abs(phi1))
    rs = np.random.RandomState(8)
    n, k = 60, 41
    L, R = rs.normal(size=(n, k)), rs.normal(size=(k, n))
    M = L @ R
    M /= np.abs(M).max(axis=1)[:, None]                                          # rows already equilibrated: r = 1
    v = rs.normal(size=n)
    x = orc.solve_svd(M, v)
    assert np.max(np.abs(M.T @ (M @ x - v))) < 1e-10 * np.linalg.norm(v) * np.linalg.norm(M, 2)
    Q, _ = np.linalg.qr(R.T, mode="complete")
    null = Q[:, k:]                                                               # R null = 0
    assert np.max(np.abs(R @ null)) < 1e-12 and np.max(np.abs(null.T @ x)) < 1e-10 * np.linalg.norm(x)


def test_push_is_axpy(orc):
    pos = np.array([[1.0, 2.0], [3.0, 4.0], [5.0, 6.0]])
    E = np.array([[1e3, 0.0], [0.0, -2e3], [4e3, 0.0]])
    out = orc.push(pos, E, mu=1.5e-4, dt=1e-9)
    assert out[0, 0] == 1.0 + 1.5e-4 * 1e3 * 1e-9 and out[1, 1] == 4.0 - 1.5e-4 * 2e3 * 1e-9 and out[2, 1] == 6.0


# ---------------------------------------------------------------------------------------------
# FastVolume and weighting field: pins for the oracle's interpolation
# ---------------------------------------------------------------------------------------------
def test_fastvol_trilinear_reproduces_products_of_linear_functions(orc):
    """Trilinear interpolation is exact for every function that is linear in each coordinate separately
    (1, x, y, z, xy, yz, zx, xyz); it returns the node values at the nodes; outside the box it gives NaN."""
    nx, ny, nz = 5, 4, 3
    o, h = np.array([0.1, -0.2, 0.3]), np.array([0.5, 0.25, 1.0])
    P = orc.fastvol_nodes(nx, ny, nz, o, h)
    assert P.shape == (3, 60) and np.allclose(P[:, 1] - P[:, 0], [h[0], 0, 0]) and np.allclose(P[:, nx] - P[:, 0], [0, h[1], 0])
    f = lambda x, y, z: (1 + 2 * x) * (3 - y) * (0.5 + z)
    vals = np.stack([f(*P), P[0] - P[2], P[1] * P[2], P[0] * P[1] * P[2]])
    rs = np.random.RandomState(0)
    pts = o[:, None] + rs.rand(3, 500) * (h * np.array([nx - 1, ny - 1, nz - 1]))[:, None]
    phi, E = orc.fastvol_eval((nx, ny, nz), o, h, vals, pts)
    assert np.max(np.abs(phi - f(*pts))) < 1e-13 * np.max(np.abs(vals[0]))
    assert np.max(np.abs(E[0] - (pts[0] - pts[2]))) < 1e-14 and np.max(np.abs(E[2] - pts[0] * pts[1] * pts[2])) < 1e-14
    phi_n, E_n = orc.fastvol_eval((nx, ny, nz), o, h, vals, P)                  # at the nodes, upper faces included
    assert np.max(np.abs(phi_n - vals[0])) < 1e-13 and np.max(np.abs(E_n - vals[1:])) < 1e-14
    out = np.array([[o[0] - 1e-6, o[0] + 0.1], [o[1] + 0.1, o[1] + 0.1], [o[2] + 0.1, o[2] + (nz - 1) * h[2] + 1e-6]])
    phi_o, E_o = orc.fastvol_eval((nx, ny, nz), o, h, vals, out)
    assert np.all(np.isnan(phi_o)) and np.all(np.isnan(E_o))


def test_fastvol_matches_scipy_regular_grid_interpolator(orc):
    from scipy.interpolate import RegularGridInterpolator
    nx, ny, nz = 7, 6, 5
    o, h = np.array([-1.0, 0.0, 2.0]), np.array([0.3, 0.7, 0.45])
    rs = np.random.RandomState(5)
    vals = rs.normal(size=(4, nx * ny * nz))
    pts = o[:, None] + rs.rand(3, 400) * (h * np.array([nx - 1, ny - 1, nz - 1]))[:, None]
    phi, E = orc.fastvol_eval((nx, ny, nz), o, h, vals, pts)
    axes = (o[2] + h[2] * np.arange(nz), o[1] + h[1] * np.arange(ny), o[0] + h[0] * np.arange(nx))
    for c, got in enumerate([phi, E[0], E[1], E[2]]):
        ref = RegularGridInterpolator(axes, vals[c].reshape(nz, ny, nx), method="linear")(pts[::-1].T)
        assert np.max(np.abs(got - ref)) < 1e-12


def test_fastvol_error_is_second_order_against_direct_evaluation(orc):
    """A FastVolume of a charged plate's field: the interpolation error against direct evaluation falls by ~4
    per halving of the grid spacing (the paper reports < 0.25 % for its map)."""
    pr = W.plate(n_side=4, m_points=0)
    g = orc.Geometry(pr)
    sig = np.full(pr.n, 1e-8)
    o = np.array([-4e-3, -4e-3, 2e-3])
    rs = np.random.RandomState(2)
    pts = o[:, None] + rs.rand(3, 200) * 8e-3
    phi_d, E_d = orc.evaluate(g, sig, pts, mode="f64")
    errs = []
    for n in (5, 9, 17):
        h = np.full(3, 8e-3 / (n - 1))
        P = orc.fastvol_nodes(n, n, n, o, h)
        ph, Ev = orc.evaluate(g, sig, P, mode="f64")
        phi_i, E_i = orc.fastvol_eval((n, n, n), o, h, np.vstack([ph[None], Ev]), pts, mode="f64")
        errs.append(np.max(np.abs(phi_i - phi_d)) / np.max(np.abs(phi_d)))
    assert errs[0] > 3.0 * errs[1] > 9.0 * errs[2] and errs[2] < 2.5e-3


def test_weighting_rhs_and_superposition(orc):
    """Weighting potentials of all conductors add up to the potential of the whole system at 1 V (linearity of
    Eq. 6): on the cube split into two read-out groups, sigma_w1 + sigma_w2 = sigma(all at 1 V)."""
    pr = W.cube(n_side=4, m_points=0)
    g = orc.Geometry(pr)
    K = orc.assemble(g, mode="f64")
    grp = (np.arange(pr.n) < pr.n // 2).astype(float)
    b1, b2 = orc.weighting_rhs(g, grp), orc.weighting_rhs(g, 1.0 - grp)
    assert np.array_equal(b1 + b2, np.ones(pr.n))
    s1, s2 = orc.solve(K, b1, mode="f64"), orc.solve(K, b2, mode="f64")
    s = orc.solve(K, orc.rhs(g, mode="f64"), mode="f64")
    assert np.max(np.abs(s1 + s2 - s)) < 1e-12 * np.max(np.abs(s))
    mixed = W.thgem(d=10, n_plane=6, n_grid=2)
    bw = orc.weighting_rhs(orc.Geometry(mixed), np.ones(mixed.n))
    assert np.all(bw[mixed.bc_kind == W.DIELECTRIC] == 0.0) and np.all(bw[mixed.bc_kind == W.DIRICHLET] == 1.0)


# ---------------------------------------------------------------------------------------------
# Alg. 3: voxelisation of point charges into line charges
# ---------------------------------------------------------------------------------------------
def test_line_charge_against_quadrature_and_limits(orc):
    """The closed form of a line charge against Gauss-Legendre quadrature of Eq. (2) P:68 along the line, against
    the (already pinned) thin-wire routine outside its radius, E = -grad Phi, and the point-charge limit."""
    lines = np.array([[0.3e-3], [-0.2e-3], [0.1e-3], [0.5e-3], [2.0e-9]])        # x, y, z1, z2, lambda
    rs = np.random.RandomState(3)
    pts = rs.normal(size=(3, 12)) * 1e-3
    phi, E = orc.line_charges(pts, lines)
    xg, wg = np.polynomial.legendre.leggauss(200)
    zc, hl = 0.5 * (lines[2, 0] + lines[3, 0]), 0.5 * (lines[3, 0] - lines[2, 0])
    for p in range(pts.shape[1]):
        zq = zc + hl * xg
        d = np.stack([np.full_like(zq, pts[0, p] - lines[0, 0]), np.full_like(zq, pts[1, p] - lines[1, 0]), pts[2, p] - zq])
        r = np.linalg.norm(d, axis=0)
        if r.min() < 5e-5:
            continue                                                              # quadrature needs distance
        phi_q = orc.K_COULOMB * lines[4, 0] * hl * np.sum(wg / r)
        E_q = orc.K_COULOMB * lines[4, 0] * hl * np.sum(wg * d / r ** 3, axis=1)
        assert abs(phi[p] - phi_q) < 1e-11 * abs(phi_q) and np.max(np.abs(E[:, p] - E_q)) < 1e-10 * np.linalg.norm(E_q)
    # the pinned wire formula (surface density sigma on radius r_w: lambda = 2 pi r_w sigma) outside the radius
    rw = 1e-6
    inf = np.array([orc.influence(W.WIRE, [lines[0, 0], lines[1, 0], lines[2, 0]], [0, 0, 2 * hl], [1, 0, 0], pts[:, p], radius=rw)
                    for p in range(pts.shape[1])])
    sig = lines[4, 0] / (2 * np.pi * rw)
    assert np.max(np.abs(orc.K_COULOMB * sig * inf[:, 0] - phi)) < 1e-12 * np.max(np.abs(phi))
    assert np.max(np.abs(orc.K_COULOMB * sig * inf[:, 1:].T - E)) < 1e-12 * np.max(np.abs(E))
    h = 1e-8
    for k in range(3):
        dp = np.zeros((3, 1)); dp[k] = h
        g = (orc.line_charges(pts + dp, lines)[0] - orc.line_charges(pts - dp, lines)[0]) / (2 * h)
        assert np.max(np.abs(E[k] + g)) < 1e-6 * np.max(np.abs(E))
    far = np.array([[0.2], [0.1], [-0.3]])
    phi_f, _ = orc.line_charges(far, lines)
    q = lines[4, 0] * 2 * hl
    assert abs(phi_f[0] - orc.K_COULOMB * q / np.linalg.norm(far[:, 0] - [lines[0, 0], lines[1, 0], zc])) < 1e-5 * abs(phi_f[0])
    on_axis = np.array([[lines[0, 0]], [lines[1, 0]], [1e-3]])                    # rho = 0: skipped
    assert orc.line_charges(on_axis, lines)[0][0] == 0.0


def test_voxelize_against_brute_force_histogram(orc):
    rs = np.random.RandomState(8)
    q = 5000
    pos = rs.normal(size=(3, q)) * 1.2e-4
    ch = rs.choice([1.0, -1.0, 2.0], size=q) * W.Q_E
    o, d, dims = np.array([-3e-4, -2e-4, -2.5e-4]), np.array([1e-4, 0.8e-4, 0.5e-4]), np.array([6, 5, 10])
    lines = orc.voxelize(pos, ch, o, d, dims)
    idx = np.stack([np.clip(np.floor((pos[a] - o[a]) / d[a]).astype(int), 0, dims[a] - 1) for a in range(3)])
    flat = (idx[2] * dims[1] + idx[1]) * dims[0] + idx[0]
    tot = np.zeros(dims.prod()); np.add.at(tot, flat, ch)
    occ = np.zeros(dims.prod(), dtype=bool); occ[flat] = True
    v = np.nonzero(occ)[0]
    assert lines.shape == (5, v.size) and v.size < q                              # N_voxels << N_points
    assert np.allclose(lines[4] * d[2], tot[v], rtol=1e-12, atol=1e-30)
    assert abs(np.sum(lines[4]) * d[2] - ch.sum()) < 1e-12 * np.abs(ch).sum()      # total charge conserved (clamped points too)
    i, j, k = v % dims[0], (v // dims[0]) % dims[1], v // (dims[0] * dims[1])
    assert np.allclose(lines[0], o[0] + (i + 0.5) * d[0], rtol=0, atol=1e-18) and np.allclose(lines[1], o[1] + (j + 0.5) * d[1], rtol=0, atol=1e-18)
    assert np.allclose(lines[2], o[2] + k * d[2], rtol=0, atol=1e-18) and np.allclose(lines[3] - lines[2], d[2], rtol=1e-12)
    assert np.any(idx[0] == 0) and (np.floor((pos[0] - o[0]) / d[0]) < 0).any()    # some points were clamped
    # far from the cloud the lines reproduce the points' field (monopole exactly, dipole up to voxel size / distance)
    pts = np.array([[3e-3, 6e-3], [1e-3, 2e-3], [-2e-3, -4e-3]])
    same = np.full(q, W.Q_E)
    l2 = orc.voxelize(pos, same, o, d, dims)
    p_pt, _ = orc.point_charges(pts, pos, same)
    p_ln, _ = orc.line_charges(pts, l2)
    err = np.abs(p_ln - p_pt) / np.abs(p_pt)
    assert np.all(err < 1e-3)


# ---------------------------------------------------------------------------------------------
# Adaptive Modelling (Table 2): far image copies as point charges
# ---------------------------------------------------------------------------------------------
def test_adaptive_modelling_limits_and_error_order(orc):
    """far_distance <= 0 or beyond every shift = the exact sum; with every shifted copy simplified the result equals
    the exact unshifted elements plus explicit point charges sigma A at the shifted centroids (written out here with
    numpy); the error against the exact sum falls as (element size / pitch)^2."""
    pr = W.random_elements(9, seed=4, kinds=(RECT, TRI, W.WIRE), size_mm=(0.02, 0.05), box_mm=0.2, m_points=40)
    sig = np.linspace(0.5, 1.5, pr.n) * 1e-6
    errs = []
    for pitch in (1.0, 2.0):
        pr.img_shift = W.image_shifts(1, pitch_mm=pitch)
        g = orc.Geometry(pr)
        phi_x, E_x = orc.evaluate(g, sig, pr.points)
        for fd in (0.0, -1.0, 10.0):
            phi0, E0 = orc.evaluate_adaptive(g, sig, pr.points, fd)
            assert np.array_equal(phi0, phi_x) and np.array_equal(E0, E_x)
        phi_a, E_a = orc.evaluate_adaptive(g, sig, pr.points, 0.5 * pitch * 1e-3)
        # by hand: unshifted elements exactly + monopoles of the 8 shifted copies
        g0 = orc.Geometry(pr); g0.img, g0.n_img = None, 0
        phi_h, E_h = orc.evaluate(g0, sig, pr.points)
        area = np.where(pr.kind == W.WIRE, 2 * np.pi * pr.radius * np.linalg.norm(pr.e1, axis=0),
                        np.linalg.norm(np.cross(pr.e1.T, pr.e2.T), axis=1) * np.where(pr.kind == RECT, 1.0, 0.5))
        cen = np.where(pr.kind == W.WIRE, pr.v0 + pr.e1 / 2, pr.v0 + (pr.e1 + pr.e2) * np.where(pr.kind == RECT, 0.5, 1 / 3))
        for s in range(pr.img_shift.shape[1]):
            sh = pr.img_shift[:, s]
            if np.linalg.norm(sh) == 0:
                continue
            d = pr.points[:, None, :] - (cen + sh[:, None])[:, :, None]            # (3, n, m)
            r = np.linalg.norm(d, axis=0)
            phi_h = phi_h + orc.K_COULOMB * np.sum((sig * area)[:, None] / r, axis=0)
            E_h = E_h + orc.K_COULOMB * np.sum((sig * area)[None, :, None] * d / r ** 3, axis=1)
        assert np.max(np.abs(phi_a - phi_h)) < 1e-12 * np.max(np.abs(phi_h)) and np.max(np.abs(E_a - E_h)) < 1e-12 * np.max(np.abs(E_h))
        errs.append(np.max(np.abs(phi_a - phi_x)) / np.max(np.abs(phi_x)))
    assert 0 < errs[1] < 0.35 * errs[0] and errs[0] < 1e-3        # (L / pitch)^2: a factor 4 per doubling (with the 1/r of the copy, 8)
