"""Writes tests/golden/quadrature_pins.txt: brute-force quadrature of the paper's DEFINING integrals.

Calls neither oracle/ nor the CUDA path.  For a fixed list of element/point cases it integrates
    Phi' = iint dx dz / r            (P:121 rectangle, P:125 right triangle with reading S2)
    E'   = iint r_vec dx dz / r^3
with mpmath's adaptive Gauss-Legendre (30 digits, intervals split at the foot of the perpendicular),
and the thin-wire line integrals  int dz / r,  int r_vec dz / r^3  (reading S24).
Elements are given in their local frame: element in the XZ plane, normal +Y.

Run:  python tests/golden/make_quadrature_pins.py
"""
import os
import mpmath as mp

mp.mp.dps = 30

# kind, (a, b) = extents along local X and Z from the corner / right-angle vertex at the origin, point (X, Y, Z)
CASES = [
    ("rect", 1.3, 0.9, (0.87, 0.21, -0.15)),      # SURVEY pin: x in [-0.5,0.8], z in [-0.3,0.6], P=(0.37,0.21,-0.45), shifted
    ("rect", 1.3, 0.9, (2.4, -0.4, 0.4)),         # SURVEY pin 2 shifted: negative y, outside the projection
    ("rect", 1.0, 1.0, (0.5, 0.3, 0.5)),          # on the axis of a square
    ("rect", 2.0, 0.5, (-0.7, 0.05, 0.2)),        # low height, outside
    ("rect", 2.0, 0.5, (1.1, 0.02, 0.3)),         # low height, above the interior
    ("rect", 0.4, 1.7, (0.2, 0.0, 2.5)),          # in plane, on the extension of nothing, outside
    ("rect", 0.4, 1.7, (0.0, 0.0, 2.5)),          # in plane, on the extension line of an edge
    ("rect", 1.0, 0.6, (7.0, -5.0, 3.0)),         # far-ish
    ("rect", 1.0, 0.6, (-31.0, 14.0, -22.0)),     # far
    ("tri", 1.0, 0.7, (0.3, 0.25, 0.4)),          # SURVEY pin
    ("tri", 1.0, 0.7, (0.2, -0.15, 0.2)),         # below, inside the projection
    ("tri", 1.0, 0.7, (0.9, 0.1, 0.6)),           # beyond the hypotenuse
    ("tri", 0.5, 2.0, (-0.4, 0.3, -0.2)),         # behind the right-angle vertex
    ("tri", 0.5, 2.0, (1.5, 0.0, 0.7)),           # in plane, outside
    ("tri", 1.0, 1.0, (-12.0, 9.0, 20.0)),        # far
    ("tri", 2.0, 0.3, (1.0, 0.04, 0.1)),          # low height above a thin triangle
    ("wire", 1.0, 0.0, (0.2, 0.0, 0.85)),         # beside the first fifth of the wire, rho = 0.85
    ("wire", 1.0, 0.0, (0.85, 0.0, 0.2)),         # SURVEY 8(c) pin: h=0.5, rho=0.2, 0.35 from the centre ALONG the axis; wire on
                                                  # the local X axis here: X = 0.5+0.35, rho along Z.  Survey values: Phi' =
                                                  # 2.84677535102197, E'_rho (here E'z) = 7.86708584166788, E'_axis (E'x) = 2.85480333137226
    ("wire", 1.0, 0.0, (1.6, 0.3, 0.4)),          # beyond the end
    ("wire", 0.3, 0.0, (-4.0, 2.0, 1.0)),         # far
]


def integrals(kind, a, b, P):
    X, Y, Z = (mp.mpf(v) for v in P)
    a, b = mp.mpf(a), mp.mpf(b)

    def split(lo, hi, c):
        pts = [lo, hi]
        if lo < c < hi:
            pts = [lo, c, hi]
        return pts

    if kind == "wire":
        # wire on the local X axis from 0 to a; per unit line density.  P = (X, Y, Z): rho^2 = Y^2 + Z^2
        f = lambda g: mp.quad(g, split(0, a, X))
        r = lambda x: mp.sqrt((X - x) ** 2 + Y ** 2 + Z ** 2)
        return [f(lambda x: 1 / r(x)), f(lambda x: (X - x) / r(x) ** 3), f(lambda x: Y / r(x) ** 3),
                f(lambda x: Z / r(x) ** 3)]

    def zmax(x):
        return b if kind == "rect" else b * (1 - x / a)

    def inner(g, x):
        return mp.quad(lambda z: g(x, z), split(0, zmax(x), Z))

    def outer(g):
        return mp.quad(lambda x: inner(g, x), split(0, a, X))

    r = lambda x, z: mp.sqrt((X - x) ** 2 + Y ** 2 + (Z - z) ** 2)
    return [outer(lambda x, z: 1 / r(x, z)), outer(lambda x, z: (X - x) / r(x, z) ** 3),
            outer(lambda x, z: Y / r(x, z) ** 3), outer(lambda x, z: (Z - z) / r(x, z) ** 3)]


def main():
    out = os.path.join(os.path.dirname(os.path.abspath(__file__)), "quadrature_pins.txt")
    with open(out, "w") as fh:
        fh.write("# Brute-force quadrature of P:121 / P:125 (reading S2) / P:131 and the wire line integrals (S24).\n")
        fh.write("# Written by tests/golden/make_quadrature_pins.py (mpmath, 30 digits); no oracle or CUDA code involved.\n")
        fh.write("# Local frame: element in the XZ plane from the origin, extents a (X) and b (Z), normal +Y; wires lie on X.\n")
        fh.write("# kind a b X Y Z Phi' E'x E'y E'z\n")
        for kind, a, b, P in CASES:
            v = integrals(kind, a, b, P)
            fh.write(" ".join([kind, repr(a), repr(b)] + [repr(c) for c in P] + [mp.nstr(c, 20) for c in v]) + "\n")
            print(kind, a, b, P, [mp.nstr(c, 17) for c in v], flush=True)


if __name__ == "__main__":
    main()
