// neb_influence.cuh — a2: exact potential and field of a uniformly charged flat rectangle, right
// triangle or thin wire at one point (integrals P:121, P:125 with reading S2,
// P:131), evaluated in the element's local frame (element in the local XZ plane, Y = normal)
// and rotated to global.  The paper does not print the closed forms; the ones used here are
// derived in DESIGN.md §3 (edge form: one logarithm per edge, one arctangent per element) and are
// branch-free: every case distinction (near/far field, foot of the perpendicular inside/outside an
// edge, on-surface and on-edge limits) is a select, so that a warp never diverges — the reason
// the paper gives for keeping this stage off the GPU does not apply.
#pragma once
#include "neb_math.cuh"

namespace neb {

// Frame-table record (a1), 20 doubles per element, stored SoA in global memory (field-major):
//   0..2  v0      corner / right-angle vertex / wire start
//   3..5  ex      unit vector along e1 (local X)
//   6..8  ey      unit normal e2 x e1 / |e2 x e1| (local Y)        [wire: unused]
//   9..11 ez      unit vector along e2 (local Z)                    [wire: unused]
//   12    a       |e1|
//   13    b       |e2|                                              [wire: radius r_w]
//   14    aux     rectangle: a b; triangle: 1/hypotenuse; wire: 2 pi r_w
//   15    w       weight: sigma_j / (4 pi eps0) for evaluation (set by neb_solve / neb_set_sigma)
//   16    far2    (2.5 Lmax + diag)^2, Lmax = longest edge, diag = sqrt(a^2+b^2): a point at least that far
//                 (squared) from v0 is >= 2.5 Lmax away from every point of the element      [wire: unused]
//   17..19 c      (v0 . ex, v0 . ey, v0 . ez): the element's origin in its own axes.  With them the local coordinates of
//                 a point are (P . ex, P . ey, P . ez) - c, and the products P . e are shared by every element that has
//                 the same axes (a whole face of a mesh): the uniform-tile path of neb_field.cu   [wire: unused]
#define NEB_REC 20

struct Infl {
  double phi, ex, ey, ez;   // primed potential and GLOBAL primed field components
};

// ln[(R+ + l+)/(R- + l-)] of one straight edge: lm < lp are the abscissae of its ends along the
// edge measured from the foot of the perpendicular from P, Rm/Rp the distances to its ends, R0sq the
// squared distance from P to the edge's line, L = lp - lm.  Three algebraically equal forms chosen by
// the position of the foot so that nothing cancels; far away (Rm+Rp > 8L) 2 atanh(L/(Rm+Rp)) keeps
// full RELATIVE accuracy of the small value (the far-field sums cancel by a factor r/L).
// om >= 0 with the sign of Y, and 0 when Y == 0 (integer operations only)
__device__ __forceinline__ double signed_or_zero(double om, double Y) {
  const int hy = __double2hiint(Y), ly = __double2loint(Y);
  const bool zero = (((hy & 0x7fffffff) | ly) == 0);
  const int ho = (__double2hiint(om) & 0x7fffffff) | (hy & 0x80000000);
  return zero ? 0.0 : __hiloint2double(ho, __double2loint(om));
}

template <class M>
__device__ __forceinline__ double edge_log(double lm, double lp, double Rm, double Rp, double R0sq, double L) {
  double s = Rm + Rp;
  double pp = Rp + fabs(lp), qq = Rm + fabs(lm);
  // sign tests on the high word (integer pipe); a zero abscissa may fall in either case, all three forms agree there
  bool cA = __double2hiint(lm) >= 0, cB = __double2hiint(lp) < 0;
  double N = cB ? qq : pp;
  N = (cA || cB) ? N : pp * qq;
  double D = cA ? qq : (cB ? pp : R0sq);
  return M::log_ratio(N, D, M::kNeedsFar && s > 8.0 * L, L, s);
}

// Rectangle [0,a] x [0,b] in the local XZ plane; (X, Y, Z) local coordinates of P.
// out: phi', local field (fx, fy, fz).
// Far field, decided per WARP (one vote, no divergence): when every lane's point is at least 2.5 Lmax away from
// the element, every edge has R- + R+ >= 5 L and the solid angle is < 0.16 sr, so the case selections of edge_log
// and the argument reduction of the arctangent are dead code; the far branch evaluates the SAME closed form
// (2 atanh(L/s) per edge, one arctangent) without them.  ~99 % of the pairs of a field map take it.
// r0sq = squared distance from the point to v0 (already needed for the corner radius).
template <class M>
__device__ __forceinline__ bool warp_is_far(double r0sq, double far2) {
  if (!M::kFarPath) return false;
  return __all_sync(0xffffffffu, r0sq >= far2);
}

// Solid angle of the rectangle [x1,x2] x [z1,z2] (u_i = x_i - X, w_j = z_j - Z, A_i = u_i^2 + y^2, B_j = w_j^2 + y^2,
// r_ij the corner distances, Nn = area x |Y|): two fan triangles (c11,c21,c22), (c11,c22,c12);
// tan(Omega_t/2) = 2A_t |d| / D_t with the triple product written as area x height (exact for a flat element: no
// far-field cancellation); products folded into the sums that use them: 14 FP64-pipe operations for D1, D2.
template <class M>
__device__ __forceinline__ double rect_omega(double u1, double u2, double w1, double w2, double yy, double A1, double A2, double B1,
                                             double B2, double r11, double r12, double r21, double r22, double Nn, bool far) {
  double d1122 = fma(u1, u2, fma(w1, w2, yy));               // r11 . r22 = r12 . r21
  double pB1 = fma(u1, u2, B1), pB2 = fma(u1, u2, B2);       // r11 . r21, r12 . r22
  double A2q = fma(w1, w2, A2), A1q = fma(w1, w2, A1);       // r21 . r22, r11 . r12
  double D1 = fma(fma(r11, r21, pB1), r22, fma(d1122, r21, A2q * r11));
  double D2 = fma(fma(r11, r22, d1122), r12, fma(A1q, r22, pB2 * r11));
  if (far) return 2.0 * M::far_atan2(Nn * (D1 + D2), fma(D1, D2, -Nn * Nn));
  return 2.0 * M::atan2_pos(Nn * (D1 + D2), fma(D1, D2, -Nn * Nn));
}

template <class M>
__device__ __forceinline__ void rect_local(double a, double b, double ab, double far2, double X, double Y, double Z, double& phi,
                                           double& fx, double& fy, double& fz) {
  double u1 = -X, u2 = a - X, w1 = -Z, w2 = b - Z, y = fabs(Y);
  double yy = y * y;
  double A1 = fma(u1, u1, yy), A2 = fma(u2, u2, yy);      // squared distances to the lines x = x_i
  double B1 = fma(w1, w1, yy), B2 = fma(w2, w2, yy);      // squared distances to the lines z = z_j
  double q11 = fma(w1, w1, A1);
  const bool far = warp_is_far<M>(q11, far2);
  double r11 = M::sqrt_nn(q11), r12 = M::sqrt_nn(fma(w2, w2, A1));
  double r21 = M::sqrt_nn(fma(w1, w1, A2)), r22 = M::sqrt_nn(fma(w2, w2, A2));
  double F1, F2, G1, G2, om;
  if (far) {
    F1 = M::far_log(b, r11 + r12);
    F2 = M::far_log(b, r21 + r22);
    G1 = M::far_log(a, r11 + r21);
    G2 = M::far_log(a, r12 + r22);
  } else {
    F1 = edge_log<M>(w1, w2, r11, r12, A1, b);            // edge x = 0
    F2 = edge_log<M>(w1, w2, r21, r22, A2, b);            // edge x = a
    G1 = edge_log<M>(u1, u2, r11, r21, B1, a);            // edge z = 0
    G2 = edge_log<M>(u1, u2, r12, r22, B2, a);            // edge z = b
  }
  om = rect_omega<M>(u1, u2, w1, w2, yy, A1, A2, B1, B2, r11, r12, r21, r22, ab * y, far);
  phi = fma(u2, F2, fma(-u1, F1, fma(w2, G2, fma(-w1, G1, -y * om))));
  fx = F2 - F1;
  fz = G2 - G1;
  fy = signed_or_zero(om, Y);                             // S5: principal value on the surface
}

// Two rectangles that share an edge — [0,a1] x [0,b] and [a1,a1+a2] x [0,b] in the FIRST one's local frame — at one
// point: the three corner-pair columns x = 0, a1, a1+a2 give 6 corner distances and 3 edge logarithms along z instead
// of 8 and 4 (the shared edge's logarithm enters both potentials with opposite outward normals): 34 of 2 x 143 FP64
// operations less.  Meshes are made of such strips (a discretised primitive is a grid of equal rectangles); which
// neighbours form a pair is decided once per table (tile_uniform_kernel), so the choice is uniform over the CTA.
template <class M>
__device__ __forceinline__ void rect_pair_local(double a1, double a2, double b, double ab1, double ab2, double far2a, double far2b,
                                                double X, double Y, double Z, double& p1, double& fx1, double& fy1, double& fz1,
                                                double& p2, double& fx2, double& fy2, double& fz2) {
  double u1 = -X, u2 = a1 - X, u3 = u2 + a2, w1 = -Z, w2 = b - Z, y = fabs(Y);
  double yy = y * y;
  double A1 = fma(u1, u1, yy), A2 = fma(u2, u2, yy), A3 = fma(u3, u3, yy);
  double B1 = fma(w1, w1, yy), B2 = fma(w2, w2, yy);
  double q11 = fma(w1, w1, A1), q21 = fma(w1, w1, A2);
  bool far = false;
  if (M::kFarPath) far = __all_sync(0xffffffffu, q11 >= far2a && q21 >= far2b);
  double r11 = M::sqrt_nn(q11), r12 = M::sqrt_nn(fma(w2, w2, A1));
  double r21 = M::sqrt_nn(q21), r22 = M::sqrt_nn(fma(w2, w2, A2));
  double r31 = M::sqrt_nn(fma(w1, w1, A3)), r32 = M::sqrt_nn(fma(w2, w2, A3));
  double F1, F2, F3, G1a, G2a, G1b, G2b;
  if (far) {
    F1 = M::far_log(b, r11 + r12);
    F2 = M::far_log(b, r21 + r22);
    F3 = M::far_log(b, r31 + r32);
    G1a = M::far_log(a1, r11 + r21);
    G2a = M::far_log(a1, r12 + r22);
    G1b = M::far_log(a2, r21 + r31);
    G2b = M::far_log(a2, r22 + r32);
  } else {
    F1 = edge_log<M>(w1, w2, r11, r12, A1, b);
    F2 = edge_log<M>(w1, w2, r21, r22, A2, b);
    F3 = edge_log<M>(w1, w2, r31, r32, A3, b);
    G1a = edge_log<M>(u1, u2, r11, r21, B1, a1);
    G2a = edge_log<M>(u1, u2, r12, r22, B2, a1);
    G1b = edge_log<M>(u2, u3, r21, r31, B1, a2);
    G2b = edge_log<M>(u2, u3, r22, r32, B2, a2);
  }
  const double om1 = rect_omega<M>(u1, u2, w1, w2, yy, A1, A2, B1, B2, r11, r12, r21, r22, ab1 * y, far);
  const double om2 = rect_omega<M>(u2, u3, w1, w2, yy, A2, A3, B1, B2, r21, r22, r31, r32, ab2 * y, far);
  p1 = fma(u2, F2, fma(-u1, F1, fma(w2, G2a, fma(-w1, G1a, -y * om1))));
  p2 = fma(u3, F3, fma(-u2, F2, fma(w2, G2b, fma(-w1, G1b, -y * om2))));
  fx1 = F2 - F1; fx2 = F3 - F2;
  fz1 = G2a - G1a; fz2 = G2b - G1b;
  fy1 = signed_or_zero(om1, Y); fy2 = signed_or_zero(om2, Y);
}

// Right triangle (0,0), (a,0), (0,b) in the local XZ plane, ih = 1/sqrt(a^2+b^2).
template <class M>
__device__ __forceinline__ void tri_local(double a, double b, double ih, double far2, double X, double Y, double Z,
                                          double& phi, double& fx, double& fy, double& fz) {
  double uA = -X, uB = a - X, wA = -Z, wC = b - Z, y = fabs(Y);
  double yy = y * y;
  double A0 = fma(uA, uA, yy), W0 = fma(wA, wA, yy);
  double qA = fma(wA, wA, A0);
  const bool far = warp_is_far<M>(qA, far2);
  double RA = M::sqrt_nn(qA), RB = M::sqrt_nn(fma(uB, uB, W0)), RC = M::sqrt_nn(fma(wC, wC, A0));
  double ca = a * ih, cb = b * ih;                        // hypotenuse B->C: t = (-ca, cb), m = (cb, ca)
  double h = (a * a + b * b) * ih;
  double P0 = fma(cb, uB, ca * wA);
  double fAB, fCA, fBC;
  if (far) {
    fAB = M::far_log(a, RA + RB);
    fCA = M::far_log(b, RA + RC);
    fBC = M::far_log(h, RB + RC);
  } else {
    fAB = edge_log<M>(uA, uB, RA, RB, W0, a);             // leg on the X axis, outward normal -Z, P0 = Z
    fCA = edge_log<M>(wA, wC, RA, RC, A0, b);             // leg on the Z axis, outward normal -X, P0 = X
    double lm = fma(-ca, uB, cb * wA);
    double lp = lm + h;
    fBC = edge_log<M>(lm, lp, RB, RC, fma(P0, P0, yy), h);
  }
  double dAB = fma(uA, uB, W0), dAC = fma(wA, wC, A0), dBC = fma(uA, uB, fma(wA, wC, yy));
  double D = fma(RA * RB, RC, fma(dAB, RC, fma(dAC, RB, dBC * RA)));
  double om = 2.0 * (far ? M::far_atan2(a * b * y, D) : M::atan2_pos(a * b * y, D));
  phi = fma(Z, fAB, fma(X, fCA, fma(P0, fBC, -y * om)));
  fx = fma(cb, fBC, -fCA);
  fz = fma(ca, fBC, -fAB);
  fy = signed_or_zero(om, Y);
}

// Element record fields of one rect/tri element, as scalars (read from shared memory by the caller).
struct Frame {
  double v0x, v0y, v0z, exx, exy, exz, eyx, eyy, eyz, ezx, ezy, ezz, a, b, aux, far2;
};

// Unit axes of a frame (rows of the local <- global rotation).
struct Axes {
  double exx, exy, exz, eyx, eyy, eyz, ezx, ezy, ezz;
};

// Rectangle or right triangle at local coordinates (X, Y, Z): phi' and the LOCAL field components.
template <class M, int KIND>
__device__ __forceinline__ void local_pair(double a, double b, double aux, double far2, double X, double Y, double Z,
                                           double& phi, double& lx, double& ly, double& lz) {
  if (KIND == 0) rect_local<M>(a, b, aux, far2, X, Y, Z, phi, lx, ly, lz);
  else tri_local<M>(a, b, aux, far2, X, Y, Z, phi, lx, ly, lz);
}

template <class M, int KIND>
__device__ __forceinline__ Infl influence(const Frame& f, double px, double py, double pz) {
  double dx = px - f.v0x, dy = py - f.v0y, dz = pz - f.v0z;
  Infl o;
  if (KIND == 2) {
    // thin wire on the local X axis from 0 to a (reading S24); line density = 2 pi r_w sigma (aux)
    double t = fma(dx, f.exx, fma(dy, f.exy, dz * f.exz));
    double qx = fma(-t, f.exx, dx), qy = fma(-t, f.exy, dy), qz = fma(-t, f.exz, dz);
    double rho2 = fma(qx, qx, fma(qy, qy, qz * qz));
    double rw = f.b;
    bool inside = rho2 < rw * rw;
    double rho2c = inside ? rw * rw : rho2;
    double lm = -t, lp = f.a - t;
    double Rm = M::sqrt_nn(fma(lm, lm, rho2c)), Rp = M::sqrt_nn(fma(lp, lp, rho2c));
    double ph = edge_log<M>(lm, lp, Rm, Rp, rho2c, f.a);
    double iRm = M::div_pos(1.0, fmax(Rm, NEB_TINY)), iRp = M::div_pos(1.0, fmax(Rp, NEB_TINY));
    double er = M::div_pos(fma(lp, iRp, -lm * iRm), fmax(rho2c, NEB_TINY));   // E'_rho / rho
    double ea = iRp - iRm;
    double sc = inside ? 0.0 : f.aux;
    o.phi = f.aux * ph;
    o.ex = sc * fma(er, qx, ea * f.exx);
    o.ey = sc * fma(er, qy, ea * f.exy);
    o.ez = sc * fma(er, qz, ea * f.exz);
    return o;
  }
  double X = fma(dx, f.exx, fma(dy, f.exy, dz * f.exz));
  double Y = fma(dx, f.eyx, fma(dy, f.eyy, dz * f.eyz));
  double Z = fma(dx, f.ezx, fma(dy, f.ezy, dz * f.ezz));
  double lx, ly, lz;
  if (KIND == 0) rect_local<M>(f.a, f.b, f.aux, f.far2, X, Y, Z, o.phi, lx, ly, lz);
  else tri_local<M>(f.a, f.b, f.aux, f.far2, X, Y, Z, o.phi, lx, ly, lz);
  o.ex = fma(lx, f.exx, fma(ly, f.eyx, lz * f.ezx));
  o.ey = fma(lx, f.exy, fma(ly, f.eyy, lz * f.ezy));
  o.ez = fma(lx, f.exz, fma(ly, f.eyz, lz * f.ezz));
  return o;
}

}  // namespace neb
