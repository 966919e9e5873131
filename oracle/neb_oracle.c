/* neb_oracle.c — TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * Plain, slow, CPU implementation of what the neBEM hot path computes, written from
 * /root/reference/PAPER.md (cited "P:line") with the readings S1..S24 of SURVEY.md §8(c) /
 * DESIGN.md §3.  It shares no code, header, table or constant with the CUDA path under
 * paper_2606_24154_b200/; only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
 * --impl reference legs may load it.
 *
 * Precision: every quantity is computed in `real`.  The default build has real = double (the
 * timed CPU baseline); -DORC_LONG_DOUBLE builds the same source with real = long double (x87
 * 80-bit), used as the truth in parity tests so that the oracle's own far-field cancellation
 * (grows as (r/L)^2 in the corner/edge forms) stays far below the 1e-10 tolerance.  Sums over
 * elements and charges are accumulated in long double in both builds (reading S17).
 *
 * Pins (tests/test_oracle_pins.py, none of them calls back into this file for its expected
 * value): brute-force Gauss-Legendre / mpmath quadrature of the defining integrals P:121, P:125,
 * P:131; far-field limit Eq.(2); E = -grad(Phi) P:75 by central differences; closed forms
 * (centre of a rectangle, axis of a square); additivity; Gauss's law on a closed cube; textbook
 * image charge over a dielectric half-space; slab capacitor; numpy.linalg.solve for the LU;
 * FastVolume interpolation: exact reproduction of products of linear functions, node values, and
 * scipy.interpolate.RegularGridInterpolator.
 * Parity unpinned: the paper's "<=1.67 % vs COMSOL" accuracy — geometry and COMSOL absent.
 *
 * Layout: all vectors are SoA, x[0..n) y[0..n) z[0..n).  SI units.  Physical values are
 * sigma/(4 pi eps0) times the primed quantities (reading S3).
 */
#include <math.h>
#include <float.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#ifdef ORC_LONG_DOUBLE
typedef long double real;
#define R_SQRT sqrtl
#define R_LOG logl
#define R_ATAN atanl
#define R_ATAN2 atan2l
#define R_FABS fabsl
#define R_ASINH asinhl
#define R_TINY 1.0e-4000L
#else
typedef double real;
#define R_SQRT sqrt
#define R_LOG log
#define R_ATAN atan
#define R_ATAN2 atan2
#define R_FABS fabs
#define R_ASINH asinh
#define R_TINY 1.0e-300
#endif

#define ORC_RECT 0
#define ORC_TRI 1
#define ORC_WIRE 2
#define ORC_DIRICHLET 0
#define ORC_DIELECTRIC 1

static const real EPS0 = 8.8541878128e-12L; /* F/m, reading S3 */
#define PI_L 3.14159265358979323846264338327950288L
#define K_COULOMB (1.0L / (4.0L * PI_L * EPS0))

int orc_real_bytes(void) { return (int)sizeof(real); }
int orc_threads(void) {
#ifdef _OPENMP
  return omp_get_max_threads();
#else
  return 1;
#endif
}

/* ------------------------------------------------------------------------------------------ */
/* a2. Influence of one element at one point: primed potential and field */
/* ------------------------------------------------------------------------------------------ */

/* ln[(l_plus + R_plus)/(l_minus + R_minus)] for a straight edge seen from a point whose squared
 * distance from the edge's line is R0sq; l_minus < l_plus are the signed abscissae of the edge's
 * ends along the edge, measured from the foot of the perpendicular.  Three algebraically equal
 * forms, chosen so that no two nearly equal numbers are subtracted (guard of the
 * 4-corner form: "when w<0 use ln(w+r) = ln((u^2+y^2)/(r-w))").  Reading S6: the denominator
 * is floored so that a point exactly on the edge gives a large finite value, never inf/NaN. */
static real edge_log(real lm, real lp, real Rm, real Rp, real R0sq) {
  real num, den;
  if (lm >= 0) { num = Rp + lp; den = Rm + lm; }
  else if (lp <= 0) { num = Rm - lm; den = Rp - lp; }
  else { num = (Rp + lp) * (Rm - lm); den = R0sq; }
  if (den < R_TINY) den = R_TINY;
  if (num < R_TINY) num = R_TINY;
  return R_LOG(num / den);
}

/* Rectangle in its local frame: element [0,a]x[0,b] in the XZ plane, Y normal.
 * 4-corner form of SURVEY §8(c), with the logs of one edge's two corners taken together:
 *   Phi' = sum_ij s_ij [ u_i ln(w_j+r_ij) + w_j ln(u_i+r_ij) - |y| atan2(u_i w_j, |y| r_ij) ]
 *   E'x  = sum_ij s_ij ln(w_j+r_ij),  E'z = sum_ij s_ij ln(u_i+r_ij),  E'y = sgn(y) sum_ij s_ij A_ij
 * u_i = x_i - X, w_j = z_j - Z, s_ij = +1 if i==j else -1. */
static void rect_local(real a, real b, real X, real Y, real Z, real out[4]) {
  real u[2] = {0 - X, a - X}, w[2] = {0 - Z, b - Z};
  real y = R_FABS(Y);
  real r[2][2];
  for (int i = 0; i < 2; ++i)
    for (int j = 0; j < 2; ++j) r[i][j] = R_SQRT(u[i] * u[i] + y * y + w[j] * w[j]);
  real phi = 0, ex = 0, ez = 0, om = 0;
  for (int i = 0; i < 2; ++i) { /* edges x = x_i, running in z: sum_j s_ij ln(w_j + r_ij) */
    real si = (i == 1) ? 1 : -1;
    real F = edge_log(w[0], w[1], r[i][0], r[i][1], u[i] * u[i] + y * y);
    ex += si * F;
    if (u[i] != 0) phi += si * u[i] * F; /* guard: u*ln(0) := 0 */
  }
  for (int j = 0; j < 2; ++j) { /* edges z = z_j, running in x */
    real sj = (j == 1) ? 1 : -1;
    real G = edge_log(u[0], u[1], r[0][j], r[1][j], w[j] * w[j] + y * y);
    ez += sj * G;
    if (w[j] != 0) phi += sj * w[j] * G;
  }
  if (y > 0) {
    for (int i = 0; i < 2; ++i)
      for (int j = 0; j < 2; ++j) om += ((i == j) ? 1 : -1) * R_ATAN2(u[i] * w[j], y * r[i][j]);
  }
  out[0] = phi - y * om;
  out[1] = ex;
  out[2] = (Y > 0) ? om : (Y < 0 ? -om : 0); /* reading S5: sgn(0) = 0, principal value on the surface */
  out[3] = ez;
}

/* Right triangle in its local frame (reading S2): vertices (0,0,0), (a,0,0), (0,0,b),
 * hypotenuse z = b(1 - x/a).  Edge form for a flat polygon (textbook potential integrals for
 * uniform sources on polygons), with the solid angle taken edge by edge:
 *   Phi' = sum_k [ P0_k f_k - |d| beta_k ],   E' = sum_k m_k f_k + sgn(d) (sum_k beta_k) n
 *   f_k    = ln[(R+ + l+)/(R- + l-)]
 *   beta_k = atan(P0 l+ / (R0^2 + |d| R+)) - atan(P0 l- / (R0^2 + |d| R-))
 * with, for edge k from v_k to v_k+1 (unit tangent t_k, in-plane outward normal m_k),
 * l-+ = (v_k,k+1 - P).t_k, P0 = (v_k - P).m_k, R0^2 = P0^2 + d^2, d = height of P above the plane. */
static void tri_local(real a, real b, real X, real Y, real Z, real out[4]) {
  /* counter-clockwise seen from +Y with (x,z) as the in-plane pair such that m = t x n points out:
   * order v0=(0,0), v1=(0,b), v2=(a,0) in (x,z)  ("triangle v0, v0+e2, v0+e1"). */
  real vx[3] = {0, 0, a}, vz[3] = {0, b, 0};
  real d = R_FABS(Y);
  real phi = 0, ex = 0, ez = 0, om = 0;
  for (int k = 0; k < 3; ++k) {
    int k1 = (k + 1) % 3;
    real Lx = vx[k1] - vx[k], Lz = vz[k1] - vz[k];
    real L = R_SQRT(Lx * Lx + Lz * Lz);
    real tx = Lx / L, tz = Lz / L;
    /* n = +Y; m = t x n: (tx,0,tz) x (0,1,0) = (-tz, 0, tx) */
    real mx = -tz, mz = tx;
    real rx0 = vx[k] - X, rz0 = vz[k] - Z, rx1 = vx[k1] - X, rz1 = vz[k1] - Z;
    real lm = rx0 * tx + rz0 * tz, lp = rx1 * tx + rz1 * tz;
    real P0 = rx0 * mx + rz0 * mz;
    real R0sq = P0 * P0 + d * d;
    real Rm = R_SQRT(rx0 * rx0 + rz0 * rz0 + d * d), Rp = R_SQRT(rx1 * rx1 + rz1 * rz1 + d * d);
    real f = edge_log(lm, lp, Rm, Rp, R0sq);
    ex += mx * f;
    ez += mz * f;
    if (P0 != 0) {
      phi += P0 * f;
      om += R_ATAN(P0 * lp / (R0sq + d * Rp)) - R_ATAN(P0 * lm / (R0sq + d * Rm));
    }
  }
  out[0] = phi - d * om;
  out[1] = ex;
  out[2] = (Y > 0) ? om : (Y < 0 ? -om : 0);
  out[3] = ez;
}

/* Thin wire (reading S24; named by BASELINE.json north_star, the paper has line charges only for
 * space charge): segment of half-length h on the local axis, rho = distance from the axis,
 *   Phi' = asinh((h-Z)/rho) + asinh((h+Z)/rho),  E'_rho = [(h-Z)/R1 + (h+Z)/R2]/rho,  E'_z = 1/R1 - 1/R2
 * per unit LINE density; the caller multiplies by 2 pi r_w to refer it to a surface density.
 * rho < r_w: rho := r_w in Phi' and E' := 0 (reading S24). out = Phi', E'_rho, E'_axis */
static void wire_local(real h, real rw, real rho, real Z, real out[3]) {
  int inside = rho < rw;
  if (inside) rho = rw;
  real R1 = R_SQRT(rho * rho + (h - Z) * (h - Z)), R2 = R_SQRT(rho * rho + (h + Z) * (h + Z));
  out[0] = R_ASINH((h - Z) / rho) + R_ASINH((h + Z) / rho);
  out[1] = inside ? 0 : ((h - Z) / R1 + (h + Z) / R2) / rho;
  out[2] = inside ? 0 : (1 / R1 - 1 / R2);
}

/* Global-frame wrapper: local frame (X,Y,Z) = (e1^, n, e2^) with n = e2 x e1 / |e2 x e1|,
 * evaluate, rotate E' back ("flux").  out4 = Phi', E'x, E'y, E'z (global, primed). */
static void influence(int kind, const real v0[3], const real e1[3], const real e2[3], real radius,
                      const real P[3], real out4[4]) {
  real a = R_SQRT(e1[0] * e1[0] + e1[1] * e1[1] + e1[2] * e1[2]);
  real ex[3] = {e1[0] / a, e1[1] / a, e1[2] / a};
  real dp[3] = {P[0] - v0[0], P[1] - v0[1], P[2] - v0[2]};
  if (kind == ORC_WIRE) {
    real h = a / 2;
    real zc = dp[0] * ex[0] + dp[1] * ex[1] + dp[2] * ex[2]; /* abscissa from the wire start */
    real pr[3] = {dp[0] - zc * ex[0], dp[1] - zc * ex[1], dp[2] - zc * ex[2]};
    real rho = R_SQRT(pr[0] * pr[0] + pr[1] * pr[1] + pr[2] * pr[2]);
    real o[3];
    wire_local(h, radius, rho, zc - h, o);
    real sc = 2 * PI_L * radius; /* lambda = 2 pi r_w sigma */
    out4[0] = sc * o[0];
    for (int c = 0; c < 3; ++c) {
      real er = (rho > 0) ? pr[c] / rho : 0;
      out4[1 + c] = sc * (o[1] * er + o[2] * ex[c]);
    }
    return;
  }
  real b = R_SQRT(e2[0] * e2[0] + e2[1] * e2[1] + e2[2] * e2[2]);
  real ez[3] = {e2[0] / b, e2[1] / b, e2[2] / b};
  real ey[3] = {ez[1] * ex[2] - ez[2] * ex[1], ez[2] * ex[0] - ez[0] * ex[2], ez[0] * ex[1] - ez[1] * ex[0]};
  real X = dp[0] * ex[0] + dp[1] * ex[1] + dp[2] * ex[2];
  real Y = dp[0] * ey[0] + dp[1] * ey[1] + dp[2] * ey[2];
  real Z = dp[0] * ez[0] + dp[1] * ez[1] + dp[2] * ez[2];
  real o[4];
  if (kind == ORC_RECT) rect_local(a, b, X, Y, Z, o);
  else tri_local(a, b, X, Y, Z, o);
  out4[0] = o[0];
  for (int c = 0; c < 3; ++c) out4[1 + c] = o[1] * ex[c] + o[2] * ey[c] + o[3] * ez[c];
}

typedef struct {
  int64_t n;
  const int32_t* kind;
  const double *v0, *e1, *e2, *radius;
} elems_t;

static void elem_influence(const elems_t* g, int64_t j, const real P[3], real out4[4]) {
  real v0[3] = {g->v0[j], g->v0[g->n + j], g->v0[2 * g->n + j]};
  real e1[3] = {g->e1[j], g->e1[g->n + j], g->e1[2 * g->n + j]};
  real e2[3] = {g->e2[j], g->e2[g->n + j], g->e2[2 * g->n + j]};
  influence(g->kind[j], v0, e1, e2, g->radius ? g->radius[j] : 0, P, out4);
}

/* One element, one point (double in/out): test entry for the pins. */
void orc_influence(int32_t kind, const double* v0, const double* e1, const double* e2, double radius,
                   const double* P, double* out4) {
  real a[3] = {v0[0], v0[1], v0[2]}, b[3] = {e1[0], e1[1], e1[2]}, c[3] = {e2[0], e2[1], e2[2]};
  real p[3] = {P[0], P[1], P[2]}, o[4];
  influence(kind, a, b, c, radius, p, o);
  for (int k = 0; k < 4; ++k) out4[k] = (double)o[k];
}

/* Sum over periodic copies (reading S12): the copy of element j shifted by +s seen from P equals
 * element j seen from P - s.  self_pv != 0 marks the pair (collocation point of element j, element j
 * itself): the unshifted copy then contributes NO field — the principal value of the normal field of
 * a flat element at a point of its own surface is zero (readings S5, S8: "self term 0 for a flat
 * element, but its image copies do contribute").  The rule is applied by index, not by testing Y == 0,
 * because the centroid of an obliquely oriented element is only in its plane up to rounding. */
static void elem_influence_images(const elems_t* g, int64_t j, const real P[3], int32_t n_img,
                                  const double* img, int self_pv, long double acc[4]) {
  for (int k = 0; k < 4; ++k) acc[k] = 0;
  int32_t copies = (n_img <= 0 || !img) ? 1 : n_img;
  for (int32_t s = 0; s < copies; ++s) {
    real sh[3] = {0, 0, 0};
    if (n_img > 0 && img) { sh[0] = (real)img[s]; sh[1] = (real)img[n_img + s]; sh[2] = (real)img[2 * n_img + s]; }
    real Ps[3] = {P[0] - sh[0], P[1] - sh[1], P[2] - sh[2]};
    real o[4];
    elem_influence(g, j, Ps, o);
    int unshifted = (sh[0] == 0 && sh[1] == 0 && sh[2] == 0);
    acc[0] += o[0];
    if (!(self_pv && unshifted))
      for (int k = 1; k < 4; ++k) acc[k] += o[k];
  }
}

static void unit_normal(const elems_t* g, int64_t i, real nrm[3]) {
  real e1[3] = {g->e1[i], g->e1[g->n + i], g->e1[2 * g->n + i]};
  real e2[3] = {g->e2[i], g->e2[g->n + i], g->e2[2 * g->n + i]};
  real c[3] = {e2[1] * e1[2] - e2[2] * e1[1], e2[2] * e1[0] - e2[0] * e1[2], e2[0] * e1[1] - e2[1] * e1[0]};
  real l = R_SQRT(c[0] * c[0] + c[1] * c[1] + c[2] * c[2]);
  nrm[0] = c[0] / l; nrm[1] = c[1] / l; nrm[2] = c[2] / l;
}

/* ------------------------------------------------------------------------------------------ */
/* a3. LHMatrix (Eq.(6)): one matrix entry                                       */
/*   Dirichlet row i  : K_ij = (1/4 pi eps0) sum_img Phi'_j(p_i)                     (Eq. 5)  */
/*   dielectric row i : K_ij = (1/4 pi eps0) sum_img n_i.E'_j(p_i) + delta_ij/(2 eps0 lambda_i) */
/*                      lambda = (eps+ - eps-)/(eps+ + eps-)                       (reading S8) */
/* ------------------------------------------------------------------------------------------ */
static real matrix_entry(const elems_t* g, const double* colloc, const int32_t* bc_kind,
                         const double* eps_plus, const double* eps_minus, int32_t n_img, const double* img,
                         int64_t i, int64_t j) {
  real P[3] = {colloc[i], colloc[g->n + i], colloc[2 * g->n + i]};
  long double acc[4];
  elem_influence_images(g, j, P, n_img, img, i == j, acc);
  if (bc_kind[i] == ORC_DIRICHLET) return (real)(K_COULOMB * acc[0]);
  real nrm[3];
  unit_normal(g, i, nrm);
  long double v = K_COULOMB * (nrm[0] * acc[1] + nrm[1] * acc[2] + nrm[2] * acc[3]);
  if (i == j) {
    long double lam = ((long double)eps_plus[i] - eps_minus[i]) / ((long double)eps_plus[i] + eps_minus[i]);
    v += 1.0L / (2.0L * EPS0 * lam);
  }
  return (real)v;
}

/* Full matrix, row-major K[i*n + j]. */
void orc_assemble(int64_t n, const int32_t* kind, const double* v0, const double* e1, const double* e2,
                  const double* radius, const double* colloc, const int32_t* bc_kind, const double* eps_plus,
                  const double* eps_minus, int32_t n_img, const double* img, double* K) {
  elems_t g = {n, kind, v0, e1, e2, radius};
#pragma omp parallel for schedule(dynamic, 4)
  for (int64_t i = 0; i < n; ++i)
    for (int64_t j = 0; j < n; ++j)
      K[i * n + j] = (double)matrix_entry(&g, colloc, bc_kind, eps_plus, eps_minus, n_img, img, i, j);
}

/* Sampled entries (rows[k], cols[k]) -> vals[k]. */
void orc_matrix_entries(int64_t n, const int32_t* kind, const double* v0, const double* e1, const double* e2,
                        const double* radius, const double* colloc, const int32_t* bc_kind,
                        const double* eps_plus, const double* eps_minus, int32_t n_img, const double* img,
                        int64_t n_s, const int64_t* rows, const int64_t* cols, double* vals) {
  elems_t g = {n, kind, v0, e1, e2, radius};
#pragma omp parallel for schedule(dynamic, 64)
  for (int64_t k = 0; k < n_s; ++k)
    vals[k] = (double)matrix_entry(&g, colloc, bc_kind, eps_plus, eps_minus, n_img, img, rows[k], cols[k]);
}

/* ------------------------------------------------------------------------------------------ */
/* a8. Known (space) charges: Eq.(2), Alg. 2; a pair with r = 0 is skipped (S11) */
/* ------------------------------------------------------------------------------------------ */
static void point_charge_sum(int64_t q, const double* pos, const double* charge, const real P[3],
                             long double acc[4]) {
  for (int k = 0; k < 4; ++k) acc[k] = 0;
  for (int64_t c = 0; c < q; ++c) {
    real dx = P[0] - (real)pos[c], dy = P[1] - (real)pos[q + c], dz = P[2] - (real)pos[2 * q + c];
    real r2 = dx * dx + dy * dy + dz * dz;
    if (r2 > 0) {
      real r = R_SQRT(r2);
      real qr = (real)charge[c] / r;
      real qr3 = qr / r2;
      acc[0] += qr;
      acc[1] += qr3 * dx;
      acc[2] += qr3 * dy;
      acc[3] += qr3 * dz;
    }
  }
  for (int k = 0; k < 4; ++k) acc[k] *= K_COULOMB;
}

/* Phi (m) and E (3*m SoA) of q point charges at m points. */
void orc_point_charges(int64_t m, const double* pts, int64_t q, const double* pos, const double* charge,
                       double* phi, double* E) {
#pragma omp parallel for schedule(dynamic, 16)
  for (int64_t p = 0; p < m; ++p) {
    real P[3] = {pts[p], pts[m + p], pts[2 * m + p]};
    long double acc[4];
    point_charge_sum(q, pos, charge, P, acc);
    if (phi) phi[p] = (double)acc[0];
    if (E) { E[p] = (double)acc[1]; E[m + p] = (double)acc[2]; E[2 * m + p] = (double)acc[3]; }
  }
}

/* ------------------------------------------------------------------------------------------ */
/* a4. RHVector + ValueKnCh (reading S10)                                        */
/*   Dirichlet: b_i = V_i - Phi_sc(p_i);  dielectric: b_i = -n_i.E_sc(p_i)                     */
/* ------------------------------------------------------------------------------------------ */
void orc_rhs(int64_t n, const double* e1, const double* e2, const double* colloc, const int32_t* bc_kind,
             const double* bc_value, int64_t q, const double* pos, const double* charge, double* b) {
  elems_t g = {n, NULL, NULL, e1, e2, NULL};
#pragma omp parallel for schedule(dynamic, 16)
  for (int64_t i = 0; i < n; ++i) {
    real P[3] = {colloc[i], colloc[n + i], colloc[2 * n + i]};
    long double acc[4] = {0, 0, 0, 0};
    if (q > 0) point_charge_sum(q, pos, charge, P, acc);
    if (bc_kind[i] == ORC_DIRICHLET) b[i] = (double)((long double)bc_value[i] - acc[0]);
    else {
      real nrm[3];
      unit_normal(&g, i, nrm);
      b[i] = (double)(-(nrm[0] * acc[1] + nrm[1] * acc[2] + nrm[2] * acc[3]));
    }
  }
}

/* ------------------------------------------------------------------------------------------ */
/* a5/a6. InvertMatrix (OptLU) + Solve (Alg. 1; readings S13, S15, S16):      */
/* rows scaled by 1/max_j|K_ij|, Gaussian elimination with partial (row) pivoting, first-max   */
/* tie-break, factors kept (no explicit inverse), forward and back substitution.               */
/* K is row-major n*n and is NOT modified; work is done in `real`.  Returns 0, or 4 if a pivot */
/* is zero/NaN.  orc_lu_factor / orc_lu_solve expose the two halves for re-solves (C4).        */
/* ------------------------------------------------------------------------------------------ */
typedef struct {
  int64_t n;
  real* lu;       /* row-major, rows already permuted */
  real* rscale;   /* row scale of the ORIGINAL row index */
  int64_t* perm;  /* perm[k] = original row now in position k */
} orc_lu_t;

orc_lu_t* orc_lu_factor(int64_t n, const double* K, int32_t* status) {
  orc_lu_t* f = (orc_lu_t*)calloc(1, sizeof(orc_lu_t));
  f->n = n;
  f->lu = (real*)malloc(sizeof(real) * (size_t)n * (size_t)n);
  f->rscale = (real*)malloc(sizeof(real) * (size_t)n);
  f->perm = (int64_t*)malloc(sizeof(int64_t) * (size_t)n);
  *status = 0;
#pragma omp parallel for
  for (int64_t i = 0; i < n; ++i) {
    real mx = 0;
    for (int64_t j = 0; j < n; ++j) { real v = R_FABS((real)K[i * n + j]); if (v > mx) mx = v; }
    f->rscale[i] = (mx > 0) ? 1 / mx : 1;
    for (int64_t j = 0; j < n; ++j) f->lu[i * n + j] = (real)K[i * n + j] * f->rscale[i];
    f->perm[i] = i;
  }
  real* a = f->lu;
  real* tmp = (real*)malloc(sizeof(real) * (size_t)n);
  for (int64_t k = 0; k < n; ++k) {
    int64_t p = k;
    real best = R_FABS(a[k * n + k]);
    for (int64_t i = k + 1; i < n; ++i) { real v = R_FABS(a[i * n + k]); if (v > best) { best = v; p = i; } }
    if (!(best > 0)) { *status = 4; break; }
    if (p != k) {
      memcpy(tmp, a + k * n, sizeof(real) * (size_t)n);
      memcpy(a + k * n, a + p * n, sizeof(real) * (size_t)n);
      memcpy(a + p * n, tmp, sizeof(real) * (size_t)n);
      int64_t t = f->perm[k]; f->perm[k] = f->perm[p]; f->perm[p] = t;
    }
    real piv = a[k * n + k];
#pragma omp parallel for schedule(static)
    for (int64_t i = k + 1; i < n; ++i) {
      real l = a[i * n + k] / piv;
      a[i * n + k] = l;
      const real* rk = a + k * n;
      real* ri = a + i * n;
      for (int64_t j = k + 1; j < n; ++j) ri[j] -= l * rk[j];
    }
  }
  free(tmp);
  return f;
}

void orc_lu_solve(const orc_lu_t* f, const double* b, double* x) {
  int64_t n = f->n;
  const real* a = f->lu;
  real* y = (real*)malloc(sizeof(real) * (size_t)n);
  for (int64_t k = 0; k < n; ++k) {
    long double s = (long double)((real)b[f->perm[k]] * f->rscale[f->perm[k]]);
    for (int64_t j = 0; j < k; ++j) s -= (long double)a[k * n + j] * y[j];
    y[k] = (real)s;
  }
  for (int64_t k = n - 1; k >= 0; --k) {
    long double s = y[k];
    for (int64_t j = k + 1; j < n; ++j) s -= (long double)a[k * n + j] * y[j];
    y[k] = (real)(s / a[k * n + k]);
  }
  for (int64_t k = 0; k < n; ++k) x[k] = (double)y[k];
  free(y);
}

void orc_lu_free(orc_lu_t* f) {
  if (!f) return;
  free(f->lu); free(f->rscale); free(f->perm); free(f);
}

int32_t orc_solve(int64_t n, const double* K, const double* b, double* x) {
  int32_t st;
  orc_lu_t* f = orc_lu_factor(n, K, &st);
  if (st == 0) orc_lu_solve(f, b, x);
  orc_lu_free(f);
  return st;
}

/* ------------------------------------------------------------------------------------------ */
/* a7. PFAtPoint = ElePFAtPoint + KnChPFAtPoint: Eq.(3),(4) P:70-78 with piecewise      */
/* constant sigma:  Phi(P) = (1/4 pi eps0) sum_j sigma_j sum_img Phi'_j(P) + Phi_sc(P),  E alike. */
/* Image copies apply to the elements only, not to the space charges (reading S12).             */
/* ------------------------------------------------------------------------------------------ */
void orc_eval(int64_t n, const int32_t* kind, const double* v0, const double* e1, const double* e2,
              const double* radius, const double* sigma, int32_t n_img, const double* img, int64_t q,
              const double* pos, const double* charge, int64_t m, const double* pts, double* phi, double* E) {
  elems_t g = {n, kind, v0, e1, e2, radius};
#pragma omp parallel for schedule(dynamic, 4)
  for (int64_t p = 0; p < m; ++p) {
    real P[3] = {pts[p], pts[m + p], pts[2 * m + p]};
    long double tot[4] = {0, 0, 0, 0};
    for (int64_t j = 0; j < n; ++j) {
      long double acc[4];
      elem_influence_images(&g, j, P, n_img, img, 0, acc);
      for (int k = 0; k < 4; ++k) tot[k] += (long double)sigma[j] * acc[k];
    }
    for (int k = 0; k < 4; ++k) tot[k] *= K_COULOMB;
    if (q > 0) {
      long double sc[4];
      point_charge_sum(q, pos, charge, P, sc);
      for (int k = 0; k < 4; ++k) tot[k] += sc[k];
    }
    if (phi) phi[p] = (double)tot[0];
    if (E) { E[p] = (double)tot[1]; E[m + p] = (double)tot[2]; E[2 * m + p] = (double)tot[3]; }
  }
}

/* Condition of the sums Eq.(3),(4) at a point: the sum of the MAGNITUDES of the terms orc_eval adds,
 *   S_Phi(P) = (1/4 pi eps0) [ sum_j |sigma_j| sum_img |Phi'_j(P)| + sum_k |q_k| / r_k ],
 *   S_E(P)   = (1/4 pi eps0) [ sum_j |sigma_j| sum_img |E'_j(P)|   + sum_k |q_k| / r_k^2 ]   (|.| = vector norm).
 * Not a result of the method: the parity tests use it as the scale of the rounding error of a cancelled sum
 * (a sum of n terms of both signs evaluated in precision eps carries an error ~ eps x S wherever it happens to
 * cancel, whatever the implementation), so that no global floor on |Phi| is needed.
 * phi / E (may be NULL): the sums of orc_eval themselves, formed in the same pass from the same terms in the same
 * order (bit-identical to orc_eval, checked in tests/test_oracle_pins.py), so that a sampled full-size parity check
 * walks the 1e6 element copies once instead of twice. */
void orc_eval_abs(int64_t n, const int32_t* kind, const double* v0, const double* e1, const double* e2,
                  const double* radius, const double* sigma, int32_t n_img, const double* img, int64_t q,
                  const double* pos, const double* charge, int64_t m, const double* pts, double* s_phi, double* s_E,
                  double* phi, double* E) {
  elems_t g = {n, kind, v0, e1, e2, radius};
  const int32_t copies = (n_img <= 0 || !img) ? 1 : n_img;
#pragma omp parallel for schedule(dynamic, 4)
  for (int64_t p = 0; p < m; ++p) {
    real P[3] = {pts[p], pts[m + p], pts[2 * m + p]};
    long double tp = 0, te = 0, tot[4] = {0, 0, 0, 0};
    for (int64_t j = 0; j < n; ++j) {
      long double ap = 0, ae = 0, acc[4] = {0, 0, 0, 0};
      for (int32_t s = 0; s < copies; ++s) {
        real sh[3] = {0, 0, 0};
        if (n_img > 0 && img) { sh[0] = (real)img[s]; sh[1] = (real)img[n_img + s]; sh[2] = (real)img[2 * n_img + s]; }
        real Ps[3] = {P[0] - sh[0], P[1] - sh[1], P[2] - sh[2]};
        real o[4];
        elem_influence(&g, j, Ps, o);
        ap += R_FABS(o[0]);
        ae += R_SQRT(o[1] * o[1] + o[2] * o[2] + o[3] * o[3]);
        for (int k = 0; k < 4; ++k) acc[k] += o[k];
      }
      tp += R_FABS((real)sigma[j]) * ap;
      te += R_FABS((real)sigma[j]) * ae;
      for (int k = 0; k < 4; ++k) tot[k] += (long double)sigma[j] * acc[k];
    }
    for (int k = 0; k < 4; ++k) tot[k] *= K_COULOMB;
    tp *= K_COULOMB;
    te *= K_COULOMB;
    if (q > 0) {
      long double sc[4];
      point_charge_sum(q, pos, charge, P, sc);
      for (int k = 0; k < 4; ++k) tot[k] += sc[k];
      long double cp = 0, ce = 0;
      for (int64_t c = 0; c < q; ++c) {
        real dx = P[0] - (real)pos[c], dy = P[1] - (real)pos[q + c], dz = P[2] - (real)pos[2 * q + c];
        real r2 = dx * dx + dy * dy + dz * dz;
        if (r2 > 0) {
          cp += R_FABS((real)charge[c]) / R_SQRT(r2);
          ce += R_FABS((real)charge[c]) / r2;
        }
      }
      tp += cp * K_COULOMB;
      te += ce * K_COULOMB;
    }
    if (s_phi) s_phi[p] = (double)tp;
    if (s_E) s_E[p] = (double)te;
    if (phi) phi[p] = (double)tot[0];
    if (E) { E[p] = (double)tot[1]; E[m + p] = (double)tot[2]; E[2 * m + p] = (double)tot[3]; }
  }
}

/* a9. Charge push of the synthetic C4 loop (reading S23): x += mu * E * dt. */
void orc_push(int64_t q, double* pos, const double* E, double mu, double dt) {
  for (int64_t k = 0; k < 3 * q; ++k) pos[k] = (double)((real)pos[k] + (real)mu * (real)E[k] * (real)dt);
}

/* ------------------------------------------------------------------------------------------------
 * FastVolume ("Fast Volume", P:222 CreateFastVolPF): the potential and field are precomputed on a
 * 3-D grid of nodal points and "rapidly estimated using a simple trilinear interpolation from the
 * values stored at the nearest nodes".  Reading (S25): uniform grid, node (i,j,k) at
 * origin + (i hx, j hy, k hz), i < nx fastest; values[c][(k*ny + j)*nx + i], c = 0..3 = Phi, Ex, Ey, Ez;
 * each of the four quantities is interpolated on its own; a point outside the grid's box gets NaN.
 * "Outside" is decided on the cell coordinate t = (x - origin)/h in DOUBLE (the precision of the CUDA
 * path, so that both sides take this yes/no decision alike) with a slack of 1e-9 cells, because a node
 * of the upper faces, computed as origin + i h, may round to t = n-1+1e-16; t is then clamped to [0, n-1].
 * Trilinear interpolation written out as its definition: the sum over the 8 corners of the cell of
 * the corner value times the product of the three 1-D hat weights.
 * ------------------------------------------------------------------------------------------------ */
void orc_fastvol_eval(int32_t nx, int32_t ny, int32_t nz, const double* origin, const double* spacing,
                      const double* values, int64_t m, const double* pts, double* phi, double* E) {
  const int64_t nn = (int64_t)nx * ny * nz;
  const int32_t dim[3] = {nx, ny, nz};
#pragma omp parallel for schedule(static)
  for (int64_t p = 0; p < m; ++p) {
    int32_t cell[3];
    real f[3];
    int inside = 1;
    for (int a = 0; a < 3; ++a) {
      const double td = (pts[a * m + p] - origin[a]) / spacing[a];
      if (!(td >= -1e-9 && td <= (double)(dim[a] - 1) + 1e-9)) { inside = 0; break; }
      real t = ((real)pts[a * m + p] - (real)origin[a]) / (real)spacing[a];
      if (t < 0) t = 0;
      if (t > (real)(dim[a] - 1)) t = (real)(dim[a] - 1);
      int32_t i = (int32_t)floorl((long double)t);
      if (i > dim[a] - 2) i = dim[a] - 2;      /* t == n-1: last cell, weight 1 on its far node */
      cell[a] = i;
      f[a] = t - (real)i;
    }
    double out[4];
    for (int c = 0; c < 4; ++c) {
      if (!inside) { out[c] = NAN; continue; }
      long double acc = 0;
      for (int dk = 0; dk < 2; ++dk)
        for (int dj = 0; dj < 2; ++dj)
          for (int di = 0; di < 2; ++di) {
            real w = (di ? f[0] : 1 - f[0]) * (dj ? f[1] : 1 - f[1]) * (dk ? f[2] : 1 - f[2]);
            int64_t node = ((int64_t)(cell[2] + dk) * ny + (cell[1] + dj)) * nx + (cell[0] + di);
            acc += (long double)(w * (real)values[c * nn + node]);
          }
      out[c] = (double)acc;
    }
    phi[p] = out[0];
    E[p] = out[1]; E[m + p] = out[2]; E[2 * m + p] = out[3];
  }
}

/* ------------------------------------------------------------------------------------------------
 * Alg. 3 "Point to Line Charge Reduction (Voxelization)": dense clusters of point charges
 * are mapped into representative line charges.  Reading (S27): the grid has dims[a] voxels of
 * size voxel[a] from origin[a]; the voxel index of a point is floor((p - origin)/voxel) per axis, clamped
 * to the grid (a point outside is counted in the nearest border voxel, so that the total charge is
 * conserved); a voxel is occupied when at least one point fell in it (Alg. 3's isOccupied), even if its
 * charges cancel; an occupied voxel becomes ONE line charge through the voxel's centre, parallel to z,
 * spanning the voxel's z extent, of line density lambda = (total charge of the voxel) / voxel[2].  Lines
 * are listed in voxel-index order (x fastest).  Kernel 1 = the scatter loop, Kernel 2 = the line loop.
 * lines: 5*cap doubles SoA  x, y, z_start, z_stop, lambda.  Returns the number of lines (<= cap), or -1
 * if cap is too small.
 * ------------------------------------------------------------------------------------------------ */
int64_t orc_voxelize(int64_t q, const double* pos, const double* charge, const double* origin, const double* voxel,
                     const int32_t* dims, int64_t cap, double* lines) {
  const int64_t nv = (int64_t)dims[0] * dims[1] * dims[2];
  long double* total = (long double*)calloc((size_t)nv, sizeof(long double));
  unsigned char* occupied = (unsigned char*)calloc((size_t)nv, 1);
  for (int64_t c = 0; c < q; ++c) {                                /* Kernel 1: Voxelize (Scatter) */
    int64_t idx[3];
    for (int a = 0; a < 3; ++a) {
      int64_t i = (int64_t)floor((pos[a * q + c] - origin[a]) / voxel[a]);   /* decided in double, like the GPU */
      if (i < 0) i = 0;
      if (i > dims[a] - 1) i = dims[a] - 1;
      idx[a] = i;
    }
    const int64_t v = (idx[2] * dims[1] + idx[1]) * dims[0] + idx[0];
    total[v] += (long double)charge[c];
    occupied[v] = 1;
  }
  int64_t nl = 0;
  for (int64_t v = 0; v < nv; ++v) {                               /* Kernel 2: Generate Lines (Reduce) */
    if (!occupied[v]) continue;
    if (nl >= cap) { nl = -1; break; }
    const int64_t i = v % dims[0], j = (v / dims[0]) % dims[1], k = v / ((int64_t)dims[0] * dims[1]);
    lines[0 * cap + nl] = origin[0] + ((double)i + 0.5) * voxel[0];
    lines[1 * cap + nl] = origin[1] + ((double)j + 0.5) * voxel[1];
    lines[2 * cap + nl] = origin[2] + (double)k * voxel[2];
    lines[3 * cap + nl] = origin[2] + (double)(k + 1) * voxel[2];
    lines[4 * cap + nl] = (double)(total[v] / (long double)voxel[2]);
    ++nl;
  }
  free(total);
  free(occupied);
  return nl;
}

/* Potential and field of nl straight line charges parallel to z (uniform line density lambda, C/m) at m
 * points: the defining integral  Phi = (1/4 pi eps0) Int lambda dz' / |r - r'|  (Eq. 2 P:68 integrated along
 * the line; the wire integral P:131 without its radius) in closed form, with l1 = z_start - Z, l2 = z_stop - Z,
 * rho^2 = dx^2 + dy^2, R_i = sqrt(rho^2 + l_i^2):
 *   Phi = k lambda [asinh(l2/rho) - asinh(l1/rho)],  E_rho = k lambda (l2/R2 - l1/R1)/rho,  E_z = k lambda (1/R2 - 1/R1).
 * A point exactly on a line's axis (rho = 0) is skipped, like r = 0 in Alg. 2 (reading S27). */
void orc_line_charges(int64_t m, const double* pts, int64_t nl, int64_t cap, const double* lines, double* phi, double* E) {
#pragma omp parallel for schedule(dynamic, 16)
  for (int64_t p = 0; p < m; ++p) {
    long double acc[4] = {0, 0, 0, 0};
    for (int64_t c = 0; c < nl; ++c) {
      real dx = (real)pts[p] - (real)lines[c], dy = (real)pts[m + p] - (real)lines[cap + c];
      real l1 = (real)lines[2 * cap + c] - (real)pts[2 * m + p], l2 = (real)lines[3 * cap + c] - (real)pts[2 * m + p];
      real rho2 = dx * dx + dy * dy;
      if (!(rho2 > 0)) continue;
      real rho = R_SQRT(rho2), R1 = R_SQRT(rho2 + l1 * l1), R2 = R_SQRT(rho2 + l2 * l2);
      real lam = (real)lines[4 * cap + c];
      real er = lam * (l2 / R2 - l1 / R1) / rho2;      /* E_rho / rho */
      acc[0] += lam * (R_ASINH(l2 / rho) - R_ASINH(l1 / rho));
      acc[1] += er * dx;
      acc[2] += er * dy;
      acc[3] += lam * (1 / R2 - 1 / R1);
    }
    if (phi) phi[p] = (double)(acc[0] * K_COULOMB);
    if (E) { E[p] = (double)(acc[1] * K_COULOMB); E[m + p] = (double)(acc[2] * K_COULOMB); E[2 * m + p] = (double)(acc[3] * K_COULOMB); }
  }
}

/* ------------------------------------------------------------------------------------------------
 * Adaptive Modelling (Table 2): "the solver is permitted to use a simplified
 * representation ... for parts of the geometry that are far away from the point of evaluation".
 * Reading (S28): the inputs here are elements, not Garfield++ primitives, so the simplified
 * representation of a FAR periodic copy of element j is its total charge sigma_j A_j as a point charge
 * at the copy's centroid (rectangle: A = |e1 x e2|, v0 + (e1+e2)/2; right triangle: A = |e1 x e2|/2,
 * v0 + (e1+e2)/3; wire: A = 2 pi r_w |e1|, v0 + e1/2); a copy is far when the length of its shift vector
 * is >= far_distance (so the unshifted element is never simplified; far_distance <= 0 means no
 * simplification).  Everything else is orc_eval.  An approximation: the error of a far copy's
 * contribution is O((element size / distance)^2) — its quadrupole term.
 * ------------------------------------------------------------------------------------------------ */
void orc_eval_adaptive(int64_t n, const int32_t* kind, const double* v0, const double* e1, const double* e2,
                       const double* radius, const double* sigma, int32_t n_img, const double* img, double far_distance,
                       int64_t q, const double* pos, const double* charge, int64_t m, const double* pts, double* phi,
                       double* E) {
  elems_t g = {n, kind, v0, e1, e2, radius};
  const int32_t copies = (n_img <= 0 || !img) ? 1 : n_img;
#pragma omp parallel for schedule(dynamic, 4)
  for (int64_t p = 0; p < m; ++p) {
    real P[3] = {pts[p], pts[m + p], pts[2 * m + p]};
    long double tot[4] = {0, 0, 0, 0};
    for (int64_t j = 0; j < n; ++j) {
      real a1[3] = {e1[j], e1[n + j], e1[2 * n + j]}, a2[3] = {e2[j], e2[n + j], e2[2 * n + j]};
      real cr[3] = {a1[1] * a2[2] - a1[2] * a2[1], a1[2] * a2[0] - a1[0] * a2[2], a1[0] * a2[1] - a1[1] * a2[0]};
      real area, cen[3];
      if (kind[j] == ORC_WIRE) {
        area = 2 * PI_L * (real)radius[j] * R_SQRT(a1[0] * a1[0] + a1[1] * a1[1] + a1[2] * a1[2]);
        for (int k = 0; k < 3; ++k) cen[k] = (real)v0[k * n + j] + a1[k] / 2;
      } else {
        real w = (kind[j] == ORC_RECT) ? (real)0.5 : (real)1 / 3;
        area = R_SQRT(cr[0] * cr[0] + cr[1] * cr[1] + cr[2] * cr[2]) * ((kind[j] == ORC_RECT) ? 1 : (real)0.5);
        for (int k = 0; k < 3; ++k) cen[k] = (real)v0[k * n + j] + w * (a1[k] + a2[k]);
      }
      long double acc[4] = {0, 0, 0, 0};
      for (int32_t s = 0; s < copies; ++s) {
        real sh[3] = {0, 0, 0};
        if (n_img > 0 && img) { sh[0] = (real)img[s]; sh[1] = (real)img[n_img + s]; sh[2] = (real)img[2 * n_img + s]; }
        real len = R_SQRT(sh[0] * sh[0] + sh[1] * sh[1] + sh[2] * sh[2]);
        if (far_distance > 0 && len >= (real)far_distance) {
          real d[3] = {P[0] - sh[0] - cen[0], P[1] - sh[1] - cen[1], P[2] - sh[2] - cen[2]};
          real r2 = d[0] * d[0] + d[1] * d[1] + d[2] * d[2];
          if (r2 > 0) {
            real r = R_SQRT(r2);
            acc[0] += area / r;
            for (int k = 0; k < 3; ++k) acc[k + 1] += area * d[k] / (r2 * r);
          }
        } else {
          real Ps[3] = {P[0] - sh[0], P[1] - sh[1], P[2] - sh[2]};
          real o[4];
          elem_influence(&g, j, Ps, o);
          for (int k = 0; k < 4; ++k) acc[k] += o[k];
        }
      }
      for (int k = 0; k < 4; ++k) tot[k] += (long double)sigma[j] * acc[k];
    }
    for (int k = 0; k < 4; ++k) tot[k] *= K_COULOMB;
    if (q > 0) {
      long double sc[4];
      point_charge_sum(q, pos, charge, P, sc);
      for (int k = 0; k < 4; ++k) tot[k] += sc[k];
    }
    if (phi) phi[p] = (double)tot[0];
    if (E) { E[p] = (double)tot[1]; E[m + p] = (double)tot[2]; E[2 * m + p] = (double)tot[3]; }
  }
}
