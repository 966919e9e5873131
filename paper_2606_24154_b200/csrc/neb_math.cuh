// neb_math.cuh — range-restricted FP64 primitives for the influence kernels (sm_100a).
//
// The influence evaluation is bound by the FP64 pipe, and CUDA's libm log /
// atan2 / sqrt / division spend most of their instructions on special-case handling (NaN, inf,
// denormals, negative arguments) that cannot occur here: every argument is a finite,
// non-negative length or product of lengths.  Two policies with the same interface:
//   MathLib  : CUDA libm (log, log1p, atan2, sqrt, /) — the reference implementation on device
//   MathFast : MUFU.RCP64H / MUFU.RSQ64H seeds + DFMA Newton steps + DFMA Horner polynomials,
//              branch-free (selects only)
// Both are exercised against the CPU oracle by the parity tests.
#pragma once
#include <cuda_runtime.h>
#include <math.h>

namespace neb {

#define NEB_TINY 1.0e-300
#define NEB_PI 3.14159265358979323846
#define NEB_HALF_PI 1.57079632679489661923

__device__ __forceinline__ double mufu_rcp(double x) {
  double r;
  asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(r) : "d"(x));
  return r;
}
__device__ __forceinline__ double mufu_rsqrt(double x) {
  double r;
  asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(r) : "d"(x));
  return r;
}

struct MathLib {
  static __device__ __forceinline__ double sqrt_nn(double x) { return sqrt(x); }
  static __device__ __forceinline__ double div_pos(double a, double b) { return a / b; }
  // ln(N/D) for N >= D > 0 in the near field, or 2 atanh(L/s) in the far field (s > 8 L)
  static __device__ __forceinline__ double log_ratio(double N, double D, bool far, double L, double s) {
    double near_v = log(fmax(N, NEB_TINY) / fmax(D, NEB_TINY));
    double far_v = log1p(2.0 * L / (s - L));
    return far ? far_v : near_v;
  }
  // atan2(|y|, x): result in [0, pi]; atan2(0,0) = 0.  y is non-negative up to rounding noise
  static __device__ __forceinline__ double atan2_pos(double y, double x) { return atan2(fabs(y), x); }
};

struct MathFast {
  // sqrt(x), x >= 0 finite (x = 0 -> 0).  One coupled Newton step on (g ~ sqrt x, h ~ 1/(2 sqrt x))
  // from the 2^-23 seed, then one residual correction: 7 DFMA-class ops + 1 DMNMX + 1 MUFU.
  static __device__ __forceinline__ double sqrt_nn(double x) {
    double y = mufu_rsqrt(fmax(x, NEB_TINY));
    double g = x * y, h = 0.5 * y;
    double r = fma(-g, h, 0.5);
    g = fma(g, r, g);
    h = fma(h, r, h);
    double d = fma(-g, g, x);
    return fma(d, h, g);
  }
  // 1/b for b > 0 finite normal: cubic step from the seed (error e^3 ~ 2^-69), 3 DFMA + 1 MUFU
  static __device__ __forceinline__ double rcp_pos(double b) {
    double r = mufu_rcp(b);
    double e = fma(-b, r, 1.0);
    double e2 = fma(e, e, e);
    return fma(r, e2, r);
  }
  static __device__ __forceinline__ double div_pos(double a, double b) {
    double r = rcp_pos(b);
    double q = a * r;
    double rem = fma(-b, q, a);
    return fma(rem, r, q);
  }
  static __device__ __forceinline__ double log_ratio(double N, double D, bool far, double L, double s) {
    N = fmax(N, NEB_TINY);
    D = fmax(D, NEB_TINY);
    // e = round(pseudo-log2(N/D)) from the exponent/mantissa bits: N/(D 2^e) in [0.666, 1.502]
    int hN = __double2hiint(N), hD = __double2hiint(D);
    int e = ((hN - hD) + 0x80000) >> 20;
    e = far ? 0 : e;
    double D2 = __hiloint2double(hD + (e << 20), __double2loint(D));
    double zn = far ? L : (N - D2);
    double zd = far ? s : (N + D2);
    double z = zn * rcp_pos(zd);                 // |z| <= 0.2004
    double w = z * z;
    // atanh(z)/z = sum_{k>=0} w^k/(2k+1); truncated after k = 11: error < 8e-19 for w <= 0.0402
    double p = 1.0 / 23.0;
    p = fma(p, w, 1.0 / 21.0);
    p = fma(p, w, 1.0 / 19.0);
    p = fma(p, w, 1.0 / 17.0);
    p = fma(p, w, 1.0 / 15.0);
    p = fma(p, w, 1.0 / 13.0);
    p = fma(p, w, 1.0 / 11.0);
    p = fma(p, w, 1.0 / 9.0);
    p = fma(p, w, 1.0 / 7.0);
    p = fma(p, w, 1.0 / 5.0);
    p = fma(p, w, 1.0 / 3.0);
    double zz = z + z;
    double t = fma(zz * w, p, zz);               // 2 atanh(z)
    // e as a double without a conversion instruction: (2^52 + 2^31 + e) - (2^52 + 2^31)
    double ed = __hiloint2double(0x43300000, e ^ 0x80000000) - 4503601774854144.0;
    return fma(ed, 0.693147180559945309417, t);
  }
  static __device__ __forceinline__ double atan2_pos(double y, double x) {
    y = fabs(y);                                          // rounding noise may make a zero numerator negative
    double ax = fabs(x);
    double mx = fmax(y, ax), mn = fmin(y, ax);
    bool big = mn > 0.26794919243112270647 * mx;          // tan(pi/12)
    double c = big ? 0.57735026918962576451 : 0.0;        // tan(pi/6)
    double num = fma(-c, mx, mn);
    double den = fmax(fma(c, mn, mx), NEB_TINY);
    double t = num * rcp_pos(den);                        // |t| <= tan(pi/12)
    double w = t * t;
    // atan(t)/t = sum (-w)^k/(2k+1), k <= 13: first omitted term < 4e-18 for w <= 0.0718
    double p = -1.0 / 27.0;
    p = fma(p, w, 1.0 / 25.0);
    p = fma(p, w, -1.0 / 23.0);
    p = fma(p, w, 1.0 / 21.0);
    p = fma(p, w, -1.0 / 19.0);
    p = fma(p, w, 1.0 / 17.0);
    p = fma(p, w, -1.0 / 15.0);
    p = fma(p, w, 1.0 / 13.0);
    p = fma(p, w, -1.0 / 11.0);
    p = fma(p, w, 1.0 / 9.0);
    p = fma(p, w, -1.0 / 7.0);
    p = fma(p, w, 1.0 / 5.0);
    p = fma(p, w, -1.0 / 3.0);
    double a = fma(t * w, p, t) + (big ? 0.52359877559829887308 : 0.0);   // + pi/6
    a = (y > ax) ? (NEB_HALF_PI - a) : a;
    a = (x < 0.0) ? (NEB_PI - a) : a;
    return a;
  }
};

}  // namespace neb
