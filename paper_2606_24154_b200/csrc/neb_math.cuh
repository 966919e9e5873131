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

// Polynomial coefficients live in the constant bank so that DFMA reads them as c[bank][offset] operands
// instead of two UMOV immediates per use.  Near-minimax fits (Chebyshev interpolation in 40-digit
// arithmetic, coefficients rounded to double and re-checked):
//   atanh(z)/z = 1 + w A(w), w = z^2 <= 0.0403, degree 7: max relative error 7.5e-19
//   atan(t)/t  = 1 + w B(w), w = t^2 <= 0.0719, degree 8: max relative error 1.3e-18
//   (stored doubled: the kernel needs 2 atanh)
static __constant__ double kAtanhC[8] = {2 * 0.3333333333333333, 2 * 0.20000000000004114, 2 * 0.14285714283573475,
                                         2 * 0.11111111534886074, 2 * 0.09090867974834849, 2 * 0.0769446730129734,
                                         2 * 0.06604199001390682, 2 * 0.06809533021415161};
static __constant__ double kAtanC[9] = {-0.3333333333333333, 0.19999999999996848, -0.14285714284542553, 0.11111110943140809,
                                        -0.09090896999665297, 0.0769181700719147, -0.06654898512832812, 0.05715903312379015,
                                        -0.03956311994071827};

// max(x, ~1e-300) for x >= 0 with one integer instruction on the high word (keeps the FP64 pipe free)
__device__ __forceinline__ double clamp_tiny(double x) {
  return __hiloint2double(max(__double2hiint(x), 0x01a56e1f), __double2loint(x));
}

// x / 2 for a normal x well inside the exponent range (here: 1/sqrt of a length squared): one integer subtraction on
// the high word instead of a DMUL on the FP64 pipe
__device__ __forceinline__ double half_of(double x) {
  return __hiloint2double(__double2hiint(x) - 0x00100000, __double2loint(x));
}

// 1/sqrt(x) for x > 0 (the caller clamps and handles x = 0): MUFU.RSQ64H seed (2^-23) + ONE cubic step
//   e = 1 - x y^2,  y <- y (1 + e/2 + 3 e^2 / 8)      (relative error ~ e^3 = 2^-69 before rounding): 5 FP64-pipe ops
__device__ __forceinline__ double rsqrt_pos(double x) {
  const double y = mufu_rsqrt(x);
  const double e = fma(-x * y, y, 1.0);
  const double p = fma(0.375, e, 0.5);
  return fma(y * e, p, y);
}

// x == 0 (either sign) by integer operations on the bit pattern
__device__ __forceinline__ bool is_zero(double x) { return (((__double2hiint(x) & 0x7fffffff) | __double2loint(x)) == 0); }

struct MathLib {
  static constexpr bool kNeedsFar = true;    // libm path: far field through log1p
  static constexpr bool kFarPath = false;    // no warp-uniform far-field shortcut: this policy is the plain reference
  static __device__ __forceinline__ double far_log(double, double) { return 0.0; }
  static __device__ __forceinline__ double far_atan2(double, double) { return 0.0; }
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
  static constexpr bool kNeedsFar = false;   // z = L/s whenever the exponent fold is zero
  static constexpr bool kFarPath = true;     // warp-uniform shortcut when every lane is >= 2.5 edge lengths away
  // sqrt(x), x >= 0 finite (x = 0 -> 0).  One coupled Newton step on (g ~ sqrt x, h ~ 1/(2 sqrt x))
  // from the 2^-23 seed, then one residual correction: 5 FP64-pipe ops (the halving is an integer
  // subtraction on the exponent) + 1 integer clamp + 1 MUFU.
  static __device__ __forceinline__ double sqrt_nn(double x) {
    double y = mufu_rsqrt(clamp_tiny(x));
    double g = x * y, h = half_of(y);
    double r = fma(-g, h, 0.5);
    g = fma(g, r, g);                 // relative error ~2^-45
    double d = fma(-g, g, x);         // residual; the seed-accurate h is enough for the correction term
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
    N = clamp_tiny(N);
    D = clamp_tiny(D);
    // e = round(pseudo-log2(N/D)) from the exponent/mantissa bits: N/(D 2^e) in [0.666, 1.502]
    int hN = __double2hiint(N), hD = __double2hiint(D);
    int e = ((hN - hD) + 0x80000) >> 20;
    // N/D = (s+L)/(s-L) identically, so (N-D)/(N+D) = L/s: whenever e = 0 (ratio within [0.666, 1.5], which
    // includes the whole far field) z is taken as L/s, which has no cancellation at all
    (void)far;
    double D2 = __hiloint2double(hD + (e << 20), __double2loint(D));
    double zn = (e == 0) ? L : (N - D2);
    double zd = (e == 0) ? s : (N + D2);
    double z = zn * rcp_pos(zd);                 // |z| <= 0.2004
    double w = z * z;
    double p = kAtanhC[7];
    p = fma(p, w, kAtanhC[6]);
    p = fma(p, w, kAtanhC[5]);
    p = fma(p, w, kAtanhC[4]);
    p = fma(p, w, kAtanhC[3]);
    p = fma(p, w, kAtanhC[2]);
    p = fma(p, w, kAtanhC[1]);
    p = fma(p, w, kAtanhC[0]);
    double t = z * fma(w, p, 2.0);               // 2 atanh(z) = z (2 + w 2A(w)); coefficients hold 2A
    // e as a double without a conversion instruction: (2^52 + 2^31 + e) - (2^52 + 2^31)
    double ed = __hiloint2double(0x43300000, e ^ 0x80000000) - 4503601774854144.0;
    return fma(ed, 0.693147180559945309417, t);
  }
  // Far field (s >= 5 L, i.e. z <= 0.2, guaranteed by the caller): ln[(s+L)/(s-L)] = 2 atanh(L/s) with the same
  // polynomial as log_ratio's e == 0 case, but no case selection, no exponent fold: 15 FP64 instructions + 1 MUFU.
  static __device__ __forceinline__ double far_log(double L, double s) {
    double z = L * rcp_pos(s);
    double w = z * z;
    double p = kAtanhC[7];
    p = fma(p, w, kAtanhC[6]);
    p = fma(p, w, kAtanhC[5]);
    p = fma(p, w, kAtanhC[4]);
    p = fma(p, w, kAtanhC[3]);
    p = fma(p, w, kAtanhC[2]);
    p = fma(p, w, kAtanhC[1]);
    p = fma(p, w, kAtanhC[0]);
    return z * fma(w, p, 2.0);
  }
  // atan(y/x) for x > 0, 0 <= y <= tan(pi/12) x (guaranteed by the caller in the far field): no argument reduction
  static __device__ __forceinline__ double far_atan2(double y, double x) {
    double t = y * rcp_pos(x);
    double w = t * t;
    double p = kAtanC[8];
    p = fma(p, w, kAtanC[7]);
    p = fma(p, w, kAtanC[6]);
    p = fma(p, w, kAtanC[5]);
    p = fma(p, w, kAtanC[4]);
    p = fma(p, w, kAtanC[3]);
    p = fma(p, w, kAtanC[2]);
    p = fma(p, w, kAtanC[1]);
    p = fma(p, w, kAtanC[0]);
    return fma(t * w, p, t);
  }
  static __device__ __forceinline__ double atan2_pos(double y, double x) {
    y = fabs(y);                                          // rounding noise may make a zero numerator negative
    double ax = fabs(x);
    double mx = fmax(y, ax), mn = fmin(y, ax);
    bool big = mn > 0.26794919243112270647 * mx;          // tan(pi/12)
    double c = big ? 0.57735026918962576451 : 0.0;        // tan(pi/6)
    double num = fma(-c, mx, mn);
    double den = clamp_tiny(fma(c, mn, mx));
    double t = num * rcp_pos(den);                        // |t| <= tan(pi/12)
    double w = t * t;
    double p = kAtanC[8];
    p = fma(p, w, kAtanC[7]);
    p = fma(p, w, kAtanC[6]);
    p = fma(p, w, kAtanC[5]);
    p = fma(p, w, kAtanC[4]);
    p = fma(p, w, kAtanC[3]);
    p = fma(p, w, kAtanC[2]);
    p = fma(p, w, kAtanC[1]);
    p = fma(p, w, kAtanC[0]);
    double a = fma(t, fma(w, p, 1.0), big ? 0.52359877559829887308 : 0.0);   // atan(t) + pi/6
    a = (y > ax) ? (NEB_HALF_PI - a) : a;
    a = (__double2hiint(x) < 0) ? (NEB_PI - a) : a;
    return a;
  }
};

}  // namespace neb
