// su2_power.cuh -- the exact SU(2) group power g -> g^omega in fp64, written for the B200's
// half-rate FP64 pipe: branch-free, bounded-range polynomials instead of the general-purpose
// libm atan2/sincos (which carry slow paths for arguments this kernel can never produce).
//
// "replacing g(x) by g^omega(x)"; reading C-8: the exact power on the
// principal branch.  For the subgroup quaternion p = (p0, pv) of K the update
// is  g = conj(p)/|p| = (cos a, -pv/|pv| sin a),  a = atan2(|pv|, p0) in [0, pi], and
//      g^omega = (cos(omega a), -pv/|pv| sin(omega a)).
//
// How a is obtained to fp64 accuracy without an fp64 atan2:
//   a~ = a cheap fp32 polynomial atan2 (error < 3e-6), widened exactly to fp64;
//   (s~, c~) = sincos(a~) by the fp64 polynomials below;
//   d = sin(a - a~) = (|pv| c~ - p0 s~)/|p|  exactly;  a = a~ + d + d^3/6   (|d|^5 < 1e-30).
// The two sincos evaluations (of a~ and of omega*a~) are independent, which gives the FP64 pipe
// four independent Horner chains; omega*a = omega*a~ + omega*(d + d^3/6) is folded in by the angle-addition
// formulas with the tiny second angle expanded to second order.
#pragma once
#include <cuda_runtime.h>
#include <math.h>
#include <stdint.h>

namespace culgt {

// Taylor coefficients of sin (odd, from -1/3! up to -1/19!) and cos (even, from -1/2! up to 1/20!).
// In constant memory so that every DFMA takes its coefficient as a constant-bank operand instead
// of two MOVs of a 64-bit immediate.
__constant__ double kSinCoef[9] = {
    -1.66666666666666666667e-01, 8.33333333333333333333e-03, -1.98412698412698412698e-04,
    2.75573192239858906526e-06,  -2.50521083854417187751e-08, 1.60590438368216145994e-10,
    -7.64716373181981647590e-13, 2.81145725434552076320e-15,  -8.22063524662432971696e-18};
__constant__ double kCosCoef[10] = {
    -0.5,                        4.16666666666666666667e-02,  -1.38888888888888888889e-03,
    2.48015873015873015873e-05,  -2.75573192239858906526e-07, 2.08767569878680989792e-09,
    -1.14707455977297247139e-11, 4.77947733238738529744e-14,  -1.56192069685862264622e-16,
    4.11031762331216485848e-19};

// sin and cos of x for 0 <= x <= ~7 (omega*a < 2*pi): Cody-Waite reduction by pi/2 (k <= 4, so two
// constants suffice) and Taylor polynomials on [-pi/4, pi/4] truncated below 1e-17.
// FULL = false stops the series at y^11/11! and y^12/12! (truncation < 7e-12): enough for fp32
// link storage, where the chain's errors are compared at 2e-5 after an amplification of <~ 1e3.
template <bool FULL>
__device__ __forceinline__ void sincos_bounded(double x, double* s, double* c) {
  constexpr int NS = FULL ? 9 : 5, NC = FULL ? 10 : 6;
  // k = rint(x * 2/pi) by the 1.5*2^52 trick: no FRND / F2I on the slow conversion pipe
  const double magic = 6755399441055744.0;
  const double kb = fma(x, 0.63661977236758134308, magic);
  const int q = __double2loint(kb);
  const double k = kb - magic;
  double y = fma(-k, 1.57079632679489655800e+00, x);            // pi/2 high part
  y = fma(-k, 6.12323399573676603587e-17, y);                   // pi/2 low part
  const double z = y * y;
  double ps = kSinCoef[NS - 1];
#pragma unroll
  for (int i = NS - 2; i >= 0; --i) ps = fma(ps, z, kSinCoef[i]);
  const double sy = fma(ps * z, y, y);
  double pc = kCosCoef[NC - 1];
#pragma unroll
  for (int i = NC - 2; i >= 0; --i) pc = fma(pc, z, kCosCoef[i]);
  const double cy = fma(pc, z, 1.0);
  const double a = (q & 1) ? cy : sy;
  const double b = (q & 1) ? sy : cy;
  *s = (q & 2) ? -a : a;
  *c = ((q + 1) & 2) ? -b : b;
}

// 1/sqrt(x) for normal positive x: the 64-bit MUFU seed (~2^-22) and two Newton steps (one when
// FULL = false: ~1e-13).
template <bool FULL>
__device__ __forceinline__ double rsqrt_newton(double x) {
  double y;
  asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(x));
  double e = fma(-x * y, y, 1.0);
  y = fma(0.5 * y, e, y);
  if (FULL) {
    e = fma(-x * y, y, 1.0);
    y = fma(0.5 * y, e, y);
  }
  return y;
}

}  // namespace culgt

#include "heatbath.cuh"   // needs kSinCoef / kCosCoef and rsqrt_newton above

namespace culgt {

// atan2(y, x) for y >= 0 and x^2 + y^2 = 1, in fp32, absolute error < 3e-6 (degree-11 odd
// polynomial on [0,1] plus octant fix-up).  It only seeds the fp64 correction below.
__device__ __forceinline__ float atan2_seed(float y, float x) {
  const float ax = fabsf(x);
  const float mx = fmaxf(ax, y), mn = fminf(ax, y);      // mx >= 0.707
  const float t = __fdividef(mn, mx);
  const float u = t * t;
  float p = -0.011686083860695362f;
  p = fmaf(p, u, 0.05254087969660759f);
  p = fmaf(p, u, -0.11629831045866013f);
  p = fmaf(p, u, 0.1934700906276703f);
  p = fmaf(p, u, -0.3326060175895691f);
  p = fmaf(p, u, 0.9999759197235107f);
  float a = p * t;
  if (y > ax) a = 1.57079632679489662f - a;
  if (x < 0.0f) a = 3.14159265358979324f - a;
  return a;
}

// q_out = (conj(p)/|p|)^omega for the un-normalised quaternion p = (p[0]; p[1], p[2], p[3]).
// Returns false (q_out untouched) when p == 0, where the update is skipped (reading C-9).
template <bool FULL>
__device__ __forceinline__ bool su2_update_power(const double* p, double omega, double* q) {
  const double r2 = p[1] * p[1] + p[2] * p[2] + p[3] * p[3];
  const double n2 = fma(p[0], p[0], r2);
  if (n2 < 1e-280) {                 // |p| = 0 skips the update; denormal-range |p| is treated alike
    return false;
  }
  if (r2 < 1e-280) {                 // g = +1 or -1: axis undefined (C-8: z axis by fiat for g = -1)
    double s = 0.0, c = 1.0;
    if (p[0] < 0.0) sincos_bounded<FULL>(omega * 3.14159265358979323846, &s, &c);
    q[0] = c; q[1] = 0.0; q[2] = 0.0; q[3] = s;
    return true;
  }
  const double rinv = rsqrt_newton<FULL>(r2);   // 1/|pv|
  const double ninv = rsqrt_newton<FULL>(n2);   // 1/|p|
  const double R = r2 * rinv;             // |pv|
  const double sn = R * ninv, cs = p[0] * ninv;      // sin a, cos a
  const double a0 = (double)atan2_seed((float)sn, (float)cs);
  double s0, c0, s1, c1;
  sincos_bounded<FULL>(a0, &s0, &c0);
  sincos_bounded<FULL>(omega * a0, &s1, &c1);
  double d = sn * c0 - cs * s0;                    // sin(a - a0), |d| < 1e-5
  d = fma(d * d * d, 1.0 / 6.0, d);                // a - a0
  const double e = omega * d;                      // omega a - omega a0
  const double ce = fma(-0.5 * e, e, 1.0);
  const double se = fma(e * e * e, -1.0 / 6.0, e);
  const double C = c1 * ce - s1 * se;
  const double S = s1 * ce + c1 * se;
  const double f = -S * rinv;
  q[0] = C; q[1] = p[1] * f; q[2] = p[2] * f; q[3] = p[3] * f;
  return true;
}

// ---- how g is raised to the power omega: a policy object passed down from the kernel parameter ----
// ExactPower: the exact group power of reading C-8 (above).  SeriesPower: the truncated binomial
// series of reading C-24,  g^omega ~ S_N = sum_{n<=N} binom(omega,n) (g-1)^n, projected back to
// SU(2).  (g-1)^n lives in span{1, i n.sigma}, so with z = (cos a - 1) + i sin a the series is the
// complex polynomial w = sum b_n z^n and the result is (Re w, n Im w)/|w|: a Horner loop, no
// transcendental function at all.  b_n = binom(omega, n) is filled in on the host.
struct ExactPower {
  double omega;
};
// Microcanonical step (reading C-26): q = g^2, the reflection that leaves Re tr[g_s K]
// unchanged.  No parameter.
struct MicroPower {
  int unused;
};
constexpr int kMaxSeriesOrder = 16;
struct SeriesPower {
  int order;
  double b[kMaxSeriesOrder + 1];
};

template <bool FULL>
__device__ __forceinline__ bool su2_update_power(const double* p, const ExactPower& pw, double* q) {
  return su2_update_power<FULL>(p, pw.omega, q);
}

template <bool FULL>
__device__ __forceinline__ bool su2_update_power(const double* p, const SeriesPower& pw, double* q) {
  const double r2 = p[1] * p[1] + p[2] * p[2] + p[3] * p[3];
  const double n2 = fma(p[0], p[0], r2);
  if (n2 < 1e-280) return false;                           // |p| = 0: the update is skipped (C-9)
  const double rinv = (r2 < 1e-280) ? 0.0 : rsqrt_newton<true>(r2);   // g = +-1: z is real, v part 0
  const double ninv = rsqrt_newton<true>(n2);
  const double zr = p[0] * ninv - 1.0;                     // cos a - 1
  const double zi = r2 * rinv * ninv;                      // sin a
  double wr = 0.0, wi = 0.0;
#pragma unroll
  for (int n = kMaxSeriesOrder; n >= 0; --n)
    if (n <= pw.order) {                                   // warp-uniform; b[n] is a compile-time slot
      const double tr = fma(wr, zr, fma(-wi, zi, pw.b[n]));
      wi = fma(wr, zi, wi * zr);
      wr = tr;
    }
  const double winv = rsqrt_newton<true>(fma(wr, wr, wi * wi));
  const double f = -wi * winv * rinv;                      // v/|v| = -pv/|pv|
  q[0] = wr * winv; q[1] = p[1] * f; q[2] = p[2] * f; q[3] = p[3] * f;
  return true;
}

// q = g^2 for g = conj(p)/|p|:  (c, v)^2 = (c^2 - v.v, 2 c v)  =  (p0^2 - pv.pv, -2 p0 pv)/|p|^2.
template <bool FULL>
__device__ __forceinline__ bool su2_update_power(const double* p, const MicroPower&, double* q) {
  const double r2 = p[1] * p[1] + p[2] * p[2] + p[3] * p[3];
  const double n2 = fma(p[0], p[0], r2);
  if (n2 < 1e-280) return false;                           // |p| = 0: the update is skipped (C-9)
  const double ninv = rsqrt_newton<true>(n2);
  const double c = p[0] * ninv;
  const double f = -2.0 * c * ninv;
  q[0] = fma(c, c, -(r2 * ninv) * ninv);
  q[1] = p[1] * f; q[2] = p[2] * f; q[3] = p[3] * f;
  return true;
}

// Uniform entry used by the solvers: (site, subgroup) select the random numbers of the heat bath
// and are ignored by the deterministic powers.
template <bool FULL>
__device__ __forceinline__ bool su2_update_at(const double* p, double omega, double* q, uint32_t, uint32_t) {
  return su2_update_power<FULL>(p, omega, q);
}
template <bool FULL>
__device__ __forceinline__ bool su2_update_at(const double* p, const ExactPower& pw, double* q, uint32_t, uint32_t) {
  return su2_update_power<FULL>(p, pw.omega, q);
}
template <bool FULL>
__device__ __forceinline__ bool su2_update_at(const double* p, const SeriesPower& pw, double* q, uint32_t, uint32_t) {
  return su2_update_power<FULL>(p, pw, q);
}
template <bool FULL>
__device__ __forceinline__ bool su2_update_at(const double* p, const MicroPower& pw, double* q, uint32_t, uint32_t) {
  return su2_update_power<FULL>(p, pw, q);
}
template <bool FULL>
__device__ __forceinline__ bool su2_update_at(const double* p, const HeatBathPower& pw, double* q, uint32_t site,
                                              uint32_t sub) {
  return su2_heatbath(p, pw, site, sub, q);
}

}  // namespace culgt
