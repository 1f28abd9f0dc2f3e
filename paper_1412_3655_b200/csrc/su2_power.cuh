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
//   a~ = atan2f(|pv|, p0) in fp32 (error <= ~1e-6), widened exactly to fp64;
//   (s~, c~) = sincos(a~) by the fp64 polynomials below;
//   d = sin(a - a~) = (|pv| c~ - p0 s~)/|p|  exactly;  a = a~ + d + d^3/6   (|d|^5 < 1e-30).
// The two sincos evaluations (of a~ and of omega*a~) are independent, which gives the FP64 pipe
// four independent Horner chains; omega*a = omega*a~ + omega*(d + d^3/6) is folded in by the angle-addition
// formulas with the tiny second angle expanded to second order.
#pragma once
#include <cuda_runtime.h>
#include <math.h>

namespace culgt {

// sin and cos of x for 0 <= x <= ~7 (omega*a < 2*pi): Cody-Waite reduction by pi/2 (k <= 4, so two
// constants suffice) and Taylor polynomials on [-pi/4, pi/4] truncated below 1e-17.
__device__ __forceinline__ void sincos_bounded(double x, double* s, double* c) {
  const double k = rint(x * 0.63661977236758134308);            // 2/pi
  double y = fma(-k, 1.57079632679489655800e+00, x);            // pi/2 high part
  y = fma(-k, 6.12323399573676603587e-17, y);                   // pi/2 low part
  const double z = y * y;
  double ps = -8.22063524662432971696e-18;                      // -1/19!
  ps = fma(ps, z, 2.81145725434552076320e-15);                  // 1/17!
  ps = fma(ps, z, -7.64716373181981647590e-13);                 // -1/15!
  ps = fma(ps, z, 1.60590438368216145994e-10);                  // 1/13!
  ps = fma(ps, z, -2.50521083854417187751e-08);                 // -1/11!
  ps = fma(ps, z, 2.75573192239858906526e-06);                  // 1/9!
  ps = fma(ps, z, -1.98412698412698412698e-04);                 // -1/7!
  ps = fma(ps, z, 8.33333333333333333333e-03);                  // 1/5!
  ps = fma(ps, z, -1.66666666666666666667e-01);                 // -1/3!
  const double sy = fma(ps * z, y, y);
  double pc = 4.11031762331216485848e-19;                       // 1/20!
  pc = fma(pc, z, -1.56192069685862264622e-16);                 // -1/18!
  pc = fma(pc, z, 4.77947733238738529744e-14);                  // 1/16!
  pc = fma(pc, z, -1.14707455977297247139e-11);                 // -1/14!
  pc = fma(pc, z, 2.08767569878680989792e-09);                  // 1/12!
  pc = fma(pc, z, -2.75573192239858906526e-07);                 // -1/10!
  pc = fma(pc, z, 2.48015873015873015873e-05);                  // 1/8!
  pc = fma(pc, z, -1.38888888888888888889e-03);                 // -1/6!
  pc = fma(pc, z, 4.16666666666666666667e-02);                  // 1/4!
  pc = fma(pc, z, -0.5);
  const double cy = fma(pc, z, 1.0);
  const int q = (int)k & 3;
  const double a = (q & 1) ? cy : sy;                           // |sin x|-carrier
  const double b = (q & 1) ? sy : cy;
  *s = (q & 2) ? -a : a;
  *c = ((q + 1) & 2) ? -b : b;
}

// q_out = (conj(p)/|p|)^omega for the un-normalised quaternion p = (p[0]; p[1], p[2], p[3]).
// Returns false (q_out untouched) when p == 0, where the update is skipped (reading C-9).
__device__ __forceinline__ bool su2_update_power(const double* p, double omega, double* q) {
  const double r2 = p[1] * p[1] + p[2] * p[2] + p[3] * p[3];
  const double n2 = fma(p[0], p[0], r2);
  if (n2 == 0.0) return false;
  if (r2 < 1e-300) {                 // g = +1 or -1: axis undefined (C-8: z axis by fiat for g = -1)
    double s = 0.0, c = 1.0;
    if (p[0] < 0.0) sincos_bounded(omega * 3.14159265358979323846, &s, &c);
    q[0] = c; q[1] = 0.0; q[2] = 0.0; q[3] = s;
    return true;
  }
  const double rinv = rsqrt(r2);     // 1/|pv|
  const double ninv = rsqrt(n2);     // 1/|p|
  const double R = r2 * rinv;        // |pv|
  const double a0 = (double)atan2f((float)R, (float)p[0]);
  double s0, c0, s1, c1;
  sincos_bounded(a0, &s0, &c0);
  sincos_bounded(omega * a0, &s1, &c1);
  double d = (R * c0 - p[0] * s0) * ninv;          // sin(a - a0)
  d = fma(d * d * d, 1.0 / 6.0, d);                // a - a0
  const double e = omega * d;                      // omega a - omega a0, |e| < 1e-5
  const double ce = fma(-0.5 * e, e, 1.0);
  const double se = fma(e * e * e, -1.0 / 6.0, e);
  const double C = c1 * ce - s1 * se;
  const double S = s1 * ce + c1 * se;
  const double f = -S * rinv;
  q[0] = C; q[1] = p[1] * f; q[2] = p[2] * f; q[3] = p[3] * f;
  return true;
}

}  // namespace culgt
