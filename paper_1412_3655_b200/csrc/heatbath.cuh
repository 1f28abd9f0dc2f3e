// heatbath.cuh -- simulated annealing: the site's gauge transformation sampled from the Boltzmann
// weight exp(Re tr[g K(x)]/T) instead of maximising it (PAPER.md L7, L11 name simulated annealing;
// DESIGN.md reading C-25).  Per SU(2) subgroup with quaternion p:  h = q * p/|p| has
// h_0 ~ sqrt(1 - h_0^2) exp(a h_0), a = |p|/T, vector part uniform on S^2;  q = h * conj(p)/|p|.
// h_0 by the Kennedy-Pendleton method for a >= 2 and by Creutz's for a < 2; random numbers from the counter-based Philox4x32-10
// generator with counter (canonical site, half-sweep counter, subgroup | draw << 8, 0) and the
// 64-bit seed as key, so a site's numbers do not depend on the thread mapping.
//
// Included from su2_power.cuh (after its Taylor coefficient tables kSinCoef / kCosCoef and rsqrt_newton).
// The transcendental functions of the sampler are bounded-range, branch-free versions: their arguments
// are uniforms u = (w + 1/2) 2^-32 or lie in (e^-4, 1], so none of libm's special cases can occur, and a
// rejection loop that the whole warp repeats until its slowest lane accepts should carry no slow path.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace culgt {

struct HeatBathPower {
  double inv_T;
  uint32_t seed_lo, seed_hi;
  uint32_t counter;          // half-sweep counter: must differ between the half-sweeps of a run
};

__device__ __forceinline__ void philox4x32_10(uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3,
                                              uint32_t k0, uint32_t k1, uint32_t* out) {
#pragma unroll
  for (int r = 0; r < 10; ++r) {
    const uint32_t hi0 = __umulhi(0xD2511F53u, c0), lo0 = 0xD2511F53u * c0;
    const uint32_t hi1 = __umulhi(0xCD9E8D57u, c2), lo1 = 0xCD9E8D57u * c2;
    const uint32_t n0 = hi1 ^ c1 ^ k0, n2 = hi0 ^ c3 ^ k1;
    c0 = n0; c1 = lo1; c2 = n2; c3 = lo0;
    k0 += 0x9E3779B9u;
    k1 += 0xBB67AE85u;
  }
  out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

// four uniforms in (0,1), u_i = (w_i + 1/2) 2^-32, from the block with draw index `draw`.  The
// 32-bit word is widened exactly by the 2^52 exponent trick (an FP64 add instead of a conversion
// on the slow XU pipe).
__device__ __forceinline__ void heatbath_uniforms(const HeatBathPower& pw, uint32_t site, uint32_t sub,
                                                  uint32_t draw, double* u) {
  uint32_t w[4];
  philox4x32_10(site, pw.counter, sub | (draw << 8), 0u, pw.seed_lo, pw.seed_hi, w);
#pragma unroll
  for (int i = 0; i < 4; ++i)
    u[i] = (__hiloint2double(0x43300000, (int)w[i]) - 4503599627370496.0 + 0.5) * (1.0 / 4294967296.0);
}

// log(x) for a normal positive x (here 2^-33 < x <= 1), to ~1e-16 relative: x = 2^e m, m in [sqrt(1/2), sqrt(2)),
// log m = 2 atanh(s), s = (m-1)/(m+1), |s| <= 0.1716, by its odd series up to s^23/23; the division by a
// MUFU reciprocal seed, two Newton steps and one residual correction.
__device__ __forceinline__ double log_bounded(double x) {
  int hi = __double2hiint(x);
  const int lo = __double2loint(x);
  int e = (hi >> 20) - 1023;
  hi = (hi & 0x000FFFFF) | 0x3FF00000;
  double m = __hiloint2double(hi, lo);                  // [1, 2)
  const bool big = m > 1.4142135623730951;
  m = big ? 0.5 * m : m;
  e = big ? e + 1 : e;
  const double num = m - 1.0, den = m + 1.0;
  double r;
  asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(r) : "d"(den));
  r = fma(r, fma(-den, r, 1.0), r);
  r = fma(r, fma(-den, r, 1.0), r);
  double s = num * r;
  s = fma(r, fma(-s, den, num), s);
  const double z = s * s;
  double p = 2.0 / 23.0;
  p = fma(p, z, 2.0 / 21.0);
  p = fma(p, z, 2.0 / 19.0);
  p = fma(p, z, 2.0 / 17.0);
  p = fma(p, z, 2.0 / 15.0);
  p = fma(p, z, 2.0 / 13.0);
  p = fma(p, z, 2.0 / 11.0);
  p = fma(p, z, 2.0 / 9.0);
  p = fma(p, z, 2.0 / 7.0);
  p = fma(p, z, 2.0 / 5.0);
  p = fma(p, z, 2.0 / 3.0);
  const double lm = fma(s * z, p, 2.0 * s);
  const double ed = (double)e;
  return fma(ed, 6.93147180369123816490e-01, fma(ed, 1.90821492927058770002e-10, lm));   // ln 2 = hi + lo
}

// sin and cos of 2 pi u for 0 < u < 1: k = rint(4u), y = u - k/4 exactly, Taylor series in 2 pi y on
// [-pi/4, pi/4] (the tables of su2_power.cuh, full length), quadrant by k.
__device__ __forceinline__ void sincos_2pi(double u, double* s, double* c) {
  const double magic = 6755399441055744.0;              // 1.5 * 2^52: rint without FRND / F2I
  const double kb = fma(u, 4.0, magic);
  const int q = __double2loint(kb);
  const double k = kb - magic;
  const double y = fma(-0.25, k, u) * 6.28318530717958647693;
  const double z = y * y;
  double ps = kSinCoef[8];
#pragma unroll
  for (int i = 7; i >= 0; --i) ps = fma(ps, z, kSinCoef[i]);
  const double sy = fma(ps * z, y, y);
  double pc = kCosCoef[9];
#pragma unroll
  for (int i = 8; i >= 0; --i) pc = fma(pc, z, kCosCoef[i]);
  const double cy = fma(pc, z, 1.0);
  const double a = (q & 1) ? cy : sy;
  const double b = (q & 1) ? sy : cy;
  *s = (q & 2) ? -a : a;
  *c = ((q + 1) & 2) ? -b : b;
}

// sqrt(x) for 0 <= x <= 1 without the libm slow path (x below 1e-280 -> 0)
__device__ __forceinline__ double sqrt_unit(double x) { return x > 1e-280 ? x * rsqrt_newton<true>(x) : 0.0; }

// q sampled for the un-normalised subgroup quaternion p; false when p == 0 (no update, C-9).
__device__ __forceinline__ bool su2_heatbath(const double* p, const HeatBathPower& pw, uint32_t site,
                                             uint32_t sub, double* q) {
  const double n2 = p[0] * p[0] + p[1] * p[1] + p[2] * p[2] + p[3] * p[3];
  if (!(n2 > 0.0) || !(n2 < 1e300)) return false;      // p = 0 (C-9); also keeps NaN/Inf out of the loop
  const double rinv = rsqrt_newton<true>(n2);
  const double n = n2 * rinv;
  const double a = n * pw.inv_T;
  uint32_t draw = 0;
  double h0;
  if (a < 2.0) {
    // Creutz's method where Kennedy-Pendleton would accept with probability ~a^{3/2}
    const double emin = exp(-2.0 * a);
    const double inv_a = 1.0 / a;
    for (;;) {
      if (draw >= (1u << 22)) { h0 = 1.0; break; }       // unreachable; never spin forever
      double u[4];
      heatbath_uniforms(pw, site, sub, draw, u);
      draw += 1;
      h0 = fma(log_bounded(emin + u[0] * (1.0 - emin)), inv_a, 1.0);
      if (u[1] * u[1] <= 1.0 - h0 * h0) break;
    }
  } else {
    double lam2;
    const double m_inv_2a = -0.5 / a;
    for (;;) {
      if (draw >= (1u << 22)) { lam2 = 0.0; break; }     // unreachable for finite a; never spin forever
      double u[4];
      heatbath_uniforms(pw, site, sub, draw, u);         // r1, r2, r3, r4: one block per trial
      draw += 1;
      double sn, c;
      sincos_2pi(u[1], &sn, &c);
      lam2 = fma(c * c, log_bounded(u[2]), log_bounded(u[0])) * m_inv_2a;
      if (u[3] * u[3] <= 1.0 - lam2) break;
    }
    h0 = 1.0 - 2.0 * lam2;
  }
  double ud[4];
  heatbath_uniforms(pw, site, sub, draw, ud);
  const double u0 = ud[0], u1 = ud[1];
  const double ct = 2.0 * u0 - 1.0;
  const double st = sqrt_unit(fma(-ct, ct, 1.0));
  double sp, cp;
  sincos_2pi(u1, &sp, &cp);
  const double r = sqrt_unit(fma(-h0, h0, 1.0));
  const double h[4] = {h0, r * st * cp, r * st * sp, r * ct};
  const double b[4] = {p[0] * rinv, -p[1] * rinv, -p[2] * rinv, -p[3] * rinv};
  q[0] = h[0] * b[0] - h[1] * b[1] - h[2] * b[2] - h[3] * b[3];
  q[1] = h[0] * b[1] + b[0] * h[1] - (h[2] * b[3] - h[3] * b[2]);
  q[2] = h[0] * b[2] + b[0] * h[2] - (h[3] * b[1] - h[1] * b[3]);
  q[3] = h[0] * b[3] + b[0] * h[3] - (h[1] * b[2] - h[2] * b[1]);
  return true;
}

}  // namespace culgt
