// su3_solve.cuh -- G(x) from K(x) for SU(3): the loop over the three SU(2) subgroups with the
// overrelaxation power (readings C-6, C-8, C-9, C-10), arranged for
// the B200 FP64 pipe.
//
// The chain K -> g_1 -> g_1 K -> g_2 -> g_2 g_1 K -> g_3 is ill-conditioned where a subgroup
// quaternion |p| is small (dg ~ dK |K|/|p|, reading C-15), so it runs in fp64 for every storage
// precision.  Only the entries of the rotated K that a later subgroup reads are updated:
//   after (0,1): row 0 (all columns) and row 1 columns 1,2     (40 DFMA instead of 48)
//   after (0,2): row 2 columns 1,2                             (16 instead of 48)
//   after (1,2): nothing                                       ( 0 instead of 48)
// The accumulated G = g_3 g_2 g_1 is formed in the type GT the caller asks for (the sweep kernels
// use double and round once to the storage precision).
#pragma once
#include "su_math.cuh"
#include "su2_power.cuh"

namespace culgt {

// p = real-quaternion part (x2) of the (I,J) block of K; q = (conj(p)/|p|)^omega.
template <int I, int J, bool FULL, typename Power>
__device__ __forceinline__ bool subgroup_quaternion(const double* K, const Power& omega, double* q, uint32_t site) {
  double p[4];
  p[0] = K[CULGT_RE(I, I)] + K[CULGT_RE(J, J)];
  p[1] = K[CULGT_IM(I, J)] + K[CULGT_IM(J, I)];
  p[2] = K[CULGT_RE(I, J)] - K[CULGT_RE(J, I)];
  p[3] = K[CULGT_IM(I, I)] - K[CULGT_IM(J, J)];
  return su2_update_at<FULL>(p, omega, q, site, (uint32_t)(I + J - 1));   // subgroups 0, 1, 2
}

// (x, y) <- (a x + b y, -conj(b) x + conj(a) y) for complex x = M[I][c], y = M[J][c];
// DO_I / DO_J select which of the two outputs are written.
template <bool DO_I, bool DO_J, typename T>
__device__ __forceinline__ void rotate_pair(T* xr_, T* xi_, T* yr_, T* yi_, T ar, T ai, T br, T bi) {
  const T xr = *xr_, xi = *xi_, yr = *yr_, yi = *yi_;
  if (DO_I) {
    *xr_ = ar * xr - ai * xi + br * yr - bi * yi;
    *xi_ = ar * xi + ai * xr + br * yi + bi * yr;
  }
  if (DO_J) {
    *yr_ = -br * xr - bi * xi + ar * yr + ai * yi;
    *yi_ = -br * xi + bi * xr + ar * yi - ai * yr;
  }
}

template <int I, int J, bool DO_I, bool DO_J, typename T>
__device__ __forceinline__ void rotate_col(T* M, int c, T ar, T ai, T br, T bi) {
  rotate_pair<DO_I, DO_J>(&M[CULGT_RE(I, c)], &M[CULGT_IM(I, c)], &M[CULGT_RE(J, c)], &M[CULGT_IM(J, c)],
                          ar, ai, br, bi);
}

// K (fp64, destroyed) -> G (type GT).  g_s embeds q = (c, v1, v2, v3) as
// [I][I] = a = c + i v3, [I][J] = b = v2 + i v1, [J][I] = -conj(b), [J][J] = conj(a)  (C-7).
// FULL selects full-length (fp64 storage) or shortened (fp32 storage) series in su2_power.cuh.
// Power = double (omega; exact power), ExactPower, SeriesPower (su2_power.cuh) or HeatBathPower
// (heatbath.cuh; `site` = canonical site index, selects its random numbers).
template <bool FULL, typename GT, typename Power>
__device__ __forceinline__ void su3_solve(double* K, GT* G, const Power& omega, uint32_t site = 0) {
  double q[4];
  // ---- subgroup (0,1)
  bool ok = subgroup_quaternion<0, 1, FULL>(K, omega, q, site);
  if (!ok) { q[0] = 1.0; q[1] = 0.0; q[2] = 0.0; q[3] = 0.0; }
  {
    const double ar = q[0], ai = q[3], br = q[2], bi = q[1];
    rotate_col<0, 1, true, false>(K, 0, ar, ai, br, bi);
    rotate_col<0, 1, true, true>(K, 1, ar, ai, br, bi);
    rotate_col<0, 1, true, true>(K, 2, ar, ai, br, bi);
  }
  // G = g_1
  const GT a1r = (GT)q[0], a1i = (GT)q[3], b1r = (GT)q[2], b1i = (GT)q[1];
  // ---- subgroup (0,2)
  ok = subgroup_quaternion<0, 2, FULL>(K, omega, q, site);
  if (!ok) { q[0] = 1.0; q[1] = 0.0; q[2] = 0.0; q[3] = 0.0; }
  {
    const double ar = q[0], ai = q[3], br = q[2], bi = q[1];
    rotate_col<0, 2, false, true>(K, 1, ar, ai, br, bi);
    rotate_col<0, 2, false, true>(K, 2, ar, ai, br, bi);
  }
  // G = g_2 g_1 with g_1 = [[a1, b1, 0], [-conj(b1), conj(a1), 0], [0, 0, 1]]:
  //   row0 = (a2 a1, a2 b1, b2), row1 = (-conj(b1), conj(a1), 0), row2 = (-conj(b2) a1, -conj(b2) b1, conj(a2))
  {
    const GT a2r = (GT)q[0], a2i = (GT)q[3], b2r = (GT)q[2], b2i = (GT)q[1];
    G[CULGT_RE(0, 0)] = a2r * a1r - a2i * a1i;  G[CULGT_IM(0, 0)] = a2r * a1i + a2i * a1r;
    G[CULGT_RE(0, 1)] = a2r * b1r - a2i * b1i;  G[CULGT_IM(0, 1)] = a2r * b1i + a2i * b1r;
    G[CULGT_RE(0, 2)] = b2r;                    G[CULGT_IM(0, 2)] = b2i;
    G[CULGT_RE(1, 0)] = -b1r;                   G[CULGT_IM(1, 0)] = b1i;
    G[CULGT_RE(1, 1)] = a1r;                    G[CULGT_IM(1, 1)] = -a1i;
    G[CULGT_RE(1, 2)] = 0;                      G[CULGT_IM(1, 2)] = 0;
    // -conj(b2) = (-b2r, +b2i)
    G[CULGT_RE(2, 0)] = -b2r * a1r - b2i * a1i; G[CULGT_IM(2, 0)] = -b2r * a1i + b2i * a1r;
    G[CULGT_RE(2, 1)] = -b2r * b1r - b2i * b1i; G[CULGT_IM(2, 1)] = -b2r * b1i + b2i * b1r;
    G[CULGT_RE(2, 2)] = a2r;                    G[CULGT_IM(2, 2)] = -a2i;
  }
  // ---- subgroup (1,2)
  ok = subgroup_quaternion<1, 2, FULL>(K, omega, q, site);
  if (ok) {
    const GT ar = (GT)q[0], ai = (GT)q[3], br = (GT)q[2], bi = (GT)q[1];
#pragma unroll
    for (int c = 0; c < 3; ++c) rotate_col<1, 2, true, true>(G, c, ar, ai, br, bi);
  }
}

}  // namespace culgt
