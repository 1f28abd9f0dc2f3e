// su_math.cuh -- register-level SU(3)/SU(2) arithmetic for the sweep kernels.
//
// A 3x3 complex matrix is T m[18], row-major, re/im interleaved: m[2*(3*r+c)] + i m[2*(3*r+c)+1].
// An SU(2) element is the quaternion (a0,a1,a2,a3) <-> [[a0+i a3, a2+i a1],[-a2+i a1, a0-i a3]]
// (reading C-7).  Everything is fully unrolled so that matrices live in registers.
#pragma once
#include <cuda_runtime.h>
#include <math.h>

namespace culgt {

#define CULGT_RE(r, c) (2 * (3 * (r) + (c)))
#define CULGT_IM(r, c) (2 * (3 * (r) + (c)) + 1)

__device__ __forceinline__ float fma_t(float a, float b, float c) { return fmaf(a, b, c); }
__device__ __forceinline__ double fma_t(double a, double b, double c) { return fma(a, b, c); }

// acc += x * y (complex), written as four fused multiply-adds so that no separate add is issued.
template <typename T>
__device__ __forceinline__ void cmac(T& accr, T& acci, T xr, T xi, T yr, T yi) {
  accr = fma_t(xr, yr, accr);
  accr = fma_t(-xi, yi, accr);
  acci = fma_t(xr, yi, acci);
  acci = fma_t(xi, yr, acci);
}
// acc += x * conj(y)
template <typename T>
__device__ __forceinline__ void cmac_conj(T& accr, T& acci, T xr, T xi, T yr, T yi) {
  accr = fma_t(xr, yr, accr);
  accr = fma_t(xi, yi, accr);
  acci = fma_t(xi, yr, acci);
  acci = fma_t(-xr, yi, acci);
}

// Third row of an SU(3) matrix from its first two: row2 = conj(row0 x row1)
// ("reconstruct the full matrix in registers", L118).
template <typename T>
__device__ __forceinline__ void reconstruct_row2(T* m) {
#pragma unroll
  for (int c = 0; c < 3; ++c) {
    const int a = (c + 1) % 3, b = (c + 2) % 3;
    // row0[a]*row1[b] - row0[b]*row1[a], then conjugated
    T re = m[CULGT_RE(0, a)] * m[CULGT_RE(1, b)];
    T im = m[CULGT_RE(0, a)] * m[CULGT_IM(1, b)];
    re = fma_t(-m[CULGT_IM(0, a)], m[CULGT_IM(1, b)], re);
    im = fma_t(m[CULGT_IM(0, a)], m[CULGT_RE(1, b)], im);
    re = fma_t(-m[CULGT_RE(0, b)], m[CULGT_RE(1, a)], re);
    im = fma_t(-m[CULGT_RE(0, b)], m[CULGT_IM(1, a)], im);
    re = fma_t(m[CULGT_IM(0, b)], m[CULGT_IM(1, a)], re);
    im = fma_t(-m[CULGT_IM(0, b)], m[CULGT_RE(1, a)], im);
    m[CULGT_RE(2, c)] = re;
    m[CULGT_IM(2, c)] = -im;
  }
}

// C(rows 0..NR-1) = A * B, 3x3 complex.
template <int NR, typename T>
__device__ __forceinline__ void mul_ab(const T* A, const T* B, T* C) {
#pragma unroll
  for (int r = 0; r < NR; ++r)
#pragma unroll
    for (int c = 0; c < 3; ++c) {
      T re = A[CULGT_RE(r, 0)] * B[CULGT_RE(0, c)];
      T im = A[CULGT_RE(r, 0)] * B[CULGT_IM(0, c)];
      re = fma_t(-A[CULGT_IM(r, 0)], B[CULGT_IM(0, c)], re);
      im = fma_t(A[CULGT_IM(r, 0)], B[CULGT_RE(0, c)], im);
#pragma unroll
      for (int k = 1; k < 3; ++k)
        cmac(re, im, A[CULGT_RE(r, k)], A[CULGT_IM(r, k)], B[CULGT_RE(k, c)], B[CULGT_IM(k, c)]);
      C[CULGT_RE(r, c)] = re;
      C[CULGT_IM(r, c)] = im;
    }
}

// C(rows 0..NR-1) = A * B^dagger.
template <int NR, typename T>
__device__ __forceinline__ void mul_abd(const T* A, const T* B, T* C) {
#pragma unroll
  for (int r = 0; r < NR; ++r)
#pragma unroll
    for (int c = 0; c < 3; ++c) {
      // sum_k A[r][k] * conj(B[c][k])
      T re = A[CULGT_RE(r, 0)] * B[CULGT_RE(c, 0)];
      T im = A[CULGT_IM(r, 0)] * B[CULGT_RE(c, 0)];
      re = fma_t(A[CULGT_IM(r, 0)], B[CULGT_IM(c, 0)], re);
      im = fma_t(-A[CULGT_RE(r, 0)], B[CULGT_IM(c, 0)], im);
#pragma unroll
      for (int k = 1; k < 3; ++k)
        cmac_conj(re, im, A[CULGT_RE(r, k)], A[CULGT_IM(r, k)], B[CULGT_RE(c, k)], B[CULGT_IM(c, k)]);
      C[CULGT_RE(r, c)] = re;
      C[CULGT_IM(r, c)] = im;
    }
}

// K += U (dagger = false) or K += U^dagger (dagger = true); U of type TU, K of type TK.
template <typename TK, typename TU>
__device__ __forceinline__ void accumulate(TK* K, const TU* U, bool dagger) {
  if (!dagger) {
#pragma unroll
    for (int i = 0; i < 18; ++i) K[i] += (TK)U[i];
  } else {
#pragma unroll
    for (int r = 0; r < 3; ++r)
#pragma unroll
      for (int c = 0; c < 3; ++c) {
        K[CULGT_RE(r, c)] += (TK)U[CULGT_RE(c, r)];
        K[CULGT_IM(r, c)] -= (TK)U[CULGT_IM(c, r)];
      }
  }
}

__device__ __forceinline__ void sincos_t(double x, double* s, double* c) { sincos(x, s, c); }
__device__ __forceinline__ void sincos_t(float x, float* s, float* c) { sincosf(x, s, c); }
__device__ __forceinline__ double atan2_t(double y, double x) { return atan2(y, x); }
__device__ __forceinline__ float atan2_t(float y, float x) { return atan2f(y, x); }
__device__ __forceinline__ double rsqrt_t(double x) { return rsqrt(x); }
__device__ __forceinline__ float rsqrt_t(float x) { return rsqrtf(x); }
__device__ __forceinline__ double sqrt_t(double x) { return sqrt(x); }
__device__ __forceinline__ float sqrt_t(float x) { return sqrtf(x); }
template <typename T> struct Tiny;
template <> struct Tiny<double> { static __device__ __forceinline__ double r2() { return 1e-300; } };
template <> struct Tiny<float> { static __device__ __forceinline__ float r2() { return 1e-36f; } };

// Exact group power q <- q^omega of a unit quaternion on the principal branch (reading C-8 of
// PAPER.md L54 "replacing g(x) by g^omega(x)"): q = cos(alpha) + i sin(alpha) n.sigma,
// alpha = atan2(|v|, c) in [0, pi]  ->  cos(omega alpha) + i sin(omega alpha) n.sigma.
template <typename T>
__device__ __forceinline__ void su2_pow(T* q, T omega) {
  const T r2 = q[1] * q[1] + q[2] * q[2] + q[3] * q[3];
  if (r2 < Tiny<T>::r2()) {
    if (q[0] > 0) { q[0] = 1; q[1] = 0; q[2] = 0; q[3] = 0; }
    else {
      T s, c;
      sincos_t(omega * (T)3.14159265358979323846, &s, &c);
      q[0] = c; q[1] = 0; q[2] = 0; q[3] = s;
    }
    return;
  }
  const T rinv = rsqrt_t(r2);
  const T alpha = atan2_t(r2 * rinv, q[0]);
  T s, c;
  sincos_t(omega * alpha, &s, &c);
  const T f = s * rinv;
  q[0] = c; q[1] *= f; q[2] *= f; q[3] *= f;
}

// One SU(2)-subgroup step (I,J) of the SU(3) site update (C-6, C-9, C-10):
// p = real-quaternion part (x2) of the (I,J) block of K, g = conj(p)/|p|, q = g^omega,
// K <- g_s K, G <- g_s G with g_s = q embedded in rows/cols I,J.
template <int I, int J, typename T>
__device__ __forceinline__ void subgroup_step(T* K, T* G, T omega) {
  T q[4];
  q[0] = K[CULGT_RE(I, I)] + K[CULGT_RE(J, J)];
  q[1] = -(K[CULGT_IM(I, J)] + K[CULGT_IM(J, I)]);
  q[2] = -(K[CULGT_RE(I, J)] - K[CULGT_RE(J, I)]);
  q[3] = -(K[CULGT_IM(I, I)] - K[CULGT_IM(J, J)]);
  const T n2 = q[0] * q[0] + q[1] * q[1] + q[2] * q[2] + q[3] * q[3];
  if (n2 == 0) return;
  const T ninv = rsqrt_t(n2);
  q[0] *= ninv; q[1] *= ninv; q[2] *= ninv; q[3] *= ninv;
  su2_pow(q, omega);
  // g_s[I][I] = a = q0 + i q3, g_s[I][J] = b = q2 + i q1, g_s[J][I] = -conj(b), g_s[J][J] = conj(a)
  const T ar = q[0], ai = q[3], br = q[2], bi = q[1];
#pragma unroll
  for (int m = 0; m < 2; ++m) {
    T* M = m ? G : K;
#pragma unroll
    for (int c = 0; c < 3; ++c) {
      const T xr = M[CULGT_RE(I, c)], xi = M[CULGT_IM(I, c)];
      const T yr = M[CULGT_RE(J, c)], yi = M[CULGT_IM(J, c)];
      M[CULGT_RE(I, c)] = ar * xr - ai * xi + br * yr - bi * yi;
      M[CULGT_IM(I, c)] = ar * xi + ai * xr + br * yi + bi * yr;
      M[CULGT_RE(J, c)] = -br * xr - bi * xi + ar * yr + ai * yi;
      M[CULGT_IM(J, c)] = -br * xi + bi * xr + ar * yi - ai * yr;
    }
  }
}

// G(x) from K(x) for SU(3): the three subgroups (0,1),(0,2),(1,2), one pass (C-6).
template <typename T>
__device__ __forceinline__ void su3_site_G(T* K, T* G, T omega) {
#pragma unroll
  for (int i = 0; i < 18; ++i) G[i] = 0;
  G[CULGT_RE(0, 0)] = 1; G[CULGT_RE(1, 1)] = 1; G[CULGT_RE(2, 2)] = 1;
  subgroup_step<0, 1>(K, G, omega);
  subgroup_step<0, 2>(K, G, omega);
  subgroup_step<1, 2>(K, G, omega);
}

// ---- SU(2) quaternion helpers ---------------------------------------------------------------
// (ab)_0 = a0 b0 - a.b ;  (ab)_vec = a0 b + b0 a - a x b     (convention C-7)
template <typename T>
__device__ __forceinline__ void quat_mul(const T* a, const T* b, T* o) {
  o[0] = a[0] * b[0] - a[1] * b[1] - a[2] * b[2] - a[3] * b[3];
  o[1] = a[0] * b[1] + b[0] * a[1] - (a[2] * b[3] - a[3] * b[2]);
  o[2] = a[0] * b[2] + b[0] * a[2] - (a[3] * b[1] - a[1] * b[3]);
  o[3] = a[0] * b[3] + b[0] * a[3] - (a[1] * b[2] - a[2] * b[1]);
}
// o = a * b^dagger
template <typename T>
__device__ __forceinline__ void quat_mul_dag(const T* a, const T* b, T* o) {
  const T bd[4] = {b[0], -b[1], -b[2], -b[3]};
  quat_mul(a, bd, o);
}

}  // namespace culgt
