// transform.cu -- a9: U_mu(x) <- g(x) U_mu(x) g(x+mu)^dagger for a user-supplied field g
// (the paper's worked code example L105-118: local = gLeft*local*gRight.hermitian()).
// g is a canonical site-major field real[V][Nc][Nc][2]; links are the internal layout, in place.
#include "lattice.cuh"
#include "su_math.cuh"
#include "kernels.h"

namespace culgt {

// The 18 reals of g at canonical site s as 9 two-element vector loads (a site is 72 / 144 bytes:
// 8- / 16-byte aligned), half the load instructions of scalar reads on a thread-strided field.
__device__ __forceinline__ void load_g3(const float* gf, int64_t s, float* out) {
  const float2* p = reinterpret_cast<const float2*>(gf + s * 18);
#pragma unroll
  for (int i = 0; i < 9; ++i) {
    const float2 v = __ldg(p + i);
    out[2 * i] = v.x;
    out[2 * i + 1] = v.y;
  }
}
__device__ __forceinline__ void load_g3(const double* gf, int64_t s, double* out) {
  const double2* p = reinterpret_cast<const double2*>(gf + s * 18);
#pragma unroll
  for (int i = 0; i < 9; ++i) {
    const double2 v = __ldg(p + i);
    out[2 * i] = v.x;
    out[2 * i + 1] = v.y;
  }
}

template <typename S, int BLOCK>
__global__ void __launch_bounds__(BLOCK)
gauge_transform_kernel(typename S::Vec* __restrict__ links, const typename S::Real* __restrict__ gf, const Geom g) {
  typedef typename S::Real Real;
  // a CTA handles BLOCK/2 half indices of BOTH parities (threads 0..BLOCK/2-1 black, the rest white):
  // together they are 2*(BLOCK/2) consecutive canonical sites, so the two halves of every cache line of
  // the site-major g field are consumed by the same CTA
  constexpr int HALF = BLOCK / 2;
  const int parity = threadIdx.x >= HALF;
  const long long t = (long long)blockIdx.x * HALF + (threadIdx.x - parity * HALF);
  if (t >= g.vh) return;
  const int h = (int)t;
  const SiteCoord sc = decode_site(g, h, parity);
  const int64_t s = canonical_site(g, h, sc);
  if (S::NC == 3) {
    Real gx[18];
    load_g3(gf, s, gx);
#pragma unroll
    for (int mu = 0; mu < 4; ++mu) {
      // forward neighbour x+mu lives in the other parity; its canonical site is 2*h' + odd'
      const int hu = up_index(g, h, sc, mu);
      const int64_t su = 2 * (int64_t)hu + (1 - sc.odd) * (mu == 0) + sc.odd * (mu != 0);
      Real gu[18], U[kLinkRegs], T[18], R[kLinkRegs];
      R[18] = 0; R[19] = 0;
      load_g3(gf, su, gu);
      typename S::Vec* p = link_base<S>(links, g, parity, mu, h);
      load_params<S>(p, g.pitch, U);
      if (S::NP == 12) reconstruct_row2(U);
      mul_ab<3>(gx, U, T);
      constexpr int NR = (S::NP == 12) ? 2 : 3;
      mul_abd<NR>(T, gu, R);
      store_params<S>(p, g.pitch, R);
    }
  } else {
    // SU(2): canonical 2x2 -> quaternion (a0,a1,a2,a3) = (Re g00, Im g01, Re g01, Im g00)
    Real gx[4] = {gf[s * 8 + 0], gf[s * 8 + 3], gf[s * 8 + 2], gf[s * 8 + 1]};
#pragma unroll
    for (int mu = 0; mu < 4; ++mu) {
      const int hu = up_index(g, h, sc, mu);
      const int64_t su = 2 * (int64_t)hu + (1 - sc.odd) * (mu == 0) + sc.odd * (mu != 0);
      Real gu[4] = {gf[su * 8 + 0], gf[su * 8 + 3], gf[su * 8 + 2], gf[su * 8 + 1]};
      Real U[4], T[4], R[4];
      typename S::Vec* p = link_base<S>(links, g, parity, mu, h);
      load_params<S>(p, g.pitch, U);
      quat_mul(gx, U, T);
      quat_mul_dag(T, gu, R);
      store_params<S>(p, g.pitch, R);
    }
  }
}

template <typename S>
static cudaError_t run_transform(const LatticeDesc& d, void* links, const void* gfield, cudaStream_t st) {
  constexpr int BLOCK = 128;
  dim3 grid((unsigned)((d.geom.vh + BLOCK / 2 - 1) / (BLOCK / 2)));
  gauge_transform_kernel<S, BLOCK><<<grid, BLOCK, 0, st>>>((typename S::Vec*)links,
                                                            (const typename S::Real*)gfield, d.geom);
  return cudaGetLastError();
}

cudaError_t launch_gauge_transform(const LatticeDesc& d, void* links, const void* g, cudaStream_t st) {
  if (d.group == 2) {
    if (d.precision == 32) return run_transform<Storage<float, 2, 4> >(d, links, g, st);
    return run_transform<Storage<double, 2, 4> >(d, links, g, st);
  }
  if (d.precision == 32) {
    if (d.params == 12) return run_transform<Storage<float, 3, 12> >(d, links, g, st);
    return run_transform<Storage<float, 3, 18> >(d, links, g, st);
  }
  if (d.params == 12) return run_transform<Storage<double, 3, 12> >(d, links, g, st);
  return run_transform<Storage<double, 3, 18> >(d, links, g, st);
}

}  // namespace culgt
