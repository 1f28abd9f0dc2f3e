// or_sweep.cu -- half-sweep dispatch (launch_or_sweep and friends), the SU(2) kernel, and the first
// generation of SU(3) kernels that keep all links in registers (variants 1-14, the measured
// alternatives of DESIGN.md 6.1).  The production SU(3) kernel is in or_sweep_staged.cu.
// (SURVEY.md 8(a) rows a1-a6.)
//
// For every site x of one parity:
//   gather the 8 links touching x, K = sum_mu U_mu(x) + U_mu(x-mu)^dagger      (eq. 3)
//   G from K by the SU(2) closed form / the SU(3) subgroup loop with g^omega   (L50-54)
//   U_mu(x) <- G U_mu(x),  U_mu(x-mu) <- U_mu(x-mu) G^dagger                   (L19-21, L48)
// Sites of one parity are independent (L54), so there is no synchronisation inside a launch.
//
// Thread-to-site mapping (the paper's 1 / 4 / 8 threads per site, L62-72, L122) is the template
// parameter TPS: each of the TPS cooperating lanes owns 8/TPS links, the partial K are summed by
// xor-shuffles (the warp-level analogue of the paper's shared-memory exchange) and every lane
// then holds the same K and computes the same G.  Which TPS each storage uses is chosen by
// measurement (profiles/).
#include "lattice.cuh"
#include "su_math.cuh"
#include "su2_power.cuh"
#include "kernels.h"

namespace culgt {

template <typename T>
__device__ __forceinline__ T shfl_xor_t(T v, int mask);
template <>
__device__ __forceinline__ float shfl_xor_t<float>(float v, int mask) { return __shfl_xor_sync(0xffffffffu, v, mask); }
template <>
__device__ __forceinline__ double shfl_xor_t<double>(double v, int mask) { return __shfl_xor_sync(0xffffffffu, v, mask); }

// ---------------------------------------------------------------------------------------------
// SU(3).  S = storage traits, Acc = type of K and of the subgroup solve, TPS threads per site.
// ---------------------------------------------------------------------------------------------
template <typename S, typename Acc, int TPS, int BLOCK>
__global__ void __launch_bounds__(BLOCK)
or_sweep_su3_kernel(typename S::Vec* __restrict__ links, const Geom g, const int parity, const Acc omega) {
  typedef typename S::Real Real;
  constexpr int LPT = 8 / TPS;   // links per thread
  const int tid = blockIdx.x * BLOCK + threadIdx.x;
  int h = tid / TPS;
  const int q = tid % TPS;
  const bool active = h < g.vh;
  if (!active) h = g.vh - 1;     // keep the lane alive for the shuffles; it stores nothing
  const SiteCoord sc = decode_site(g, h, parity);

  Real U[LPT][kLinkRegs];
  typename S::Vec* ptr[LPT];
#pragma unroll
  for (int l = 0; l < LPT; ++l) {
    const int slot = q * LPT + l;          // slot = 2*mu + (0: U_mu(x), 1: U_mu(x-mu))
    const int mu = slot >> 1;
    const bool dn = slot & 1;
    const int idx = dn ? down_index(g, h, sc, mu) : h;
    ptr[l] = link_base<S>(links, g, dn ? 1 - parity : parity, mu, idx);
  }
#pragma unroll
  for (int l = 0; l < LPT; ++l) load_params<S>(ptr[l], g.vh, U[l]);
  if (S::NP == 12) {
#pragma unroll
    for (int l = 0; l < LPT; ++l) reconstruct_row2(U[l]);
  }

  Acc K[18];
#pragma unroll
  for (int i = 0; i < 18; ++i) K[i] = 0;
#pragma unroll
  for (int l = 0; l < LPT; ++l) accumulate(K, U[l], ((q * LPT + l) & 1) != 0);
#pragma unroll
  for (int m = 1; m < TPS; m <<= 1) {
#pragma unroll
    for (int i = 0; i < 18; ++i) K[i] += shfl_xor_t<Acc>(K[i], m);
  }

  Acc Ga[18];
  su3_site_G(K, Ga, omega);
  Real G[18];
#pragma unroll
  for (int i = 0; i < 18; ++i) G[i] = (Real)Ga[i];

  if (!active) return;
  constexpr int NR = (S::NP == 12) ? 2 : 3;   // rows that are stored
#pragma unroll
  for (int l = 0; l < LPT; ++l) {
    Real R[kLinkRegs];
    R[18] = 0; R[19] = 0;
    if (((q * LPT + l) & 1) == 0) mul_ab<NR>(G, U[l], R);
    else mul_abd<NR>(U[l], G, R);
    store_params<S>(ptr[l], g.vh, R);
  }
}

// ---------------------------------------------------------------------------------------------
// SU(2), 4-parameter storage, one thread per site.  8 links = 32 (fp32) / 64 (fp64) registers, so
// they stay in registers.  K(x) and the closed-form update g = K^dagger/sqrt(det K^dagger)
// (PAPER.md L52), g^omega, in fp64 for both storage precisions (the same conditioning argument as
// for SU(3), reading C-15); the 8 quaternion products in the storage precision.  Odd-parity
// launches walk the site blocks in descending order (L2 carry-over, as the SU(3) kernel).
// ---------------------------------------------------------------------------------------------
template <typename S, int BLOCK, bool COULOMB, typename Power>
__global__ void __launch_bounds__(BLOCK)
or_sweep_su2_kernel(typename S::Vec* __restrict__ links, const Geom g, const int parity,
                    const Power omega, const int reverse) {
  typedef typename S::Real Real;
  const int blk = reverse ? (int)gridDim.x - 1 - (int)blockIdx.x : (int)blockIdx.x;
  const int h = blk * BLOCK + threadIdx.x;
  if (h >= g.vh) return;
  const SiteCoord sc = decode_site(g, h, parity);
  if (COULOMB && g.slice_active != nullptr && g.slice_active[sc.x3] == 0) return;   // frozen slice
  Real U[8][4];
  typename S::Vec* ptr[8];
#pragma unroll
  for (int mu = 0; mu < 4; ++mu) {
    ptr[2 * mu] = link_base<S>(links, g, parity, mu, h);
    ptr[2 * mu + 1] = link_base<S>(links, g, 1 - parity, mu, down_index(g, h, sc, mu));
  }
  pdl_prologue_done();    // lattice.cuh: the next half-sweep may be scheduled; the previous one is complete
#pragma unroll
  for (int l = 0; l < 8; ++l) load_params<S>(ptr[l], g.vh, U[l]);
  // K = k0 + i k.sigma = sum_mu u_up + conj(u_dn)
  double k[4] = {0, 0, 0, 0};
#pragma unroll
  for (int mu = 0; mu < (COULOMB ? 3 : 4); ++mu) {     // Coulomb gauge: spatial links only (C-22)
    k[0] += (double)U[2 * mu][0] + (double)U[2 * mu + 1][0];
#pragma unroll
    for (int i = 1; i < 4; ++i) k[i] += (double)U[2 * mu][i] - (double)U[2 * mu + 1][i];
  }
  // the subgroup quaternion of the 2x2 K is p = 2k (the scale only matters to the heat bath, a = |p|/T)
#pragma unroll
  for (int i = 0; i < 4; ++i) k[i] *= 2.0;
  double Gd[4];
  if (!su2_update_at<(sizeof(Real) == 8)>(k, omega, Gd, (uint32_t)canonical_site(g, h, sc), 0u)) return;   // K = 0: skip (C-9)
  const Real G[4] = {(Real)Gd[0], (Real)Gd[1], (Real)Gd[2], (Real)Gd[3]};
#pragma unroll
  for (int l = 0; l < 8; ++l) {
    Real R[4];
    if ((l & 1) == 0) quat_mul(G, U[l], R);
    else quat_mul_dag(U[l], G, R);
    store_params<S>(ptr[l], g.vh, R);
  }
}

// ---------------------------------------------------------------------------------------------
// host-side launchers
// ---------------------------------------------------------------------------------------------
template <typename S, typename Acc, int TPS>
static cudaError_t launch_su3(void* links, const Geom& g, int parity, double omega, cudaStream_t st) {
  constexpr int BLOCK = 128;
  const long long threads = (long long)g.vh * TPS;
  const unsigned grid = (unsigned)((threads + BLOCK - 1) / BLOCK);
  or_sweep_su3_kernel<S, Acc, TPS, BLOCK><<<grid, BLOCK, 0, st>>>(
      (typename S::Vec*)links, g, parity, (Acc)omega);
  return cudaGetLastError();
}

template <typename S, typename Power>
static cudaError_t launch_su2(void* links, const Geom& g, int parity, Power omega, bool coulomb, cudaStream_t st) {
  constexpr int BLOCK = 128;
  const unsigned grid = (unsigned)((g.vh + BLOCK - 1) / BLOCK);
  if (coulomb)
    return launch_pdl(or_sweep_su2_kernel<S, BLOCK, true, Power>, dim3(grid), dim3(BLOCK), 0, st,
                      (typename S::Vec*)links, g, parity, omega, parity);
  return launch_pdl(or_sweep_su2_kernel<S, BLOCK, false, Power>, dim3(grid), dim3(BLOCK), 0, st,
                    (typename S::Vec*)links, g, parity, omega, parity);
}

// Truncated-series overrelaxation (reading C-24): b_n = binom(omega, n) by the recurrence
// b_n = b_{n-1} (omega - n + 1)/n; production mappings only.
cudaError_t launch_or_sweep_series(const LatticeDesc& d, void* links, int parity, double omega, int order,
                                   cudaStream_t st) {
  if (order < 0 || order > kMaxSeriesOrder) return cudaErrorInvalidValue;
  SeriesPower pw;
  pw.order = order;
  pw.b[0] = 1.0;
  for (int n = 1; n <= kMaxSeriesOrder; ++n) pw.b[n] = n <= order ? pw.b[n - 1] * ((omega - (double)(n - 1)) / (double)n) : 0.0;
  if (d.group == 2) {
    if (d.precision == 32) return launch_su2<Storage<float, 2, 4> >(links, d.geom, parity, pw, false, st);
    return launch_su2<Storage<double, 2, 4> >(links, d.geom, parity, pw, false, st);
  }
  return launch_or_sweep_staged_series(d, links, parity, pw, st);
}

// Simulated-annealing half-sweep at temperature T (reading C-25); production mappings only.
cudaError_t launch_sa_sweep(const LatticeDesc& d, void* links, int parity, double T, unsigned long long seed,
                            unsigned counter, cudaStream_t st) {
  HeatBathPower pw;
  pw.inv_T = 1.0 / T;
  pw.seed_lo = (uint32_t)seed;
  pw.seed_hi = (uint32_t)(seed >> 32);
  pw.counter = counter;
  if (d.group == 2) {
    if (d.precision == 32) return launch_su2<Storage<float, 2, 4> >(links, d.geom, parity, pw, false, st);
    return launch_su2<Storage<double, 2, 4> >(links, d.geom, parity, pw, false, st);
  }
  return launch_or_sweep_staged_heatbath(d, links, parity, pw, st);
}

// Microcanonical half-sweep (reading C-26); production mappings only.
cudaError_t launch_micro_sweep(const LatticeDesc& d, void* links, int parity, cudaStream_t st) {
  if (d.group == 2) {
    if (d.precision == 32) return launch_su2<Storage<float, 2, 4> >(links, d.geom, parity, MicroPower{0}, false, st);
    return launch_su2<Storage<double, 2, 4> >(links, d.geom, parity, MicroPower{0}, false, st);
  }
  return launch_or_sweep_staged_micro(d, links, parity, st);
}

cudaError_t launch_or_full_sweep(const LatticeDesc& d, void* links, double omega, int variant, cudaStream_t st) {
  if (variant >= 40 && variant < 60) {
    const cudaError_t e = launch_or_sweep_staged_slabbed(d, links, omega, 1 << (variant % 10), variant >= 50, st);
    if (e != cudaErrorNotSupported) return e;
    variant = 0;                                         // lattice does not fit the slab schedule
  }
  for (int parity = 0; parity < 2; ++parity) {
    const cudaError_t e = launch_or_sweep(d, links, parity, omega, variant, st);
    if (e != cudaSuccess) return e;
  }
  return cudaSuccess;
}

cudaError_t launch_or_sweep(const LatticeDesc& d, void* links, int parity, double omega,
                            int variant, cudaStream_t st, bool coulomb) {
  const Geom& g = d.geom;
  if (variant >= 40 && variant < 60) variant = 0;       // slab schedules exist for full sweeps only
  if (d.group == 2) {
    if (d.precision == 32) return launch_su2<Storage<float, 2, 4> >(links, g, parity, omega, coulomb, st);
    return launch_su2<Storage<double, 2, 4> >(links, g, parity, omega, coulomb, st);
  }
  // variant 0 = the production mapping (or_sweep_staged.cu); 20+ select staged mappings
  if (variant == 0) {
    const int best = 20;   // the production mapping of each storage format (or_sweep_staged.cu)
    return launch_or_sweep_staged(d, links, parity, omega, best, coulomb, st);
  }
  if (coulomb) return cudaErrorInvalidValue;   // Coulomb gauge: production mapping (variant 0) only
  if (variant >= 20) return launch_or_sweep_staged(d, links, parity, omega, variant, false, st);
  if (d.precision == 32) {
    // fp32 storage: K and the subgroup solve in fp64 (reading C-15); variants 10+ are
    // all-fp32 arithmetic, kept for the precision/throughput comparison in profiles/.
    if (d.params == 12) {
      switch (variant) {
        case 1: return launch_su3<Storage<float, 3, 12>, double, 1>(links, g, parity, omega, st);
        case 2: return launch_su3<Storage<float, 3, 12>, double, 2>(links, g, parity, omega, st);
        case 4: return launch_su3<Storage<float, 3, 12>, double, 4>(links, g, parity, omega, st);
        case 11: return launch_su3<Storage<float, 3, 12>, float, 1>(links, g, parity, omega, st);
        case 14: return launch_su3<Storage<float, 3, 12>, float, 4>(links, g, parity, omega, st);
        default: return cudaErrorInvalidValue;
      }
    }
    switch (variant) {
      case 2: return launch_su3<Storage<float, 3, 18>, double, 2>(links, g, parity, omega, st);
      case 4: return launch_su3<Storage<float, 3, 18>, double, 4>(links, g, parity, omega, st);
      default: return cudaErrorInvalidValue;
    }
  }
  if (d.params == 12) {
    switch (variant) {
      case 4: return launch_su3<Storage<double, 3, 12>, double, 4>(links, g, parity, omega, st);
      case 2: return launch_su3<Storage<double, 3, 12>, double, 2>(links, g, parity, omega, st);
      case 8: return launch_su3<Storage<double, 3, 12>, double, 8>(links, g, parity, omega, st);
      default: return cudaErrorInvalidValue;
    }
  }
  switch (variant) {
    case 4: return launch_su3<Storage<double, 3, 18>, double, 4>(links, g, parity, omega, st);
    case 8: return launch_su3<Storage<double, 3, 18>, double, 8>(links, g, parity, omega, st);
    default: return cudaErrorInvalidValue;
  }
}

}  // namespace culgt
