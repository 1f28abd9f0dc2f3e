// or_sweep.cu -- half-sweep and full-sweep dispatch (launch_or_sweep, launch_or_full_sweeps and
// friends) and the SU(2) kernel.  The production SU(3) kernel is in or_sweep_staged.cu, the fused
// full-sweep kernel in or_sweep_fused.cu, the measured alternatives in or_sweep_measure.cu.
// (SURVEY.md 8(a) rows a1-a6.)
//
// For every site x of one parity:
//   gather the 8 links touching x, K = sum_mu U_mu(x) + U_mu(x-mu)^dagger      (eq. 3)
//   G from K by the SU(2) closed form / the SU(3) subgroup loop with g^omega   (L50-54)
//   U_mu(x) <- G U_mu(x),  U_mu(x-mu) <- U_mu(x-mu) G^dagger                   (L19-21, L48)
// Sites of one parity are independent (L54), so there is no synchronisation inside a launch.
#include "lattice.cuh"
#include "su_math.cuh"
#include "su2_power.cuh"
#include "kernels.h"

namespace culgt {

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
                    const Power omega, const int reverse, const int* __restrict__ stop_flag) {
  typedef typename S::Real Real;
  const int blk = reverse ? (int)gridDim.x - 1 - (int)blockIdx.x : (int)blockIdx.x;
  const int h = blk * BLOCK + threadIdx.x;
  if (h >= g.vh) return;
  const SiteCoord sc = decode_site(g, h, parity);
  Real U[8][4];
  typename S::Vec* ptr[8];
#pragma unroll
  for (int mu = 0; mu < 4; ++mu) {
    ptr[2 * mu] = link_base<S>(links, g, parity, mu, h);
    ptr[2 * mu + 1] = link_base<S>(links, g, 1 - parity, mu, down_index(g, h, sc, mu));
  }
  pdl_prologue_done();    // lattice.cuh: the next half-sweep may be scheduled; the previous one is complete
  if (stop_flag != nullptr && *stop_flag != 0) return;                               // driver loop has stopped
  if (COULOMB && g.slice_active != nullptr && g.slice_active[sc.x3] == 0) return;   // frozen slice
#pragma unroll
  for (int l = 0; l < 8; ++l) load_params<S>(ptr[l], g.pitch, U[l]);
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
    store_params<S>(ptr[l], g.pitch, R);
  }
}

// ---------------------------------------------------------------------------------------------
// host-side launchers
// ---------------------------------------------------------------------------------------------
template <typename S, typename Power>
static cudaError_t launch_su2(void* links, const Geom& g, int parity, Power omega, bool coulomb, const int* stop_flag,
                              cudaStream_t st) {
  constexpr int BLOCK = 128;
  const unsigned grid = (unsigned)((g.vh + BLOCK - 1) / BLOCK);
  if (coulomb)
    return launch_pdl(or_sweep_su2_kernel<S, BLOCK, true, Power>, dim3(grid), dim3(BLOCK), 0, st,
                      (typename S::Vec*)links, g, parity, omega, parity, stop_flag);
  return launch_pdl(or_sweep_su2_kernel<S, BLOCK, false, Power>, dim3(grid), dim3(BLOCK), 0, st,
                    (typename S::Vec*)links, g, parity, omega, parity, stop_flag);
}

template <typename Power>
static cudaError_t launch_su2_any(const LatticeDesc& d, void* links, int parity, const Power& pw, bool coulomb,
                                  const int* stop_flag, cudaStream_t st) {
  if (d.precision == 32) return launch_su2<Storage<float, 2, 4> >(links, d.geom, parity, pw, coulomb, stop_flag, st);
  return launch_su2<Storage<double, 2, 4> >(links, d.geom, parity, pw, coulomb, stop_flag, st);
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
  if (d.group == 2) return launch_su2_any(d, links, parity, pw, false, nullptr, st);
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
  if (d.group == 2) return launch_su2_any(d, links, parity, pw, false, nullptr, st);
  return launch_or_sweep_staged_heatbath(d, links, parity, pw, st);
}

// Microcanonical half-sweep (reading C-26); production mappings only.
cudaError_t launch_micro_sweep(const LatticeDesc& d, void* links, int parity, cudaStream_t st) {
  if (d.group == 2) return launch_su2_any(d, links, parity, MicroPower{0}, false, nullptr, st);
  return launch_or_sweep_staged_micro(d, links, parity, st);
}

// Variant numbers (culgt_set_sweep_variant):
//   product:  0 production (20 is its explicit name), 24 / 33 / 34 the same kernel without the reversed
//             traversal / programmatic dependent launch / L2 hints;
//   -DCULGT_MEASURE only: 1-14, 21-32 (or_sweep_measure.cu), 41-44 launch-level slab schedules, 60 the
//             fused one-kernel full sweep (or_sweep_fused.cu; needs a workspace), >= 100000 its parameter
//             sweeps (100000 + 50000*alternate + 1000*lag + hints code).
bool sweep_variant_known(int variant) {
  switch (variant) {
    case 0: case 20: case 24: case 33: case 34: return true;
    default: break;
  }
#ifdef CULGT_MEASURE
  if ((variant >= 1 && variant <= 14) || (variant >= 21 && variant <= 32) || (variant >= 41 && variant <= 44) ||
      variant == 60 || (variant >= 100000 && variant < 200000))
    return true;
#endif
  return false;
}

cudaError_t launch_or_sweep(const LatticeDesc& d, void* links, int parity, double omega,
                            int variant, cudaStream_t st, bool coulomb, const int* stop_flag) {
  if (d.group == 2) return launch_su2_any(d, links, parity, omega, coulomb, stop_flag, st);
  // full-sweep schedules (fused, slab-blocked) have no half-sweep form: the production mapping
  if (variant == 0 || variant >= 40) variant = 20;
  if (variant == 20 || variant == 24 || variant == 33 || variant == 34)
    return launch_or_sweep_staged(d, links, parity, omega, variant, coulomb, stop_flag, st);
#ifdef CULGT_MEASURE
  if (!coulomb && stop_flag == nullptr) return launch_or_sweep_measure(d, links, parity, omega, variant, st);
#endif
  return cudaErrorInvalidValue;
}

cudaError_t launch_or_full_sweeps(const LatticeDesc& d, void* links, double* workspace, int n_sweeps, double omega,
                                  int variant, const int* stop_flag, cudaStream_t st) {
  if (n_sweeps <= 0) return cudaSuccess;
#ifdef CULGT_MEASURE
  if ((variant == 60 || variant >= 100000) && workspace != nullptr) {
    int lag = 0, hints = kFusedDefaultHints;
    bool alternate = true;
    if (variant >= 100000) {
      const int v = variant - 100000;
      alternate = v >= 50000;
      lag = (v % 50000) / 1000;
      int code = v % 1000;                     // base-3 digits: black load, black store, white load, white store
      hints = 0;
      for (int i = 0; i < 4; ++i) { hints |= (code % 3) << (2 * i); code /= 3; }
    }
    void* ctl = workspace + fused_ctl_offset_doubles(d.geom);
    const cudaError_t e = launch_or_sweeps_fused(d, links, omega, ctl, n_sweeps, lag, hints, alternate, stop_flag, st);
    if (e != cudaErrorNotSupported) return e;     // lattice does not fit the fused schedule: two launches
  }
  if (variant >= 41 && variant <= 44) {
    bool fits = true;                          // cudaErrorNotSupported depends on the lattice only: first call
    for (int i = 0; i < n_sweeps && fits; ++i) {
      const cudaError_t e = launch_or_sweep_measure_slabbed(d, links, omega, 1 << (variant - 40), st);
      if (e == cudaErrorNotSupported) fits = false;
      else if (e != cudaSuccess) return e;
    }
    if (fits) return cudaSuccess;
  }
#else
  (void)workspace;
#endif
  const int half_variant = (variant >= 40) ? 0 : variant;
  for (int i = 0; i < n_sweeps; ++i)
    for (int parity = 0; parity < 2; ++parity) {
      const cudaError_t e = launch_or_sweep(d, links, parity, omega, half_variant, st, false, stop_flag);
      if (e != cudaSuccess) return e;
    }
  return cudaSuccess;
}

}  // namespace culgt
