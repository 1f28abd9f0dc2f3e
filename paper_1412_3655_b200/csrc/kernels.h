// kernels.h -- internal (C++) interface between the C-ABI layer (api.cu) and the kernel files.
#pragma once
#include <cuda_runtime.h>
#include "lattice.cuh"

namespace culgt {

struct LatticeDesc {
  Geom geom;
  int group;      // 2 or 3
  int precision;  // 32 or 64
  int params;     // 18, 12 or 4
  long long V;
};

constexpr int kReduceBlock = 256;       // threads per block of the reduction kernels
// CTAs (= partials per quantity) of the fused theta+F kernel: `half` sites of each parity per CTA
// (128 for the register path, 64 for the staged fp32 12-parameter path; the workspace is sized for 64)
inline int reduce_blocks_fused(int vh, int half = 64) { return (vh + half - 1) / half; }
// doubles in the reduction workspace: block partials (Landau: 2 * vh/128; Coulomb: 2 * N3 *
// slice/128; never below 4096) followed by 2 * N3 result slots that the *_host / *_fix paths
// read back (Landau uses the first two).
inline size_t reduce_partial_doubles(const Geom& g) {
  size_t n = 2 * (size_t)reduce_blocks_fused(g.vh);
  const size_t c = 2 * (size_t)g.n[3] * (size_t)reduce_blocks_fused(g.stride[3]);
  if (c > n) n = c;
  return n > 4096 ? n : 4096;
}
// ... and N3 bytes (rounded up to doubles) for the Coulomb driver's per-slice activity mask
inline size_t reduce_workspace_doubles(const Geom& g) {
  return reduce_partial_doubles(g) + 2 * (size_t)g.n[3] + ((size_t)g.n[3] + 7) / 8;
}

// coulomb = true: Coulomb-gauge half-sweep (K from the spatial links; production mapping only)
cudaError_t launch_or_sweep(const LatticeDesc& d, void* links, int parity, double omega,
                            int variant, cudaStream_t st, bool coulomb = false);
struct SeriesPower;
struct HeatBathPower;
// simulated-annealing half-sweep (reading C-25), production mappings only
cudaError_t launch_sa_sweep(const LatticeDesc& d, void* links, int parity, double T, unsigned long long seed,
                            unsigned counter, cudaStream_t st);
cudaError_t launch_or_sweep_staged_heatbath(const LatticeDesc& d, void* links, int parity, const HeatBathPower& pw,
                                            cudaStream_t st);
// microcanonical half-sweep (reading C-26), production mappings only
cudaError_t launch_micro_sweep(const LatticeDesc& d, void* links, int parity, cudaStream_t st);
cudaError_t launch_or_sweep_staged_micro(const LatticeDesc& d, void* links, int parity, cudaStream_t st);
// truncated-series overrelaxation (reading C-24), production mappings only
cudaError_t launch_or_sweep_series(const LatticeDesc& d, void* links, int parity, double omega, int order,
                                   cudaStream_t st);
cudaError_t launch_or_sweep_staged_series(const LatticeDesc& d, void* links, int parity, const SeriesPower& pw,
                                          cudaStream_t st);
// One FULL sweep (black then white).  Variants 40..59 select the slab-blocked schedule of
// or_sweep_staged.cu (40 + log2(slab slices): one stream; 50 + log2(slab slices): white windows on a
// second stream); every other variant, and any lattice the slab schedule does not fit, is the two
// whole half-sweeps of launch_or_sweep.
cudaError_t launch_or_full_sweep(const LatticeDesc& d, void* links, double omega, int variant, cudaStream_t st);
cudaError_t launch_or_sweep_staged_slabbed(const LatticeDesc& d, void* links, double omega, int slab_slices,
                                           bool overlap, cudaStream_t st);
cudaError_t launch_or_sweep_staged(const LatticeDesc& d, void* links, int parity, double omega,
                                   int variant, bool coulomb, cudaStream_t st);
cudaError_t launch_pack(const LatticeDesc& d, const void* canonical, void* links, cudaStream_t st);
cudaError_t launch_reunitarize(const LatticeDesc& d, void* links, cudaStream_t st);
cudaError_t launch_unpack(const LatticeDesc& d, const void* links, void* canonical, cudaStream_t st);
// fused theta + F; workspace holds 2 * reduce_blocks_fused(vh) partials
cudaError_t launch_theta_functional(const LatticeDesc& d, const void* links, double* workspace,
                                    double* out_theta, double* out_F, cudaStream_t st);
// Coulomb gauge: per-slice theta_t, F_t (N3 doubles each)
cudaError_t launch_coulomb_theta_functional(const LatticeDesc& d, const void* links, double* workspace,
                                            double* out_theta_t, double* out_F_t, cudaStream_t st);
cudaError_t launch_gauge_transform(const LatticeDesc& d, void* links, const void* g, cudaStream_t st);

}  // namespace culgt
