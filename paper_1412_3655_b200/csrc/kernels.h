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
// CTAs (= partials per quantity) of the fused theta+F kernel: 128 sites of each parity per CTA
inline int reduce_blocks_fused(int vh) { return (vh + 127) / 128; }
// doubles in the reduction workspace: partials + the two scalars the *_host paths read back
inline size_t reduce_workspace_doubles(int vh) {
  const size_t fused = 2 * (size_t)reduce_blocks_fused(vh);
  return (fused > 4096 ? fused : 4096) + 2;   // never below 32 KiB
}

cudaError_t launch_or_sweep(const LatticeDesc& d, void* links, int parity, double omega,
                            int variant, cudaStream_t st);
cudaError_t launch_or_sweep_staged(const LatticeDesc& d, void* links, int parity, double omega,
                                   int variant, cudaStream_t st);
cudaError_t launch_pack(const LatticeDesc& d, const void* canonical, void* links, cudaStream_t st);
cudaError_t launch_unpack(const LatticeDesc& d, const void* links, void* canonical, cudaStream_t st);
// fused theta + F; workspace holds 2 * reduce_blocks_fused(vh) partials
cudaError_t launch_theta_functional(const LatticeDesc& d, const void* links, double* workspace,
                                    double* out_theta, double* out_F, cudaStream_t st);
cudaError_t launch_gauge_transform(const LatticeDesc& d, void* links, const void* g, cudaStream_t st);

}  // namespace culgt
