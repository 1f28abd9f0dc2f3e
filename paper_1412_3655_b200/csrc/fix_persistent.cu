// fix_persistent.cu -- the paper's whole driver loop (black half-sweep, white half-sweep,
// "iterated until the discrete gauge condition (1) is satisfied up to a given numerical precision")
// as ONE cooperative kernel, for SU(3) lattices small enough that every site block of a parity has
// its own resident CTA (4^4 ... 16^4: SURVEY.md 7.1 step 7, 7.4 item 6).
//
// Such lattices are bound by latency, not bandwidth: a half-sweep is one wave of CTAs, and a launch
// per half-sweep plus two per check costs more than the work (BASELINE.json configs[0]: theta every
// sweep on 256 sites).  Here CTA b owns site block b of BOTH parities for the whole run:
//     loop:  theta, F of the current field (per-CTA partial -> grid barrier -> every CTA adds the
//            partials in the same fixed order, so all CTAs take the same decision without another
//            barrier);  stop if theta < target or max_sweeps is reached;
//            check_every x ( black half-sweep of my block; grid barrier; white; grid barrier ).
// The per-site update is the production body (staged.cuh) unchanged, so the links are bit-identical
// to the launch-per-half-sweep path.  Links are read with L2-coherent accesses only (cp.async.cg in
// the sweep, ld.global.cg in the reduction): another SM's stores of the previous phase are visible
// after the barrier (__threadfence before the arrival, ld.acquire.gpu on the polling side).
// The grid barrier is a monotone arrival counter in the caller's workspace; the launch is
// cooperative (cudaLaunchCooperativeKernel), which guarantees that all CTAs are resident.
#include "staged.cuh"
#include "kernels.h"

namespace culgt {

__device__ __forceinline__ unsigned ld_acquire_u32(const unsigned* p) {
  unsigned v;
  asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
  return v;
}

// every thread of every CTA calls this the same number of times
__device__ __forceinline__ void grid_barrier(unsigned* counter, unsigned& target) {
  __syncthreads();
  if (threadIdx.x == 0) {
    target += gridDim.x;
    __threadfence();                       // my CTA's stores are visible before I arrive
    atomicAdd(counter, 1u);
    while ((int)(ld_acquire_u32(counter) - target) < 0) {}     // wrap-safe: the counter is monotone mod 2^32
  }
  __syncthreads();
}

template <int BLOCK>
__device__ __forceinline__ double block_sum_p(double v, double* warp_part) {
#pragma unroll
  for (int m = 16; m > 0; m >>= 1) v += __shfl_xor_sync(0xffffffffu, v, m);
  if ((threadIdx.x & 31) == 0) warp_part[threadIdx.x >> 5] = v;
  __syncthreads();
  double t = 0;
#pragma unroll
  for (int w = 0; w < BLOCK / 32; ++w) t += warp_part[w];     // every thread: the same order, the same bits
  __syncthreads();
  return t;
}

// theta and F contributions of site (parity, h): the anti-Hermitian parts of its 8 links (reading C-11;
// reduce.cu add_antihermitian_parts restated for L2-coherent loads).
template <typename S>
__device__ __forceinline__ void site_theta_F(const typename S::Vec* links, const Geom& g, int parity, int h,
                                             double* th, double* f) {
  typedef typename S::Real Real;
  typedef typename S::Vec Vec;
  const SiteCoord sc = decode_site(g, h, parity);
  double a[9];
#pragma unroll
  for (int i = 0; i < 9; ++i) a[i] = 0;
#pragma unroll 2                          // two links' loads in flight; more would spill the fp64 formats
  for (int l = 0; l < 8; ++l) {
    const int mu = l >> 1;
    const bool down = l & 1;
    const Vec* p = link_base<S>(links, g, down ? 1 - parity : parity, mu, down ? down_index(g, h, sc, mu) : h);
    Real U[kLinkRegs];
#pragma unroll
    for (int j = 0; j < S::NV; ++j) {
      const Vec v = __ldcg(p + (size_t)j * (size_t)g.pitch);
      vec_get(v, U + j * S::VL);
    }
    double m[18];
#pragma unroll
    for (int i = 0; i < S::NP; ++i) m[i] = (double)U[i];
    if (S::NP == 12) reconstruct_row2(m);
    const double sign = down ? -1.0 : 1.0;
    a[0] = fma(sign, m[CULGT_IM(0, 0)], a[0]);
    a[1] = fma(sign, m[CULGT_IM(1, 1)], a[1]);
    a[2] = fma(sign, m[CULGT_IM(2, 2)], a[2]);
    a[3] = fma(sign, m[CULGT_IM(0, 1)] + m[CULGT_IM(1, 0)], a[3]);
    a[4] = fma(sign, m[CULGT_RE(0, 1)] - m[CULGT_RE(1, 0)], a[4]);
    a[5] = fma(sign, m[CULGT_IM(0, 2)] + m[CULGT_IM(2, 0)], a[5]);
    a[6] = fma(sign, m[CULGT_RE(0, 2)] - m[CULGT_RE(2, 0)], a[6]);
    a[7] = fma(sign, m[CULGT_IM(1, 2)] + m[CULGT_IM(2, 1)], a[7]);
    a[8] = fma(sign, m[CULGT_RE(1, 2)] - m[CULGT_RE(2, 1)], a[8]);
    if (!down) *f += m[CULGT_RE(0, 0)] + m[CULGT_RE(1, 1)] + m[CULGT_RE(2, 2)];
  }
  const double tr = (a[0] + a[1] + a[2]) * (1.0 / 3.0);
  double sum = 0;
#pragma unroll
  for (int c = 0; c < 3; ++c) sum += (a[c] - tr) * (a[c] - tr);
#pragma unroll
  for (int c = 3; c < 9; ++c) sum = fma(0.5 * a[c], a[c], sum);
  *th += sum;
}

template <typename S, int BLOCK>
__global__ void __launch_bounds__(BLOCK, 1)       // at most one CTA per SM is ever launched: all registers are its own
landau_fix_persistent_kernel(typename S::Vec* links, const Geom g, const double omega, const double theta_target,
                             const int max_sweeps, const int check_every, double* partial, PersistCtl* ctl,
                             const double scale_theta, const double scale_F) {
  typedef typename S::Vec Vec;
  extern __shared__ __align__(16) unsigned char smem_raw[];
  Vec* const sm = reinterpret_cast<Vec*>(smem_raw) + threadIdx.x;
  const unsigned sm_addr = (unsigned)__cvta_generic_to_shared(sm);
  __shared__ double warp_part[BLOCK / 32];
  const int nb = (int)gridDim.x;
  const int h = (int)blockIdx.x * BLOCK + (int)threadIdx.x;
  unsigned target = 0;
  int done = 0;
  double theta = 0, F = 0;
  for (;;) {
    // ---- theta and F of the current field
    double th = 0, f = 0;
    if (h < g.vh) {
      site_theta_F<S>(links, g, 0, h, &th, &f);
      site_theta_F<S>(links, g, 1, h, &th, &f);
    }
    const double st = block_sum_p<BLOCK>(th, warp_part);
    const double sf = block_sum_p<BLOCK>(f, warp_part);
    if (threadIdx.x == 0) {
      __stcg(&partial[blockIdx.x], st);
      __stcg(&partial[nb + blockIdx.x], sf);
    }
    grid_barrier(&ctl->barrier, target);
    double at = 0, af = 0;
    for (int i = threadIdx.x; i < nb; i += BLOCK) {
      at += __ldcg(&partial[i]);
      af += __ldcg(&partial[nb + i]);
    }
    theta = block_sum_p<BLOCK>(at, warp_part) * scale_theta;
    F = block_sum_p<BLOCK>(af, warp_part) * scale_F;
    if (theta < theta_target || done >= max_sweeps) break;     // the same bits in every CTA: a uniform decision
    // ---- check_every full sweeps
    int n = check_every;
    if (done + n > max_sweeps) n = max_sweeps - done;
    for (int i = 0; i < n; ++i) {
#pragma unroll 1
      for (int parity = 0; parity < 2; ++parity) {
        const SiteRef<8> r = locate<BLOCK, 1>(g, parity, (int)blockIdx.x, 0);
        issue_site_loads<S, BLOCK, false>(links, g, parity, r, sm, 0);
        cp_async_wait<0>();
        update_site<S, BLOCK, false, false>(links, g, parity, omega, r, sm_addr, 0);
        grid_barrier(&ctl->barrier, target);
      }
    }
    done += n;
  }
  if (blockIdx.x == 0 && threadIdx.x == 0) {
    ctl->sweeps_done = done;
    ctl->theta = theta;
    ctl->F = F;
  }
}

template <typename S, int BLOCK>
static cudaError_t run_persistent(void* links, const LatticeDesc& d, double omega, double theta_target, int max_sweeps,
                                  int check_every, double* partial, PersistCtl* ctl, cudaStream_t st) {
  typedef typename S::Vec Vec;
  const Geom& g = d.geom;
  auto kern = landau_fix_persistent_kernel<S, BLOCK>;
  constexpr size_t smem = staged_smem_bytes<S, BLOCK>();
  const int nb = (g.vh + BLOCK - 1) / BLOCK;
  static bool configured[kMaxDevices] = {false};
  static int capacity[kMaxDevices] = {0};
  int dev = 0;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) return e;
  if (dev < 0 || dev >= kMaxDevices) return cudaErrorNotSupported;
  if (!configured[dev]) {
    if ((e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem)) != cudaSuccess) return e;
    int per_sm = 0, coop = 0;
    if ((e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, kern, BLOCK, smem)) != cudaSuccess) return e;
    if ((e = cudaDeviceGetAttribute(&coop, cudaDevAttrCooperativeLaunch, dev)) != cudaSuccess) return e;
    capacity[dev] = coop ? per_sm * device_sm_count() : 0;
    configured[dev] = true;
  }
  // one CTA per SM at most: beyond that the launch-per-half-sweep path is as fast (measured)
  if (nb > capacity[dev] || nb > device_sm_count()) return cudaErrorNotSupported;
  if ((e = cudaMemsetAsync(ctl, 0, sizeof(PersistCtl), st)) != cudaSuccess) return e;
  Vec* lp = (Vec*)links;
  Geom gg = g;
  double scale_theta = 1.0 / (3.0 * (double)d.V), scale_F = 1.0 / (12.0 * (double)d.V);
  void* args[] = {&lp, &gg, &omega, &theta_target, &max_sweeps, &check_every, &partial, &ctl, &scale_theta, &scale_F};
  return cudaLaunchCooperativeKernel((const void*)kern, dim3((unsigned)nb), dim3(BLOCK), args, smem, st);
}

// cudaErrorNotSupported: the lattice is not SU(3) or has more site blocks per parity than SMs.
cudaError_t launch_landau_fix_persistent(const LatticeDesc& d, void* links, double omega, double theta_target,
                                         int max_sweeps, int check_every, double* partial, PersistCtl* ctl,
                                         cudaStream_t st) {
  if (d.group != 3) return cudaErrorNotSupported;
  if (d.precision == 32 && d.params == 12)
    return run_persistent<Storage<float, 3, 12>, 128>(links, d, omega, theta_target, max_sweeps, check_every, partial, ctl, st);
  if (d.precision == 32)
    return run_persistent<Storage<float, 3, 18>, 64>(links, d, omega, theta_target, max_sweeps, check_every, partial, ctl, st);
  if (d.params == 12)
    return run_persistent<Storage<double, 3, 12>, 64>(links, d, omega, theta_target, max_sweeps, check_every, partial, ctl, st);
  return run_persistent<Storage<double, 3, 18>, 64>(links, d, omega, theta_target, max_sweeps, check_every, partial, ctl, st);
}

}  // namespace culgt
