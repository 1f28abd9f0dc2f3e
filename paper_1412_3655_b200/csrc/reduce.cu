// reduce.cu -- a7 functional F and a8 gauge precision theta, one fused pass.
//
//   F     = 1/(4 Nc V) sum_x sum_mu Re tr U_mu(x)                      PAPER.md eq. (2) at g = 1
//   theta = 1/(Nc V) sum_x tr[Delta(x) Delta(x)^dagger],  Delta(x) = [(K(x) - K(x)^dagger)/(2i)]_traceless
//           which equals sum_mu A_mu(x) - A_mu(x-mu) of eq. (1) (reading C-11).
// Reduction: per-thread fp64 partial -> warp xor-shuffles -> one shared-memory slot per warp ->
// one partial per block in the workspace -> a single block per quantity sums the partials in a
// fixed order.  Deterministic: no atomics, the same launch always produces the same bits.
// All arithmetic is fp64 on the stored values (12-parameter storage: third row rebuilt in fp64).
#include "lattice.cuh"
#include "su_math.cuh"
#include "kernels.h"

namespace culgt {

template <int BLOCK>
__device__ __forceinline__ double block_sum(double v) {
  __shared__ double warp_part[BLOCK / 32];
#pragma unroll
  for (int m = 16; m > 0; m >>= 1) v += __shfl_xor_sync(0xffffffffu, v, m);
  if ((threadIdx.x & 31) == 0) warp_part[threadIdx.x >> 5] = v;
  __syncthreads();
  double t = 0;
  if (threadIdx.x < 32) {
    t = threadIdx.x < BLOCK / 32 ? warp_part[threadIdx.x] : 0.0;
#pragma unroll
    for (int m = 16; m > 0; m >>= 1) t += __shfl_xor_sync(0xffffffffu, t, m);
  }
  return t;   // valid in thread 0
}

// sum_ab |Delta_ab|^2 with Delta = [(K - K^dagger)/(2i)]_traceless (reading C-11):
// D_ab = (K_ab - conj(K_ba))/(2i);  re(D_ab) = (im K_ab + im K_ba)/2, im(D_ab) = -(re K_ab - re K_ba)/2.
__device__ __forceinline__ double theta_from_K(const double* K) {
  double dre[3];
#pragma unroll
  for (int a = 0; a < 3; ++a) dre[a] = K[CULGT_IM(a, a)];
  const double tr = (dre[0] + dre[1] + dre[2]) * (1.0 / 3.0);
  double sum = 0;
#pragma unroll
  for (int a = 0; a < 3; ++a) sum += (dre[a] - tr) * (dre[a] - tr);
#pragma unroll
  for (int a = 0; a < 3; ++a)
#pragma unroll
    for (int b = a + 1; b < 3; ++b) {
      const double re = 0.5 * (K[CULGT_IM(a, b)] + K[CULGT_IM(b, a)]);
      const double im = -0.5 * (K[CULGT_RE(a, b)] - K[CULGT_RE(b, a)]);
      sum += 2.0 * (re * re + im * im);     // |D_ab|^2 + |D_ba|^2, D Hermitian
    }
  return sum;
}

// Fused theta + F in one pass over the field (what the driver loop needs at every check).
// CTA b handles the BLOCK/2 sites h in [b*BLOCK/2, (b+1)*BLOCK/2) of BOTH parities (threads
// 0..BLOCK/2-1 black, the rest white): a link is read once as U_mu(x) by its own site and once
// as U_mu(x'-mu) by the neighbour x' = x+mu of the other parity, and with both parities in one
// CTA the second read comes from L1/L2 instead of HBM (mu = 0: same CTA; mu = 1,2: a few CTAs
// away; mu = 3: one time-slice of CTAs away, far below the L2 size).  F = sum of Re tr over the
// 4 up links of every site of both parities = every link exactly once.
//
// COULOMB = true (reading C-22): mu runs over the 3 spatial directions only and the sums are kept
// per time-slice: blockIdx.y = t, the CTA's sites are the BLOCK/2 sites [bx*BLOCK/2, ...) of each
// parity INSIDE slice t (a slice is the contiguous index range [t*stride3, (t+1)*stride3) of each
// parity's sublattice), partials are laid out [t][bx].
template <typename S, int BLOCK, bool COULOMB>
__global__ void __launch_bounds__(BLOCK)
theta_functional_kernel(const typename S::Vec* __restrict__ links, const Geom g,
                        double* __restrict__ partial_theta, double* __restrict__ partial_F) {
  typedef typename S::Real Real;
  constexpr int HALF = BLOCK / 2;
  constexpr int ND = COULOMB ? 3 : 4;
  const int parity = threadIdx.x >= HALF;
  const int in_group = blockIdx.x * HALF + (int)threadIdx.x - parity * HALF;   // index inside the slice / lattice
  const int group_size = COULOMB ? g.stride[3] : g.vh;
  const int h = COULOMB ? (int)blockIdx.y * g.stride[3] + in_group : in_group;
  double th = 0, f = 0;
  if (in_group < group_size) {
    const SiteCoord sc = decode_site(g, h, parity);
    if (S::NC == 3) {
      double K[18];
#pragma unroll
      for (int i = 0; i < 18; ++i) K[i] = 0;
      // the loads of a batch of directions are issued before any of them is used (memory-level
      // parallelism); fp32 storage batches 2 directions = 4 links, fp64 storage 1 direction
      constexpr int MU_BATCH = (sizeof(Real) == 4) ? 2 : 1;
#pragma unroll
      for (int mu0 = 0; mu0 < ND; mu0 += MU_BATCH) {
        Real U[2 * MU_BATCH][kLinkRegs];
#pragma unroll
        for (int b = 0; b < MU_BATCH; ++b)
          if (mu0 + b < ND) {
            load_params<S>(link_base<S>(links, g, parity, mu0 + b, h), g.vh, U[2 * b]);
            load_params<S>(link_base<S>(links, g, 1 - parity, mu0 + b, down_index(g, h, sc, mu0 + b)), g.vh,
                           U[2 * b + 1]);
          }
#pragma unroll
        for (int b = 0; b < MU_BATCH; ++b)
          if (mu0 + b < ND) {
            double Ud[18];                   // widened first: the third row is rebuilt in fp64
#pragma unroll
            for (int i = 0; i < S::NP; ++i) Ud[i] = (double)U[2 * b][i];
            if (S::NP == 12) reconstruct_row2(Ud);
            f += Ud[CULGT_RE(0, 0)] + Ud[CULGT_RE(1, 1)] + Ud[CULGT_RE(2, 2)];
            accumulate(K, Ud, false);
#pragma unroll
            for (int i = 0; i < S::NP; ++i) Ud[i] = (double)U[2 * b + 1][i];
            if (S::NP == 12) reconstruct_row2(Ud);
            accumulate(K, Ud, true);
          }
      }
      th = theta_from_K(K);
    } else {
      double d[3] = {0, 0, 0};
#pragma unroll
      for (int mu = 0; mu < ND; ++mu) {
        Real u[4], w[4];
        load_params<S>(link_base<S>(links, g, parity, mu, h), g.vh, u);
        load_params<S>(link_base<S>(links, g, 1 - parity, mu, down_index(g, h, sc, mu)), g.vh, w);
        f += 2.0 * (double)u[0];
#pragma unroll
        for (int i = 0; i < 3; ++i) d[i] += (double)u[i + 1] - (double)w[i + 1];
      }
      th = 2.0 * (d[0] * d[0] + d[1] * d[1] + d[2] * d[2]);
    }
  }
  const double st = block_sum<BLOCK>(th);
  __syncthreads();                       // block_sum's shared slots are reused
  const double sf = block_sum<BLOCK>(f);
  if (threadIdx.x == 0) {
    const size_t slot = (size_t)blockIdx.y * gridDim.x + blockIdx.x;
    partial_theta[slot] = st;
    partial_F[slot] = sf;
  }
}

// Final pass: block (group, quantity) sums the n partials of that group in a fixed order and
// scales.  partial = [quantity][group][n]; quantity 0 = theta, 1 = F; group = time-slice for the
// Coulomb sums, a single group for the Landau sums.
template <int BLOCK>
__global__ void __launch_bounds__(BLOCK)
final_sum_kernel(const double* __restrict__ partial, int n, double scale0, double scale1,
                 double* __restrict__ out0, double* __restrict__ out1) {
  const double* p = partial + ((size_t)blockIdx.y * gridDim.x + blockIdx.x) * (size_t)n;
  double acc = 0;
  for (int i = threadIdx.x; i < n; i += BLOCK) acc += p[i];
  const double s = block_sum<BLOCK>(acc);
  if (threadIdx.x == 0) {
    if (blockIdx.y == 0) out0[blockIdx.x] = s * scale0;
    else out1[blockIdx.x] = s * scale1;
  }
}

template <typename S>
static cudaError_t run_theta_functional(const LatticeDesc& d, const void* links, double* ws, double* out_theta,
                                        double* out_F, cudaStream_t st) {
  constexpr int BLOCK = 256;
  const int nblk = reduce_blocks_fused(d.geom.vh);
  theta_functional_kernel<S, BLOCK, false><<<nblk, BLOCK, 0, st>>>((const typename S::Vec*)links, d.geom, ws, ws + nblk);
  cudaError_t e = cudaGetLastError();
  if (e != cudaSuccess) return e;
  final_sum_kernel<kReduceBlock><<<dim3(1, 2), kReduceBlock, 0, st>>>(
      ws, nblk, 1.0 / ((double)S::NC * (double)d.V), 1.0 / (4.0 * S::NC * (double)d.V), out_theta, out_F);
  return cudaGetLastError();
}

// Coulomb gauge: theta_t and F_t for every time-slice t (arrays of N3 doubles).
template <typename S>
static cudaError_t run_coulomb_theta_functional(const LatticeDesc& d, const void* links, double* ws,
                                                double* out_theta_t, double* out_F_t, cudaStream_t st) {
  constexpr int BLOCK = 256;
  const int n3 = d.geom.n[3];
  const int nbx = reduce_blocks_fused(d.geom.stride[3]);
  const size_t per_quantity = (size_t)n3 * nbx;
  theta_functional_kernel<S, BLOCK, true><<<dim3(nbx, n3), BLOCK, 0, st>>>((const typename S::Vec*)links, d.geom,
                                                                           ws, ws + per_quantity);
  cudaError_t e = cudaGetLastError();
  if (e != cudaSuccess) return e;
  const double vs = (double)d.V / (double)n3;
  final_sum_kernel<kReduceBlock><<<dim3(n3, 2), kReduceBlock, 0, st>>>(
      ws, nbx, 1.0 / ((double)S::NC * vs), 1.0 / (3.0 * S::NC * vs), out_theta_t, out_F_t);
  return cudaGetLastError();
}

#define CULGT_DISPATCH(FN, ...)                                                                   \
  if (d.group == 2) {                                                                             \
    if (d.precision == 32) return FN<Storage<float, 2, 4> >(__VA_ARGS__);                         \
    return FN<Storage<double, 2, 4> >(__VA_ARGS__);                                               \
  }                                                                                               \
  if (d.precision == 32) {                                                                        \
    if (d.params == 12) return FN<Storage<float, 3, 12> >(__VA_ARGS__);                           \
    return FN<Storage<float, 3, 18> >(__VA_ARGS__);                                               \
  }                                                                                               \
  if (d.params == 12) return FN<Storage<double, 3, 12> >(__VA_ARGS__);                            \
  return FN<Storage<double, 3, 18> >(__VA_ARGS__);

cudaError_t launch_theta_functional(const LatticeDesc& d, const void* links, double* workspace,
                                    double* out_theta, double* out_F, cudaStream_t st) {
  CULGT_DISPATCH(run_theta_functional, d, links, workspace, out_theta, out_F, st)
}

cudaError_t launch_coulomb_theta_functional(const LatticeDesc& d, const void* links, double* workspace,
                                            double* out_theta_t, double* out_F_t, cudaStream_t st) {
  CULGT_DISPATCH(run_coulomb_theta_functional, d, links, workspace, out_theta_t, out_F_t, st)
}

}  // namespace culgt
