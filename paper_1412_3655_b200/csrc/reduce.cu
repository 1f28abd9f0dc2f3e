// reduce.cu -- a7 functional F and a8 gauge precision theta, one fused pass.
//
//   F     = 1/(4 Nc V) sum_x sum_mu Re tr U_mu(x)                      PAPER.md eq. (2) at g = 1
//   theta = 1/(Nc V) sum_x tr[Delta(x) Delta(x)^dagger],  Delta(x) = [(K(x) - K(x)^dagger)/(2i)]_traceless
//           which equals sum_mu A_mu(x) - A_mu(x-mu) of eq. (1) (reading C-11).
// Reduction: per-thread fp64 partial -> warp xor-shuffles -> one shared-memory slot per warp ->
// one partial per block in the workspace -> a single block per quantity sums the partials in a
// fixed order.  Deterministic: no atomics, the same launch always produces the same bits.
// All arithmetic is fp64 on the stored values (12-parameter storage: third row rebuilt in fp64).
#include <stdlib.h>
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

__device__ __forceinline__ void cp_async16(void* smem, const void* gmem) {
  const unsigned s = (unsigned)__cvta_generic_to_shared(smem);
  asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(s), "l"(gmem) : "memory");
}


// What theta and F need of one link (reading C-11: Delta = [(K - K^dagger)/(2i)]_traceless depends only
// on the anti-Hermitian part of K, to which U_mu(x) and U_mu(x-mu)^dagger contribute with opposite signs):
//   a[0..2] = Im U_aa;   a[3], a[4] = Im U_01 + Im U_10, Re U_01 - Re U_10;   a[5], a[6]: (0,2);   a[7], a[8]: (1,2)
// and Re tr U.  acc += sign * a.  The stored rows are widened first; the third row of 12-parameter
// storage is rebuilt in fp64.
template <typename S>
__device__ __forceinline__ double add_antihermitian_parts(const typename S::Real* U, double sign, double* acc) {
  double m[18];
#pragma unroll
  for (int i = 0; i < S::NP; ++i) m[i] = (double)U[i];
  if (S::NP == 12) reconstruct_row2(m);
  acc[0] = fma(sign, m[CULGT_IM(0, 0)], acc[0]);
  acc[1] = fma(sign, m[CULGT_IM(1, 1)], acc[1]);
  acc[2] = fma(sign, m[CULGT_IM(2, 2)], acc[2]);
  acc[3] = fma(sign, m[CULGT_IM(0, 1)] + m[CULGT_IM(1, 0)], acc[3]);
  acc[4] = fma(sign, m[CULGT_RE(0, 1)] - m[CULGT_RE(1, 0)], acc[4]);
  acc[5] = fma(sign, m[CULGT_IM(0, 2)] + m[CULGT_IM(2, 0)], acc[5]);
  acc[6] = fma(sign, m[CULGT_RE(0, 2)] - m[CULGT_RE(2, 0)], acc[6]);
  acc[7] = fma(sign, m[CULGT_IM(1, 2)] + m[CULGT_IM(2, 1)], acc[7]);
  acc[8] = fma(sign, m[CULGT_RE(1, 2)] - m[CULGT_RE(2, 1)], acc[8]);
  return m[CULGT_RE(0, 0)] + m[CULGT_RE(1, 1)] + m[CULGT_RE(2, 2)];
}

// tr[Delta Delta^dagger] from the accumulated parts: the diagonal with its trace removed, and
// |D_ab|^2 + |D_ba|^2 = (s^2 + r^2)/2 for D_ab = (s - i r)/2.
__device__ __forceinline__ double theta_from_parts(const double* a) {
  const double tr = (a[0] + a[1] + a[2]) * (1.0 / 3.0);
  double sum = 0;
#pragma unroll
  for (int c = 0; c < 3; ++c) sum += (a[c] - tr) * (a[c] - tr);
#pragma unroll
  for (int c = 3; c < 9; ++c) sum = fma(0.5 * a[c], a[c], sum);
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
// STAGED = false: the links are loaded straight into registers, a batch of directions at a time.
// STAGED = true (SU(3)): all 2*ND links of the site are first copied into thread-private shared-memory
// slots by cp.async.cg, `[vector][thread]` so that a warp's copy of one vector is 512 contiguous bytes
// on both sides, one commit group per direction, and then widened and accumulated one link at a time
// as its direction lands: every load of the site is in flight at once without holding registers (the
// half-sweep's staging), and the conversions of direction mu overlap the loads of the
// later ones.  No __syncthreads: cp.async.wait_group orders a thread against its own copies.
// Measured and rejected: four threads per site with the parts exchanged through shared
// memory (commit 7e9a7e2: 72 us against 59 at 32^4 fp32-12 -- a third of the bytes in flight per SM),
// part of the fp32 -> fp64 conversions moved from the XU to the integer pipe (no change: the kernel is
// not bound by a pipe), staging through the L1 with cp.async.ca (82 us), a 4-D site tile per CTA in which
// every link is fetched and converted once (theta_functional_tile_kernel below: 79 us).
template <typename S, int BLOCK, bool COULOMB, bool STAGED>
__global__ void __launch_bounds__(BLOCK, STAGED ? 512 / BLOCK : 0)
theta_functional_kernel(const typename S::Vec* __restrict__ links, const Geom g,
                        double* __restrict__ partial_theta, double* __restrict__ partial_F,
                        const int* __restrict__ stop_flag) {
  typedef typename S::Real Real;
  if (stop_flag != nullptr && *stop_flag != 0) return;   // driver loop: this check is no longer wanted
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
      double a[9];
#pragma unroll
      for (int i = 0; i < 9; ++i) a[i] = 0;
      if constexpr (STAGED) {
        typedef typename S::Vec Vec;
        extern __shared__ __align__(16) unsigned char smem_raw[];
        Vec* const sm = reinterpret_cast<Vec*>(smem_raw) + threadIdx.x;   // vector v of link l at sm[(l*NV+v)*BLOCK]
#pragma unroll
        for (int mu = 0; mu < ND; ++mu) {
          const Vec* up = link_base<S>(links, g, parity, mu, h);
          const Vec* dn = link_base<S>(links, g, 1 - parity, mu, down_index(g, h, sc, mu));
#pragma unroll
          for (int j = 0; j < S::NV; ++j) {
            cp_async16(sm + ((2 * mu) * S::NV + j) * BLOCK, up + (size_t)j * (size_t)g.pitch);
            cp_async16(sm + ((2 * mu + 1) * S::NV + j) * BLOCK, dn + (size_t)j * (size_t)g.pitch);
          }
          asm volatile("cp.async.commit_group;" ::: "memory");   // one group per direction
        }
#pragma unroll
        for (int l = 0; l < 2 * ND; ++l) {
          if ((l & 1) == 0) {                    // direction l/2 has landed; the later ones are still in flight
            if (ND - 1 - l / 2 == 3) asm volatile("cp.async.wait_group 3;" ::: "memory");
            else if (ND - 1 - l / 2 == 2) asm volatile("cp.async.wait_group 2;" ::: "memory");
            else if (ND - 1 - l / 2 == 1) asm volatile("cp.async.wait_group 1;" ::: "memory");
            else asm volatile("cp.async.wait_group 0;" ::: "memory");
          }
          Real U[kLinkRegs];
#pragma unroll
          for (int j = 0; j < S::NV; ++j) vec_get(sm[(l * S::NV + j) * BLOCK], U + j * S::VL);
          const double tr = add_antihermitian_parts<S>(U, (l & 1) ? -1.0 : 1.0, a);
          if ((l & 1) == 0) f += tr;
        }
      } else {
      // the loads of a batch of directions are issued before any of them is used (memory-level
      // parallelism); fp32 storage batches 2 directions = 4 links, fp64 storage 1 direction
      constexpr int MU_BATCH = (sizeof(Real) == 4) ? 2 : 1;
#pragma unroll
      for (int mu0 = 0; mu0 < ND; mu0 += MU_BATCH) {
        Real U[2 * MU_BATCH][kLinkRegs];
#pragma unroll
        for (int b = 0; b < MU_BATCH; ++b)
          if (mu0 + b < ND) {
            load_params<S>(link_base<S>(links, g, parity, mu0 + b, h), g.pitch, U[2 * b]);
            load_params<S>(link_base<S>(links, g, 1 - parity, mu0 + b, down_index(g, h, sc, mu0 + b)), g.pitch,
                           U[2 * b + 1]);
          }
#pragma unroll
        for (int b = 0; b < MU_BATCH; ++b)
          if (mu0 + b < ND) {
            f += add_antihermitian_parts<S>(U[2 * b], 1.0, a);
            add_antihermitian_parts<S>(U[2 * b + 1], -1.0, a);
          }
      }
      }
      th = theta_from_parts(a);
    } else {
      double d[3] = {0, 0, 0};
#pragma unroll
      for (int mu = 0; mu < ND; ++mu) {
        Real u[4], w[4];
        load_params<S>(link_base<S>(links, g, parity, mu, h), g.pitch, u);
        load_params<S>(link_base<S>(links, g, 1 - parity, mu, down_index(g, h, sc, mu)), g.pitch, w);
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


// ---------------------------------------------------------------------------------------------------
// Landau gauge, SU(3): a 4-D SITE TILE per CTA, every link widened and reduced ONCE.
//
// theta needs, per site, the anti-Hermitian parts (9 reals, add_antihermitian_parts) of its 4 up links
// minus those of its 4 down links; a link is the up link of one site and the down link of the
// neighbouring site of the other parity.  The kernels above fetch and widen it twice.  Here a CTA owns
// the TX x T1 x T2 x T3 block of half indices (hx, x1, x2, x3) of BOTH parities (2*NT sites, one thread
// each): a thread loads its 4 up links, reduces each to its 9 reals, keeps them for its own sum and
// parks them in shared memory ([component][parity*4+mu][site], conflict-free); after one barrier it
// subtracts the parts of its down links, which its neighbours parked -- except on the tile's lower
// faces, where the down link belongs to another tile and is fetched and reduced directly (issued with
// the up links, before the barrier).  Link fetches per site: 4 + (1/(2 TX) + 1/T1 + 1/T2 + 1/T3)
// instead of 8; conversions and third-row rebuilds likewise.  Threads are ordered hx-fastest, so a
// warp reads runs of TX consecutive vectors of a plane.
// Requires nh0 % TX == 0, N1 % T1 == 0, N2 % T2 == 0, N3 % T3 == 0 (else the kernels above).
// ---------------------------------------------------------------------------------------------------
#ifdef CULGT_MEASURE
template <typename S>
__device__ __forceinline__ double link_parts(const typename S::Real* U, double* pr) {
#pragma unroll
  for (int c = 0; c < 9; ++c) pr[c] = 0;
  return add_antihermitian_parts<S>(U, 1.0, pr);
}

template <typename S, int TX, int T1, int T2, int T3, int MINB>
__global__ void __launch_bounds__(2 * TX * T1 * T2 * T3, MINB)
theta_functional_tile_kernel(const typename S::Vec* __restrict__ links, const Geom g, const int nbx, const int nb1,
                             const int nb2, double* __restrict__ partial_theta, double* __restrict__ partial_F,
                             const int* __restrict__ stop_flag) {
  typedef typename S::Real Real;
  constexpr int NT = TX * T1 * T2 * T3;          // sites of one parity per tile
  if (stop_flag != nullptr && *stop_flag != 0) return;
  extern __shared__ __align__(16) unsigned char smem_raw[];
  double* const parts = reinterpret_cast<double*>(smem_raw);      // [9][8 * NT]
  // tile origin
  int b = (int)blockIdx.x;
  const int bx = b % nbx; b /= nbx;
  const int b1 = b % nb1; b /= nb1;
  const int b2 = b % nb2;
  const int b3 = b / nb2;
  // my site
  const int p = (int)threadIdx.x / NT;
  const int lh = (int)threadIdx.x % NT;
  const int lhx = lh % TX, l1 = (lh / TX) % T1, l2 = (lh / (TX * T1)) % T2, l3 = lh / (TX * T1 * T2);
  SiteCoord sc;
  sc.hx = bx * TX + lhx;
  sc.x1 = b1 * T1 + l1;
  sc.x2 = b2 * T2 + l2;
  sc.x3 = b3 * T3 + l3;
  sc.odd = (sc.x1 + sc.x2 + sc.x3 + p) & 1;
  const int h = sc.hx + g.nh0 * (sc.x1 + g.n[1] * (sc.x2 + g.n[2] * sc.x3));
  // local index of the down neighbour inside the tile, or -1 when it belongs to another tile
  int nb_local[4];
  nb_local[0] = sc.odd ? lh : (lhx > 0 ? lh - 1 : -1);
  nb_local[1] = l1 > 0 ? lh - TX : -1;
  nb_local[2] = l2 > 0 ? lh - TX * T1 : -1;
  nb_local[3] = l3 > 0 ? lh - TX * T1 * T2 : -1;

  double a[9];
#pragma unroll
  for (int c = 0; c < 9; ++c) a[c] = 0;
  double f = 0;
  // all loads first: the 4 up links, and the down links that come from outside the tile
  Real Uu[4][kLinkRegs];
#pragma unroll
  for (int mu = 0; mu < 4; ++mu) load_params<S>(link_base<S>(links, g, p, mu, h), g.pitch, Uu[mu]);
#pragma unroll
  for (int mu = 0; mu < 4; ++mu) {
    if (nb_local[mu] < 0) {
      Real Ud[kLinkRegs];
      load_params<S>(link_base<S>(links, g, 1 - p, mu, down_index(g, h, sc, mu)), g.pitch, Ud);
      add_antihermitian_parts<S>(Ud, -1.0, a);
    }
  }
#pragma unroll
  for (int mu = 0; mu < 4; ++mu) {
    double pr[9];
    f += link_parts<S>(Uu[mu], pr);
#pragma unroll
    for (int c = 0; c < 9; ++c) {
      a[c] += pr[c];
      parts[(c * 8 + p * 4 + mu) * NT + lh] = pr[c];
    }
  }
  __syncthreads();
#pragma unroll
  for (int mu = 0; mu < 4; ++mu) {
    if (nb_local[mu] >= 0) {
#pragma unroll
      for (int c = 0; c < 9; ++c) a[c] -= parts[(c * 8 + (1 - p) * 4 + mu) * NT + nb_local[mu]];
    }
  }
  const double th = theta_from_parts(a);
  __syncthreads();
  const double st = block_sum<2 * NT>(th);
  __syncthreads();                       // block_sum's shared slots are reused
  const double sf = block_sum<2 * NT>(f);
  if (threadIdx.x == 0) {
    partial_theta[blockIdx.x] = st;
    partial_F[blockIdx.x] = sf;
  }
}
#endif  // CULGT_MEASURE

// Final pass of the per-slice (Coulomb) sums: block (group, quantity) sums the n partials of that group
// in a fixed order and scales.  partial = [quantity][group][n]; quantity 0 = theta, 1 = F; group = time-slice for the
// Coulomb sums, a single group for the Landau sums.
template <int BLOCK>
__global__ void __launch_bounds__(BLOCK)
final_sum_kernel(const double* __restrict__ partial, int n, double scale0, double scale1,
                 double* __restrict__ out0, double* __restrict__ out1, const int* __restrict__ stop_flag) {
  if (stop_flag != nullptr && *stop_flag != 0) return;   // driver loop has stopped: keep the last results
  const double* p = partial + ((size_t)blockIdx.y * gridDim.x + blockIdx.x) * (size_t)n;
  double acc = 0;
  for (int i = threadIdx.x; i < n; i += BLOCK) acc += p[i];
  const double s = block_sum<BLOCK>(acc);
  if (threadIdx.x == 0) {
    if (blockIdx.y == 0) out0[blockIdx.x] = s * scale0;
    else out1[blockIdx.x] = s * scale1;
  }
}

// Coulomb driver loop on the device (culgt_coulomb_fix): after a check, slice t stays active iff NOT
// theta_t < target (a NaN keeps it active); when no slice is active the stop word is raised and every
// sweep and check enqueued behind it returns at entry.  Slices decouple (reading C-22), so a frozen
// slice's theta_t never changes again.
__global__ void coulomb_mask_kernel(const double* __restrict__ theta_t, int n3, double target,
                                    unsigned char* __restrict__ mask, FixCtl* __restrict__ ctl, int sweeps_before) {
  if (ctl->stop != 0) return;
  __shared__ int any_active;
  if (threadIdx.x == 0) any_active = 0;
  __syncthreads();
  for (int t = threadIdx.x; t < n3; t += blockDim.x) {
    const bool active = !(theta_t[t] < target);
    mask[t] = active ? 1 : 0;
    if (active) any_active = 1;            // benign race: every writer stores 1
  }
  __syncthreads();
  if (threadIdx.x == 0) {
    ctl->checks_done += 1;
    if (!any_active) {
      ctl->sweeps_at_stop = sweeps_before;
      ctl->stop = 1;
    }
  }
}

// Landau gauge: ONE block sums the theta partials, then the F partials, each in a fixed order, scales,
// writes both scalars and -- when a driver loop is attached (FixCtl, kernels.h) -- does the loop's
// bookkeeping on the device: records theta and F, and raises `stop` once theta < theta_target, after
// which every sweep and check enqueued behind this one returns at entry ("iterated until the
// discrete gauge condition (1) is satisfied up to a given numerical precision").  A NaN theta never
// satisfies the test, so a non-finite field runs to max_sweeps.
template <int BLOCK>
__global__ void __launch_bounds__(BLOCK)
final_sum_landau_kernel(const double* __restrict__ partial, int n, double scale_theta, double scale_F,
                        double* __restrict__ out_theta, double* __restrict__ out_F, FixCtl* __restrict__ ctl,
                        double theta_target, int sweeps_before) {
  if (ctl != nullptr && ctl->stop != 0) return;
  // both quantities at once, four partials of each in flight per thread (the loads are what this
  // kernel waits for: one block, a few thousand partials)
  double at = 0, af = 0;
#pragma unroll 4
  for (int i = threadIdx.x; i < n; i += BLOCK) {
    at += partial[i];
    af += partial[(size_t)n + i];
  }
  const double st = block_sum<BLOCK>(at);
  __syncthreads();
  const double sf = block_sum<BLOCK>(af);
  if (threadIdx.x == 0) {
    const double theta = st * scale_theta, F = sf * scale_F;
    *out_theta = theta;
    *out_F = F;
    if (ctl != nullptr) {
      ctl->theta = theta;
      ctl->F = F;
      ctl->checks_done += 1;
      if (theta < theta_target) {
        ctl->sweeps_at_stop = sweeps_before;
        ctl->stop = 1;
      }
    }
  }
}

constexpr int kFinalBlock = 1024;      // threads of the single block that sums the Landau partials

template <typename S, int BLOCK, bool COULOMB>
static cudaError_t launch_theta_staged(dim3 grid, const void* links, const Geom& g, double* p_theta, double* p_F,
                                       const int* stop_flag, cudaStream_t st) {
  auto kern = theta_functional_kernel<S, BLOCK, COULOMB, true>;
  constexpr size_t smem = (size_t)8 * S::NV * BLOCK * sizeof(typename S::Vec);
  static bool configured[kMaxDevices] = {false};
  int dev = 0;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) return e;
  if (dev < 0 || dev >= kMaxDevices || !configured[dev]) {
    e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    if (dev >= 0 && dev < kMaxDevices) configured[dev] = true;
  }
  kern<<<grid, BLOCK, smem, st>>>((const typename S::Vec*)links, g, p_theta, p_F, stop_flag);
  return cudaGetLastError();
}

// fp32 12-parameter storage takes the staged kernel (measured); the others the register path
// fp32 12-parameter storage takes the staged kernel, 64 sites of each parity per 128-thread CTA, 4 CTAs
// per SM (measured at 32^4: 67 -> 60 us per check inside the sweep loop, 91 -> 56 us back to back;
// DESIGN.md 6.3); the other formats the register path with 128 sites of each parity per CTA.
// The 4-D tile kernel (theta_functional_tile_kernel) was measured and rejected (78.7 us
// against 57.5 us at 32^4 fp32-12, 697 against 482 us at 48^3 x 96): it fetches 5.3 instead of 8 links per
// site and converts each once, but keeps only a third of the bytes in flight per SM.  It is compiled only
// into the measurement build, where CULGT_THETA_TILE=1 selects it.
static bool theta_tile_enabled() {
#ifdef CULGT_MEASURE
  static int v = -1;
  if (v < 0) {
    const char* e = getenv("CULGT_THETA_TILE");
    v = e ? (e[0] != '0') : 0;
  }
  return v != 0;
#else
  return false;
#endif
}

template <typename S>
static constexpr bool theta_is_staged() { return S::NC == 3 && S::NP == 12 && sizeof(typename S::Real) == 4; }

// group_size sites of each parity per y-slot of the grid (the sublattice, or one time-slice of it);
// the partials of quantity 1 start at p_theta + ny * blocks
template <typename S, bool COULOMB>
static cudaError_t launch_theta_pass(int group_size, int ny, const void* links, const Geom& g, double* p_theta,
                                     const int* stop_flag, cudaStream_t st, int* blocks_out) {
#ifdef CULGT_MEASURE
  if constexpr (!COULOMB && S::NC == 3 && sizeof(typename S::Real) == 4 && S::NP == 12) {
    constexpr int TX = 8, T1 = 4, T2 = 2, T3 = 2, NT = TX * T1 * T2 * T3, MINB = 2;
    if (theta_tile_enabled() && g.nh0 % TX == 0 && g.n[1] % T1 == 0 && g.n[2] % T2 == 0 && g.n[3] % T3 == 0) {
      auto kern = theta_functional_tile_kernel<S, TX, T1, T2, T3, MINB>;
      constexpr size_t smem = (size_t)9 * 8 * NT * sizeof(double);
      static bool configured[kMaxDevices] = {false};
      int dev = 0;
      cudaError_t e = cudaGetDevice(&dev);
      if (e != cudaSuccess) return e;
      if (dev < 0 || dev >= kMaxDevices || !configured[dev]) {
        e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e != cudaSuccess) return e;
        if (dev >= 0 && dev < kMaxDevices) configured[dev] = true;
      }
      const int nbx = g.nh0 / TX, nb1 = g.n[1] / T1, nb2 = g.n[2] / T2, nb3 = g.n[3] / T3;
      const int nb = nbx * nb1 * nb2 * nb3;             // = vh / NT
      *blocks_out = nb;
      kern<<<nb, 2 * NT, smem, st>>>((const typename S::Vec*)links, g, nbx, nb1, nb2, p_theta, p_theta + nb, stop_flag);
      return cudaGetLastError();
    }
  }
#endif
  const int nb = reduce_blocks_fused(group_size, theta_is_staged<S>() ? 64 : 128);
  *blocks_out = nb;
  double* p_F = p_theta + (size_t)ny * nb;
  const dim3 grid(nb, ny);
  if constexpr (theta_is_staged<S>()) {
    return launch_theta_staged<S, 128, COULOMB>(grid, links, g, p_theta, p_F, stop_flag, st);
  } else {
    theta_functional_kernel<S, 256, COULOMB, false><<<grid, 256, 0, st>>>((const typename S::Vec*)links, g, p_theta,
                                                                                p_F, stop_flag);
    return cudaGetLastError();
  }
}

template <typename S>
static cudaError_t run_theta_functional(const LatticeDesc& d, const void* links, double* ws, double* out_theta,
                                        double* out_F, cudaStream_t st, const FixCheck* fix) {
  int nblk = 0;
  FixCtl* ctl = fix ? fix->ctl : nullptr;
  cudaError_t e = launch_theta_pass<S, false>(d.geom.vh, 1, links, d.geom, ws, ctl ? &ctl->stop : nullptr, st, &nblk);
  if (e != cudaSuccess) return e;
  final_sum_landau_kernel<kFinalBlock><<<1, kFinalBlock, 0, st>>>(
      ws, nblk, 1.0 / ((double)S::NC * (double)d.V), 1.0 / (4.0 * S::NC * (double)d.V), out_theta, out_F, ctl,
      fix ? fix->theta_target : 0.0, fix ? fix->sweeps_before : 0);
  return cudaGetLastError();
}

// Coulomb gauge: theta_t and F_t for every time-slice t (arrays of N3 doubles).
template <typename S>
static cudaError_t run_coulomb_theta_functional(const LatticeDesc& d, const void* links, double* ws,
                                                double* out_theta_t, double* out_F_t, cudaStream_t st,
                                                const CoulombCheck* chk) {
  const int n3 = d.geom.n[3];
  int nbx = 0;
  const int* stop = chk ? &chk->ctl->stop : nullptr;
  cudaError_t e = launch_theta_pass<S, true>(d.geom.stride[3], n3, links, d.geom, ws, stop, st, &nbx);
  if (e != cudaSuccess) return e;
  const double vs = (double)d.V / (double)n3;
  final_sum_kernel<kReduceBlock><<<dim3(n3, 2), kReduceBlock, 0, st>>>(
      ws, nbx, 1.0 / ((double)S::NC * vs), 1.0 / (3.0 * S::NC * vs), out_theta_t, out_F_t, stop);
  if ((e = cudaGetLastError()) != cudaSuccess || chk == nullptr) return e;
  coulomb_mask_kernel<<<1, 128, 0, st>>>(out_theta_t, n3, chk->theta_target, chk->mask, chk->ctl, chk->sweeps_before);
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
                                    double* out_theta, double* out_F, cudaStream_t st, const FixCheck* fix) {
  CULGT_DISPATCH(run_theta_functional, d, links, workspace, out_theta, out_F, st, fix)
}

// Raw sums of one time slab (scale 1): the caller combines the slabs (slab.cu).
template <typename S>
static cudaError_t run_theta_functional_sums(const LatticeDesc& d, const void* links, double* ws, double* out2,
                                             cudaStream_t st) {
  int nblk = 0;
  cudaError_t e = launch_theta_pass<S, false>(d.geom.vh, 1, links, d.geom, ws, nullptr, st, &nblk);
  if (e != cudaSuccess) return e;
  final_sum_landau_kernel<kFinalBlock><<<1, kFinalBlock, 0, st>>>(ws, nblk, 1.0, 1.0, out2, out2 + 1, nullptr, 0.0, 0);
  return cudaGetLastError();
}

cudaError_t launch_theta_functional_sums(const LatticeDesc& d, const void* links, double* workspace, double* out2,
                                         cudaStream_t st) {
  CULGT_DISPATCH(run_theta_functional_sums, d, links, workspace, out2, st)
}

cudaError_t launch_coulomb_theta_functional(const LatticeDesc& d, const void* links, double* workspace,
                                            double* out_theta_t, double* out_F_t, cudaStream_t st,
                                            const CoulombCheck* chk) {
  CULGT_DISPATCH(run_coulomb_theta_functional, d, links, workspace, out_theta_t, out_F_t, st, chk)
}

// ---------------------------------------------------------------------------------------------------
// theta + F for callers that cannot allocate (code under CUDA graph capture, serving loops, harnesses
// that forbid cudaMalloc): the same fused pass and the same kernels as launch_theta_functional, but the
// block partials live in a file-scope device array instead of a caller-supplied workspace.
//   * kNoAllocPartials doubles = 2 MiB, held by every GPU that loads the library until the process
//     exits.  It covers 2 quantities x V/128 partials (V/64 for fp32 12-parameter storage) up to
//     V = 2^24 sites (64^4) in every storage format; larger lattices are refused.
//   * In host code `g_noalloc_partials` is a host-side stand-in, NOT a device address: the device
//     address is resolved once per device, with that device current, by cudaGetSymbolAddress, and that
//     pointer is what the kernels get.
//   * Nothing in the array has to start at zero: every slot the final sum reads has been written by
//     the partial kernel of the same call, so the previous call's contents are simply overwritten.
//   * Every call on a device shares the array: two calls that overlap on the GPU (different streams)
//     race on it.  Calls on one stream are ordered and safe.
// No cudaMalloc / cudaFree / allocating library routine is called here or below.
// ---------------------------------------------------------------------------------------------------
constexpr size_t kNoAllocPartials = (size_t)1 << 18;                 // doubles: 2 MiB
static __device__ __align__(256) double g_noalloc_partials[kNoAllocPartials];

size_t noalloc_partials_needed(const LatticeDesc& d) {
  const bool staged = d.group == 3 && d.precision == 32 && d.params == 12;      // theta_is_staged
  return 2 * (size_t)reduce_blocks_fused(d.geom.vh, staged ? 64 : 128);
}

cudaError_t launch_theta_functional_noalloc(const LatticeDesc& d, const void* links, double* out_theta, double* out_F,
                                            cudaStream_t st) {
  if (noalloc_partials_needed(d) > kNoAllocPartials) return cudaErrorMemoryAllocation;   // mapped to CULGT_ERR_TOO_LARGE
  static double* scratch[kMaxDevices] = {nullptr};
  int dev = 0;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) return e;
  if (dev < 0 || dev >= kMaxDevices) return cudaErrorInvalidDevice;
  if (scratch[dev] == nullptr) {                 // set-up, once per device, with that device current
    double* ptr = nullptr;
    e = cudaGetSymbolAddress((void**)&ptr, g_noalloc_partials);
    if (e != cudaSuccess) return e;
    if (ptr == nullptr) return cudaErrorInvalidSymbol;
    scratch[dev] = ptr;
  }
  return launch_theta_functional(d, links, scratch[dev], out_theta, out_F, st, nullptr);
}

}  // namespace culgt
