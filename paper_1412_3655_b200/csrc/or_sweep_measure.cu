// or_sweep_measure.cu -- the MEASURED ALTERNATIVES of the SU(3) half-sweep (DESIGN.md 6.1,
// profiles/r1_variant_sweep.md), compiled only with -DCULGT_MEASURE (python -m
// paper_1412_3655_b200.build --measure).  None of this is in the product library:
//   * other thread-to-site mappings (2 / 4 / 8 threads per site with K(x) summed by xor-shuffles --
//     the paper's L62-72, L122 -- in registers or staged), persistent grid-stride grids, a 2-stage
//     software pipeline, L2 prefetch, chunked traversal, st.global.cs stores;
//   * measurement-only kernels that do NOT compute the method: all-fp32 arithmetic (misses the
//     2e-5 link tolerance), G = 1 (memory pattern only), K without the subgroup solve;
//   * the launch-level slab-blocked full sweep (variants 41-44, 51-54).
// They share the staging helpers of staged.cuh with the production kernel.
#ifdef CULGT_MEASURE
#include "staged.cuh"
#include "kernels.h"

namespace culgt {

// omega as a plain double for the all-fp32 measurement kernels (which only know the exact power)
__device__ __forceinline__ double power_omega(double w) { return w; }

// Option bits of the OPT template parameter.
constexpr int OPT_PREFETCH = 1;    // persistent only: prefetch.global.L2 of the next site block
constexpr int OPT_CHUNKED = 4;     // persistent only: contiguous chunk of site blocks per CTA
constexpr int OPT_NOMATH = 8;      // measurement only: G = 1 (memory pattern + products, no K / solve)
constexpr int OPT_FLAT = 16;       // one CTA per site block (hardware block scheduler), not persistent
constexpr int OPT_STREAM_ST = 32;  // st.global.cs stores
constexpr int OPT_NOSOLVE = 256;   // measurement only: K is accumulated but G = 1 (no subgroup solve)

template <typename S, typename Acc, int TPS, int BLOCK, int STAGES, int MINB, int OPT, typename Power>
__global__ void __launch_bounds__(BLOCK, MINB)
or_sweep_su3_measure_kernel(typename S::Vec* __restrict__ links, const Geom g, const int parity,
                           const Power omega, const int n_site_blocks, const int reverse,
                           const int block_lo) {
  typedef typename S::Real Real;
  typedef typename S::Vec Vec;
  constexpr int LPT = 8 / TPS;          // links per thread
  constexpr int NV = S::NV;             // vectors per link
  constexpr int NVT = LPT * NV;         // vectors per thread per stage
  constexpr int NR = (S::NP == 12) ? 2 : 3;
  extern __shared__ __align__(16) unsigned char smem_raw[];
  Vec* const sm = reinterpret_cast<Vec*>(smem_raw) + threadIdx.x;   // (stage, v) at sm[(stage*NVT+v)*BLOCK]
  const unsigned sm_addr = (unsigned)__cvta_generic_to_shared(sm);
  const int q = (int)threadIdx.x % TPS;

  // site blocks of this CTA: strided (b, b + grid, ...) or, with OPT bit 2, one contiguous chunk
  const int per_cta = (n_site_blocks + (int)gridDim.x - 1) / (int)gridDim.x;
  auto block_of = [&](int it) {
    const int b = (OPT & OPT_CHUNKED) ? (int)blockIdx.x * per_cta + it : it * (int)gridDim.x + (int)blockIdx.x;
    return block_lo + (reverse ? n_site_blocks - 1 - b : b);   // window [block_lo, block_lo + n_site_blocks)
  };
  auto issue = [&](const SiteRef<LPT>& r, int stage) {
    if (r.active) {
#pragma unroll
      for (int l = 0; l < LPT; ++l) {
#pragma unroll
        for (int j = 0; j < NV; ++j) {
          cp_async_vec(sm + (size_t)((stage * NVT + l * NV + j) * BLOCK),
                       vec_ptr<S, LPT>(links, g, parity, r, q, l, j));
        }
      }
    }
    cp_async_commit();
  };
  auto load_link = [&](int stage, int l, Real* U, auto vol) {
#pragma unroll
    for (int j = 0; j < NV; ++j) {
      Vec v;
      lds_vec<decltype(vol)::value>(sm_addr + (unsigned)((stage * NVT + l * NV + j) * BLOCK * (int)sizeof(Vec)), v);
      vec_get(v, U + j * S::VL);
    }
  };

  const int n_it = (OPT & OPT_CHUNKED) ? min(per_cta, n_site_blocks - (int)blockIdx.x * per_cta)
                            : (n_site_blocks - (int)blockIdx.x + (int)gridDim.x - 1) / (int)gridDim.x;
  if (n_it <= 0) return;

  // prologue: STAGES-1 sites in flight
  SiteRef<LPT> cur = locate<BLOCK, TPS>(g, parity, block_of(0), q);
  SiteRef<LPT> nxt = cur;
  if (STAGES == 1) {
    // nothing in flight yet
  } else {
    issue(cur, 0);
  }

  for (int it = 0; it < n_it; ++it) {
    const int stage = (STAGES == 1) ? 0 : (it & 1);
    if (STAGES == 1) {
      issue(cur, 0);
      if ((OPT & OPT_PREFETCH) && it + 1 < n_it) {
        // pull the NEXT site block's lines into L2 while this one is computed: the blocking
        // cp.async of the next iteration then pays L2 latency, not HBM latency
        nxt = locate<BLOCK, TPS>(g, parity, block_of(it + 1), q);
        if (nxt.active) {
#pragma unroll
          for (int l = 0; l < LPT; ++l)
#pragma unroll
            for (int j = 0; j < NV; ++j) prefetch_l2(vec_ptr<S, LPT>(links, g, parity, nxt, q, l, j));
        }
      }
      cp_async_wait<0>();
    } else {
      if (it + 1 < n_it) {
        nxt = locate<BLOCK, TPS>(g, parity, block_of(it + 1), q);
        issue(nxt, stage ^ 1);
        cp_async_wait<1>();
      } else {
        cp_async_wait<0>();
      }
    }

    Real G[18];
    if (OPT & OPT_NOMATH) {   // measurement only: memory pattern + apply, no K / solve (G = 1)
#pragma unroll
      for (int i = 0; i < 18; ++i) G[i] = (i == 0 || i == 8 || i == 16) ? (Real)1 : (Real)0;
    } else {
    // ---- K(x) = sum_mu U_mu(x) + U_mu(x-mu)^dagger                     (eq. 3)
    Acc K[18];
#pragma unroll
    for (int i = 0; i < 18; ++i) K[i] = 0;
#pragma unroll
    for (int l = 0; l < LPT; ++l) {
      Real U[kLinkRegs];
      asm volatile("" ::: "memory");   // keep the shared-memory reads of link l behind link l-1's use
      load_link(stage, l, U, std::false_type());
      if (S::NP == 12 && sizeof(Real) < sizeof(Acc)) {
        // fp32 12-parameter storage: widen the two stored rows and rebuild the third row in
        // fp64 for K.  A third row rebuilt in fp32 puts ~1e-7 into K, which the small-|p| sites
        // of a hot 10^7-site lattice amplify past the 2e-5 link tolerance; it also
        // needs 12 instead of 18 fp32->fp64 conversions per link.
        Acc Ua[18];
#pragma unroll
        for (int i = 0; i < 12; ++i) Ua[i] = (Acc)U[i];
        reconstruct_row2(Ua);
        accumulate(K, Ua, ((q * LPT + l) & 1) != 0);
      } else {
        if (S::NP == 12) reconstruct_row2(U);
        accumulate(K, U, ((q * LPT + l) & 1) != 0);
      }
    }
#pragma unroll
    for (int m = 1; m < TPS; m <<= 1) {
#pragma unroll
      for (int i = 0; i < 18; ++i) K[i] += __shfl_xor_sync(0xffffffffu, K[i], m);
    }

    // ---- G(x): subgroup loop with g^omega                              (L50-54)
    if (sizeof(Acc) == 8) {
      double Kd[18];
#pragma unroll
      for (int i = 0; i < 18; ++i) Kd[i] = (double)K[i];
      // G = g_3 g_2 g_1 is accumulated in fp64 and rounded once: accumulating it in fp32 costs
      // 0.7 % less time but doubles the worst link error at 32^4 (1.08e-5 vs 5.8e-6)
      double Gd[18];
      if (OPT & OPT_NOSOLVE) {
        double acc = 0;
#pragma unroll
        for (int i = 0; i < 18; ++i) { acc += Kd[i]; Gd[i] = (i == 0 || i == 8 || i == 16) ? 1.0 : 0.0; }
        Gd[1] = acc * 1e-300;      // keeps K alive
      } else if (cur.active) {
        // idle lanes of a ragged last block hold uninitialised shared memory: they must not enter
        // the solve (the heat bath's rejection loop would never end on NaN input)
        su3_solve<(sizeof(Real) == 8), double>(Kd, Gd, omega, cur.site);
      } else {
#pragma unroll
        for (int i = 0; i < 18; ++i) Gd[i] = 0.0;
      }
#pragma unroll
      for (int i = 0; i < 18; ++i) G[i] = (Real)Gd[i];
    } else {
      Acc Ga[18];
      su3_site_G(K, Ga, (Acc)power_omega(omega));
#pragma unroll
      for (int i = 0; i < 18; ++i) G[i] = (Real)Ga[i];
    }

    }
    // ---- U_mu(x) <- G U_mu(x),  U_mu(x-mu) <- U_mu(x-mu) G^dagger      (L19-21, L48)
    if (cur.active) {
#pragma unroll
      for (int l = 0; l < LPT; ++l) {
        Real U[kLinkRegs], R[kLinkRegs];
        R[18] = 0; R[19] = 0;
        asm volatile("" ::: "memory");
        load_link(stage, l, U, std::true_type());
        if (((q * LPT + l) & 1) == 0) {
          if (S::NP == 12) reconstruct_row2(U);
          mul_ab<NR>(G, U, R);
        } else {
          mul_abd<NR>(U, G, R);
        }
#pragma unroll
        for (int j = 0; j < NV; ++j) {
          Vec v;
          vec_set(v, R + j * S::VL);
          if (OPT & OPT_STREAM_ST) st_cs(vec_ptr<S, LPT>(links, g, parity, cur, q, l, j), v);
          else *vec_ptr<S, LPT>(links, g, parity, cur, q, l, j) = v;
        }
      }
    }
    if (STAGES == 1 && !(OPT & OPT_PREFETCH)) {
      if (it + 1 < n_it) cur = locate<BLOCK, TPS>(g, parity, block_of(it + 1), q);
    } else {
      cur = nxt;
    }
  }
}

// ---------------------------------------------------------------------------------------------
// host side
// ---------------------------------------------------------------------------------------------
template <typename S, typename Acc, int TPS, int BLOCK, int STAGES, int MINB, int OPT>
static cudaError_t launch_measure(void* links, const Geom& g, int parity, double omega, bool reverse_odd,
                                  cudaStream_t st, int win_lo = 0, int win_n = -1, int win_reverse = -1) {
  typedef typename S::Vec Vec;
  auto kern = or_sweep_su3_measure_kernel<S, Acc, TPS, BLOCK, STAGES, MINB, OPT, double>;
  constexpr size_t smem = (size_t)STAGES * (8 / TPS) * S::NV * BLOCK * sizeof(Vec);
  cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
  if (e != cudaSuccess) return e;
  constexpr int SITES = BLOCK / TPS;
  const int n_site_blocks = win_n >= 0 ? win_n : (g.vh + SITES - 1) / SITES;
  if (n_site_blocks == 0) return cudaSuccess;
  int grid = (OPT & OPT_FLAT) ? n_site_blocks : device_sm_count() * MINB;
  if (grid > n_site_blocks) grid = n_site_blocks;
  const int rev = win_reverse >= 0 ? win_reverse : ((reverse_odd && parity) ? 1 : 0);
  kern<<<grid, BLOCK, smem, st>>>((Vec*)links, g, parity, omega, n_site_blocks, rev, win_lo);
  return cudaGetLastError();
}

// Staged alternatives.  "AxB" = A threads per CTA, B CTAs per SM; "flat" = one CTA per site block,
// "pers" = persistent grid-stride loop; tps = threads per site.
static cudaError_t launch_measure_staged(const LatticeDesc& d, void* links, int parity, double omega, int variant,
                                         cudaStream_t st) {
  const Geom& g = d.geom;
  if (d.precision == 32 && d.params == 12) {
    typedef Storage<float, 3, 12> S;
    switch (variant) {
      case 21: return launch_measure<S, double, 1, 256, 1, 2, 0>(links, g, parity, omega, true, st);          // pers
      case 22: return launch_measure<S, double, 1, 128, 2, 2, 0>(links, g, parity, omega, true, st);          // pers, 2 stages
      case 23: return launch_measure<S, double, 2, 256, 1, 2, 0>(links, g, parity, omega, true, st);          // 2 tps, pers
      case 25: return launch_measure<S, float, 1, 128, 1, 4, OPT_FLAT>(links, g, parity, omega, true, st);    // all-fp32
      case 26: return launch_measure<S, double, 1, 256, 1, 2, OPT_PREFETCH>(links, g, parity, omega, true, st);
      case 27: return launch_measure<S, double, 1, 256, 1, 2, OPT_CHUNKED>(links, g, parity, omega, true, st);
      case 28: return launch_measure<S, double, 1, 128, 1, 4, OPT_FLAT | OPT_NOMATH>(links, g, parity, omega, true, st);
      case 29: return launch_measure<S, double, 1, 128, 1, 4, OPT_FLAT | OPT_STREAM_ST>(links, g, parity, omega, true, st);
      case 30: return launch_measure<S, double, 1, 256, 1, 2, OPT_FLAT>(links, g, parity, omega, true, st);
      case 31: return launch_measure<S, double, 1, 32, 1, 16, OPT_FLAT>(links, g, parity, omega, true, st);
      case 32: return launch_measure<S, double, 1, 128, 1, 4, OPT_FLAT | OPT_NOSOLVE>(links, g, parity, omega, true, st);
      default: return cudaErrorInvalidValue;
    }
  }
  if (d.precision == 32) {
    typedef Storage<float, 3, 18> S;
    switch (variant) {
      case 21: return launch_measure<S, double, 1, 128, 1, 2, 0>(links, g, parity, omega, true, st);          // pers
      case 22: return launch_measure<S, double, 2, 256, 1, 2, 0>(links, g, parity, omega, true, st);          // 2 tps, pers
      case 23: return launch_measure<S, double, 2, 256, 1, 2, OPT_FLAT>(links, g, parity, omega, true, st);
      case 30: return launch_measure<S, double, 1, 128, 1, 2, OPT_FLAT>(links, g, parity, omega, true, st);
      default: return cudaErrorInvalidValue;
    }
  }
  if (d.params == 12) {
    typedef Storage<double, 3, 12> S;
    switch (variant) {
      case 21: return launch_measure<S, double, 1, 128, 1, 2, 0>(links, g, parity, omega, true, st);          // pers
      case 22: return launch_measure<S, double, 2, 256, 1, 2, 0>(links, g, parity, omega, true, st);          // 2 tps, pers
      case 23: return launch_measure<S, double, 4, 256, 1, 2, 0>(links, g, parity, omega, true, st);          // 4 tps, pers
      case 30: return launch_measure<S, double, 1, 128, 1, 2, OPT_FLAT>(links, g, parity, omega, true, st);
      default: return cudaErrorInvalidValue;
    }
  }
  typedef Storage<double, 3, 18> S;
  switch (variant) {
    case 21: return launch_measure<S, double, 1, 192, 1, 1, 0>(links, g, parity, omega, true, st);            // pers
    case 22: return launch_measure<S, double, 2, 192, 1, 2, 0>(links, g, parity, omega, true, st);            // 2 tps, pers
    case 23: return launch_measure<S, double, 4, 256, 1, 2, 0>(links, g, parity, omega, true, st);            // 4 tps, pers
    case 26: return launch_measure<S, double, 1, 192, 1, 1, OPT_PREFETCH>(links, g, parity, omega, true, st);
    case 27: return launch_measure<S, double, 1, 192, 1, 1, OPT_CHUNKED>(links, g, parity, omega, true, st);
    case 28: return launch_measure<S, double, 1, 64, 1, 3, OPT_FLAT | OPT_NOMATH>(links, g, parity, omega, true, st);
    case 30: return launch_measure<S, double, 1, 192, 1, 1, OPT_FLAT>(links, g, parity, omega, true, st);
    case 31: return launch_measure<S, double, 1, 32, 1, 6, OPT_FLAT>(links, g, parity, omega, true, st);
    case 32: return launch_measure<S, double, 1, 96, 2, 1, 0>(links, g, parity, omega, true, st);             // pers, 2 stages
    default: return cudaErrorInvalidValue;
  }
}

// ---------------------------------------------------------------------------------------------
// First-generation kernels: all links of a site in registers, TPS threads per site (the paper's
// 1 / 4 / 8 threads per site, L62-72, L122): each of the TPS cooperating lanes owns 8/TPS links,
// the partial K are summed by xor-shuffles (the warp-level analogue of the paper's shared-memory
// exchange) and every lane then holds the same K and computes the same G.
// ---------------------------------------------------------------------------------------------
template <typename T>
__device__ __forceinline__ T shfl_xor_t(T v, int mask);
template <>
__device__ __forceinline__ float shfl_xor_t<float>(float v, int mask) { return __shfl_xor_sync(0xffffffffu, v, mask); }
template <>
__device__ __forceinline__ double shfl_xor_t<double>(double v, int mask) { return __shfl_xor_sync(0xffffffffu, v, mask); }

template <typename S, typename Acc, int TPS, int BLOCK>
__global__ void __launch_bounds__(BLOCK)
or_sweep_su3_direct_kernel(typename S::Vec* __restrict__ links, const Geom g, const int parity, const Acc omega) {
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
  for (int l = 0; l < LPT; ++l) load_params<S>(ptr[l], g.pitch, U[l]);
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
    store_params<S>(ptr[l], g.pitch, R);
  }
}

template <typename S, typename Acc, int TPS>
static cudaError_t launch_direct(void* links, const Geom& g, int parity, double omega, cudaStream_t st) {
  constexpr int BLOCK = 128;
  const long long threads = (long long)g.vh * TPS;
  const unsigned grid = (unsigned)((threads + BLOCK - 1) / BLOCK);
  or_sweep_su3_direct_kernel<S, Acc, TPS, BLOCK><<<grid, BLOCK, 0, st>>>(
      (typename S::Vec*)links, g, parity, (Acc)omega);
  return cudaGetLastError();
}

// fp32 storage: K and the subgroup solve in fp64 (reading C-15); variants 10+ are
// all-fp32 arithmetic, kept for the precision/throughput comparison in profiles/.
cudaError_t launch_or_sweep_measure(const LatticeDesc& d, void* links, int parity, double omega, int variant,
                                    cudaStream_t st) {
  const Geom& g = d.geom;
  if (d.group != 3) return cudaErrorInvalidValue;
  if (variant >= 20) return launch_measure_staged(d, links, parity, omega, variant, st);
  if (d.precision == 32) {
    if (d.params == 12) {
      switch (variant) {
        case 1: return launch_direct<Storage<float, 3, 12>, double, 1>(links, g, parity, omega, st);
        case 2: return launch_direct<Storage<float, 3, 12>, double, 2>(links, g, parity, omega, st);
        case 4: return launch_direct<Storage<float, 3, 12>, double, 4>(links, g, parity, omega, st);
        case 11: return launch_direct<Storage<float, 3, 12>, float, 1>(links, g, parity, omega, st);
        case 14: return launch_direct<Storage<float, 3, 12>, float, 4>(links, g, parity, omega, st);
        default: return cudaErrorInvalidValue;
      }
    }
    switch (variant) {
      case 2: return launch_direct<Storage<float, 3, 18>, double, 2>(links, g, parity, omega, st);
      case 4: return launch_direct<Storage<float, 3, 18>, double, 4>(links, g, parity, omega, st);
      default: return cudaErrorInvalidValue;
    }
  }
  if (d.params == 12) {
    switch (variant) {
      case 4: return launch_direct<Storage<double, 3, 12>, double, 4>(links, g, parity, omega, st);
      case 2: return launch_direct<Storage<double, 3, 12>, double, 2>(links, g, parity, omega, st);
      case 8: return launch_direct<Storage<double, 3, 12>, double, 8>(links, g, parity, omega, st);
      default: return cudaErrorInvalidValue;
    }
  }
  switch (variant) {
    case 4: return launch_direct<Storage<double, 3, 18>, double, 4>(links, g, parity, omega, st);
    case 8: return launch_direct<Storage<double, 3, 18>, double, 8>(links, g, parity, omega, st);
    default: return cudaErrorInvalidValue;
  }
}

// ---------------------------------------------------------------------------------------------
// Launch-level slab-blocked FULL sweep (variants 40 + k: slabs of 2^k time-slices): the black and
// the white half-sweep interleaved slab by slab along t as windowed launches of the production
// kernel.  With slab ends e_k = min((k+1)*sl, N3):
//     for k:  black slices [k*sl, e_k)  ascending;   white slices [max(1, k*sl - 1), e_k - 1)  descending
//     then    white slice N3-1, white slice 0.
// Measured and rejected (every windowed launch pays its own ramp-up and drain); the
// one-kernel version of the same idea is or_sweep_fused.cu.
// Returns cudaErrorNotSupported when the lattice does not split into whole site blocks per slice.
// ---------------------------------------------------------------------------------------------
cudaError_t launch_or_sweep_measure_slabbed(const LatticeDesc& d, void* links, double omega, int sl, cudaStream_t st) {
  const Geom& g = d.geom;
  const int n3 = g.n[3];
  if (d.group != 3 || sl < 2 || n3 < 4 || sl > n3 - 2) return cudaErrorNotSupported;
  cudaError_t e;
  for (int k = 0; k * sl < n3; ++k) {
    const int s_k = k * sl, e_k = (k + 1) * sl < n3 ? (k + 1) * sl : n3;
    if ((e = launch_or_sweep_window(d, links, 0, omega, s_k, e_k, st)) != cudaSuccess) return e;
    if ((e = launch_or_sweep_window(d, links, 1, omega, s_k > 1 ? s_k - 1 : 1, e_k - 1, st)) != cudaSuccess) return e;
  }
  if ((e = launch_or_sweep_window(d, links, 1, omega, n3 - 1, n3, st)) != cudaSuccess) return e;
  return launch_or_sweep_window(d, links, 1, omega, 0, 1, st);
}

}  // namespace culgt
#endif  // CULGT_MEASURE
