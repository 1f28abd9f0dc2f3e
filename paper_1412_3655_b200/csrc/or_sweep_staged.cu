// or_sweep_staged.cu -- the production SU(3) half-sweep kernel.
//
// Same mathematics as or_sweep.cu (eq. 3; L19-21), different machine mapping:
//
//  * The 8 links of a site are moved global -> shared memory by per-thread cp.async (LDGSTS)
//    into slots that only the issuing thread reads back (slot layout [stage][vector][thread],
//    16-byte vectors, so every LDS.128 / cp.async of a warp is 512 contiguous bytes and
//    conflict-free).  No block barrier is needed: cp.async.wait_group orders a thread against its
//    own copies.  The paper's obstacle (L72: 8 x 18 link registers do not fit a thread) is solved
//    on B200 by parking the links in the 228 KB of shared memory per SM instead of splitting the
//    site over 4 or 8 threads and paying the K(x) exchange.
//  * Registers then hold only K (fp64), G and one link at a time: 126 registers for fp32
//    storage, no spills in any format.
//  * Grid: ONE small CTA per site block (128 threads x 4 CTAs/SM for fp32-12, 64 x 3 for fp64-18),
//    handed out in order by the hardware block scheduler.  A persistent grid-stride loop (kept as
//    a variant) keeps every CTA of an SM in the same load-then-compute phase and measures 8-23 %
//    slower; small CTAs that retire and are replaced one at a time keep loads, arithmetic and
//    stores of different CTAs overlapped.  Odd-parity launches map blockIdx to site blocks in
//    DESCENDING order so that the white half-sweep starts on the links the black half-sweep
//    touched last, which are still in the 126 MB L2.
//  * One thread per site for every storage format (TPS = 1); TPS = 2, 4 (partial K by
//    xor-shuffle, the subgroup solve repeated per thread) are kept as measured alternatives.
//  * K accumulation, the subgroup chain and G in fp64 (su3_solve.cuh); reconstruction and link
//    products in the storage precision.
#include <type_traits>
#include "lattice.cuh"
#include "su_math.cuh"
#include "su3_solve.cuh"
#include "kernels.h"

namespace culgt {

// omega as a plain double for the all-fp32 measurement kernels (which only know the exact power)
__device__ __forceinline__ double power_omega(double w) { return w; }
__device__ __forceinline__ double power_omega(const ExactPower& p) { return p.omega; }
__device__ __forceinline__ double power_omega(const SeriesPower&) { return 0.0; }
__device__ __forceinline__ double power_omega(const HeatBathPower&) { return 0.0; }
__device__ __forceinline__ double power_omega(const MicroPower&) { return 0.0; }

// Option bits of the OPT template parameter.
constexpr int OPT_PREFETCH = 1;    // persistent only: prefetch.global.L2 of the next site block
constexpr int OPT_CHUNKED = 4;     // persistent only: contiguous chunk of site blocks per CTA
constexpr int OPT_NOMATH = 8;      // measurement only: G = 1 (memory pattern + products, no K / solve)
constexpr int OPT_FLAT = 16;       // one CTA per site block (hardware block scheduler), not persistent
constexpr int OPT_STREAM_ST = 32;  // st.global.cs stores
constexpr int OPT_NOSOLVE = 256;   // measurement only: K is accumulated but G = 1 (no subgroup solve)
constexpr int OPT_PDL = 512;       // programmatic dependent launch: the next half-sweep's CTAs are scheduled
                                   // (index arithmetic done) while this one's last wave drains
constexpr int OPT_L2HINT = 1024;   // flat grid only: L2 eviction hints by position in the traversal.  The CTAs from
                                   // `late_from` on (the last ~90 MB of links a launch touches, which the next,
                                   // reversed launch revisits first) store with evict_last and load normally; the
                                   // earlier ones load with evict_first (their lines cannot survive until they are
                                   // revisited) and store normally.  late_from < 0: no preference anywhere.
constexpr int OPT_COULOMB = 64;    // Coulomb gauge (reading C-22): K(x) from the 6 spatial links only

__device__ __forceinline__ void cp_async_vec(float4* smem, const float4* gmem) {
  const unsigned s = (unsigned)__cvta_generic_to_shared(smem);
  asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(s), "l"(gmem) : "memory");
}
__device__ __forceinline__ void cp_async_vec(double2* smem, const double2* gmem) {
  const unsigned s = (unsigned)__cvta_generic_to_shared(smem);
  asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(s), "l"(gmem) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
// Shared-memory reads as asm.  VOL = true emits ld.volatile: ptxas otherwise recognises the apply
// pass's reads as repeats of the K pass's reads and keeps all 8 links live in registers across the
// subgroup solve (spilling them), which is exactly what the staging exists to avoid.
template <bool VOL>
__device__ __forceinline__ void lds_vec(unsigned addr, float4& v) {
  if (VOL) asm volatile("ld.volatile.shared.v4.f32 {%0, %1, %2, %3}, [%4];" : "=f"(v.x), "=f"(v.y), "=f"(v.z), "=f"(v.w) : "r"(addr));
  else asm volatile("ld.shared.v4.f32 {%0, %1, %2, %3}, [%4];" : "=f"(v.x), "=f"(v.y), "=f"(v.z), "=f"(v.w) : "r"(addr));
}
template <bool VOL>
__device__ __forceinline__ void lds_vec(unsigned addr, double2& v) {
  if (VOL) asm volatile("ld.volatile.shared.v2.f64 {%0, %1}, [%2];" : "=d"(v.x), "=d"(v.y) : "r"(addr));
  else asm volatile("ld.shared.v2.f64 {%0, %1}, [%2];" : "=d"(v.x), "=d"(v.y) : "r"(addr));
}
__device__ __forceinline__ void st_cs(float4* p, const float4& v) {
  asm volatile("st.global.cs.v4.f32 [%0], {%1, %2, %3, %4};" ::"l"(p), "f"(v.x), "f"(v.y), "f"(v.z), "f"(v.w) : "memory");
}
__device__ __forceinline__ void st_cs(double2* p, const double2& v) {
  asm volatile("st.global.cs.v2.f64 [%0], {%1, %2};" ::"l"(p), "d"(v.x), "d"(v.y) : "memory");
}
__device__ __forceinline__ void st_hint(float4* p, const float4& v, uint64_t pol) {
  asm volatile("st.global.L2::cache_hint.v4.f32 [%0], {%1, %2, %3, %4}, %5;" ::"l"(p), "f"(v.x), "f"(v.y), "f"(v.z),
               "f"(v.w), "l"(pol) : "memory");
}
__device__ __forceinline__ void st_hint(double2* p, const double2& v, uint64_t pol) {
  asm volatile("st.global.L2::cache_hint.v2.f64 [%0], {%1, %2}, %3;" ::"l"(p), "d"(v.x), "d"(v.y), "l"(pol) : "memory");
}
template <typename V>
__device__ __forceinline__ void cp_async_vec_hint(V* smem, const V* gmem, uint64_t pol) {
  const unsigned s = (unsigned)__cvta_generic_to_shared(smem);
  asm volatile("cp.async.cg.shared.global.L2::cache_hint [%0], [%1], 16, %2;" ::"r"(s), "l"(gmem), "l"(pol) : "memory");
}
__device__ __forceinline__ void prefetch_l2(const void* gmem) {
  asm volatile("prefetch.global.L2 [%0];" ::"l"(gmem));
}
template <int N>
__device__ __forceinline__ void cp_async_wait() { asm volatile("cp.async.wait_group %0;" ::"n"(N) : "memory"); }

// What one thread needs to know about the site it works on: the half index of each of its LPT
// links (slot = q*LPT + l = 2*mu + down; up links sit at the site's own index h in this parity's
// sublattice, down links at the index of x - mu in the other parity's).
template <int LPT>
struct SiteRef {
  int idx[LPT];
  unsigned site;   // canonical site index (selects the heat bath's random numbers)
  bool active;
};

template <int BLOCK, int TPS, bool MASKED>
__device__ __forceinline__ SiteRef<8 / TPS> locate(const Geom& g, int parity, int site_block, int q) {
  constexpr int LPT = 8 / TPS;
  SiteRef<LPT> r;
  int h = site_block * (BLOCK / TPS) + (int)threadIdx.x / TPS;
  r.active = h < g.vh;
  if (!r.active) h = g.vh - 1;
  const SiteCoord sc = decode_site(g, h, parity);
  r.site = (unsigned)canonical_site(g, h, sc);
  if (MASKED && g.slice_active != nullptr && g.slice_active[sc.x3] == 0) r.active = false;   // frozen slice
#pragma unroll
  for (int l = 0; l < LPT; ++l) {
    const int slot = q * LPT + l;
    r.idx[l] = (slot & 1) ? down_index(g, h, sc, slot >> 1) : h;
  }
  return r;
}

// Global address of vector j of this thread's link l: a plane base that does not depend on the
// thread (for TPS = 1 it is uniform over the grid, so it lives in uniform registers) plus the
// 32-bit half index -- this keeps 64-bit per-thread address arithmetic out of the inner loops.
template <typename S, int LPT>
__device__ __forceinline__ typename S::Vec* vec_ptr(typename S::Vec* links, const Geom& g, int parity,
                                                    const SiteRef<LPT>& r, int q, int l, int j) {
  const int slot = q * LPT + l;
  const int plane = (((slot & 1) ? 1 - parity : parity) * 4 + (slot >> 1)) * S::NV + j;
  typename S::Vec* base = links + (size_t)plane * (size_t)g.vh;
  return base + (unsigned)r.idx[l];
}

template <typename S, typename Acc, int TPS, int BLOCK, int STAGES, int MINB, int OPT, typename Power>
__global__ void __launch_bounds__(BLOCK, MINB)
or_sweep_su3_staged_kernel(typename S::Vec* __restrict__ links, const Geom g, const int parity,
                           const Power omega, const int n_site_blocks, const int reverse,
                           const int block_lo, const int late_from) {
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
  constexpr bool L2HINT = (OPT & OPT_L2HINT) != 0;
  uint64_t pol = 0, pol_st = 0;
  if (L2HINT) {
    uint64_t pf, pn, pl;
    asm("createpolicy.fractional.L2::evict_first.b64 %0, 1.0;" : "=l"(pf));
    asm("createpolicy.fractional.L2::evict_normal.b64 %0, 1.0;" : "=l"(pn));
    asm("createpolicy.fractional.L2::evict_last.b64 %0, 1.0;" : "=l"(pl));
    const bool late = (int)blockIdx.x >= late_from;
    pol = (late_from < 0 || late) ? pn : pf;
    pol_st = (late_from >= 0 && late) ? pl : pn;
  }
  auto issue = [&](const SiteRef<LPT>& r, int stage) {
    if (r.active) {
#pragma unroll
      for (int l = 0; l < LPT; ++l) {
#pragma unroll
        for (int j = 0; j < NV; ++j) {
          if (L2HINT) cp_async_vec_hint(sm + (size_t)((stage * NVT + l * NV + j) * BLOCK),
                                        (const Vec*)vec_ptr<S, LPT>(links, g, parity, r, q, l, j), pol);
          else cp_async_vec(sm + (size_t)((stage * NVT + l * NV + j) * BLOCK),
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
  SiteRef<LPT> cur = locate<BLOCK, TPS, (OPT & OPT_COULOMB) != 0>(g, parity, block_of(0), q);
  SiteRef<LPT> nxt = cur;
  if (OPT & OPT_PDL) {
    // let the next launch of the stream be scheduled as soon as every CTA of this one has started,
    // then wait until the previous launch has completed and its stores are visible
    pdl_prologue_done();
  }
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
        nxt = locate<BLOCK, TPS, (OPT & OPT_COULOMB) != 0>(g, parity, block_of(it + 1), q);
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
        nxt = locate<BLOCK, TPS, (OPT & OPT_COULOMB) != 0>(g, parity, block_of(it + 1), q);
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
      if ((OPT & OPT_COULOMB) && ((q * LPT + l) >> 1) == 3) continue;   // time links do not enter K_C
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
          if (L2HINT) st_hint(vec_ptr<S, LPT>(links, g, parity, cur, q, l, j), v, pol_st);
          else if (OPT & OPT_STREAM_ST) st_cs(vec_ptr<S, LPT>(links, g, parity, cur, q, l, j), v);
          else *vec_ptr<S, LPT>(links, g, parity, cur, q, l, j) = v;
        }
      }
    }
    if (STAGES == 1 && !(OPT & OPT_PREFETCH)) {
      if (it + 1 < n_it) cur = locate<BLOCK, TPS, (OPT & OPT_COULOMB) != 0>(g, parity, block_of(it + 1), q);
    } else {
      cur = nxt;
    }
  }
}

// ---------------------------------------------------------------------------------------------
// host side
// ---------------------------------------------------------------------------------------------
static int sm_count() {
  static int n = 0;
  if (n == 0) {
    int dev = 0;
    cudaGetDevice(&dev);
    if (cudaDeviceGetAttribute(&n, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess || n <= 0) n = 148;
  }
  return n;
}

template <typename S, typename Acc, int TPS, int BLOCK, int STAGES, int MINB, int OPT, typename Power>
static cudaError_t launch_staged(void* links, const Geom& g, int parity, Power omega, bool reverse_odd,
                                 cudaStream_t st, int win_lo = 0, int win_n = -1, int win_reverse = -1) {
  typedef typename S::Vec Vec;
  if constexpr ((OPT & OPT_L2HINT) != 0) {
    // The hints pay where the field is a small multiple of the 126 MB L2 (measured: 201 MB 58.4 -> 55.0 us,
    // 604 MB 177.3 -> 176.9, 2.0 GB 617 -> 627, 9.7 GB 2863 -> 2924): elsewhere, and for the windowed
    // (slab) launches, the same mapping without them.
    const double field_bytes = 8.0 * (double)g.vh * S::NV * sizeof(Vec);
    if (win_n >= 0 || field_bytes < 110e6 || field_bytes > 700e6)
      return launch_staged<S, Acc, TPS, BLOCK, STAGES, MINB, OPT & ~OPT_L2HINT, Power>(links, g, parity, omega, reverse_odd,
                                                                                       st, win_lo, win_n, win_reverse);
  }
  auto kern = or_sweep_su3_staged_kernel<S, Acc, TPS, BLOCK, STAGES, MINB, OPT, Power>;
  constexpr size_t smem = (size_t)STAGES * (8 / TPS) * S::NV * BLOCK * sizeof(Vec);
  static bool configured = false;
  if (!configured) {
    cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    configured = true;
  }
  constexpr int SITES = BLOCK / TPS;
  // the whole parity sublattice, or (slab-blocked schedule) the window [win_lo, win_lo + win_n) of it
  const int n_site_blocks = win_n >= 0 ? win_n : (g.vh + SITES - 1) / SITES;
  if (n_site_blocks == 0) return cudaSuccess;
  // OPT bit 16: one CTA per site block (the hardware block scheduler hands out blocks in order)
  // instead of a persistent grid-stride loop
  int grid = (OPT & OPT_FLAT) ? n_site_blocks : sm_count() * MINB;
  if (grid > n_site_blocks) grid = n_site_blocks;
  const int rev = win_reverse >= 0 ? win_reverse : ((reverse_odd && parity) ? 1 : 0);
  // the last ~90 MB of links of the traversal are kept in L2 for the next (reversed) launch
  int late_from = -1;
  if (OPT & OPT_L2HINT) late_from = grid - (int)((double)grid * (90e6 / (8.0 * (double)g.vh * S::NV * sizeof(Vec))));
  if (OPT & OPT_PDL) {
    return launch_pdl(kern, dim3((unsigned)grid), dim3(BLOCK), smem, st, (Vec*)links, g, parity, omega,
                      n_site_blocks, rev, win_lo, late_from);
  }
  kern<<<grid, BLOCK, smem, st>>>((Vec*)links, g, parity, omega, n_site_blocks, rev, win_lo, late_from);
  return cudaGetLastError();
}

// Variant table (measured in profiles/r1_variant_sweep.md).  20 is the production
// mapping of each storage format; the others are the measured alternatives and stay callable
// (culgt_set_sweep_variant) and parity-tested.  "AxB" = A threads per CTA, B CTAs per SM;
// "flat" = one CTA per site block, "pers" = persistent grid-stride loop; tps = threads per site.
cudaError_t launch_or_sweep_staged(const LatticeDesc& d, void* links, int parity, double omega,
                                   int variant, bool coulomb, cudaStream_t st) {
  const Geom& g = d.geom;
  if (d.group != 3) return cudaErrorInvalidValue;
  if (coulomb) {   // Coulomb gauge: the production mapping of each format with K from spatial links
    if (variant != 20) return cudaErrorInvalidValue;
    if (d.precision == 32 && d.params == 12)
      return launch_staged<Storage<float, 3, 12>, double, 1, 128, 1, 4, OPT_FLAT | OPT_PDL | OPT_L2HINT | OPT_COULOMB>(links, g, parity, omega, true, st);
    if (d.precision == 32)
      return launch_staged<Storage<float, 3, 18>, double, 1, 64, 1, 5, OPT_FLAT | OPT_PDL | OPT_L2HINT | OPT_COULOMB>(links, g, parity, omega, true, st);
    if (d.params == 12)
      return launch_staged<Storage<double, 3, 12>, double, 1, 64, 1, 4, OPT_FLAT | OPT_PDL | OPT_L2HINT | OPT_COULOMB>(links, g, parity, omega, true, st);
    return launch_staged<Storage<double, 3, 18>, double, 1, 64, 1, 3, OPT_FLAT | OPT_PDL | OPT_L2HINT | OPT_COULOMB>(links, g, parity, omega, true, st);
  }
  if (d.precision == 32 && d.params == 12) {
    typedef Storage<float, 3, 12> S;
    switch (variant) {
      case 20: return launch_staged<S, double, 1, 128, 1, 4, OPT_FLAT | OPT_PDL | OPT_L2HINT>(links, g, parity, omega, true, st);
      case 21: return launch_staged<S, double, 1, 256, 1, 2, 0>(links, g, parity, omega, true, st);          // pers
      case 22: return launch_staged<S, double, 1, 128, 2, 2, 0>(links, g, parity, omega, true, st);          // pers, 2 stages
      case 23: return launch_staged<S, double, 2, 256, 1, 2, 0>(links, g, parity, omega, true, st);          // 2 tps, pers
      case 24: return launch_staged<S, double, 1, 128, 1, 4, OPT_FLAT>(links, g, parity, omega, false, st);  // no reversal
      case 25: return launch_staged<S, float, 1, 128, 1, 4, OPT_FLAT>(links, g, parity, omega, true, st);    // all-fp32
      case 26: return launch_staged<S, double, 1, 256, 1, 2, OPT_PREFETCH>(links, g, parity, omega, true, st);
      case 27: return launch_staged<S, double, 1, 256, 1, 2, OPT_CHUNKED>(links, g, parity, omega, true, st);
      case 28: return launch_staged<S, double, 1, 128, 1, 4, OPT_FLAT | OPT_NOMATH>(links, g, parity, omega, true, st);
      case 29: return launch_staged<S, double, 1, 128, 1, 4, OPT_FLAT | OPT_STREAM_ST>(links, g, parity, omega, true, st);
      case 32: return launch_staged<S, double, 1, 128, 1, 4, OPT_FLAT | OPT_NOSOLVE>(links, g, parity, omega, true, st);
      case 30: return launch_staged<S, double, 1, 256, 1, 2, OPT_FLAT>(links, g, parity, omega, true, st);
      case 31: return launch_staged<S, double, 1, 32, 1, 16, OPT_FLAT>(links, g, parity, omega, true, st);
      case 33: return launch_staged<S, double, 1, 128, 1, 4, OPT_FLAT>(links, g, parity, omega, true, st);            // no PDL
      case 34: return launch_staged<S, double, 1, 128, 1, 4, OPT_FLAT | OPT_PDL>(links, g, parity, omega, true, st);  // no L2 hints
      default: return cudaErrorInvalidValue;
    }
  }
  if (d.precision == 32) {
    typedef Storage<float, 3, 18> S;
    switch (variant) {
      case 20: return launch_staged<S, double, 1, 64, 1, 5, OPT_FLAT | OPT_PDL | OPT_L2HINT>(links, g, parity, omega, true, st);
      case 21: return launch_staged<S, double, 1, 128, 1, 2, 0>(links, g, parity, omega, true, st);          // pers
      case 22: return launch_staged<S, double, 2, 256, 1, 2, 0>(links, g, parity, omega, true, st);          // 2 tps, pers
      case 23: return launch_staged<S, double, 2, 256, 1, 2, OPT_FLAT>(links, g, parity, omega, true, st);
      case 24: return launch_staged<S, double, 1, 128, 1, 2, OPT_FLAT>(links, g, parity, omega, true, st);
      default: return cudaErrorInvalidValue;
    }
  }
  if (d.params == 12) {
    typedef Storage<double, 3, 12> S;
    switch (variant) {
      case 20: return launch_staged<S, double, 1, 64, 1, 4, OPT_FLAT | OPT_PDL | OPT_L2HINT>(links, g, parity, omega, true, st);
      case 21: return launch_staged<S, double, 1, 128, 1, 2, 0>(links, g, parity, omega, true, st);          // pers
      case 22: return launch_staged<S, double, 2, 256, 1, 2, 0>(links, g, parity, omega, true, st);          // 2 tps, pers
      case 23: return launch_staged<S, double, 4, 256, 1, 2, 0>(links, g, parity, omega, true, st);          // 4 tps, pers
      case 24: return launch_staged<S, double, 1, 128, 1, 2, OPT_FLAT>(links, g, parity, omega, true, st);
      default: return cudaErrorInvalidValue;
    }
  }
  typedef Storage<double, 3, 18> S;
  switch (variant) {
    case 20: return launch_staged<S, double, 1, 64, 1, 3, OPT_FLAT | OPT_PDL | OPT_L2HINT>(links, g, parity, omega, true, st);
    case 21: return launch_staged<S, double, 1, 192, 1, 1, 0>(links, g, parity, omega, true, st);            // pers
    case 22: return launch_staged<S, double, 2, 192, 1, 2, 0>(links, g, parity, omega, true, st);            // 2 tps, pers
    case 23: return launch_staged<S, double, 4, 256, 1, 2, 0>(links, g, parity, omega, true, st);            // 4 tps, pers
    case 24: return launch_staged<S, double, 1, 64, 1, 3, OPT_FLAT>(links, g, parity, omega, false, st);     // no reversal
    case 26: return launch_staged<S, double, 1, 192, 1, 1, OPT_PREFETCH>(links, g, parity, omega, true, st);
    case 27: return launch_staged<S, double, 1, 192, 1, 1, OPT_CHUNKED>(links, g, parity, omega, true, st);
    case 28: return launch_staged<S, double, 1, 64, 1, 3, OPT_FLAT | OPT_NOMATH>(links, g, parity, omega, true, st);
    case 30: return launch_staged<S, double, 1, 192, 1, 1, OPT_FLAT>(links, g, parity, omega, true, st);
    case 31: return launch_staged<S, double, 1, 32, 1, 6, OPT_FLAT>(links, g, parity, omega, true, st);
    case 33: return launch_staged<S, double, 1, 64, 1, 3, OPT_FLAT>(links, g, parity, omega, true, st);              // no PDL
    case 34: return launch_staged<S, double, 1, 64, 1, 3, OPT_FLAT | OPT_PDL>(links, g, parity, omega, true, st);    // no L2 hints
    case 32: return launch_staged<S, double, 1, 96, 2, 1, 0>(links, g, parity, omega, true, st);             // pers, 2 stages
    default: return cudaErrorInvalidValue;
  }
}

// ---------------------------------------------------------------------------------------------
// Slab-blocked FULL sweep: the black and the white half-sweep interleaved slab by
// slab along t, so that a white site finds the links its black neighbours have just written still
// in the 126 MB L2 -- the field then crosses HBM about once per full sweep instead of twice.
// Time-slice t is the contiguous half-index range [t*stride3, (t+1)*stride3) of each parity, i.e.
// a contiguous window of site blocks.  With slab ends e_k = min((k+1)*sl, N3):
//     for k:  black slices [k*sl, e_k)  ascending;   white slices [max(1, k*sl - 1), e_k - 1)  descending
//     then    white slice N3-1, white slice 0.
// A white site of slice t needs its black neighbours of slices t-1, t, t+1 done: t <= e_k - 2 and
// t >= 1 guarantee it; slices N3-1 and 0 wait for the last / first black slab (periodic wrap).
// Sites of one parity do not interact, so the result is bit-identical to two whole half-sweeps.
// overlap: the white windows run on a second stream, concurrently with the next black slab -- they
// touch disjoint links (black slab k+1 writes links stored at slices >= e_k - 1, the white window
// links stored at slices <= e_k - 2) -- so neither launch's tail leaves the GPU idle.
// Returns cudaErrorNotSupported when the lattice does not split into whole site blocks per slice.
// ---------------------------------------------------------------------------------------------
struct SlabStreams {
  cudaStream_t white = nullptr;
  cudaEvent_t black_done[64];
  cudaEvent_t white_done = nullptr;
  bool ready = false;
};
static SlabStreams g_slab;

static cudaError_t slab_streams_init() {
  if (g_slab.ready) return cudaSuccess;
  cudaError_t e = cudaStreamCreateWithFlags(&g_slab.white, cudaStreamNonBlocking);
  if (e != cudaSuccess) return e;
  for (int i = 0; i < 64; ++i)
    if ((e = cudaEventCreateWithFlags(&g_slab.black_done[i], cudaEventDisableTiming)) != cudaSuccess) return e;
  if ((e = cudaEventCreateWithFlags(&g_slab.white_done, cudaEventDisableTiming)) != cudaSuccess) return e;
  g_slab.ready = true;
  return cudaSuccess;
}

template <typename S, int BLOCK, int MINB>
static cudaError_t slab_sweep(void* links, const Geom& g, double omega, int sl, bool overlap, cudaStream_t st) {
  const int n3 = g.n[3];
  if (g.stride[3] % BLOCK != 0 || sl < 2 || n3 < 4 || sl > n3 - 2) return cudaErrorNotSupported;
  const int bps = g.stride[3] / BLOCK;                  // site blocks per time-slice (per parity)
  const int ns = (n3 + sl - 1) / sl;
  if (ns > 64) return cudaErrorNotSupported;
  cudaError_t e;
  cudaStream_t wst = st;
  if (overlap) {
    if ((e = slab_streams_init()) != cudaSuccess) return e;
    wst = g_slab.white;
    // the previous work on the caller's stream (e.g. the previous sweep's black slabs) precedes our white windows
  }
  auto launch = [&](int parity, int t_lo, int t_hi, cudaStream_t s) {   // slices [t_lo, t_hi)
    if (t_hi <= t_lo) return cudaSuccess;
    return launch_staged<S, double, 1, BLOCK, 1, MINB, OPT_FLAT>(links, g, parity, omega, true, s, t_lo * bps,
                                                                (t_hi - t_lo) * bps, parity);
  };
  for (int k = 0; k < ns; ++k) {
    const int s_k = k * sl, e_k = (k + 1) * sl < n3 ? (k + 1) * sl : n3;
    if ((e = launch(0, s_k, e_k, st)) != cudaSuccess) return e;
    if (overlap) {
      if ((e = cudaEventRecord(g_slab.black_done[k], st)) != cudaSuccess) return e;
      if ((e = cudaStreamWaitEvent(wst, g_slab.black_done[k], 0)) != cudaSuccess) return e;
    }
    if ((e = launch(1, s_k > 1 ? s_k - 1 : 1, e_k - 1, wst)) != cudaSuccess) return e;
  }
  if ((e = launch(1, n3 - 1, n3, wst)) != cudaSuccess) return e;
  if ((e = launch(1, 0, 1, wst)) != cudaSuccess) return e;
  if (overlap) {     // join: whatever follows on the caller's stream sees the finished sweep
    if ((e = cudaEventRecord(g_slab.white_done, wst)) != cudaSuccess) return e;
    if ((e = cudaStreamWaitEvent(st, g_slab.white_done, 0)) != cudaSuccess) return e;
  }
  return cudaSuccess;
}

cudaError_t launch_or_sweep_staged_slabbed(const LatticeDesc& d, void* links, double omega, int slab_slices,
                                           bool overlap, cudaStream_t st) {
  const Geom& g = d.geom;
  if (d.group != 3) return cudaErrorNotSupported;
  if (d.precision == 32 && d.params == 12) return slab_sweep<Storage<float, 3, 12>, 128, 4>(links, g, omega, slab_slices, overlap, st);
  if (d.precision == 32) return slab_sweep<Storage<float, 3, 18>, 64, 5>(links, g, omega, slab_slices, overlap, st);
  if (d.params == 12) return slab_sweep<Storage<double, 3, 12>, 64, 4>(links, g, omega, slab_slices, overlap, st);
  return slab_sweep<Storage<double, 3, 18>, 64, 3>(links, g, omega, slab_slices, overlap, st);
}

// Truncated-series overrelaxation (reading C-24) / simulated annealing (C-25) / the
// microcanonical step (C-26) on the production
// mapping of each format.
template <typename Power>
static cudaError_t launch_production(const LatticeDesc& d, void* links, int parity, const Power& pw, cudaStream_t st) {
  const Geom& g = d.geom;
  if (d.group != 3) return cudaErrorInvalidValue;
  if (d.precision == 32 && d.params == 12)
    return launch_staged<Storage<float, 3, 12>, double, 1, 128, 1, 4, OPT_FLAT | OPT_PDL | OPT_L2HINT>(links, g, parity, pw, true, st);
  if (d.precision == 32)
    return launch_staged<Storage<float, 3, 18>, double, 1, 64, 1, 5, OPT_FLAT | OPT_PDL | OPT_L2HINT>(links, g, parity, pw, true, st);
  if (d.params == 12)
    return launch_staged<Storage<double, 3, 12>, double, 1, 64, 1, 4, OPT_FLAT | OPT_PDL | OPT_L2HINT>(links, g, parity, pw, true, st);
  return launch_staged<Storage<double, 3, 18>, double, 1, 64, 1, 3, OPT_FLAT | OPT_PDL | OPT_L2HINT>(links, g, parity, pw, true, st);
}

cudaError_t launch_or_sweep_staged_series(const LatticeDesc& d, void* links, int parity, const SeriesPower& pw,
                                          cudaStream_t st) {
  return launch_production(d, links, parity, pw, st);
}
cudaError_t launch_or_sweep_staged_micro(const LatticeDesc& d, void* links, int parity, cudaStream_t st) {
  return launch_production(d, links, parity, MicroPower{0}, st);
}
cudaError_t launch_or_sweep_staged_heatbath(const LatticeDesc& d, void* links, int parity, const HeatBathPower& pw,
                                            cudaStream_t st) {
  return launch_production(d, links, parity, pw, st);
}

}  // namespace culgt
