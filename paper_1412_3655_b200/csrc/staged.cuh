// staged.cuh -- the per-site-block body of the production SU(3) half-sweep (SURVEY.md 8(a) rows
// a1-a6) and the shared-memory staging helpers, shared by the launch-per-half-sweep kernel
// (or_sweep_staged.cu) and the fused full-sweep kernel (or_sweep_fused.cu).
//
// One thread per site.  The 8 links of the site are moved global -> shared memory by per-thread
// cp.async (LDGSTS, 16 bytes) into slots that only the issuing thread reads back (slot layout
// [vector][thread], so every LDS.128 / cp.async of a warp is 512 contiguous bytes and
// conflict-free); cp.async.wait_group orders a thread against its own copies, so no block barrier
// is needed.  Registers hold only K (fp64), G and one link at a time.
#pragma once
#include <type_traits>
#include "lattice.cuh"
#include "su_math.cuh"
#include "su3_solve.cuh"

namespace culgt {

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

// The three L2 eviction policies as 64-bit descriptors (createpolicy.fractional, fraction 1).
struct L2Policies {
  uint64_t first, normal, last;
  __device__ __forceinline__ void create() {
    asm("createpolicy.fractional.L2::evict_first.b64 %0, 1.0;" : "=l"(first));
    asm("createpolicy.fractional.L2::evict_normal.b64 %0, 1.0;" : "=l"(normal));
    asm("createpolicy.fractional.L2::evict_last.b64 %0, 1.0;" : "=l"(last));
  }
  // 0 = evict_first, 1 = evict_normal, 2 = evict_last
  __device__ __forceinline__ uint64_t pick(int which) const { return which == 0 ? first : (which == 2 ? last : normal); }
};

// What one thread needs to know about the site it works on: the half index of each of its LPT
// links (slot = q*LPT + l = 2*mu + down; up links sit at the site's own index h in this parity's
// sublattice, down links at the index of x - mu in the other parity's).
template <int LPT>
struct SiteRef {
  int idx[LPT];
  unsigned site;   // canonical site index (selects the heat bath's random numbers)
  int x3;          // time coordinate (Coulomb gauge: the slice whose activity byte decides)
  bool active;
};

// Index arithmetic only: no global memory is touched here (under programmatic dependent launch
// this runs BEFORE griddepcontrol.wait, i.e. possibly while the previous kernel of the stream is
// still writing).
template <int BLOCK, int TPS>
__device__ __forceinline__ SiteRef<8 / TPS> locate(const Geom& g, int parity, int site_block, int q) {
  constexpr int LPT = 8 / TPS;
  SiteRef<LPT> r;
  int h = site_block * (BLOCK / TPS) + (int)threadIdx.x / TPS;
  r.active = h < g.vh;
  if (!r.active) h = g.vh - 1;
  const SiteCoord sc = decode_site(g, h, parity);
  r.site = (unsigned)canonical_site(g, h, sc);
  r.x3 = sc.x3;
#pragma unroll
  for (int l = 0; l < LPT; ++l) {
    const int slot = q * LPT + l;
    r.idx[l] = (slot & 1) ? down_index(g, h, sc, slot >> 1) : h;
  }
  return r;
}

// Coulomb gauge with a per-slice activity mask (reading C-22): a site of a frozen slice is left
// alone.  Reads global memory, so it must run AFTER griddepcontrol.wait.
template <int LPT>
__device__ __forceinline__ void apply_slice_mask(const Geom& g, SiteRef<LPT>& r) {
  if (g.slice_active != nullptr && g.slice_active[r.x3] == 0) r.active = false;
}

// Global address of vector j of this thread's link l: a plane base that does not depend on the
// thread (for TPS = 1 it is uniform over the CTA, so it lives in uniform registers) plus the
// 32-bit half index -- this keeps 64-bit per-thread address arithmetic out of the inner loops.
template <typename S, int LPT>
__device__ __forceinline__ typename S::Vec* vec_ptr(typename S::Vec* links, const Geom& g, int parity,
                                                    const SiteRef<LPT>& r, int q, int l, int j) {
  const int slot = q * LPT + l;
  const int plane = (((slot & 1) ? 1 - parity : parity) * 4 + (slot >> 1)) * S::NV + j;
  typename S::Vec* base = links + (size_t)plane * (size_t)g.pitch;
  return base + (unsigned)r.idx[l];
}

// ---- the production body: one thread per site, one stage ---------------------------------------
// issue_site_loads: the 8 links of the located site, global -> this thread's shared-memory slots.
// HINT = true: cp.async with the L2 eviction policy `pol`.
template <typename S, int BLOCK, bool HINT>
__device__ __forceinline__ void issue_site_loads(typename S::Vec* __restrict__ links, const Geom& g, int parity,
                                                 const SiteRef<8>& r, typename S::Vec* sm, uint64_t pol) {
  typedef typename S::Vec Vec;
  constexpr int NV = S::NV;
  if (r.active) {
#pragma unroll
    for (int l = 0; l < 8; ++l) {
#pragma unroll
      for (int j = 0; j < NV; ++j) {
        if (HINT) cp_async_vec_hint(sm + (size_t)((l * NV + j) * BLOCK), (const Vec*)vec_ptr<S, 8>(links, g, parity, r, 0, l, j), pol);
        else cp_async_vec(sm + (size_t)((l * NV + j) * BLOCK), vec_ptr<S, 8>(links, g, parity, r, 0, l, j));
      }
    }
  }
  cp_async_commit();
}

// update_site: K(x) from the staged links (eq. 3), G(x) by the subgroup loop with g^omega
// (P:L50-54), U_mu(x) <- G U_mu(x), U_mu(x-mu) <- U_mu(x-mu) G^dagger stored in
// place.  The caller has waited for the thread's cp.async group.  COULOMB: the time links do not
// enter K (reading C-22).  HINT: stores carry the L2 eviction policy `pol_st`.
template <typename S, int BLOCK, bool COULOMB, bool HINT, typename Power>
__device__ __forceinline__ void update_site(typename S::Vec* __restrict__ links, const Geom& g, int parity,
                                            const Power& omega, const SiteRef<8>& r, unsigned sm_addr,
                                            uint64_t pol_st) {
  typedef typename S::Real Real;
  typedef typename S::Vec Vec;
  constexpr int NV = S::NV;
  constexpr int NR = (S::NP == 12) ? 2 : 3;
  auto load_link = [&](int l, Real* U, auto vol) {
#pragma unroll
    for (int j = 0; j < NV; ++j) {
      Vec v;
      lds_vec<decltype(vol)::value>(sm_addr + (unsigned)((l * NV + j) * BLOCK * (int)sizeof(Vec)), v);
      vec_get(v, U + j * S::VL);
    }
  };
  Real G[18];
  {
    // ---- K(x) = sum_mu U_mu(x) + U_mu(x-mu)^dagger                     (eq. 3)
    double K[18];
#pragma unroll
    for (int i = 0; i < 18; ++i) K[i] = 0;
#pragma unroll
    for (int l = 0; l < 8; ++l) {
      if (COULOMB && (l >> 1) == 3) continue;   // time links do not enter K_C
      Real U[kLinkRegs];
      asm volatile("" ::: "memory");   // keep the shared-memory reads of link l behind link l-1's use
      load_link(l, U, std::false_type());
      if (S::NP == 12 && sizeof(Real) == 4) {
        // fp32 12-parameter storage: widen the two stored rows and rebuild the third row in
        // fp64 for K.  A third row rebuilt in fp32 puts ~1e-7 into K, which the small-|p| sites
        // of a hot 10^7-site lattice amplify past the 2e-5 link tolerance; it also
        // needs 12 instead of 18 fp32->fp64 conversions per link.
        double Ua[18];
#pragma unroll
        for (int i = 0; i < 12; ++i) Ua[i] = (double)U[i];
        reconstruct_row2(Ua);
        accumulate(K, Ua, (l & 1) != 0);
      } else {
        if (S::NP == 12) reconstruct_row2(U);
        accumulate(K, U, (l & 1) != 0);
      }
    }
    // ---- G(x): subgroup loop with g^omega                              (L50-54)
    // G = g_3 g_2 g_1 is accumulated in fp64 and rounded once: accumulating it in fp32 costs
    // 0.7 % less time but doubles the worst link error at 32^4 (1.08e-5 vs 5.8e-6)
    double Gd[18];
    if (r.active) {
      // idle lanes of a ragged last block hold uninitialised shared memory: they must not enter
      // the solve (the heat bath's rejection loop would never end on NaN input)
      su3_solve<(sizeof(Real) == 8), double>(K, Gd, omega, r.site);
    } else {
#pragma unroll
      for (int i = 0; i < 18; ++i) Gd[i] = 0.0;
    }
#pragma unroll
    for (int i = 0; i < 18; ++i) G[i] = (Real)Gd[i];
  }
  // ---- U_mu(x) <- G U_mu(x),  U_mu(x-mu) <- U_mu(x-mu) G^dagger      (L19-21, L48)
  if (r.active) {
#pragma unroll
    for (int l = 0; l < 8; ++l) {
      Real U[kLinkRegs], R[kLinkRegs];
      R[18] = 0; R[19] = 0;
      asm volatile("" ::: "memory");
      load_link(l, U, std::true_type());
      if ((l & 1) == 0) {
        if (S::NP == 12) reconstruct_row2(U);
        mul_ab<NR>(G, U, R);
      } else {
        mul_abd<NR>(U, G, R);
      }
#pragma unroll
      for (int j = 0; j < NV; ++j) {
        Vec v;
        vec_set(v, R + j * S::VL);
        if (HINT) st_hint(vec_ptr<S, 8>(links, g, parity, r, 0, l, j), v, pol_st);
        else *vec_ptr<S, 8>(links, g, parity, r, 0, l, j) = v;
      }
    }
  }
}

// Shared memory of one CTA of the production body.
template <typename S, int BLOCK>
constexpr size_t staged_smem_bytes() { return (size_t)8 * S::NV * BLOCK * sizeof(typename S::Vec); }

}  // namespace culgt
