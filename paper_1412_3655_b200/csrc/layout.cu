// layout.cu -- a0: canonical (site-major, full matrices) <-> internal (parity-split, site-fastest
// SoA of 12/18/4-parameter vectors).  PAPER.md L64 (reordering into black/white sublattices),
// L95 (canonical linear array), L118 (pack discards the third row; unpack reconstructs it).
#include "lattice.cuh"
#include "su_math.cuh"
#include "kernels.h"

namespace culgt {

// two reals as one 8- / 16-byte shared-memory access
template <typename Real> struct HalfVec;
template <> struct HalfVec<float> {
  typedef float2 type;
  __device__ static __forceinline__ float2 make(float a, float b) { return make_float2(a, b); }
  __device__ static __forceinline__ void split(const float2& v, float& a, float& b) { a = v.x; b = v.y; }
};
template <> struct HalfVec<double> {
  typedef double2 type;
  __device__ static __forceinline__ double2 make(double a, double b) { return make_double2(a, b); }
  __device__ static __forceinline__ void split(const double2& v, double& a, double& b) { a = v.x; b = v.y; }
};

// A CTA converts TILE consecutive canonical sites (= TILE/2 consecutive half indices h of BOTH
// parities, 4*TILE links).  The canonical side of the tile is one contiguous run of
// TILE*4*NFULL reals and moves with coalesced 16-byte accesses through shared memory; the internal
// side is written / read with consecutive threads on consecutive h of one (parity, mu) plane set.
// (A thread per link touching its 18 canonical reals directly reached 40 % of the copy rate.)
//
// Shared-memory layout: consecutive h are one SITE PAIR = 8*NFULL reals apart (144 reals for SU(3)),
// a multiple of 32 four-byte banks for every format, so the link threads of a warp would all hit the
// same banks.  Two reals of padding behind every site pair make the pair stride an odd number of
// 8-byte (fp32) / 16-byte (fp64) units: the link threads' 64- / 128-bit accesses are conflict-free.
// A 16-byte canonical vector never straddles a pair, so the copy side only splits it into its two
// 8-byte halves (fp32) or moves it whole (fp64).
template <typename S, int TILE>
struct TileLayout {
  static constexpr int PAIR = 8 * S::NFULL;                    // reals of one site pair
  static constexpr int PAD = 2;                                // reals of padding behind it
  static constexpr int REALS = (TILE / 2) * (PAIR + PAD);
  __device__ static __forceinline__ int at(int real_index) { return real_index + PAD * (real_index / PAIR); }
};

template <typename S, bool PACK, int TILE, int BLOCK>
__global__ void __launch_bounds__(BLOCK)
layout_tiled_kernel(typename S::Real* __restrict__ canonical, typename S::Vec* __restrict__ links, const Geom g,
                    const long long V) {
  typedef typename S::Real Real;
  typedef typename S::Vec Vec;
  typedef TileLayout<S, TILE> TL;
  typedef typename HalfVec<Real>::type HV;
  constexpr int NF = S::NFULL;
  constexpr int VL = S::VL;                                    // reals per 16-byte vector: 4 or 2
  extern __shared__ __align__(16) unsigned char tile_raw[];
  Real* tile = reinterpret_cast<Real*>(tile_raw);              // [site in tile][mu][NF], padded per site pair
  const long long s0 = (long long)blockIdx.x * TILE;
  const int nsite = (int)((V - s0 < TILE) ? (V - s0) : TILE);  // even: every extent is even
  const int nvec = nsite * 4 * NF / VL;
  Vec* can_v = reinterpret_cast<Vec*>(canonical + s0 * 4 * NF);
  // one canonical vector <-> its padded place, as 8-byte halves (fp32) or whole (fp64: VL = 2 reals = PAD)
  auto put = [&](int i, const Vec& v) {
    Real r[VL];
    vec_get(v, r);
    Real* d = tile + TL::at(i * VL);
#pragma unroll
    for (int k = 0; k < VL; k += 2) *reinterpret_cast<HV*>(d + k) = HalfVec<Real>::make(r[k], r[k + 1]);
  };
  auto get = [&](int i) {
    Real r[VL];
    const Real* d = tile + TL::at(i * VL);
#pragma unroll
    for (int k = 0; k < VL; k += 2) HalfVec<Real>::split(*reinterpret_cast<const HV*>(d + k), r[k], r[k + 1]);
    Vec v;
    vec_set(v, r);
    return v;
  };
  if (PACK) {
    for (int i = threadIdx.x; i < nvec; i += BLOCK) put(i, can_v[i]);
    __syncthreads();
  }
  const int h0 = (int)(s0 >> 1);
  const int nh = nsite >> 1;
  for (int L = threadIdx.x; L < 8 * (TILE / 2); L += BLOCK) {   // link = (parity, mu, hl)
    const int hl = L % (TILE / 2);
    const int pm = L / (TILE / 2);
    const int parity = pm >> 2, mu = pm & 3;
    if (hl >= nh) continue;
    const int h = h0 + hl;
    const SiteCoord sc = decode_site(g, h, parity);
    Real* c = tile + hl * (TL::PAIR + TL::PAD) + (sc.odd * 4 + mu) * NF;   // canonical site 2h + odd, local index
    Vec* lptr = link_base<S>(links, g, parity, mu, h);
    if (PACK) {
      Real m[kLinkRegs];
#pragma unroll
      for (int i = 0; i < kLinkRegs; ++i) m[i] = (Real)0;                   // pad reals stay 0
#pragma unroll
      for (int i = 0; i < NF; i += 2) HalfVec<Real>::split(*reinterpret_cast<const HV*>(c + i), m[i], m[i + 1]);
      if (S::NC == 3) {
        store_params<S>(lptr, g.pitch, m);              // first NP reals = first NP/6 rows (L118)
      } else {
        // SU(2): [[a0+i a3, a2+i a1],[..]] -> (a0,a1,a2,a3)   (C-7)
        Real a[4] = {m[0], m[3], m[2], m[1]};
        store_params<S>(lptr, g.pitch, a);
      }
    } else {
      if (S::NC == 3) {
        Real m[kLinkRegs];
        load_params<S>(lptr, g.pitch, m);
        if (S::NP == 12) reconstruct_row2(m);
#pragma unroll
        for (int i = 0; i < 18; i += 2) *reinterpret_cast<HV*>(c + i) = HalfVec<Real>::make(m[i], m[i + 1]);
      } else {
        Real a[4];
        load_params<S>(lptr, g.pitch, a);
        *reinterpret_cast<HV*>(c + 0) = HalfVec<Real>::make(a[0], a[3]);     // a0 + i a3
        *reinterpret_cast<HV*>(c + 2) = HalfVec<Real>::make(a[2], a[1]);     // a2 + i a1
        *reinterpret_cast<HV*>(c + 4) = HalfVec<Real>::make(-a[2], a[1]);    // -a2 + i a1
        *reinterpret_cast<HV*>(c + 6) = HalfVec<Real>::make(a[0], -a[3]);    // a0 - i a3
      }
    }
  }
  if (!PACK) {
    __syncthreads();
    for (int i = threadIdx.x; i < nvec; i += BLOCK) can_v[i] = get(i);
  }
}

template <typename S, bool PACK>
static cudaError_t launch_layout(void* canonical, void* links, const Geom& g, cudaStream_t st) {
  constexpr int BLOCK = 256;
  constexpr int TILE = (sizeof(typename S::Real) == 8 && S::NC == 3) ? 64 : 128;   // <= 36 KB of shared memory
  constexpr size_t smem = (size_t)TileLayout<S, TILE>::REALS * sizeof(typename S::Real);
  const long long V = 2ll * g.vh;
  const unsigned grid = (unsigned)((V + TILE - 1) / TILE);
  layout_tiled_kernel<S, PACK, TILE, BLOCK><<<grid, BLOCK, smem, st>>>((typename S::Real*)canonical,
                                                                       (typename S::Vec*)links, g, V);
  return cudaGetLastError();
}

template <bool PACK>
static cudaError_t dispatch_layout(const LatticeDesc& d, void* canonical, void* links, cudaStream_t st) {
  const Geom& g = d.geom;
  if (d.group == 2) {
    if (d.precision == 32) return launch_layout<Storage<float, 2, 4>, PACK>(canonical, links, g, st);
    return launch_layout<Storage<double, 2, 4>, PACK>(canonical, links, g, st);
  }
  if (d.precision == 32) {
    if (d.params == 12) return launch_layout<Storage<float, 3, 12>, PACK>(canonical, links, g, st);
    return launch_layout<Storage<float, 3, 18>, PACK>(canonical, links, g, st);
  }
  if (d.params == 12) return launch_layout<Storage<double, 3, 12>, PACK>(canonical, links, g, st);
  return launch_layout<Storage<double, 3, 18>, PACK>(canonical, links, g, st);
}

// ---------------------------------------------------------------------------------------------
// Re-unitarisation (reading C-23): Gram-Schmidt on the stored rows of every link, in
// fp64, rounded once to the storage precision.  One thread per (parity, mu, h) link.
//   r0 <- r0/|r0|;  r1 <- r1 - <r0,r1> r0;  r1 <- r1/|r1|;  (18-parameter: r2 <- conj(r0 x r1));
//   SU(2): (a0..a3) <- (a0..a3)/|a|.
// ---------------------------------------------------------------------------------------------
template <typename S, int BLOCK>
__global__ void __launch_bounds__(BLOCK)
reunitarize_kernel(typename S::Vec* __restrict__ links, const Geom g) {
  typedef typename S::Real Real;
  const long long t = (long long)blockIdx.x * BLOCK + threadIdx.x;     // (parity*4 + mu)*vh + h
  if (t >= 8ll * g.vh) return;
  const int pm = (int)(t / g.vh);
  const int h = (int)(t - (long long)pm * g.vh);
  typename S::Vec* p = links + ((size_t)pm * S::NV) * (size_t)g.pitch + (size_t)h;
  Real r[kLinkRegs];
  load_params<S>(p, g.pitch, r);
  if (S::NC == 2) {
    double a[4] = {(double)r[0], (double)r[1], (double)r[2], (double)r[3]};
    const double inv = 1.0 / sqrt(a[0] * a[0] + a[1] * a[1] + a[2] * a[2] + a[3] * a[3]);
#pragma unroll
    for (int i = 0; i < 4; ++i) r[i] = (Real)(a[i] * inv);
  } else {
    double m[18];
#pragma unroll
    for (int i = 0; i < 12; ++i) m[i] = (double)r[i];
    double n0 = 0;
#pragma unroll
    for (int i = 0; i < 6; ++i) n0 += m[i] * m[i];
    const double i0 = 1.0 / sqrt(n0);
#pragma unroll
    for (int i = 0; i < 6; ++i) m[i] *= i0;
    double ipr = 0, ipi = 0;                       // <r0, r1> = sum conj(r0_k) r1_k
#pragma unroll
    for (int c = 0; c < 3; ++c) {
      ipr += m[CULGT_RE(0, c)] * m[CULGT_RE(1, c)] + m[CULGT_IM(0, c)] * m[CULGT_IM(1, c)];
      ipi += m[CULGT_RE(0, c)] * m[CULGT_IM(1, c)] - m[CULGT_IM(0, c)] * m[CULGT_RE(1, c)];
    }
#pragma unroll
    for (int c = 0; c < 3; ++c) {
      m[CULGT_RE(1, c)] -= ipr * m[CULGT_RE(0, c)] - ipi * m[CULGT_IM(0, c)];
      m[CULGT_IM(1, c)] -= ipr * m[CULGT_IM(0, c)] + ipi * m[CULGT_RE(0, c)];
    }
    double n1 = 0;
#pragma unroll
    for (int i = 6; i < 12; ++i) n1 += m[i] * m[i];
    const double i1 = 1.0 / sqrt(n1);
#pragma unroll
    for (int i = 6; i < 12; ++i) m[i] *= i1;
    if (S::NP == 18) reconstruct_row2(m);
#pragma unroll
    for (int i = 0; i < S::NP; ++i) r[i] = (Real)m[i];
  }
  store_params<S>(p, g.pitch, r);
}

template <typename S>
static cudaError_t run_reunitarize(void* links, const Geom& g, cudaStream_t st) {
  constexpr int BLOCK = 256;
  const unsigned grid = (unsigned)((8ll * g.vh + BLOCK - 1) / BLOCK);
  reunitarize_kernel<S, BLOCK><<<grid, BLOCK, 0, st>>>((typename S::Vec*)links, g);
  return cudaGetLastError();
}

cudaError_t launch_reunitarize(const LatticeDesc& d, void* links, cudaStream_t st) {
  const Geom& g = d.geom;
  if (d.group == 2) {
    if (d.precision == 32) return run_reunitarize<Storage<float, 2, 4> >(links, g, st);
    return run_reunitarize<Storage<double, 2, 4> >(links, g, st);
  }
  if (d.precision == 32) {
    if (d.params == 12) return run_reunitarize<Storage<float, 3, 12> >(links, g, st);
    return run_reunitarize<Storage<float, 3, 18> >(links, g, st);
  }
  if (d.params == 12) return run_reunitarize<Storage<double, 3, 12> >(links, g, st);
  return run_reunitarize<Storage<double, 3, 18> >(links, g, st);
}

cudaError_t launch_pack(const LatticeDesc& d, const void* canonical, void* links, cudaStream_t st) {
  return dispatch_layout<true>(d, const_cast<void*>(canonical), links, st);
}
cudaError_t launch_unpack(const LatticeDesc& d, const void* links, void* canonical, cudaStream_t st) {
  return dispatch_layout<false>(d, canonical, const_cast<void*>(links), st);
}

}  // namespace culgt
