// layout.cu -- a0: canonical (site-major, full matrices) <-> internal (parity-split, site-fastest
// SoA of 12/18/4-parameter vectors).  PAPER.md L64 (reordering into black/white sublattices),
// L95 (canonical linear array), L118 (pack discards the third row; unpack reconstructs it).
#include "lattice.cuh"
#include "su_math.cuh"
#include "kernels.h"

namespace culgt {

// One thread per (parity, h, mu).  Canonical link (s, mu) is NFULL contiguous reals.
template <typename S, bool PACK, int BLOCK>
__global__ void __launch_bounds__(BLOCK)
layout_kernel(typename S::Real* __restrict__ canonical, typename S::Vec* __restrict__ links, const Geom g) {
  typedef typename S::Real Real;
  const long long t = (long long)blockIdx.x * BLOCK + threadIdx.x;   // t = (h*4 + mu) within a parity
  const int parity = blockIdx.y;
  if (t >= 4ll * g.vh) return;
  const int h = (int)(t >> 2);
  const int mu = (int)(t & 3);
  const SiteCoord sc = decode_site(g, h, parity);
  const int64_t s = canonical_site(g, h, sc);
  Real* cptr = canonical + (s * 4 + mu) * S::NFULL;
  typename S::Vec* lptr = link_base<S>(links, g, parity, mu, h);
  if (PACK) {
    Real m[S::NFULL];
#pragma unroll
    for (int i = 0; i < S::NFULL; ++i) m[i] = cptr[i];
    if (S::NC == 3) {
      store_params<S>(lptr, g.vh, m);              // first NP reals = first NP/6 rows
    } else {
      // SU(2): [[a0+i a3, a2+i a1],[..]] -> (a0,a1,a2,a3)   (C-7)
      Real a[4] = {m[0], m[3], m[2], m[1]};
      store_params<S>(lptr, g.vh, a);
    }
  } else {
    if (S::NC == 3) {
      Real m[18];
      load_params<S>(lptr, g.vh, m);
      if (S::NP == 12) reconstruct_row2(m);
#pragma unroll
      for (int i = 0; i < 18; ++i) cptr[i] = m[i];
    } else {
      Real a[4];
      load_params<S>(lptr, g.vh, a);
      cptr[0] = a[0];  cptr[1] = a[3];     // a0 + i a3
      cptr[2] = a[2];  cptr[3] = a[1];     // a2 + i a1
      cptr[4] = -a[2]; cptr[5] = a[1];     // -a2 + i a1
      cptr[6] = a[0];  cptr[7] = -a[3];    // a0 - i a3
    }
  }
}

template <typename S, bool PACK>
static cudaError_t launch_layout(void* canonical, void* links, const Geom& g, cudaStream_t st) {
  constexpr int BLOCK = 256;
  dim3 grid((unsigned)((4ll * g.vh + BLOCK - 1) / BLOCK), 2);
  layout_kernel<S, PACK, BLOCK><<<grid, BLOCK, 0, st>>>((typename S::Real*)canonical,
                                                         (typename S::Vec*)links, g);
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

cudaError_t launch_pack(const LatticeDesc& d, const void* canonical, void* links, cudaStream_t st) {
  return dispatch_layout<true>(d, const_cast<void*>(canonical), links, st);
}
cudaError_t launch_unpack(const LatticeDesc& d, const void* links, void* canonical, cudaStream_t st) {
  return dispatch_layout<false>(d, canonical, const_cast<void*>(links), st);
}

}  // namespace culgt
