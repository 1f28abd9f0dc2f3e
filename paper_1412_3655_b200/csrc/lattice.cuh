// lattice.cuh -- geometry of the parity-split internal layout and vector load/store helpers.
//
// Internal field ("reorder the lattice into its black and white sublattices ...
// the site index runs faster than Lorentz and matrix indices"; L103: "three float4"):
//     links[parity][mu][j][h]   vectors of 16 bytes (fp32 18-parameter: 5 float4, the last half used),
// h = canonical_site >> 1 = x0/2 + (N0/2)*(x1 + N1*(x2 + N2*x3)), valid because N0 is even.
// Every [parity][mu][j] plane is a contiguous run of V/2 vectors, so a warp that walks
// consecutive h reads consecutive addresses in every plane.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace culgt {

// n / d for 0 <= n < 2^31 by multiply-shift (Granlund-Montgomery, 31-bit dividend).
struct FastDiv {
  uint32_t d, mul, shift;
  __host__ void init(uint32_t div) {
    d = div;
    uint32_t l = 0;
    while ((1u << l) < div) ++l;
    shift = 31 + l;
    mul = (uint32_t)(((1ull << shift) + div - 1) / div);
  }
  __device__ __forceinline__ uint32_t div(uint32_t n) const {
    return (uint32_t)(((uint64_t)n * mul) >> shift);
  }
};

struct Geom {
  int32_t n[4];      // N0..N3
  int32_t nh0;       // N0/2
  int32_t vh;        // V/2 sites per parity
  int32_t pitch;     // vectors per [parity][mu][j] plane: vh, or vh + stride[3] for a time slab that
                     // carries a ghost slice behind its last slice (slab.cu)
  int32_t wrap3;     // x3 = 0: index offset of the neighbour x - t_hat.  Periodic lattice:
                     // stride[3]*(N3-1) (its own last slice); time slab: stride[3]*N3 = the ghost slice
  int32_t stride[4]; // half-index strides: 1 (unused for mu=0), N0/2, N0/2*N1, N0/2*N1*N2
  FastDiv d_nh0, d_n1, d_n2;
  // Coulomb gauge only: device array of N3 bytes, a site of time-slice t is swept iff
  // slice_active[t] != 0; nullptr = every slice (set by the API layer per call)
  const unsigned char* slice_active;
};

inline Geom make_geom(const int32_t dims[4]) {
  Geom g;
  for (int i = 0; i < 4; ++i) g.n[i] = dims[i];
  g.nh0 = dims[0] / 2;
  g.stride[0] = 1;
  g.stride[1] = g.nh0;
  g.stride[2] = g.nh0 * dims[1];
  g.stride[3] = g.nh0 * dims[1] * dims[2];
  g.vh = g.stride[3] * dims[3];
  g.pitch = g.vh;
  g.wrap3 = g.stride[3] * (dims[3] - 1);
  g.d_nh0.init((uint32_t)g.nh0);
  g.d_n1.init((uint32_t)dims[1]);
  g.d_n2.init((uint32_t)dims[2]);
  g.slice_active = nullptr;
  return g;
}

// Coordinates of the site with half index h in the sublattice `parity`.
struct SiteCoord {
  int hx, x1, x2, x3;  // hx = x0 >> 1
  int odd;             // x0 & 1  = (x1+x2+x3+parity) & 1
};

__device__ __forceinline__ SiteCoord decode_site(const Geom& g, int h, int parity) {
  SiteCoord c;
  uint32_t t = g.d_nh0.div((uint32_t)h);
  c.hx = h - (int)t * g.nh0;
  uint32_t t2 = g.d_n1.div(t);
  c.x1 = (int)t - (int)t2 * g.n[1];
  uint32_t t3 = g.d_n2.div(t2);
  c.x2 = (int)t2 - (int)t3 * g.n[2];
  c.x3 = (int)t3;
  c.odd = (c.x1 + c.x2 + c.x3 + parity) & 1;
  return c;
}

// Half index (in the OTHER parity's sublattice) of the neighbour x - mu_hat, periodic.
__device__ __forceinline__ int down_index(const Geom& g, int h, const SiteCoord& c, int mu) {
  if (mu == 0) {
    // x0 odd: x0-1 = 2*hx has the same hx.  x0 even: x0-1 -> hx-1, wrapping to N0/2-1.
    if (c.odd) return h;
    return c.hx > 0 ? h - 1 : h + g.nh0 - 1;
  }
  // selects instead of g.stride[mu] / g.n[mu]: a run-time index into the kernel-parameter struct
  // would make the compiler copy it to local memory
  const int x = (mu == 1) ? c.x1 : (mu == 2) ? c.x2 : c.x3;
  const int st = (mu == 1) ? g.stride[1] : (mu == 2) ? g.stride[2] : g.stride[3];
  const int wrap = (mu == 1) ? g.stride[1] * (g.n[1] - 1) : (mu == 2) ? g.stride[2] * (g.n[2] - 1) : g.wrap3;
  return x > 0 ? h - st : h + wrap;
}

// Half index (other parity) of x + mu_hat, periodic.
__device__ __forceinline__ int up_index(const Geom& g, int h, const SiteCoord& c, int mu) {
  if (mu == 0) {
    if (!c.odd) return h;
    return c.hx + 1 < g.nh0 ? h + 1 : h - (g.nh0 - 1);
  }
  int x = (mu == 1) ? c.x1 : (mu == 2) ? c.x2 : c.x3;
  int st = g.stride[mu];
  return x + 1 < g.n[mu] ? h + st : h - st * (g.n[mu] - 1);
}

// Canonical site index s = x0 + N0*(x1 + N1*(x2 + N2*x3)) of (parity, h).
__device__ __forceinline__ int64_t canonical_site(const Geom& g, int h, const SiteCoord& c) {
  return 2 * (int64_t)h + c.odd;   // h enumerates pairs (2k, 2k+1) of the canonical order
}

// Registers of a link as loaded / stored through its vectors (>= 18 matrix reals, >= NPAD).
constexpr int kLinkRegs = 20;

// ---- storage traits: how one link is cut into vectors ---------------------------------------
template <typename Real, int NP> struct VecOf;
template <> struct VecOf<float, 12> { typedef float4 type; };
template <> struct VecOf<float, 4>  { typedef float4 type; };
template <> struct VecOf<float, 18> { typedef float4 type; };   // 18 floats in 5 float4 (2 pad floats)
template <> struct VecOf<double, 12> { typedef double2 type; };
template <> struct VecOf<double, 18> { typedef double2 type; };
template <> struct VecOf<double, 4>  { typedef double2 type; };

template <typename Real_, int NC_, int NP_>
struct Storage {
  typedef Real_ Real;
  typedef typename VecOf<Real_, NP_>::type Vec;
  static constexpr int NC = NC_;                       // 2 or 3
  static constexpr int NP = NP_;                       // reals stored per link
  static constexpr int VL = sizeof(Vec) / sizeof(Real_);  // reals per vector
  static constexpr int NV = (NP_ + VL - 1) / VL;       // vectors per link (fp32-18: 5, last half used)
  static constexpr int NPAD = NV * VL;                 // reals moved per link (= NP except fp32-18: 20)
  static constexpr int NFULL = 2 * NC_ * NC_;          // reals of the full matrix
};

__device__ __forceinline__ void vec_get(const float4& v, float* r) { r[0] = v.x; r[1] = v.y; r[2] = v.z; r[3] = v.w; }
__device__ __forceinline__ void vec_get(const double2& v, double* r) { r[0] = v.x; r[1] = v.y; }
__device__ __forceinline__ void vec_set(float4& v, const float* r) { v = make_float4(r[0], r[1], r[2], r[3]); }
__device__ __forceinline__ void vec_set(double2& v, const double* r) { v = make_double2(r[0], r[1]); }

// Pointer to vector j=0 of link (parity, mu, h); vector j is at +j*pitch.
template <typename S>
__device__ __forceinline__ typename S::Vec* link_base(typename S::Vec* links, const Geom& g,
                                                      int parity, int mu, int h) {
  return links + ((size_t)((parity * 4 + mu) * S::NV)) * (size_t)g.pitch + (size_t)h;
}
template <typename S>
__device__ __forceinline__ const typename S::Vec* link_base(const typename S::Vec* links, const Geom& g,
                                                            int parity, int mu, int h) {
  return links + ((size_t)((parity * 4 + mu) * S::NV)) * (size_t)g.pitch + (size_t)h;
}

// Load the NP stored reals of a link into r[0..NP).
template <typename S>
__device__ __forceinline__ void load_params(const typename S::Vec* p, int pitch, typename S::Real* r) {
#pragma unroll
  for (int j = 0; j < S::NV; ++j) {
    typename S::Vec v = p[(size_t)j * (size_t)pitch];
    vec_get(v, r + j * S::VL);
  }
}
template <typename S>
__device__ __forceinline__ void store_params(typename S::Vec* p, int pitch, const typename S::Real* r) {
#pragma unroll
  for (int j = 0; j < S::NV; ++j) {
    typename S::Vec v;
    vec_set(v, r + j * S::VL);
    p[(size_t)j * (size_t)pitch] = v;
  }
}

// ---- programmatic dependent launch (sm_90+) ----------------------------------------------------
// A kernel that calls pdl_prologue_done() before its first global access, launched through
// launch_pdl(), lets the NEXT such launch of the stream be scheduled as soon as all of its own CTAs
// have started, instead of after its last CTA has drained: the next grid's CTAs take the SM slots
// the tail frees, do their index arithmetic, and block in griddepcontrol.wait until this grid has
// completed and its stores are visible.  Stream order is preserved exactly.
__device__ __forceinline__ void pdl_prologue_done() {
  asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
  asm volatile("griddepcontrol.wait;" ::: "memory");
}

template <typename... KArgs, typename... Args>
inline cudaError_t launch_pdl(void (*kern)(KArgs...), dim3 grid, dim3 block, size_t smem, cudaStream_t st,
                              Args... args) {
  cudaLaunchConfig_t cfg = {};
  cfg.gridDim = grid;
  cfg.blockDim = block;
  cfg.dynamicSmemBytes = smem;
  cfg.stream = st;
  cudaLaunchAttribute attr[1];
  attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
  attr[0].val.programmaticStreamSerializationAllowed = 1;
  cfg.attrs = attr;
  cfg.numAttrs = 1;
  return cudaLaunchKernelEx(&cfg, kern, static_cast<KArgs>(args)...);
}

}  // namespace culgt
