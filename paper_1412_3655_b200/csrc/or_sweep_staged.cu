// or_sweep_staged.cu -- the production SU(3) half-sweep kernel.
//
// PAPER.md L44-54, eq. 3; L19-21.  Machine mapping (the per-site body is in staged.cuh):
//
//  * The 8 links of a site are moved global -> shared memory by per-thread cp.async (LDGSTS)
//    into slots that only the issuing thread reads back.  The paper's obstacle (L72: 8 x 18 link
//    registers do not fit a thread) is solved on B200 by parking the links in the 228 KB of shared
//    memory per SM instead of splitting the site over 4 or 8 threads and paying the K(x) exchange.
//  * Registers then hold only K (fp64), G and one link at a time: 126 registers for fp32
//    storage, no spills in any format.
//  * Grid: ONE small CTA per site block (128 threads x 4 CTAs/SM for fp32-12, 64 x 3 for fp64-18),
//    handed out in order by the hardware block scheduler.  Small CTAs that retire and are replaced
//    one at a time keep loads, arithmetic and stores of different CTAs overlapped (a persistent
//    grid-stride loop measured 8-23 % slower).  Odd-parity launches map blockIdx to
//    site blocks in DESCENDING order so that the white half-sweep starts on the links the black
//    half-sweep touched last, which are still in the L2.
//  * K accumulation, the subgroup chain and G in fp64 (su3_solve.cuh); reconstruction and link
//    products in the storage precision.
//
// The measured alternatives (2/4/8 threads per site, persistent grids, two stages, prefetch, the
// all-fp32 and no-solve measurement kernels, slab-blocked launch schedules) live in
// or_sweep_measure.cu and are compiled only with -DCULGT_MEASURE.
#include "staged.cuh"
#include "kernels.h"

namespace culgt {

// Launch options of the production kernel.
constexpr int OPT_PDL = 512;       // programmatic dependent launch: the next half-sweep's CTAs are scheduled
                                   // (index arithmetic done) while this one's last wave drains
constexpr int OPT_L2HINT = 1024;   // L2 eviction hints by position in the traversal.  The CTAs from
                                   // `late_from` on (the last part of the field a launch touches, which the next,
                                   // reversed launch revisits first) store with evict_last and load normally; the
                                   // earlier ones load with evict_first (their lines cannot survive until they are
                                   // revisited) and store normally.  late_from < 0: no preference anywhere.
constexpr int OPT_COULOMB = 64;    // Coulomb gauge (reading C-22): K(x) from the 6 spatial links only

// One CTA per site block: blockIdx b works on site block block_lo + (reverse ? n - 1 - b : b) of
// the sublattice `parity`.  stop_flag (may be null): a device word that a driver loop sets once
// its stopping criterion is met; every CTA of a launch enqueued after that returns at entry
// (api.cu, culgt_landau_fix).
template <typename S, int BLOCK, int MINB, int OPT, typename Power>
__global__ void __launch_bounds__(BLOCK, MINB)
or_sweep_su3_staged_kernel(typename S::Vec* __restrict__ links, const Geom g, const int parity,
                           const Power omega, const int n_site_blocks, const int reverse,
                           const int block_lo, const int late_from, const int* __restrict__ stop_flag) {
  typedef typename S::Vec Vec;
  extern __shared__ __align__(16) unsigned char smem_raw[];
  Vec* const sm = reinterpret_cast<Vec*>(smem_raw) + threadIdx.x;   // vector v of link l at sm[(l*NV+v)*BLOCK]
  const unsigned sm_addr = (unsigned)__cvta_generic_to_shared(sm);
  constexpr bool L2HINT = (OPT & OPT_L2HINT) != 0;
  uint64_t pol = 0, pol_st = 0;
  if (L2HINT) {
    L2Policies p;
    p.create();
    const bool late = (int)blockIdx.x >= late_from;
    pol = (late_from < 0 || late) ? p.normal : p.first;
    pol_st = (late_from >= 0 && late) ? p.last : p.normal;
  }
  const int site_block = block_lo + (reverse ? n_site_blocks - 1 - (int)blockIdx.x : (int)blockIdx.x);
  SiteRef<8> r = locate<BLOCK, 1>(g, parity, site_block, 0);
  if (OPT & OPT_PDL) {
    // let the next launch of the stream be scheduled as soon as every CTA of this one has started,
    // then wait until the previous launch has completed and its stores are visible
    pdl_prologue_done();
  }
  if (stop_flag != nullptr && *stop_flag != 0) return;
  if (OPT & OPT_COULOMB) apply_slice_mask(g, r);
  issue_site_loads<S, BLOCK, L2HINT>(links, g, parity, r, sm, pol);
  cp_async_wait<0>();
  update_site<S, BLOCK, (OPT & OPT_COULOMB) != 0, L2HINT>(links, g, parity, omega, r, sm_addr, pol_st);
}

// ---------------------------------------------------------------------------------------------
// host side
// ---------------------------------------------------------------------------------------------

// Per-device properties (a process may drive several devices).
int device_sm_count() {
  static int cache[kMaxDevices] = {0};
  int dev = 0;
  if (cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev >= kMaxDevices) return 148;
  if (cache[dev] == 0) {
    int n = 0;
    if (cudaDeviceGetAttribute(&n, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess || n <= 0) n = 148;
    cache[dev] = n;
  }
  return cache[dev];
}
double device_l2_bytes() {
  static double cache[kMaxDevices] = {0};
  int dev = 0;
  if (cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev >= kMaxDevices) return 126e6;
  if (cache[dev] == 0) {
    int n = 0;
    if (cudaDeviceGetAttribute(&n, cudaDevAttrL2CacheSize, dev) != cudaSuccess || n <= 0) n = 126 * 1000 * 1000;
    cache[dev] = (double)n;
  }
  return cache[dev];
}

// win_n >= 0: only the window [win_lo, win_lo + win_n) of site blocks (time-slab launches, slab.cu),
// traversed descending iff win_reverse.
template <typename S, int BLOCK, int MINB, int OPT, typename Power>
static cudaError_t launch_staged(void* links, const Geom& g, int parity, Power omega, bool reverse_odd,
                                 const int* stop_flag, cudaStream_t st, int win_lo = 0, int win_n = -1,
                                 int win_reverse = -1) {
  typedef typename S::Vec Vec;
  const double field_bytes = 8.0 * (double)g.vh * S::NV * sizeof(Vec);
  const double l2 = device_l2_bytes();
  if constexpr ((OPT & OPT_L2HINT) != 0) {
    // The hints pay where the field is a small multiple of the L2 (measured on the 126 MB L2 of B200:
    // 201 MB 58.4 -> 55.0 us, 604 MB 177.3 -> 176.9, 2.0 GB 617 -> 627, 9.7 GB 2863 -> 2924, i.e. between
    // 0.87 and 5.5 L2 sizes): elsewhere, and for windowed launches, the same mapping without them.
    if (win_n >= 0 || field_bytes < 0.87 * l2 || field_bytes > 5.5 * l2)
      return launch_staged<S, BLOCK, MINB, OPT & ~OPT_L2HINT, Power>(links, g, parity, omega, reverse_odd, stop_flag, st,
                                                                    win_lo, win_n, win_reverse);
  }
  auto kern = or_sweep_su3_staged_kernel<S, BLOCK, MINB, OPT, Power>;
  constexpr size_t smem = staged_smem_bytes<S, BLOCK>();
  static bool configured[kMaxDevices] = {false};
  int dev = 0;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) return e;
  if (dev < 0 || dev >= kMaxDevices || !configured[dev]) {
    e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    if (dev >= 0 && dev < kMaxDevices) configured[dev] = true;
  }
  // the whole parity sublattice, or the window [win_lo, win_lo + win_n) of it
  const int n_site_blocks = win_n >= 0 ? win_n : (g.vh + BLOCK - 1) / BLOCK;
  if (n_site_blocks == 0) return cudaSuccess;
  const int grid = n_site_blocks;
  const int rev = win_reverse >= 0 ? win_reverse : ((reverse_odd && parity) ? 1 : 0);
  // the last 0.71 L2 sizes of links of the traversal (90 MB on B200) are kept for the next (reversed) launch
  int late_from = -1;
  if (OPT & OPT_L2HINT) late_from = grid - (int)((double)grid * (0.71 * l2 / field_bytes));
  if (OPT & OPT_PDL) {
    return launch_pdl(kern, dim3((unsigned)grid), dim3(BLOCK), smem, st, (Vec*)links, g, parity, omega,
                      n_site_blocks, rev, win_lo, late_from, stop_flag);
  }
  kern<<<grid, BLOCK, smem, st>>>((Vec*)links, g, parity, omega, n_site_blocks, rev, win_lo, late_from, stop_flag);
  return cudaGetLastError();
}

// The production mapping of each storage format ("AxB" = A threads per CTA, B CTAs per SM):
// fp32-12 128x4, fp32-18 64x5, fp64-12 64x4, fp64-18 64x3 (profiles/r1_variant_sweep.md).
template <int OPT, typename Power>
static cudaError_t launch_format(const LatticeDesc& d, void* links, int parity, const Power& pw, bool reverse_odd,
                                 const int* stop_flag, cudaStream_t st, int win_lo = 0, int win_n = -1,
                                 int win_reverse = -1) {
  const Geom& g = d.geom;
  if (d.group != 3) return cudaErrorInvalidValue;
  if (d.precision == 32 && d.params == 12)
    return launch_staged<Storage<float, 3, 12>, 128, 4, OPT>(links, g, parity, pw, reverse_odd, stop_flag, st, win_lo, win_n, win_reverse);
  if (d.precision == 32)
    return launch_staged<Storage<float, 3, 18>, 64, 5, OPT>(links, g, parity, pw, reverse_odd, stop_flag, st, win_lo, win_n, win_reverse);
  if (d.params == 12)
    return launch_staged<Storage<double, 3, 12>, 64, 4, OPT>(links, g, parity, pw, reverse_odd, stop_flag, st, win_lo, win_n, win_reverse);
  return launch_staged<Storage<double, 3, 18>, 64, 3, OPT>(links, g, parity, pw, reverse_odd, stop_flag, st, win_lo, win_n, win_reverse);
}

// Name of the kernel instantiation that variant 0 launches for this lattice (what a committed ncu
// capture must have been taken on to describe it: bench.py, profiles/roofline_traffic.csv).  The
// numbers are the ones launch_format uses.
const char* sweep_kernel_name(const LatticeDesc& d) {
  if (d.group == 2) return d.precision == 32 ? "or_sweep_su2_kernel<f32-4,128,pdl>" : "or_sweep_su2_kernel<f64-4,128,pdl>";
  if (d.precision == 32 && d.params == 12) return "or_sweep_su3_staged_kernel<f32-12,128x4,pdl+l2hint,r2>";
  if (d.precision == 32) return "or_sweep_su3_staged_kernel<f32-18,64x5,pdl+l2hint,r2>";
  if (d.params == 12) return "or_sweep_su3_staged_kernel<f64-12,64x4,pdl+l2hint,r2>";
  return "or_sweep_su3_staged_kernel<f64-18,64x3,pdl+l2hint,r2>";
}

// Product variants of the SU(3) half-sweep: all the same per-site arithmetic (bit-identical
// results), different launch options.  0 / 20 production; 24 without the reversed odd-parity
// traversal; 33 without programmatic dependent launch; 34 without L2 hints.
cudaError_t launch_or_sweep_staged(const LatticeDesc& d, void* links, int parity, double omega,
                                   int variant, bool coulomb, const int* stop_flag, cudaStream_t st) {
  if (d.group != 3) return cudaErrorInvalidValue;
  if (coulomb) {   // Coulomb gauge: the production mapping of each format with K from spatial links
    if (variant != 20) return cudaErrorInvalidValue;
    return launch_format<OPT_PDL | OPT_L2HINT | OPT_COULOMB>(d, links, parity, omega, true, stop_flag, st);
  }
  switch (variant) {
    case 20: return launch_format<OPT_PDL | OPT_L2HINT>(d, links, parity, omega, true, stop_flag, st);
    case 24: return launch_format<0>(d, links, parity, omega, false, stop_flag, st);
    case 33: return launch_format<0>(d, links, parity, omega, true, stop_flag, st);
    case 34: return launch_format<OPT_PDL>(d, links, parity, omega, true, stop_flag, st);
    default: return cudaErrorInvalidValue;
  }
}

// Windowed half-sweep over the time-slices [t_lo, t_hi) of the sublattice `parity` (time-slab
// decomposition, slab.cu): the production mapping without L2 hints, ascending.  The lattice must
// hold whole site blocks per slice (cudaErrorNotSupported otherwise).
cudaError_t launch_or_sweep_window(const LatticeDesc& d, void* links, int parity, double omega, int t_lo, int t_hi,
                                   cudaStream_t st) {
  const Geom& g = d.geom;
  if (d.group != 3) return cudaErrorNotSupported;
  const int block = (d.precision == 32 && d.params == 12) ? 128 : 64;
  if (g.stride[3] % block != 0) return cudaErrorNotSupported;
  if (t_hi <= t_lo) return cudaSuccess;
  const int bps = g.stride[3] / block;
  return launch_format<OPT_PDL>(d, links, parity, omega, false, nullptr, st, t_lo * bps, (t_hi - t_lo) * bps, 0);
}

// Truncated-series overrelaxation (reading C-24) / simulated annealing (C-25) / the
// microcanonical step (C-26) on the production mapping of each format.
cudaError_t launch_or_sweep_staged_series(const LatticeDesc& d, void* links, int parity, const SeriesPower& pw,
                                          cudaStream_t st) {
  return launch_format<OPT_PDL | OPT_L2HINT>(d, links, parity, pw, true, nullptr, st);
}
cudaError_t launch_or_sweep_staged_micro(const LatticeDesc& d, void* links, int parity, cudaStream_t st) {
  return launch_format<OPT_PDL | OPT_L2HINT>(d, links, parity, MicroPower{0}, true, nullptr, st);
}
cudaError_t launch_or_sweep_staged_heatbath(const LatticeDesc& d, void* links, int parity, const HeatBathPower& pw,
                                            cudaStream_t st) {
  return launch_format<OPT_PDL | OPT_L2HINT>(d, links, parity, pw, true, nullptr, st);
}

}  // namespace culgt
