// kernels.h -- internal (C++) interface between the C-ABI layer (api.cu) and the kernel files.
#pragma once
#include <cuda_runtime.h>
#include <stddef.h>
#include "lattice.cuh"

namespace culgt {

struct LatticeDesc {
  Geom geom;
  int group;      // 2 or 3
  int precision;  // 32 or 64
  int params;     // 18, 12 or 4
  long long V;
};

constexpr int kMaxDevices = 64;         // per-device caches (function attributes, SM count, L2 size)
int device_sm_count();                  // of the current device
double device_l2_bytes();

constexpr int kReduceBlock = 256;       // threads per block of the reduction kernels
// CTAs (= partials per quantity) of the fused theta+F kernel: `half` sites of each parity per CTA
// (128 for the register path, 64 for the staged fp32 12-parameter path; the workspace is sized for 64)
inline int reduce_blocks_fused(int vh, int half = 64) { return (vh + half - 1) / half; }
// doubles in the reduction workspace: block partials (Landau: 2 * vh/128; Coulomb: 2 * N3 *
// slice/128; never below 4096) followed by 2 * N3 result slots that the *_host / *_fix paths
// read back (Landau uses the first two).
inline size_t reduce_partial_doubles(const Geom& g) {
  size_t n = 2 * (size_t)reduce_blocks_fused(g.vh) + 8;      // + 8 spare slots
  const size_t c = 2 * (size_t)g.n[3] * (size_t)reduce_blocks_fused(g.stride[3]);
  if (c > n) n = c;
  return n > 4096 ? n : 4096;
}
// ... and N3 bytes (rounded up to doubles) for the Coulomb driver's per-slice activity mask
inline size_t reduce_workspace_doubles(const Geom& g) {
  return reduce_partial_doubles(g) + 2 * (size_t)g.n[3] + ((size_t)g.n[3] + 7) / 8;
}

// ---- control blocks that live behind the reduction part of the caller's workspace ---------------
// The library keeps no device state of its own: whatever a kernel needs to remember between
// launches sits in the workspace the caller hands in, and is (re)initialised by the call that uses it.

// Driver loop (culgt_landau_fix): written by the final reduction kernel of every check, read by
// the sweep and reduction kernels enqueued behind it (they return at entry once `stop` is set).
struct FixCtl {
  int stop;            // 1 once a check found theta < theta_target
  int checks_done;     // checks that ran (not skipped) so far
  int sweeps_at_stop;  // value of `sweeps_before` of the check that set `stop`
  int pad;
  double theta, F;     // of the last check that ran
};

// Persistent driver loop for small lattices (fix_persistent.cu); shares FixCtl's slot.
struct PersistCtl {
  unsigned barrier;    // grid barrier: arrivals so far (monotone)
  int sweeps_done;
  double theta, F;
};

// Fused full sweep (or_sweep_fused.cu; -DCULGT_MEASURE builds only -- the struct is declared
// unconditionally so that both builds lay the workspace out the same way).
constexpr int kFusedMaxSlices = 512;
struct FusedCtl {
  unsigned ticket;                           // next ticket of the running launch
  unsigned exited;                           // CTAs of the running launch that have left
  unsigned pad[30];
  unsigned done[2][kFusedMaxSlices];         // completed site blocks per (parity, time-slice)
  unsigned task[2][2 * kFusedMaxSlices];     // [direction][u] = parity << 31 | slice: slice-task order
};

// L2 eviction policies of the fused sweep (2 bits each: black loads, black stores, white loads, white
// stores; 0 evict_first, 1 evict_normal, 2 evict_last), chosen by measurement
constexpr int kFusedDefaultHints = 1 | (1 << 2) | (1 << 4) | (1 << 6);

inline size_t ctl_offset_doubles(const Geom& g) { return (reduce_workspace_doubles(g) + 15) / 16 * 16; }
inline size_t fix_ctl_offset_doubles(const Geom& g) { return ctl_offset_doubles(g); }
inline size_t fused_ctl_offset_doubles(const Geom& g) { return ctl_offset_doubles(g) + 16; }
inline size_t workspace_doubles(const Geom& g) { return fused_ctl_offset_doubles(g) + sizeof(FusedCtl) / 8; }
static_assert(sizeof(FixCtl) <= 16 * 8 && sizeof(PersistCtl) <= 16 * 8, "the driver-loop control blocks share a 16-double slot");
static_assert(sizeof(FusedCtl) % 8 == 0, "FusedCtl is addressed in doubles");

// ---- half-sweeps ----------------------------------------------------------------------------------
// Product variants: 0 (= 20) production mapping; 24 no reversed odd-parity traversal; 33 no programmatic
// dependent launch; 34 no L2 hints -- identical arithmetic, bit-identical results.  With
// -DCULGT_MEASURE also the measured alternatives of or_sweep_measure.cu.  Others: cudaErrorInvalidValue.
// coulomb = true: Coulomb-gauge half-sweep (K from the spatial links; production mapping only).
// stop_flag (device, may be null): the launch does nothing if *stop_flag != 0 when it starts.
bool sweep_variant_known(int variant);
const char* sweep_kernel_name(const LatticeDesc& d);
cudaError_t launch_or_sweep(const LatticeDesc& d, void* links, int parity, double omega,
                            int variant, cudaStream_t st, bool coulomb = false, const int* stop_flag = nullptr);
cudaError_t launch_or_sweep_staged(const LatticeDesc& d, void* links, int parity, double omega,
                                   int variant, bool coulomb, const int* stop_flag, cudaStream_t st);
// production half-sweep restricted to the time-slices [t_lo, t_hi) (time-slab decomposition)
cudaError_t launch_or_sweep_window(const LatticeDesc& d, void* links, int parity, double omega, int t_lo, int t_hi,
                                   cudaStream_t st);
struct SeriesPower;
struct HeatBathPower;
// simulated-annealing half-sweep (reading C-25), production mappings only
cudaError_t launch_sa_sweep(const LatticeDesc& d, void* links, int parity, double T, unsigned long long seed,
                            unsigned counter, cudaStream_t st);
cudaError_t launch_or_sweep_staged_heatbath(const LatticeDesc& d, void* links, int parity, const HeatBathPower& pw,
                                            cudaStream_t st);
// microcanonical half-sweep (reading C-26), production mappings only
cudaError_t launch_micro_sweep(const LatticeDesc& d, void* links, int parity, cudaStream_t st);
cudaError_t launch_or_sweep_staged_micro(const LatticeDesc& d, void* links, int parity, cudaStream_t st);
// truncated-series overrelaxation (reading C-24), production mappings only
cudaError_t launch_or_sweep_series(const LatticeDesc& d, void* links, int parity, double omega, int order,
                                   cudaStream_t st);
cudaError_t launch_or_sweep_staged_series(const LatticeDesc& d, void* links, int parity, const SeriesPower& pw,
                                          cudaStream_t st);

// ---- full sweeps ------------------------------------------------------------------------------------
// n_sweeps FULL sweeps (black then white), two half-sweep launches each.  `workspace` (may be null)
// is the caller's reduction workspace; only the -DCULGT_MEASURE build uses it here (variant 60: the
// fused one-kernel schedule of or_sweep_fused.cu).
cudaError_t launch_or_full_sweeps(const LatticeDesc& d, void* links, double* workspace, int n_sweeps, double omega,
                                  int variant, const int* stop_flag, cudaStream_t st);
#ifdef CULGT_MEASURE
// the fused schedule itself: cudaErrorNotSupported when the lattice does not qualify.
// lag <= 0: default; hints: L2 policy bits (or_sweep_fused.cu); alternate: every other sweep descending.
cudaError_t launch_or_sweeps_fused(const LatticeDesc& d, void* links, double omega, void* ctl, int n_sweeps,
                                   int lag, int hints, bool alternate, const int* stop_flag, cudaStream_t st);
void fused_schedule(int n3, int lag, int dir, unsigned* out);   // host: the slice-task order (2 * n3 entries)
cudaError_t launch_or_sweep_measure(const LatticeDesc& d, void* links, int parity, double omega, int variant,
                                    cudaStream_t st);
cudaError_t launch_or_sweep_measure_slabbed(const LatticeDesc& d, void* links, double omega, int slab_slices,
                                            cudaStream_t st);
#endif

// The whole driver loop as one cooperative kernel (fix_persistent.cu): SU(3) lattices with at most one
// site block per SM and parity; cudaErrorNotSupported otherwise.  partial: 2 * (site blocks) doubles.
cudaError_t launch_landau_fix_persistent(const LatticeDesc& d, void* links, double omega, double theta_target,
                                         int max_sweeps, int check_every, double* partial, PersistCtl* ctl,
                                         cudaStream_t st);

// ---- layout, reductions, transform ----------------------------------------------------------------
cudaError_t launch_pack(const LatticeDesc& d, const void* canonical, void* links, cudaStream_t st);
cudaError_t launch_reunitarize(const LatticeDesc& d, void* links, cudaStream_t st);
cudaError_t launch_unpack(const LatticeDesc& d, const void* links, void* canonical, cudaStream_t st);
// fused theta + F; workspace holds 2 * reduce_blocks_fused(vh) partials.
// fix (may be null): driver-loop bookkeeping done by the final kernel -- see FixCtl; the pass is
// skipped when fix->stop is already set.
struct FixCheck {
  FixCtl* ctl;
  double theta_target;
  int sweeps_before;     // sweeps completed when this check runs
};
cudaError_t launch_theta_functional(const LatticeDesc& d, const void* links, double* workspace,
                                    double* out_theta, double* out_F, cudaStream_t st,
                                    const FixCheck* fix = nullptr);
// the same pass with the block partials in the library's own file-scope device array (reduce.cu): allocates
// nothing; cudaErrorMemoryAllocation when the lattice needs more partials than the array holds
size_t noalloc_partials_needed(const LatticeDesc& d);
cudaError_t launch_theta_functional_noalloc(const LatticeDesc& d, const void* links, double* out_theta, double* out_F,
                                            cudaStream_t st);
// Coulomb gauge: per-slice theta_t, F_t (N3 doubles each).  chk (may be null): driver-loop bookkeeping on
// the device -- the per-slice activity mask is recomputed from theta_t, the stop word raised when no slice
// is active; the pass is skipped when the stop word is already set.
struct CoulombCheck {
  FixCtl* ctl;
  unsigned char* mask;   // N3 bytes, device
  double theta_target;
  int sweeps_before;
};
cudaError_t launch_coulomb_theta_functional(const LatticeDesc& d, const void* links, double* workspace,
                                            double* out_theta_t, double* out_F_t, cudaStream_t st,
                                            const CoulombCheck* chk = nullptr);
cudaError_t launch_gauge_transform(const LatticeDesc& d, void* links, const void* g, cudaStream_t st);

// ---- time-slab decomposition (slab.cu) ------------------------------------------------------------------
void make_slab_geom(Geom* g);     // pitch and wrap3 of a slab with a ghost slice
int slab_vectors_per_link(const LatticeDesc& d);
void slab_halo_chunks(const LatticeDesc& d, int parity, int which, size_t* offsets, size_t* chunk_bytes, int* n_chunks);
cudaError_t slab_halo_copy(const LatticeDesc& d, const void* src, void* dst, int parity, int direction, cudaStream_t st);
cudaError_t slab_theta_F_combine(const LatticeDesc& global, const double* sums, int n_slabs, double* theta, double* F,
                                 cudaStream_t st);
// fused theta + F of one slab as RAW sums (sum_x tr[Delta Delta^dagger], sum_{x,mu} Re tr U): out2[0], out2[1]
cudaError_t launch_theta_functional_sums(const LatticeDesc& slab, const void* links, double* workspace, double* out2,
                                         cudaStream_t st);
void slab_halo_peers(int rank, int n_ranks, int direction, int* send_to, int* recv_from);
bool slab_nccl_available();
const char* slab_nccl_error(int code);
int slab_comm_id(void* id128);
int slab_comm_create(const void* id128, int rank, int n_ranks, void** out);
int slab_comm_destroy(void* comm);
void slab_comm_info(void* comm, int* rank, int* n_ranks);
int slab_halo_exchange(void* comm, const LatticeDesc& d, void* links, int parity, int direction, cudaStream_t st);
int slab_allgather_sums(void* comm, const double* sums2, double* all, cudaStream_t st);

}  // namespace culgt
