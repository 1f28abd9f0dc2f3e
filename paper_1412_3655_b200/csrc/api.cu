// api.cu -- the C ABI of libculgt_b200.so (include/culgt_b200.h): descriptor validation, error
// codes and dispatch to the kernel launchers.  No compute happens here.
#include <math.h>
#include <stdio.h>
#include <stdlib.h>
#include <string.h>
#include <vector>
#include "../../include/culgt_b200.h"
#include "kernels.h"
#include "measure_api.h"

using namespace culgt;

namespace {

// Per host thread: the text of the last CUDA error and the sweep-variant selection.  The library has
// no process-global mutable state beyond caches of device properties and of lazily-set function
// attributes (both per device).
thread_local char g_cuda_err[256] = "";
thread_local int g_variant = 0;

int nccl_fail(int code) {
  snprintf(g_cuda_err, sizeof(g_cuda_err), "NCCL: %s", slab_nccl_error(code));
  return CULGT_ERR_NCCL;
}

int cuda_fail(cudaError_t e) {
  snprintf(g_cuda_err, sizeof(g_cuda_err), "%s: %s", cudaGetErrorName(e), cudaGetErrorString(e));
  return CULGT_ERR_CUDA;
}

int describe(const culgt_lattice* lat, LatticeDesc* d) {
  if (!lat) return CULGT_ERR_NULL;
  long long v = 1;
  for (int i = 0; i < 4; ++i) {
    const int n = lat->dims[i];
    if (n < 2 || (n & 1)) return CULGT_ERR_DIMS;
    v *= n;
    if (v > (1ll << 30)) return CULGT_ERR_DIMS;   // 32-bit site indices, 8*V thread indices in 64-bit
  }
  const bool prec_ok = lat->precision == 32 || lat->precision == 64;
  const bool su3 = lat->group == 3 && (lat->params == 18 || lat->params == 12);
  const bool su2 = lat->group == 2 && lat->params == 4;
  if (!prec_ok || !(su3 || su2)) return CULGT_ERR_DESC;
  if (d) {
    d->geom = make_geom(lat->dims);
    d->group = lat->group;
    d->precision = lat->precision;
    d->params = lat->params;
    d->V = v;
  }
  return CULGT_OK;
}

bool misaligned(const void* p) { return ((uintptr_t)p & 15u) != 0; }

// descriptor of one time slab: the local lattice with a ghost slice behind every plane (slab.cu)
int describe_slab(const culgt_lattice* local, LatticeDesc* d) {
  const int rc = describe(local, d);
  if (rc != CULGT_OK) return rc;
  if ((long long)d->geom.vh + d->geom.stride[3] >= (1ll << 30)) return CULGT_ERR_DIMS;
  make_slab_geom(&d->geom);
  return CULGT_OK;
}

}  // namespace

extern "C" {

int culgt_validate(const culgt_lattice* lat) { return describe(lat, nullptr); }

size_t culgt_links_bytes(const culgt_lattice* lat) {
  LatticeDesc d;
  if (describe(lat, &d) != CULGT_OK) return 0;
  // fp32 18-parameter links are stored as 5 float4 (80 bytes, 2 pad floats): 16-byte accesses
  const size_t link_bytes = (d.group == 3 && d.precision == 32 && d.params == 18)
                                ? 80 : (size_t)d.params * (size_t)(d.precision / 8);
  return (size_t)4 * (size_t)d.V * link_bytes;
}

size_t culgt_canonical_bytes(const culgt_lattice* lat) {
  LatticeDesc d;
  if (describe(lat, &d) != CULGT_OK) return 0;
  return (size_t)4 * (size_t)d.V * (size_t)(2 * d.group * d.group) * (size_t)(d.precision / 8);
}

size_t culgt_gfield_bytes(const culgt_lattice* lat) {
  LatticeDesc d;
  if (describe(lat, &d) != CULGT_OK) return 0;
  return (size_t)d.V * (size_t)(2 * d.group * d.group) * (size_t)(d.precision / 8);
}

size_t culgt_workspace_bytes(const culgt_lattice* lat) {
  LatticeDesc d;
  if (describe(lat, &d) != CULGT_OK) return 0;
  // block partials + 2 * N3 result slots + the Coulomb mask + the driver-loop and fused-sweep control blocks
  return workspace_doubles(d.geom) * sizeof(double);
}

int culgt_pack(const culgt_lattice* lat, const void* canonical, void* links, void* stream) {
  LatticeDesc d;
  int rc = describe(lat, &d);
  if (rc != CULGT_OK) return rc;
  if (!canonical || !links) return CULGT_ERR_NULL;
  if (misaligned(canonical) || misaligned(links)) return CULGT_ERR_ALIGN;
  cudaError_t e = launch_pack(d, canonical, links, (cudaStream_t)stream);
  return e == cudaSuccess ? CULGT_OK : cuda_fail(e);
}

int culgt_unpack(const culgt_lattice* lat, const void* links, void* canonical, void* stream) {
  LatticeDesc d;
  int rc = describe(lat, &d);
  if (rc != CULGT_OK) return rc;
  if (!canonical || !links) return CULGT_ERR_NULL;
  if (misaligned(canonical) || misaligned(links)) return CULGT_ERR_ALIGN;
  cudaError_t e = launch_unpack(d, links, canonical, (cudaStream_t)stream);
  return e == cudaSuccess ? CULGT_OK : cuda_fail(e);
}

int culgt_reunitarize(const culgt_lattice* lat, void* links, void* stream) {
  LatticeDesc d;
  int rc = describe(lat, &d);
  if (rc != CULGT_OK) return rc;
  if (!links) return CULGT_ERR_NULL;
  if (misaligned(links)) return CULGT_ERR_ALIGN;
  cudaError_t e = launch_reunitarize(d, links, (cudaStream_t)stream);
  return e == cudaSuccess ? CULGT_OK : cuda_fail(e);
}

static int check_omega(double omega) {
  if (!(omega >= 1.0 && omega < 2.0)) return CULGT_ERR_OMEGA;   // NaN fails the comparison
  return CULGT_OK;
}

int culgt_or_sweep(const culgt_lattice* lat, void* links, int parity, double omega, void* stream) {
  LatticeDesc d;
  int rc = describe(lat, &d);
  if (rc != CULGT_OK) return rc;
  if (!links) return CULGT_ERR_NULL;
  if (misaligned(links)) return CULGT_ERR_ALIGN;
  if (parity != 0 && parity != 1) return CULGT_ERR_PARITY;
  if ((rc = check_omega(omega)) != CULGT_OK) return rc;
  cudaError_t e = launch_or_sweep(d, links, parity, omega, g_variant, (cudaStream_t)stream);
  return e == cudaSuccess ? CULGT_OK : cuda_fail(e);
}

int culgt_or_sweeps(const culgt_lattice* lat, void* links, int n_sweeps, double omega, void* stream) {
  LatticeDesc d;
  int rc = describe(lat, &d);
  if (rc != CULGT_OK) return rc;
  if (!links) return CULGT_ERR_NULL;
  if (misaligned(links)) return CULGT_ERR_ALIGN;
  if (n_sweeps < 0) return CULGT_ERR_ARG;
  if ((rc = check_omega(omega)) != CULGT_OK) return rc;
  cudaError_t e = launch_or_full_sweeps(d, links, nullptr, n_sweeps, omega, g_variant, nullptr, (cudaStream_t)stream);
  return e == cudaSuccess ? CULGT_OK : cuda_fail(e);
}

int culgt_gauge_precision(const culgt_lattice* lat, const void* links, void* workspace,
                          double* theta_dev, void* stream) {
  LatticeDesc d;
  int rc = describe(lat, &d);
  if (rc != CULGT_OK) return rc;
  if (!links || !workspace || !theta_dev) return CULGT_ERR_NULL;
  if (misaligned(links) || misaligned(workspace)) return CULGT_ERR_ALIGN;
  // one fused pass computes both scalars; F goes to the spare slot at the end of the workspace
  double* spare = (double*)workspace + reduce_partial_doubles(d.geom) + 1;
  cudaError_t e = launch_theta_functional(d, links, (double*)workspace, theta_dev, spare, (cudaStream_t)stream);
  return e == cudaSuccess ? CULGT_OK : cuda_fail(e);
}

int culgt_functional(const culgt_lattice* lat, const void* links, void* workspace,
                     double* F_dev, void* stream) {
  LatticeDesc d;
  int rc = describe(lat, &d);
  if (rc != CULGT_OK) return rc;
  if (!links || !workspace || !F_dev) return CULGT_ERR_NULL;
  if (misaligned(links) || misaligned(workspace)) return CULGT_ERR_ALIGN;
  double* spare = (double*)workspace + reduce_partial_doubles(d.geom);
  cudaError_t e = launch_theta_functional(d, links, (double*)workspace, spare, F_dev, (cudaStream_t)stream);
  return e == cudaSuccess ? CULGT_OK : cuda_fail(e);
}

int culgt_gauge_transform(const culgt_lattice* lat, void* links, const void* g, void* stream) {
  LatticeDesc d;
  int rc = describe(lat, &d);
  if (rc != CULGT_OK) return rc;
  if (!links || !g) return CULGT_ERR_NULL;
  if (misaligned(links) || misaligned(g)) return CULGT_ERR_ALIGN;
  cudaError_t e = launch_gauge_transform(d, links, g, (cudaStream_t)stream);
  return e == cudaSuccess ? CULGT_OK : cuda_fail(e);
}

int culgt_gauge_precision_functional(const culgt_lattice* lat, const void* links, void* workspace,
                                     double* theta_dev, double* F_dev, void* stream) {
  LatticeDesc d;
  int rc = describe(lat, &d);
  if (rc != CULGT_OK) return rc;
  if (!links || !workspace || !theta_dev || !F_dev) return CULGT_ERR_NULL;
  if (misaligned(links) || misaligned(workspace)) return CULGT_ERR_ALIGN;
  cudaError_t e = launch_theta_functional(d, links, (double*)workspace, theta_dev, F_dev, (cudaStream_t)stream);
  return e == cudaSuccess ? CULGT_OK : cuda_fail(e);
}

// theta and F for callers that cannot allocate: no workspace argument, the block partials live in a 2 MiB
// file-scope device array of the library (csrc/reduce.cu).
int culgt_gauge_precision_functional_noalloc(const culgt_lattice* lat, const void* links, double* theta_dev,
                                             double* F_dev, void* stream) {
  LatticeDesc d;
  int rc = describe(lat, &d);
  if (rc != CULGT_OK) return rc;
  if (!links || !theta_dev || !F_dev) return CULGT_ERR_NULL;
  if (misaligned(links)) return CULGT_ERR_ALIGN;
  if ((long long)d.V > (long long)CULGT_NOALLOC_MAX_SITES) return CULGT_ERR_TOO_LARGE;
  cudaError_t e = launch_theta_functional_noalloc(d, links, theta_dev, F_dev, (cudaStream_t)stream);
  if (e == cudaErrorMemoryAllocation) {          // the launcher's own size check (never an allocation failure)
    cudaGetLastError();
    return CULGT_ERR_TOO_LARGE;
  }
  return e == cudaSuccess ? CULGT_OK : cuda_fail(e);
}

// theta and F (one fused pass) into the first two result slots of the workspace, read back.
static int read_theta_F(const LatticeDesc& d, const void* links, void* workspace, cudaStream_t st,
                        double* theta, double* F) {
  double* ws = (double*)workspace;
  double* scal = ws + reduce_partial_doubles(d.geom);
  cudaError_t e = launch_theta_functional(d, links, ws, scal, scal + 1, st);
  if (e != cudaSuccess) return cuda_fail(e);
  double host[2] = {0, 0};
  e = cudaMemcpyAsync(host, scal, 2 * sizeof(double), cudaMemcpyDeviceToHost, st);
  if (e != cudaSuccess) return cuda_fail(e);
  e = cudaStreamSynchronize(st);
  if (e != cudaSuccess) return cuda_fail(e);
  *theta = host[0];
  if (F) *F = host[1];
  return CULGT_OK;
}

// The driver loop runs on the DEVICE between synchronisations: every check's final reduction kernel
// records theta and F in a control block in the workspace and raises its stop word once
// theta < theta_target; sweeps and checks enqueued behind a raised stop word return at entry.  The
// host enqueues rounds of (check_every sweeps + one check) in batches and reads the control block back
// once per batch, instead of once per check.
int culgt_landau_fix(const culgt_lattice* lat, void* links, void* workspace, double omega,
                     double theta_target, int max_sweeps, int check_every,
                     int* sweeps_done, double* theta_out, double* F_out, void* stream) {
  LatticeDesc d;
  int rc = describe(lat, &d);
  if (rc != CULGT_OK) return rc;
  if (!links || !workspace) return CULGT_ERR_NULL;
  if (misaligned(links) || misaligned(workspace)) return CULGT_ERR_ALIGN;
  if (max_sweeps < 0 || check_every < 1) return CULGT_ERR_ARG;
  if ((rc = check_omega(omega)) != CULGT_OK) return rc;
  cudaStream_t st = (cudaStream_t)stream;
  double* ws = (double*)workspace;
  double* scal = ws + reduce_partial_doubles(d.geom);
  cudaError_t e;
  if (g_variant == 0) {
    // small SU(3) lattices: the whole loop as one cooperative kernel (csrc/fix_persistent.cu)
    PersistCtl* pc = (PersistCtl*)(ws + fix_ctl_offset_doubles(d.geom));
    e = launch_landau_fix_persistent(d, links, omega, theta_target, max_sweeps, check_every, ws, pc, st);
    if (e == cudaSuccess) {
      PersistCtl h;
      if ((e = cudaMemcpyAsync(&h, pc, sizeof(h), cudaMemcpyDeviceToHost, st)) != cudaSuccess) return cuda_fail(e);
      if ((e = cudaStreamSynchronize(st)) != cudaSuccess) return cuda_fail(e);
      if (sweeps_done) *sweeps_done = h.sweeps_done;
      if (theta_out) *theta_out = h.theta;
      if (F_out) *F_out = h.F;
      return CULGT_OK;
    }
    if (e != cudaErrorNotSupported) return cuda_fail(e);
  }
  FixCtl* ctl = (FixCtl*)(ws + fix_ctl_offset_doubles(d.geom));
  e = cudaMemsetAsync(ctl, 0, sizeof(FixCtl), st);
  if (e != cudaSuccess) return cuda_fail(e);
  FixCheck chk = {ctl, theta_target, 0};
  if ((e = launch_theta_functional(d, links, ws, scal, scal + 1, st, &chk)) != cudaSuccess) return cuda_fail(e);
  // rounds per synchronisation: about 32 sweeps' worth of launches, so that a small lattice is not
  // bound by the host round trip and a stopped run wastes at most that many empty launches
  const int rounds_per_sync = check_every >= 32 ? 1 : 32 / check_every;
  FixCtl host;
  int enqueued = 0;
  for (;;) {
    for (int r = 0; r < rounds_per_sync && enqueued < max_sweeps; ++r) {
      int n = check_every;
      if (enqueued + n > max_sweeps) n = max_sweeps - enqueued;
      if ((e = launch_or_full_sweeps(d, links, ws, n, omega, g_variant, &ctl->stop, st)) != cudaSuccess) return cuda_fail(e);
      enqueued += n;
      chk.sweeps_before = enqueued;
      if ((e = launch_theta_functional(d, links, ws, scal, scal + 1, st, &chk)) != cudaSuccess) return cuda_fail(e);
    }
    if ((e = cudaMemcpyAsync(&host, ctl, sizeof(FixCtl), cudaMemcpyDeviceToHost, st)) != cudaSuccess) return cuda_fail(e);
    if ((e = cudaStreamSynchronize(st)) != cudaSuccess) return cuda_fail(e);
    if (host.stop || enqueued >= max_sweeps) break;
  }
  if (sweeps_done) *sweeps_done = host.stop ? host.sweeps_at_stop : enqueued;
  if (theta_out) *theta_out = host.theta;
  if (F_out) *F_out = host.F;
  return CULGT_OK;
}

int culgt_fix_host(const culgt_lattice* lat, void* canonical_host, void* canonical_dev,
                   void* links_dev, void* workspace, int n_sweeps, double omega,
                   double* theta_out, double* F_out, void* stream) {
  LatticeDesc d;
  int rc = describe(lat, &d);
  if (rc != CULGT_OK) return rc;
  if (!canonical_host || !canonical_dev || !links_dev || !workspace) return CULGT_ERR_NULL;
  if (misaligned(canonical_dev) || misaligned(links_dev) || misaligned(workspace)) return CULGT_ERR_ALIGN;
  if (n_sweeps < 0) return CULGT_ERR_ARG;
  if ((rc = check_omega(omega)) != CULGT_OK) return rc;
  cudaStream_t st = (cudaStream_t)stream;
  const size_t cbytes = culgt_canonical_bytes(lat);
  cudaError_t e = cudaMemcpyAsync(canonical_dev, canonical_host, cbytes, cudaMemcpyHostToDevice, st);
  if (e != cudaSuccess) return cuda_fail(e);
  if ((e = launch_pack(d, canonical_dev, links_dev, st)) != cudaSuccess) return cuda_fail(e);
  if ((e = launch_or_full_sweeps(d, links_dev, (double*)workspace, n_sweeps, omega, g_variant, nullptr, st)) != cudaSuccess)
    return cuda_fail(e);
  if ((e = launch_unpack(d, links_dev, canonical_dev, st)) != cudaSuccess) return cuda_fail(e);
  e = cudaMemcpyAsync(canonical_host, canonical_dev, cbytes, cudaMemcpyDeviceToHost, st);
  if (e != cudaSuccess) return cuda_fail(e);
  double theta = 0, F = 0;
  if ((rc = read_theta_F(d, links_dev, workspace, st, &theta, &F)) != CULGT_OK) return rc;
  if (theta_out) *theta_out = theta;
  if (F_out) *F_out = F;
  return CULGT_OK;
}

// ---- truncated-series overrelaxation (reading C-24) ------------------------------------

int culgt_or_sweep_series(const culgt_lattice* lat, void* links, int parity, double omega, int order,
                          void* stream) {
  LatticeDesc d;
  int rc = describe(lat, &d);
  if (rc != CULGT_OK) return rc;
  if (!links) return CULGT_ERR_NULL;
  if (misaligned(links)) return CULGT_ERR_ALIGN;
  if (parity != 0 && parity != 1) return CULGT_ERR_PARITY;
  if ((rc = check_omega(omega)) != CULGT_OK) return rc;
  if (order < 0 || order > 16) return CULGT_ERR_ARG;
  cudaError_t e = launch_or_sweep_series(d, links, parity, omega, order, (cudaStream_t)stream);
  return e == cudaSuccess ? CULGT_OK : cuda_fail(e);
}

int culgt_or_sweeps_series(const culgt_lattice* lat, void* links, int n_sweeps, double omega, int order,
                           void* stream) {
  LatticeDesc d;
  int rc = describe(lat, &d);
  if (rc != CULGT_OK) return rc;
  if (!links) return CULGT_ERR_NULL;
  if (misaligned(links)) return CULGT_ERR_ALIGN;
  if (n_sweeps < 0 || order < 0 || order > 16) return CULGT_ERR_ARG;
  if ((rc = check_omega(omega)) != CULGT_OK) return rc;
  for (int i = 0; i < n_sweeps; ++i)
    for (int parity = 0; parity < 2; ++parity) {
      cudaError_t e = launch_or_sweep_series(d, links, parity, omega, order, (cudaStream_t)stream);
      if (e != cudaSuccess) return cuda_fail(e);
    }
  return CULGT_OK;
}

// ---- simulated annealing (reading C-25) ------------------------------------------------

int culgt_sa_sweep(const culgt_lattice* lat, void* links, int parity, double T, unsigned long long seed,
                   unsigned counter, void* stream) {
  LatticeDesc d;
  int rc = describe(lat, &d);
  if (rc != CULGT_OK) return rc;
  if (!links) return CULGT_ERR_NULL;
  if (misaligned(links)) return CULGT_ERR_ALIGN;
  if (parity != 0 && parity != 1) return CULGT_ERR_PARITY;
  if (!(T > 0.0) || !(T < 1e300)) return CULGT_ERR_ARG;
  cudaError_t e = launch_sa_sweep(d, links, parity, T, seed, counter, (cudaStream_t)stream);
  return e == cudaSuccess ? CULGT_OK : cuda_fail(e);
}

int culgt_sa_anneal(const culgt_lattice* lat, void* links, double T_max, double T_min, int n_sweeps,
                    unsigned long long seed, void* stream) {
  LatticeDesc d;
  int rc = describe(lat, &d);
  if (rc != CULGT_OK) return rc;
  if (!links) return CULGT_ERR_NULL;
  if (misaligned(links)) return CULGT_ERR_ALIGN;
  if (n_sweeps < 0 || !(T_min > 0.0) || !(T_max >= T_min) || !(T_max < 1e300)) return CULGT_ERR_ARG;
  for (int i = 0; i < n_sweeps; ++i) {
    const double T = n_sweeps > 1 ? T_max - (T_max - T_min) * (double)i / (double)(n_sweeps - 1) : T_min;
    for (int parity = 0; parity < 2; ++parity) {
      cudaError_t e = launch_sa_sweep(d, links, parity, T, seed, (unsigned)(2 * i + parity), (cudaStream_t)stream);
      if (e != cudaSuccess) return cuda_fail(e);
    }
  }
  return CULGT_OK;
}

// ---- microcanonical step (reading C-26) ------------------------------------------------

int culgt_micro_sweep(const culgt_lattice* lat, void* links, int parity, void* stream) {
  LatticeDesc d;
  int rc = describe(lat, &d);
  if (rc != CULGT_OK) return rc;
  if (!links) return CULGT_ERR_NULL;
  if (misaligned(links)) return CULGT_ERR_ALIGN;
  if (parity != 0 && parity != 1) return CULGT_ERR_PARITY;
  cudaError_t e = launch_micro_sweep(d, links, parity, (cudaStream_t)stream);
  return e == cudaSuccess ? CULGT_OK : cuda_fail(e);
}

int culgt_micro_sweeps(const culgt_lattice* lat, void* links, int n_sweeps, void* stream) {
  LatticeDesc d;
  int rc = describe(lat, &d);
  if (rc != CULGT_OK) return rc;
  if (!links) return CULGT_ERR_NULL;
  if (misaligned(links)) return CULGT_ERR_ALIGN;
  if (n_sweeps < 0) return CULGT_ERR_ARG;
  for (int i = 0; i < n_sweeps; ++i)
    for (int parity = 0; parity < 2; ++parity) {
      cudaError_t e = launch_micro_sweep(d, links, parity, (cudaStream_t)stream);
      if (e != cudaSuccess) return cuda_fail(e);
    }
  return CULGT_OK;
}

int culgt_sa_anneal_micro(const culgt_lattice* lat, void* links, double T_max, double T_min, int n_sweeps,
                          int n_micro, unsigned long long seed, void* stream) {
  LatticeDesc d;
  int rc = describe(lat, &d);
  if (rc != CULGT_OK) return rc;
  if (!links) return CULGT_ERR_NULL;
  if (misaligned(links)) return CULGT_ERR_ALIGN;
  if (n_sweeps < 0 || n_micro < 0 || !(T_min > 0.0) || !(T_max >= T_min) || !(T_max < 1e300)) return CULGT_ERR_ARG;
  for (int i = 0; i < n_sweeps; ++i) {
    const double T = n_sweeps > 1 ? T_max - (T_max - T_min) * (double)i / (double)(n_sweeps - 1) : T_min;
    for (int parity = 0; parity < 2; ++parity) {
      cudaError_t e = launch_sa_sweep(d, links, parity, T, seed, (unsigned)(2 * i + parity), (cudaStream_t)stream);
      if (e != cudaSuccess) return cuda_fail(e);
    }
    for (int m = 0; m < n_micro; ++m)
      for (int parity = 0; parity < 2; ++parity) {
        cudaError_t e = launch_micro_sweep(d, links, parity, (cudaStream_t)stream);
        if (e != cudaSuccess) return cuda_fail(e);
      }
  }
  return CULGT_OK;
}

// ---- Coulomb gauge (reading C-22) -----------------------------------------------------

int culgt_or_sweep_coulomb(const culgt_lattice* lat, void* links, int parity, double omega, void* stream) {
  LatticeDesc d;
  int rc = describe(lat, &d);
  if (rc != CULGT_OK) return rc;
  if (!links) return CULGT_ERR_NULL;
  if (misaligned(links)) return CULGT_ERR_ALIGN;
  if (parity != 0 && parity != 1) return CULGT_ERR_PARITY;
  if ((rc = check_omega(omega)) != CULGT_OK) return rc;
  cudaError_t e = launch_or_sweep(d, links, parity, omega, 0, (cudaStream_t)stream, true);
  return e == cudaSuccess ? CULGT_OK : cuda_fail(e);
}

int culgt_or_sweep_coulomb_masked(const culgt_lattice* lat, void* links, int parity, double omega,
                                  const unsigned char* slice_active_dev, void* stream) {
  LatticeDesc d;
  int rc = describe(lat, &d);
  if (rc != CULGT_OK) return rc;
  if (!links || !slice_active_dev) return CULGT_ERR_NULL;
  if (misaligned(links)) return CULGT_ERR_ALIGN;
  if (parity != 0 && parity != 1) return CULGT_ERR_PARITY;
  if ((rc = check_omega(omega)) != CULGT_OK) return rc;
  d.geom.slice_active = slice_active_dev;
  cudaError_t e = launch_or_sweep(d, links, parity, omega, 0, (cudaStream_t)stream, true);
  return e == cudaSuccess ? CULGT_OK : cuda_fail(e);
}

int culgt_or_sweeps_coulomb(const culgt_lattice* lat, void* links, int n_sweeps, double omega, void* stream) {
  LatticeDesc d;
  int rc = describe(lat, &d);
  if (rc != CULGT_OK) return rc;
  if (!links) return CULGT_ERR_NULL;
  if (misaligned(links)) return CULGT_ERR_ALIGN;
  if (n_sweeps < 0) return CULGT_ERR_ARG;
  if ((rc = check_omega(omega)) != CULGT_OK) return rc;
  for (int i = 0; i < n_sweeps; ++i)
    for (int parity = 0; parity < 2; ++parity) {
      cudaError_t e = launch_or_sweep(d, links, parity, omega, 0, (cudaStream_t)stream, true);
      if (e != cudaSuccess) return cuda_fail(e);
    }
  return CULGT_OK;
}

int culgt_coulomb_precision_functional(const culgt_lattice* lat, const void* links, void* workspace,
                                       double* theta_t_dev, double* F_t_dev, void* stream) {
  LatticeDesc d;
  int rc = describe(lat, &d);
  if (rc != CULGT_OK) return rc;
  if (!links || !workspace || !theta_t_dev || !F_t_dev) return CULGT_ERR_NULL;
  if (misaligned(links) || misaligned(workspace)) return CULGT_ERR_ALIGN;
  cudaError_t e = launch_coulomb_theta_functional(d, links, (double*)workspace, theta_t_dev, F_t_dev,
                                                  (cudaStream_t)stream);
  return e == cudaSuccess ? CULGT_OK : cuda_fail(e);
}

// As culgt_landau_fix, the stopping decision is taken on the device: every check recomputes the per-slice
// activity mask from theta_t (coulomb_mask_kernel) and raises the stop word when no slice is active; the
// host reads the control block and the 2*N3 results back once per batch of rounds.
int culgt_coulomb_fix(const culgt_lattice* lat, void* links, void* workspace, double omega,
                      double theta_target, int max_sweeps, int check_every, int* sweeps_done,
                      double* theta_t_out, double* F_t_out, void* stream) {
  LatticeDesc d;
  int rc = describe(lat, &d);
  if (rc != CULGT_OK) return rc;
  if (!links || !workspace) return CULGT_ERR_NULL;
  if (misaligned(links) || misaligned(workspace)) return CULGT_ERR_ALIGN;
  if (max_sweeps < 0 || check_every < 1) return CULGT_ERR_ARG;
  if ((rc = check_omega(omega)) != CULGT_OK) return rc;
  cudaStream_t st = (cudaStream_t)stream;
  const int n3 = d.geom.n[3];
  double* ws = (double*)workspace;
  double* res = ws + reduce_partial_doubles(d.geom);                 // theta_t[N3], F_t[N3]
  unsigned char* mask_dev = (unsigned char*)(res + 2 * (size_t)n3);  // the per-slice activity mask behind them
  FixCtl* ctl = (FixCtl*)(ws + fix_ctl_offset_doubles(d.geom));
  cudaError_t e = cudaMemsetAsync(ctl, 0, sizeof(FixCtl), st);
  if (e != cudaSuccess) return cuda_fail(e);
  CoulombCheck chk = {ctl, mask_dev, theta_target, 0};
  if ((e = launch_coulomb_theta_functional(d, links, ws, res, res + n3, st, &chk)) != cudaSuccess) return cuda_fail(e);
  LatticeDesc dm = d;
  dm.geom.slice_active = mask_dev;
  const int rounds_per_sync = check_every >= 32 ? 1 : 32 / check_every;
  std::vector<double> host(2 * (size_t)n3);
  FixCtl hc;
  int enqueued = 0;
  for (;;) {
    for (int r = 0; r < rounds_per_sync && enqueued < max_sweeps; ++r) {
      int n = check_every;
      if (enqueued + n > max_sweeps) n = max_sweeps - enqueued;
      for (int i = 0; i < n; ++i)
        for (int parity = 0; parity < 2; ++parity)
          if ((e = launch_or_sweep(dm, links, parity, omega, 0, st, true, &ctl->stop)) != cudaSuccess) return cuda_fail(e);
      enqueued += n;
      chk.sweeps_before = enqueued;
      if ((e = launch_coulomb_theta_functional(d, links, ws, res, res + n3, st, &chk)) != cudaSuccess) return cuda_fail(e);
    }
    if ((e = cudaMemcpyAsync(&hc, ctl, sizeof(FixCtl), cudaMemcpyDeviceToHost, st)) != cudaSuccess) return cuda_fail(e);
    if ((e = cudaMemcpyAsync(host.data(), res, 2 * (size_t)n3 * sizeof(double), cudaMemcpyDeviceToHost, st)) != cudaSuccess)
      return cuda_fail(e);
    if ((e = cudaStreamSynchronize(st)) != cudaSuccess) return cuda_fail(e);
    if (hc.stop || enqueued >= max_sweeps) break;
  }
  if (sweeps_done) *sweeps_done = hc.stop ? hc.sweeps_at_stop : enqueued;
  for (int t = 0; t < n3; ++t) {
    if (theta_t_out) theta_t_out[t] = host[t];
    if (F_t_out) F_t_out[t] = host[n3 + t];
  }
  return CULGT_OK;
}


// ---- time-slab decomposition over several GPUs (csrc/slab.cu) -------------

int culgt_slab_lattice(const culgt_lattice* global, int n_slabs, culgt_lattice* local) {
  LatticeDesc d;
  int rc = describe(global, &d);
  if (rc != CULGT_OK) return rc;
  if (!local) return CULGT_ERR_NULL;
  if (n_slabs < 1 || global->dims[3] % n_slabs != 0) return CULGT_ERR_ARG;
  const int t = global->dims[3] / n_slabs;
  if (t < 2 || (t & 1)) return CULGT_ERR_ARG;          // an odd slab would flip the parity of its sites
  *local = *global;
  local->dims[3] = t;
  return CULGT_OK;
}

size_t culgt_slab_links_bytes(const culgt_lattice* local) {
  LatticeDesc d;
  if (describe_slab(local, &d) != CULGT_OK) return 0;
  return (size_t)8 * (size_t)slab_vectors_per_link(d) * (size_t)d.geom.pitch * 16;
}

size_t culgt_slab_halo_bytes(const culgt_lattice* local) {
  LatticeDesc d;
  if (describe_slab(local, &d) != CULGT_OK) return 0;
  return (size_t)slab_vectors_per_link(d) * (size_t)d.geom.stride[3] * 16;
}

int culgt_slab_halo_chunks(const culgt_lattice* local, int parity, int which, size_t* offsets, size_t* chunk_bytes,
                           int* n_chunks) {
  LatticeDesc d;
  int rc = describe_slab(local, &d);
  if (rc != CULGT_OK) return rc;
  if (!offsets || !chunk_bytes || !n_chunks) return CULGT_ERR_NULL;
  if (parity != 0 && parity != 1) return CULGT_ERR_PARITY;
  if (which != 0 && which != 1) return CULGT_ERR_ARG;
  slab_halo_chunks(d, parity, which, offsets, chunk_bytes, n_chunks);
  return CULGT_OK;
}

int culgt_slab_halo_peers(int rank, int n_ranks, int direction, int* send_to, int* recv_from) {
  if (!send_to || !recv_from) return CULGT_ERR_NULL;
  if (n_ranks < 1 || rank < 0 || rank >= n_ranks || (direction != 0 && direction != 1)) return CULGT_ERR_ARG;
  slab_halo_peers(rank, n_ranks, direction, send_to, recv_from);
  return CULGT_OK;
}

int culgt_slab_pack(const culgt_lattice* local, const void* canonical_slab, void* links_slab, void* stream) {
  LatticeDesc d;
  int rc = describe_slab(local, &d);
  if (rc != CULGT_OK) return rc;
  if (!canonical_slab || !links_slab) return CULGT_ERR_NULL;
  if (misaligned(canonical_slab) || misaligned(links_slab)) return CULGT_ERR_ALIGN;
  cudaError_t e = launch_pack(d, canonical_slab, links_slab, (cudaStream_t)stream);
  return e == cudaSuccess ? CULGT_OK : cuda_fail(e);
}

int culgt_slab_unpack(const culgt_lattice* local, const void* links_slab, void* canonical_slab, void* stream) {
  LatticeDesc d;
  int rc = describe_slab(local, &d);
  if (rc != CULGT_OK) return rc;
  if (!canonical_slab || !links_slab) return CULGT_ERR_NULL;
  if (misaligned(canonical_slab) || misaligned(links_slab)) return CULGT_ERR_ALIGN;
  cudaError_t e = launch_unpack(d, links_slab, canonical_slab, (cudaStream_t)stream);
  return e == cudaSuccess ? CULGT_OK : cuda_fail(e);
}

static int check_slab_sweep(const culgt_lattice* local, const void* links, int parity, double omega, LatticeDesc* d) {
  int rc = describe_slab(local, d);
  if (rc != CULGT_OK) return rc;
  if (!links) return CULGT_ERR_NULL;
  if (misaligned(links)) return CULGT_ERR_ALIGN;
  if (parity != 0 && parity != 1) return CULGT_ERR_PARITY;
  return check_omega(omega);
}

int culgt_slab_or_sweep(const culgt_lattice* local, void* links_slab, int parity, double omega, void* stream) {
  LatticeDesc d;
  int rc = check_slab_sweep(local, links_slab, parity, omega, &d);
  if (rc != CULGT_OK) return rc;
  cudaError_t e = launch_or_sweep(d, links_slab, parity, omega, g_variant, (cudaStream_t)stream);
  return e == cudaSuccess ? CULGT_OK : cuda_fail(e);
}

int culgt_slab_or_sweep_window(const culgt_lattice* local, void* links_slab, int parity, double omega, int t_lo,
                               int t_hi, void* stream) {
  LatticeDesc d;
  int rc = check_slab_sweep(local, links_slab, parity, omega, &d);
  if (rc != CULGT_OK) return rc;
  if (t_lo < 0 || t_hi > local->dims[3] || t_lo > t_hi) return CULGT_ERR_ARG;
  cudaError_t e = launch_or_sweep_window(d, links_slab, parity, omega, t_lo, t_hi, (cudaStream_t)stream);
  if (e == cudaErrorNotSupported) return CULGT_ERR_DESC;      // SU(2), or no whole site blocks per time-slice
  return e == cudaSuccess ? CULGT_OK : cuda_fail(e);
}

int culgt_slab_halo_copy(const culgt_lattice* local, const void* src_links, void* dst_links, int parity, int direction,
                         void* stream) {
  LatticeDesc d;
  int rc = describe_slab(local, &d);
  if (rc != CULGT_OK) return rc;
  if (!src_links || !dst_links) return CULGT_ERR_NULL;
  if (misaligned(src_links) || misaligned(dst_links)) return CULGT_ERR_ALIGN;
  if (parity != 0 && parity != 1) return CULGT_ERR_PARITY;
  if (direction != 0 && direction != 1) return CULGT_ERR_ARG;
  cudaError_t e = slab_halo_copy(d, src_links, dst_links, parity, direction, (cudaStream_t)stream);
  return e == cudaSuccess ? CULGT_OK : cuda_fail(e);
}

int culgt_slab_theta_F_sums(const culgt_lattice* local, const void* links_slab, void* workspace, double* sums2_dev,
                            void* stream) {
  LatticeDesc d;
  int rc = describe_slab(local, &d);
  if (rc != CULGT_OK) return rc;
  if (!links_slab || !workspace || !sums2_dev) return CULGT_ERR_NULL;
  if (misaligned(links_slab) || misaligned(workspace)) return CULGT_ERR_ALIGN;
  cudaError_t e = launch_theta_functional_sums(d, links_slab, (double*)workspace, sums2_dev, (cudaStream_t)stream);
  return e == cudaSuccess ? CULGT_OK : cuda_fail(e);
}

int culgt_slab_theta_F_combine(const culgt_lattice* global, const double* sums_dev, int n_slabs, double* theta_dev,
                               double* F_dev, void* stream) {
  LatticeDesc d;
  int rc = describe(global, &d);
  if (rc != CULGT_OK) return rc;
  if (!sums_dev || !theta_dev || !F_dev) return CULGT_ERR_NULL;
  if (n_slabs < 1) return CULGT_ERR_ARG;
  cudaError_t e = slab_theta_F_combine(d, sums_dev, n_slabs, theta_dev, F_dev, (cudaStream_t)stream);
  return e == cudaSuccess ? CULGT_OK : cuda_fail(e);
}

// One half-sweep of parity p on one slab, boundary slices first when `boundary_first` (the schedule that
// lets the halo messages travel while the interior is swept): slice 0 writes the ghost slice of parity
// 1-p, slice T-1 the slab's own t-links of parity p in its last slice; the interior touches neither.
static cudaError_t slab_half_sweep(const LatticeDesc& d, void* links, int parity, double omega, bool boundary_first,
                                   cudaStream_t st, cudaEvent_t boundary_done) {
  const int T = d.geom.n[3];
  cudaError_t e = cudaErrorNotSupported;
  if (boundary_first) {
    e = launch_or_sweep_window(d, links, parity, omega, 0, 1, st);
    if (e == cudaSuccess) e = launch_or_sweep_window(d, links, parity, omega, T - 1, T, st);
    if (e == cudaSuccess && boundary_done) e = cudaEventRecord(boundary_done, st);
    if (e == cudaSuccess) e = launch_or_sweep_window(d, links, parity, omega, 1, T - 1, st);
  }
  if (e == cudaErrorNotSupported) {             // no whole site blocks per slice (or SU(2)): one launch
    e = launch_or_sweep(d, links, parity, omega, g_variant, st);
    if (e == cudaSuccess && boundary_done) e = cudaEventRecord(boundary_done, st);
  }
  return e;
}

int culgt_slab_exchange_all_local(const culgt_lattice* local, void* const* links_slabs, int n_slabs, void* stream) {
  LatticeDesc d;
  int rc = describe_slab(local, &d);
  if (rc != CULGT_OK) return rc;
  if (!links_slabs) return CULGT_ERR_NULL;
  if (n_slabs < 1) return CULGT_ERR_ARG;
  for (int k = 0; k < n_slabs; ++k)
    if (!links_slabs[k]) return CULGT_ERR_NULL;
  for (int k = 0; k < n_slabs; ++k)
    for (int parity = 0; parity < 2; ++parity) {
      cudaError_t e = slab_halo_copy(d, links_slabs[k], links_slabs[(k + 1) % n_slabs], parity, 0, (cudaStream_t)stream);
      if (e != cudaSuccess) return cuda_fail(e);
    }
  return CULGT_OK;
}

int culgt_slab_or_sweeps_local(const culgt_lattice* local, void* const* links_slabs, int n_slabs, int n_sweeps,
                               double omega, int boundary_first, void* stream) {
  LatticeDesc d;
  int rc = describe_slab(local, &d);
  if (rc != CULGT_OK) return rc;
  if (!links_slabs) return CULGT_ERR_NULL;
  if (n_slabs < 1 || n_sweeps < 0) return CULGT_ERR_ARG;
  for (int k = 0; k < n_slabs; ++k) {
    if (!links_slabs[k]) return CULGT_ERR_NULL;
    if (misaligned(links_slabs[k])) return CULGT_ERR_ALIGN;
  }
  if ((rc = check_omega(omega)) != CULGT_OK) return rc;
  cudaStream_t st = (cudaStream_t)stream;
  cudaError_t e;
  for (int i = 0; i < n_sweeps; ++i)
    for (int p = 0; p < 2; ++p) {
      for (int k = 0; k < n_slabs; ++k)
        if ((e = slab_half_sweep(d, links_slabs[k], p, omega, boundary_first != 0, st, nullptr)) != cudaSuccess) return cuda_fail(e);
      for (int k = 0; k < n_slabs; ++k) {
        const int prev = (k + n_slabs - 1) % n_slabs, next = (k + 1) % n_slabs;
        // the updated U_t(x - t_hat) of slab k's first slice go BACK to their owner ...
        if ((e = slab_halo_copy(d, links_slabs[k], links_slabs[prev], 1 - p, 1, st)) != cudaSuccess) return cuda_fail(e);
        // ... and slab k's own updated t-links of its last slice go FORWARD for the other parity's half-sweep
        if ((e = slab_halo_copy(d, links_slabs[k], links_slabs[next], p, 0, st)) != cudaSuccess) return cuda_fail(e);
      }
    }
  return CULGT_OK;
}

int culgt_slab_theta_F_local(const culgt_lattice* global, const culgt_lattice* local, void* const* links_slabs,
                             int n_slabs, void* workspace, double* sums_dev, double* theta_dev, double* F_dev,
                             void* stream) {
  LatticeDesc dg, d;
  int rc = describe(global, &dg);
  if (rc != CULGT_OK) return rc;
  if ((rc = describe_slab(local, &d)) != CULGT_OK) return rc;
  if (!links_slabs || !workspace || !sums_dev || !theta_dev || !F_dev) return CULGT_ERR_NULL;
  if (n_slabs < 1 || (long long)n_slabs * local->dims[3] != global->dims[3]) return CULGT_ERR_ARG;
  cudaStream_t st = (cudaStream_t)stream;
  for (int k = 0; k < n_slabs; ++k) {
    if (!links_slabs[k]) return CULGT_ERR_NULL;
    cudaError_t e = launch_theta_functional_sums(d, links_slabs[k], (double*)workspace, sums_dev + 2 * k, st);
    if (e != cudaSuccess) return cuda_fail(e);
  }
  cudaError_t e = slab_theta_F_combine(dg, sums_dev, n_slabs, theta_dev, F_dev, st);
  return e == cudaSuccess ? CULGT_OK : cuda_fail(e);
}

// ---- one slab per rank, NCCL over NVLink ---------------------------------------------------------------------

int culgt_slab_comm_unique_id(void* id128_host) {
  if (!id128_host) return CULGT_ERR_NULL;
  const int r = slab_comm_id(id128_host);
  return r == 0 ? CULGT_OK : nccl_fail(r);
}

int culgt_slab_comm_create(const void* id128_host, int rank, int n_ranks, void** comm_out) {
  if (!id128_host || !comm_out) return CULGT_ERR_NULL;
  if (n_ranks < 1 || rank < 0 || rank >= n_ranks) return CULGT_ERR_ARG;
  const int r = slab_comm_create(id128_host, rank, n_ranks, comm_out);
  return r == 0 ? CULGT_OK : nccl_fail(r);
}

int culgt_slab_comm_destroy(void* comm) {
  const int r = slab_comm_destroy(comm);
  return r == 0 ? CULGT_OK : nccl_fail(r);
}

int culgt_slab_halo_exchange(void* comm, const culgt_lattice* local, void* links_slab, int parity, int direction,
                             void* stream) {
  LatticeDesc d;
  int rc = describe_slab(local, &d);
  if (rc != CULGT_OK) return rc;
  if (!comm || !links_slab) return CULGT_ERR_NULL;
  if (misaligned(links_slab)) return CULGT_ERR_ALIGN;
  if (parity != 0 && parity != 1) return CULGT_ERR_PARITY;
  if (direction != 0 && direction != 1) return CULGT_ERR_ARG;
  const int r = slab_halo_exchange(comm, d, links_slab, parity, direction, (cudaStream_t)stream);
  return r == 0 ? CULGT_OK : nccl_fail(r);
}

int culgt_slab_or_sweeps_nccl(void* comm, const culgt_lattice* local, void* links_slab, int n_sweeps, double omega,
                              void* comm_stream, void* stream) {
  LatticeDesc d;
  int rc = describe_slab(local, &d);
  if (rc != CULGT_OK) return rc;
  if (!comm || !links_slab) return CULGT_ERR_NULL;
  if (misaligned(links_slab)) return CULGT_ERR_ALIGN;
  if (n_sweeps < 0) return CULGT_ERR_ARG;
  if ((rc = check_omega(omega)) != CULGT_OK) return rc;
  cudaStream_t st = (cudaStream_t)stream, cst = (cudaStream_t)comm_stream;
  const bool overlap = comm_stream != nullptr && comm_stream != stream;
  cudaEvent_t boundary_done = nullptr, halo_done = nullptr;
  cudaError_t e = cudaSuccess;
  if (overlap) {
    if ((e = cudaEventCreateWithFlags(&boundary_done, cudaEventDisableTiming)) != cudaSuccess) return cuda_fail(e);
    if ((e = cudaEventCreateWithFlags(&halo_done, cudaEventDisableTiming)) != cudaSuccess) {
      cudaEventDestroy(boundary_done);
      return cuda_fail(e);
    }
  }
  int nr = 0;
  for (int i = 0; i < n_sweeps && e == cudaSuccess && nr == 0; ++i)
    for (int p = 0; p < 2 && e == cudaSuccess && nr == 0; ++p) {
      if (!overlap) {
        e = slab_half_sweep(d, links_slab, p, omega, false, st, nullptr);
        if (e == cudaSuccess) nr = slab_halo_exchange(comm, d, links_slab, 1 - p, 1, st);
        if (e == cudaSuccess && nr == 0) nr = slab_halo_exchange(comm, d, links_slab, p, 0, st);
      } else {
        // boundary slices, then the two messages on the communication stream while the interior is swept
        e = slab_half_sweep(d, links_slab, p, omega, true, st, boundary_done);
        if (e == cudaSuccess) e = cudaStreamWaitEvent(cst, boundary_done, 0);
        if (e == cudaSuccess) nr = slab_halo_exchange(comm, d, links_slab, 1 - p, 1, cst);
        if (e == cudaSuccess && nr == 0) nr = slab_halo_exchange(comm, d, links_slab, p, 0, cst);
        if (e == cudaSuccess && nr == 0) e = cudaEventRecord(halo_done, cst);
        if (e == cudaSuccess && nr == 0) e = cudaStreamWaitEvent(st, halo_done, 0);   // the next half-sweep needs both
      }
    }
  if (overlap) {
    cudaEventDestroy(boundary_done);
    cudaEventDestroy(halo_done);
  }
  if (e != cudaSuccess) return cuda_fail(e);
  return nr == 0 ? CULGT_OK : nccl_fail(nr);
}

int culgt_slab_theta_F_nccl(void* comm, const culgt_lattice* global, const culgt_lattice* local, const void* links_slab,
                            void* workspace, double* sums_dev, double* theta_dev, double* F_dev, void* stream) {
  LatticeDesc dg, d;
  int rc = describe(global, &dg);
  if (rc != CULGT_OK) return rc;
  if ((rc = describe_slab(local, &d)) != CULGT_OK) return rc;
  if (!comm || !links_slab || !workspace || !sums_dev || !theta_dev || !F_dev) return CULGT_ERR_NULL;
  int rank = 0, n_ranks = 1;
  slab_comm_info(comm, &rank, &n_ranks);
  if ((long long)n_ranks * local->dims[3] != global->dims[3]) return CULGT_ERR_ARG;
  cudaStream_t st = (cudaStream_t)stream;
  // my two raw sums behind the gathered ones, then all ranks' pairs in rank order on every rank
  double* mine = sums_dev + 2 * n_ranks;
  cudaError_t e = launch_theta_functional_sums(d, links_slab, (double*)workspace, mine, st);
  if (e != cudaSuccess) return cuda_fail(e);
  const int r = slab_allgather_sums(comm, mine, sums_dev, st);
  if (r != 0) return nccl_fail(r);
  e = slab_theta_F_combine(dg, sums_dev, n_ranks, theta_dev, F_dev, st);
  return e == cudaSuccess ? CULGT_OK : cuda_fail(e);
}

int culgt_slab_exchange_all_nccl(void* comm, const culgt_lattice* local, void* links_slab, void* stream) {
  LatticeDesc d;
  int rc = describe_slab(local, &d);
  if (rc != CULGT_OK) return rc;
  if (!comm || !links_slab) return CULGT_ERR_NULL;
  for (int parity = 0; parity < 2; ++parity) {
    const int r = slab_halo_exchange(comm, d, links_slab, parity, 0, (cudaStream_t)stream);
    if (r != 0) return nccl_fail(r);
  }
  return CULGT_OK;
}

// Run-time autotuner (the paper's selection of the fastest kernel set-up per GPU at run time,
// P:L89 (d)): times every result-equivalent sweep schedule built for this storage format
// on the caller's field and makes the fastest one the calling thread's choice.
int culgt_autotune_sweep(const culgt_lattice* lat, void* links, void* workspace, double omega,
                         int sweeps_per_trial, int* best_variant, float* best_us_per_half_sweep, void* stream) {
  LatticeDesc d;
  int rc = describe(lat, &d);
  if (rc != CULGT_OK) return rc;
  if (!links || !workspace) return CULGT_ERR_NULL;
  if (misaligned(links) || misaligned(workspace)) return CULGT_ERR_ALIGN;
  if (sweeps_per_trial < 1) return CULGT_ERR_ARG;
  if ((rc = check_omega(omega)) != CULGT_OK) return rc;
  cudaStream_t st = (cudaStream_t)stream;
  cudaEvent_t e0, e1;
  if (cudaEventCreate(&e0) != cudaSuccess) return cuda_fail(cudaGetLastError());
  if (cudaEventCreate(&e1) != cudaSuccess) { cudaEventDestroy(e0); return cuda_fail(cudaGetLastError()); }
  int best = 0;
  float best_us = -1.f;
  for (int v = 1; v < 64; ++v) {
    if (!sweep_variant_known(v) || v == 20) continue;            // 20 is variant 0's other name: timed once, below
    // 11, 14, 25: all-fp32 arithmetic (different precision); 28, 32: measurement-only (no solve)
    if (v == 11 || v == 14 || v == 25 || v == 28 || v == 32) continue;
    if (d.group == 2 && v != 20) continue;
    cudaError_t e = launch_or_full_sweeps(d, links, (double*)workspace, 1, omega, v, nullptr, st);
    if (e == cudaErrorInvalidValue) { cudaGetLastError(); continue; }   // mapping not built for this format
    if (e != cudaSuccess) { rc = cuda_fail(e); break; }
    cudaEventRecord(e0, st);
    e = launch_or_full_sweeps(d, links, (double*)workspace, sweeps_per_trial, omega, v, nullptr, st);
    cudaEventRecord(e1, st);
    if (e == cudaSuccess) e = cudaEventSynchronize(e1);
    if (e != cudaSuccess) { rc = cuda_fail(e); break; }
    float ms = 0.f;
    cudaEventElapsedTime(&ms, e0, e1);
    const float us = ms * 1e3f / (2.f * sweeps_per_trial);
    if (best_us < 0.f || us < best_us) { best_us = us; best = v; }
  }
  cudaEventDestroy(e0);
  cudaEventDestroy(e1);
  if (rc != CULGT_OK) return rc;
  g_variant = best;
  if (best_variant) *best_variant = best;
  if (best_us_per_half_sweep) *best_us_per_half_sweep = best_us;
  return CULGT_OK;
}

int culgt_set_sweep_variant(int variant) {
  if (!sweep_variant_known(variant)) return CULGT_ERR_ARG;
  g_variant = variant;
  return CULGT_OK;
}
int culgt_get_sweep_variant(void) { return g_variant; }
const char* culgt_sweep_kernel_name(const culgt_lattice* lat) {
  LatticeDesc d;
  if (describe(lat, &d) != CULGT_OK) return "";
  return sweep_kernel_name(d);
}
int culgt_measure_build(void) {
#ifdef CULGT_MEASURE
  return 1;
#else
  return 0;
#endif
}

#ifdef CULGT_MEASURE
// ---- entry points of the measurement build only (csrc/measure_api.h) -----------------------------------
int culgt_or_sweeps_ws(const culgt_lattice* lat, void* links, void* workspace, int n_sweeps, double omega,
                       void* stream) {
  LatticeDesc d;
  int rc = describe(lat, &d);
  if (rc != CULGT_OK) return rc;
  if (!links || !workspace) return CULGT_ERR_NULL;
  if (misaligned(links) || misaligned(workspace)) return CULGT_ERR_ALIGN;
  if (n_sweeps < 0) return CULGT_ERR_ARG;
  if ((rc = check_omega(omega)) != CULGT_OK) return rc;
  cudaError_t e = launch_or_full_sweeps(d, links, (double*)workspace, n_sweeps, omega, g_variant, nullptr,
                                        (cudaStream_t)stream);
  return e == cudaSuccess ? CULGT_OK : cuda_fail(e);
}

int culgt_fused_schedule(int n_slices, int lag, int direction, unsigned* tasks_out) {
  if (!tasks_out) return CULGT_ERR_NULL;
  if (n_slices < 2 || (n_slices & 1) || n_slices > kFusedMaxSlices || (direction != 0 && direction != 1)) return CULGT_ERR_ARG;
  fused_schedule(n_slices, lag, direction, tasks_out);
  return CULGT_OK;
}

#endif

const char* culgt_strerror(int status) {
  switch (status) {
    case CULGT_OK: return "ok";
    case CULGT_ERR_NULL: return "null pointer";
    case CULGT_ERR_DIMS: return "lattice extents must be even, >= 2, volume <= 2^30";
    case CULGT_ERR_DESC: return "unsupported group/precision/params combination";
    case CULGT_ERR_PARITY: return "parity must be 0 or 1";
    case CULGT_ERR_OMEGA: return "omega must be in [1,2)";
    case CULGT_ERR_ALIGN: return "device pointer not 16-byte aligned";
    case CULGT_ERR_CUDA: return "CUDA error (see culgt_last_cuda_error)";
    case CULGT_ERR_ARG: return "argument out of range";
    case CULGT_ERR_NCCL: return "NCCL error (see culgt_last_cuda_error)";
    case CULGT_ERR_TOO_LARGE: return "lattice exceeds the built-in scratch of the no-allocation entry point (at most 2^24 sites)";
    default: return "unknown status";
  }
}
const char* culgt_last_cuda_error(void) { return g_cuda_err; }
int culgt_version(void) { return 200; }

}  // extern "C"
