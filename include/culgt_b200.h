/* culgt_b200.h -- C ABI of libculgt_b200.so: the checkerboard overrelaxation sweep for lattice
 * Landau gauge fixing (arXiv:1412.3655 "cuLGT: Lattice Gauge Fixing on GPUs"), hand-written
 * CUDA for sm_100a (NVIDIA B200).
 *
 * Citations: P:Lnn = PAPER.md line nn of the reference text; C-n = reading n in DESIGN.md.
 *
 * General rules
 *   - Every function returns an int status (CULGT_OK = 0, errors < 0) unless it returns a size.
 *     Nothing throws, aborts, prints or allocates device memory.
 *   - The library keeps NO state between calls except, per device, lazily-set kernel attributes and
 *     cached device properties, and, per HOST THREAD, the sweep-variant selection
 *     (culgt_set_sweep_variant) and the text of the last CUDA error.  Whatever a kernel must remember
 *     between launches (the driver loop's stop word) lives in the
 *     caller's `workspace` and is re-initialised by the call that uses it; a workspace must therefore
 *     not be shared by calls that run concurrently.  One process may drive several devices: every call
 *     acts on the CURRENT device (cudaSetDevice), to which its pointers and stream must belong.
 *   - "device pointer" = address in the current CUDA device's global memory, 16-byte aligned,
 *     owned (allocated and freed) by the caller.  "host pointer" = ordinary host memory owned
 *     by the caller (pinned memory makes the *_host calls faster but is not required).
 *   - `stream` is a cudaStream_t passed as void* (NULL = the legacy default stream).  Calls
 *     taking a stream only ENQUEUE work and return without synchronising, except where stated.
 *   - There is no CPU fallback: without a CUDA device every compute call returns CULGT_ERR_CUDA.
 *   - Non-unitary input is not detected (garbage in, garbage out).
 *
 * Lattice and layouts
 *   dims = {N0,N1,N2,N3} = x,y,z,t extents, periodic in all directions (C-2); every extent must
 *   be even and >= 2 (an odd extent breaks the checkerboard across the wrap).
 *   Canonical site index  s = x0 + N0*(x1 + N1*(x2 + N2*x3));  parity(x) = (x0+x1+x2+x3)&1,
 *   0 = "black", 1 = "white" (C-1); mu = 0..3 <-> x,y,z,t (C-3).
 *   CANONICAL field  : real[V][4][Nc][Nc][2]  site-major, full Nc x Nc complex matrices,
 *                      row-major, re/im interleaved (the interchange format a host framework
 *                      hands over, "linear float or double array of length V*Nd*2Nc^2").
 *   CANONICAL g field: real[V][Nc][Nc][2].
 *   INTERNAL field   : links[parity][mu][j][h], parity-split, site-fastest structure of arrays
 *                      ("site index runs faster than Lorentz and matrix indices") of
 *                      vectors: SU(3) 12-parameter fp32 = 3 x float4, fp64 = 6 x double2;
 *                      18-parameter fp32 = 5 x float4 (the last half used), fp64 = 9 x double2; SU(2) 4-parameter
 *                      fp32 = 1 x float4 (a0,a1,a2,a3), fp64 = 2 x double2.  h = s>>1 is the
 *                      index of the site inside its parity.  Opaque to the caller: use
 *                      culgt_pack / culgt_unpack.  `real` = float (precision 32) or double (64)
 *                      for BOTH the canonical and the internal field.
 */
#ifndef CULGT_B200_H
#define CULGT_B200_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define CULGT_OK            0
#define CULGT_ERR_NULL     -1  /* a required pointer is NULL                                  */
#define CULGT_ERR_DIMS     -2  /* an extent is odd, < 2, or the volume overflows int32 indices */
#define CULGT_ERR_DESC     -3  /* group / precision / params combination not provided         */
#define CULGT_ERR_PARITY   -4  /* parity is not 0 or 1                                         */
#define CULGT_ERR_OMEGA    -5  /* omega is NaN or outside [1,2)                        */
#define CULGT_ERR_ALIGN    -6  /* a device pointer is not 16-byte aligned                      */
#define CULGT_ERR_CUDA     -7  /* CUDA runtime / launch failure (see culgt_last_cuda_error)    */
#define CULGT_ERR_ARG      -8  /* another argument is out of range                             */
#define CULGT_ERR_NCCL     -9  /* NCCL failure, or libnccl.so.2 not found (culgt_last_cuda_error) */
#define CULGT_ERR_TOO_LARGE -10 /* lattice larger than the no-allocation entry point's built-in scratch */

typedef struct {
  int32_t dims[4];    /* N0..N3, x fastest in the canonical site index                        */
  int32_t group;      /* 2 = SU(2), 3 = SU(3)                                                 */
  int32_t precision;  /* 32 or 64                                                             */
  int32_t params;     /* SU(3): 18 (full) or 12 (first two rows); SU(2): 4             */
} culgt_lattice;

/* Sizes in bytes; 0 if the descriptor is invalid. */
size_t culgt_links_bytes(const culgt_lattice* lat);      /* internal field: 4*V*params*sizeof(real)
                                                            (fp32 18-parameter: 4*V*80, 2 pad floats) */
size_t culgt_canonical_bytes(const culgt_lattice* lat);  /* V*4*Nc*Nc*2*sizeof(real)                */
size_t culgt_gfield_bytes(const culgt_lattice* lat);     /* V*Nc*Nc*2*sizeof(real)                  */
size_t culgt_workspace_bytes(const culgt_lattice* lat);  /* reductions: block partials + result slots
                                                            (V/64 doubles), plus ~12 KB of control
                                                            blocks (driver loop)                     */

/* Validate a descriptor: CULGT_OK, CULGT_ERR_NULL, CULGT_ERR_DIMS or CULGT_ERR_DESC. */
int culgt_validate(const culgt_lattice* lat);

/* a0: canonical <-> internal (P:L64 reordering into black/white sublattices; "discarding
 * the third line" on pack, implicit reconstruction row2 = conj(row0 x row1) on unpack).
 * canonical, links: device pointers (distinct buffers).  Asynchronous on `stream`. */
int culgt_pack(const culgt_lattice* lat, const void* canonical, void* links, void* stream);
int culgt_unpack(const culgt_lattice* lat, const void* links, void* canonical, void* stream);

/* Re-unitarisation (reading C-23; not in the paper's text): projects every stored link
 * back onto the group by Gram-Schmidt on its stored rows (r0 <- r0/|r0|, r1 <- r1 - <r0,r1> r0,
 * r1 <- r1/|r1|; 18-parameter: r2 <- conj(r0 x r1); SU(2): quaternion normalisation), in fp64,
 * in place.  For long fp32 runs, whose stored rows drift slowly off SU(3) (C-13).  Asynchronous. */
int culgt_reunitarize(const culgt_lattice* lat, void* links, void* stream);

/* a1-a6: ONE HALF sweep of overrelaxation over all sites x of `parity`, in place:
 *   K(x) = sum_mu [ U_mu(x) + U_mu(x-mu)^dagger ]                         eq. (3)
 *   SU(2): g = K^dagger/sqrt(det K^dagger), G = g^omega
 *   SU(3): for the subgroups (0,1),(0,2),(1,2): g_s from the block of the current K, raised to
 *          omega, K <- g_s K, G <- g_s G  (C-6, C-10); g^omega is the exact group power (C-8)
 *   U_mu(x) <- G U_mu(x),  U_mu(x-mu) <- U_mu(x-mu) G^dagger
 * links: device pointer to the internal field.  omega in [1,2).  Asynchronous on `stream`.
 * Arithmetic: precision 64 -> all fp64.  precision 32 -> link storage, reconstruction and the 8
 * link products in fp32; K accumulation and the subgroup solve in fp64 (C-15). */
int culgt_or_sweep(const culgt_lattice* lat, void* links, int parity, double omega, void* stream);

/* n_sweeps full sweeps (black then white half-sweep each; C-12), enqueued back to back. */
int culgt_or_sweeps(const culgt_lattice* lat, void* links, int n_sweeps, double omega, void* stream);

/* a8: theta = 1/(Nc V) sum_x tr[Delta(x) Delta(x)^dagger],  Delta = sum_mu A_mu(x) - A_mu(x-mu),
 * A_mu = [(U_mu - U_mu^dagger)/(2i)]_traceless with a*g = 1 (eq. (1); C-4, C-5).
 * a7: F = 1/(4 Nc V) sum_x sum_mu Re tr U_mu(x) (eq. (2) at g = 1).
 * workspace: device pointer, >= culgt_workspace_bytes.  The fp64 scalar is written to the DEVICE
 * address *_dev; the reduction is deterministic (fixed order, fp64).  Asynchronous on `stream`. */
int culgt_gauge_precision(const culgt_lattice* lat, const void* links, void* workspace,
                          double* theta_dev, void* stream);
int culgt_functional(const culgt_lattice* lat, const void* links, void* workspace,
                     double* F_dev, void* stream);

/* a7 + a8 in ONE pass over the field (what the driver loop needs at every check): both
 * scalars as above, written to the DEVICE addresses theta_dev and F_dev.  Same workspace. */
int culgt_gauge_precision_functional(const culgt_lattice* lat, const void* links, void* workspace,
                                     double* theta_dev, double* F_dev, void* stream);

/* a7 + a8 for callers that CANNOT ALLOCATE device memory (code under CUDA graph capture, tight serving
 * loops, harnesses that forbid cudaMalloc): the same fused pass, the same kernels and the same bits as
 * culgt_gauge_precision_functional, without a workspace argument -- the block partials live in a
 * file-scope device array of the library: 2 MiB, held by every GPU that loads the library until the
 * process exits.  Limit: V = N0*N1*N2*N3 <= CULGT_NOALLOC_MAX_SITES = 2^24 sites (64^4) in every
 * storage format; a larger lattice returns CULGT_ERR_TOO_LARGE and launches nothing.  The call
 * allocates nothing (no cudaMalloc, cudaFree or allocating library routine).  The first call on each
 * device resolves the array's device address (cudaGetSymbolAddress; no allocation): make it before
 * starting a stream capture.  All calls on a device share the array, which keeps the last call's
 * contents; nothing in it has to start at zero (every slot read has been written by the same call).
 * Calls on one stream are ordered and safe; calls that OVERLAP on the GPU (different streams, no event
 * between them) race on the array -- do not do that.  theta_dev, F_dev: DEVICE addresses, as above.
 * Asynchronous on `stream`. */
#define CULGT_NOALLOC_MAX_SITES (1 << 24)
int culgt_gauge_precision_functional_noalloc(const culgt_lattice* lat, const void* links, double* theta_dev,
                                             double* F_dev, void* stream);

/* a9: U_mu(x) <- g(x) U_mu(x) g(x+mu)^dagger for all x, mu (the paper's worked code
 * example P:L105-118).  g: device pointer to a canonical g field (read-only); links in place. */
int culgt_gauge_transform(const culgt_lattice* lat, void* links, const void* g, void* stream);

/* The paper's driver loop ("iterated until the discrete gauge condition (1) is satisfied
 * up to a given numerical precision"): full sweeps until theta < theta_target or max_sweeps,
 * theta checked every check_every sweeps (and before the first).  The stopping decision is taken
 * ON THE DEVICE (a stop word in the workspace, raised by the check's reduction kernel, turns every
 * launch enqueued behind it into a no-op), so the host synchronises only once per batch of about 32
 * sweeps' worth of launches, not at each check; the field, sweeps_done, theta and F are exactly
 * those of the loop that stops at the first check with theta < theta_target.  A NaN theta never
 * satisfies the test (the loop then runs to max_sweeps).  SU(3) lattices with at most one site block
 * (128 sites for fp32 12-parameter storage, 64 otherwise) per SM and parity run the WHOLE loop as one
 * cooperative kernel (grid barriers between half-sweeps, theta and F reduced inside it); the links
 * are the same bit for bit, theta and F agree to rounding (the partial sums are grouped differently).
 * SYNCHRONISES.  Outputs are HOST pointers (any may be NULL). */
int culgt_landau_fix(const culgt_lattice* lat, void* links, void* workspace, double omega,
                     double theta_target, int max_sweeps, int check_every,
                     int* sweeps_done, double* theta_out, double* F_out, void* stream);

/* End-to-end call with HOST buffers: copies the canonical field host->device, packs, runs
 * n_sweeps full sweeps, computes theta and F, unpacks and copies the fixed field back to the
 * host (canonical_host is updated in place).  Device scratch is supplied by the caller:
 * canonical_dev >= culgt_canonical_bytes, links_dev >= culgt_links_bytes, workspace >=
 * culgt_workspace_bytes.  SYNCHRONISES before returning.  theta_out / F_out: host pointers. */
int culgt_fix_host(const culgt_lattice* lat, void* canonical_host, void* canonical_dev,
                   void* links_dev, void* workspace, int n_sweeps, double omega,
                   double* theta_out, double* F_out, void* stream);

/* ---- Truncated-series overrelaxation (reading C-24; the paper says only "replacing g(x)
 * by g^omega(x)"): the same half-sweep with g^omega replaced by the binomial series
 * sum_{n<=order} binom(omega,n) (g-1)^n projected back to SU(2) (order 0..16; the series converges
 * to the exact power only while |g-1| < 1, i.e. on smooth fields).  Landau gauge. */
int culgt_or_sweep_series(const culgt_lattice* lat, void* links, int parity, double omega, int order,
                          void* stream);
int culgt_or_sweeps_series(const culgt_lattice* lat, void* links, int n_sweeps, double omega, int order,
                           void* stream);

/* ---- Simulated annealing (named by the paper beside overrelaxation, P:L7; DESIGN.md reading
 * C-25): a half-sweep in which the site's transformation is a SAMPLE of exp(Re tr[g K(x)]/T) dg
 * (per SU(2) subgroup for SU(3); Kennedy-Pendleton heat bath) instead of its maximiser.  Random
 * numbers: Philox4x32-10 with counter (canonical site, `counter`, subgroup | draw << 8, 0) and key
 * `seed`; `counter` must differ between the half-sweeps of a run.  T > 0.  Landau gauge.
 * culgt_sa_anneal: n_sweeps full sweeps with T going linearly from T_max to T_min, half-sweep
 * counters 0, 1, 2, ...; asynchronous (follow it with overrelaxation to converge). */
int culgt_sa_sweep(const culgt_lattice* lat, void* links, int parity, double T, unsigned long long seed,
                   unsigned counter, void* stream);
int culgt_sa_anneal(const culgt_lattice* lat, void* links, double T_max, double T_min, int n_sweeps,
                    unsigned long long seed, void* stream);

/* ---- Microcanonical step (SURVEY.md 8(f) NEXT-3 pairs it with simulated annealing; DESIGN.md
 * reading C-26): the half-sweep whose per-subgroup update is the reflection q = g^2 of the maximiser
 * g = K^dagger/sqrt(det K^dagger) -- Re tr[g_s K], hence F, is unchanged while the links move
 * (the omega -> 2 end of "replacing g(x) by g^omega(x)", which culgt_or_sweep excludes).
 * Deterministic, in place, asynchronous; Landau gauge.
 * culgt_micro_sweeps: n_sweeps full (black + white) sweeps.
 * culgt_sa_anneal_micro: the schedule of culgt_sa_anneal with n_micro >= 0 microcanonical full
 * sweeps after every annealing sweep (annealing half-sweep counters stay 2i, 2i+1). */
int culgt_micro_sweep(const culgt_lattice* lat, void* links, int parity, void* stream);
int culgt_micro_sweeps(const culgt_lattice* lat, void* links, int n_sweeps, void* stream);
int culgt_sa_anneal_micro(const culgt_lattice* lat, void* links, double T_max, double T_min, int n_sweeps,
                          int n_micro, unsigned long long seed, void* stream);

/* ---- Coulomb gauge (named by the paper, P:L7; reading C-22): the same update
 * with mu restricted to the 3 spatial directions, time-slice by time-slice:
 *   K_C(x) = sum_{i<3} [ U_i(x) + U_i(x-i)^dagger ],  G from K_C as above,
 *   U_mu(x) <- G U_mu(x),  U_mu(x-mu) <- U_mu(x-mu) G^dagger  for ALL 4 mu (a gauge transformation
 *   acts on every link touching x, time links included).
 *   F_t = 1/(3 Nc Vs) sum_{x in slice t} sum_{i<3} Re tr U_i(x),
 *   theta_t = 1/(Nc Vs) sum_{x in slice t} tr[Delta_C Delta_C^dagger],  Delta_C = sum_{i<3} A_i(x) - A_i(x-i),
 *   t = x3 = 0..N3-1, Vs = N0*N1*N2.
 * culgt_or_sweep_coulomb / culgt_or_sweeps_coulomb: as the Landau calls.
 * culgt_coulomb_precision_functional: theta_t_dev, F_t_dev are DEVICE arrays of dims[3] doubles.
 * culgt_or_sweep_coulomb_masked: the half-sweep over the time-slices t with slice_active_dev[t] != 0
 *   only (DEVICE array of dims[3] bytes); slices decouple, so frozen slices keep their spatial links.
 * culgt_coulomb_fix: every slice is swept until ITS theta_t < theta_target (checked every
 *   check_every sweeps; converged slices are frozen, the others go on) or max_sweeps.  As in
 *   culgt_landau_fix the decisions are taken on the device (the mask is recomputed by the check, a stop
 *   word raised when no slice is active) and the host synchronises once per batch of checks;
 *   SYNCHRONISES; sweeps_done = sweeps of the slowest slice; theta_t_out / F_t_out: HOST arrays of
 *   dims[3] doubles (may be NULL). */
int culgt_or_sweep_coulomb(const culgt_lattice* lat, void* links, int parity, double omega, void* stream);
int culgt_or_sweeps_coulomb(const culgt_lattice* lat, void* links, int n_sweeps, double omega, void* stream);
int culgt_or_sweep_coulomb_masked(const culgt_lattice* lat, void* links, int parity, double omega,
                                  const unsigned char* slice_active_dev, void* stream);
int culgt_coulomb_precision_functional(const culgt_lattice* lat, const void* links, void* workspace,
                                       double* theta_t_dev, double* F_t_dev, void* stream);
int culgt_coulomb_fix(const culgt_lattice* lat, void* links, void* workspace, double omega,
                      double theta_target, int max_sweeps, int check_every, int* sweeps_done,
                      double* theta_t_out, double* F_t_out, void* stream);

/* ---- Time-slab decomposition over several GPUs (the paper's only hook is
 * the title of its ref. [2], "... with Multi-GPUs").  The lattice is cut along t into n_slabs
 * slabs of T = dims[3] / n_slabs time-slices (T even >= 2).  A slab is described by the LOCAL lattice
 * (dims[3] = T; culgt_slab_lattice) and stored as an internal field whose planes carry one extra GHOST
 * slice (culgt_slab_links_bytes): it holds the t-links U_t(y), y in the previous slab's last slice, i.e.
 * the links U_t(x - t_hat) that the sites x of the slab's first slice read AND write.
 * Sites of one parity are independent: a half-sweep of parity p runs on all slabs at once with
 * the unchanged kernels (the links come out bit-identical to the undivided sweep), followed by ONE halo
 * message each way per boundary, culgt_slab_halo_bytes = N0*N1*N2/2 links each:
 *     BACK    (direction 1): my ghost slice, parity 1-p  ->  the previous slab's last slice;
 *     FORWARD (direction 0): my last slice,  parity p    ->  the next slab's ghost slice.
 * Before the first half-sweep (and before theta/F on freshly packed slabs) both parities go FORWARD once
 * (culgt_slab_exchange_all_*).  The slab holding time-slices [k*T, (k+1)*T) is slab k; "previous" is
 * k-1 (mod n_slabs).  The canonical field of slab k is the contiguous part [k*V/n_slabs, (k+1)*V/n_slabs)
 * of the global canonical field (t is the slowest coordinate).
 *
 * culgt_slab_halo_chunks (host only): a message is n_chunks (= vectors per link, <= 9) runs of chunk_bytes
 *   bytes; offsets[j] = byte offset of run j from the start of the slab's links, for the ghost slice
 *   (which = 0) or the last slice (which = 1) of the t-links of `parity`.
 * culgt_slab_halo_peers (host only): the ranks a message of `direction` is sent to / received from
 *   (FORWARD: to rank+1 from rank-1; BACK: to rank-1 from rank+1; periodic).
 * culgt_slab_or_sweep / _window: the half-sweep on one slab (all of it / time-slices [t_lo, t_hi) only --
 *   CULGT_ERR_DESC when the slab holds no whole site blocks per time-slice, or for SU(2)).  Sweeping the
 *   boundary slices 0 and T-1 first lets both messages travel while the interior [1, T-1) is swept.
 * culgt_slab_halo_copy: one message between two slabs of this process (same or peer devices).
 * culgt_slab_theta_F_sums: the slab's RAW sums (sum_x tr[Delta Delta^dagger], sum_{x,mu} Re tr U) as two
 *   doubles at sums2_dev; culgt_slab_theta_F_combine adds the n_slabs pairs at sums_dev in slab order and
 *   normalises with the GLOBAL volume (eq. (1), (2)): bit-reproducible for a given n_slabs.
 * culgt_slab_*_local: drivers for n_slabs slabs held by ONE process (links_slabs: host array of device
 *   pointers, slab order): n_sweeps full sweeps with the exchanges as device copies on `stream`
 *   (boundary_first != 0: boundary slices first, as the overlapped schedule orders them); theta and F
 *   (sums_dev: 2*n_slabs doubles of device scratch).
 * culgt_slab_comm_*: one slab per rank over NCCL (resolved at run time from the process, normally the
 *   libnccl torch loaded; CULGT_ERR_NCCL if absent).  unique_id: 128 bytes of HOST memory, made on rank
 *   0 and distributed by the caller (e.g. torch.distributed broadcast); create is collective.
 * culgt_slab_or_sweeps_nccl: n_sweeps full sweeps of my slab with ncclSend/ncclRecv halo messages
 *   around the ring.  comm_stream NULL or == stream: messages on `stream` after each half-sweep;
 *   otherwise the boundary slices are swept first and the messages travel on comm_stream while the
 *   interior is swept (the next half-sweep waits for them).
 * culgt_slab_theta_F_nccl: every rank's raw sums are all-gathered (sums_dev: 2*n_ranks + 2 doubles of
 *   device scratch) and combined in rank order on every rank. */
int culgt_slab_lattice(const culgt_lattice* global, int n_slabs, culgt_lattice* local);
size_t culgt_slab_links_bytes(const culgt_lattice* local);
size_t culgt_slab_halo_bytes(const culgt_lattice* local);
int culgt_slab_halo_chunks(const culgt_lattice* local, int parity, int which, size_t* offsets, size_t* chunk_bytes,
                           int* n_chunks);
int culgt_slab_halo_peers(int rank, int n_ranks, int direction, int* send_to, int* recv_from);
int culgt_slab_pack(const culgt_lattice* local, const void* canonical_slab, void* links_slab, void* stream);
int culgt_slab_unpack(const culgt_lattice* local, const void* links_slab, void* canonical_slab, void* stream);
int culgt_slab_or_sweep(const culgt_lattice* local, void* links_slab, int parity, double omega, void* stream);
int culgt_slab_or_sweep_window(const culgt_lattice* local, void* links_slab, int parity, double omega, int t_lo,
                               int t_hi, void* stream);
int culgt_slab_halo_copy(const culgt_lattice* local, const void* src_links, void* dst_links, int parity, int direction,
                         void* stream);
int culgt_slab_theta_F_sums(const culgt_lattice* local, const void* links_slab, void* workspace, double* sums2_dev,
                            void* stream);
int culgt_slab_theta_F_combine(const culgt_lattice* global, const double* sums_dev, int n_slabs, double* theta_dev,
                               double* F_dev, void* stream);
int culgt_slab_exchange_all_local(const culgt_lattice* local, void* const* links_slabs, int n_slabs, void* stream);
int culgt_slab_or_sweeps_local(const culgt_lattice* local, void* const* links_slabs, int n_slabs, int n_sweeps,
                               double omega, int boundary_first, void* stream);
int culgt_slab_theta_F_local(const culgt_lattice* global, const culgt_lattice* local, void* const* links_slabs,
                             int n_slabs, void* workspace, double* sums_dev, double* theta_dev, double* F_dev,
                             void* stream);
int culgt_slab_comm_unique_id(void* id128_host);
int culgt_slab_comm_create(const void* id128_host, int rank, int n_ranks, void** comm_out);
int culgt_slab_comm_destroy(void* comm);
int culgt_slab_halo_exchange(void* comm, const culgt_lattice* local, void* links_slab, int parity, int direction,
                             void* stream);
int culgt_slab_exchange_all_nccl(void* comm, const culgt_lattice* local, void* links_slab, void* stream);
int culgt_slab_or_sweeps_nccl(void* comm, const culgt_lattice* local, void* links_slab, int n_sweeps, double omega,
                              void* comm_stream, void* stream);
int culgt_slab_theta_F_nccl(void* comm, const culgt_lattice* global, const culgt_lattice* local, const void* links_slab,
                            void* workspace, double* sums_dev, double* theta_dev, double* F_dev, void* stream);

/* Sweep-schedule selection of the CALLING HOST THREAD.  Every value the product
 * library accepts computes the same update, bit for bit:
 *    0  the default chosen by measurement (20 is its explicit name for the half-sweep kernel);
 *   24 / 33 / 34  the production kernel without the reversed odd-parity traversal / without
 *       programmatic dependent launch / without L2 eviction hints.
 * Anything else returns CULGT_ERR_ARG.  (A library built with -DCULGT_MEASURE -- python -m
 * paper_1412_3655_b200.build --measure; culgt_measure_build() == 1 -- additionally accepts the
 * measured alternatives of csrc/or_sweep_measure.cu and csrc/or_sweep_fused.cu, some of which
 * deliberately do NOT compute the method; they are never part of the product build.) */
int culgt_set_sweep_variant(int variant);
int culgt_get_sweep_variant(void);
int culgt_measure_build(void);
/* Name of the half-sweep kernel instantiation variant 0 launches for this lattice (static string; ""
 * for an invalid descriptor).  bench.py stamps its committed ncu captures with it. */
const char* culgt_sweep_kernel_name(const culgt_lattice* lat);

/* Run-time autotuner (the paper's per-GPU selection of the fastest set-up, P:L89 (d)):
 * times every result-equivalent sweep schedule with `sweeps_per_trial` REAL full sweeps each on
 * `links` (the field is gauge-fixed further by them), makes the fastest the calling thread's
 * variant and reports it.  workspace: device pointer, >= culgt_workspace_bytes.  SYNCHRONISES.  best_variant,
 * best_us_per_half_sweep: host pointers, may be NULL. */
int culgt_autotune_sweep(const culgt_lattice* lat, void* links, void* workspace, double omega,
                         int sweeps_per_trial, int* best_variant, float* best_us_per_half_sweep, void* stream);

const char* culgt_strerror(int status);
const char* culgt_last_cuda_error(void);
int culgt_version(void);

#ifdef __cplusplus
}
#endif
#endif /* CULGT_B200_H */
