// or_sweep_fused.cu -- ONE persistent kernel for a FULL overrelaxation sweep (black + white,
// PAPER.md L54) in which the two half-sweeps are interleaved time-slice by time-slice, so that a
// white site finds the links its black neighbours have just written still in the 126 MB L2: the
// field then crosses HBM about once per full sweep instead of twice (DESIGN.md 6.1 "fused sweep").
//
// Work is cut into site blocks of BLOCK sites of one parity (the unit of the per-half-sweep
// kernel); a time-slice holds `bps` whole site blocks of each parity.  Resident CTAs draw
// TICKETS from a global counter.  Ticket k is block (k mod bps) of slice-task k / bps, and the
// slice-tasks are ordered (host-built list, FusedCtl::task)
//     B(0) .. B(L+1),  W(1), B(L+2), W(2), ... , B(N3-1), W(N3-2-L),  W(N3-1-L) .. W(N3-2),  W(N3-1), W(0)
// (B = black, W = white, argument = time-slice; L = lag in slices; the descending direction is the
// mirror image t -> N3-1-t with the blocks of a slice descending).  A white site of slice t reads
// and writes links that the black sites of slices t-1, t, t+1 (periodic) also touch, and no
// others; so a W(t) block starts once the completion counters of B(t-1), B(t), B(t+1) have
// reached bps.  Counters are incremented with release semantics after a block's stores
// (__syncthreads, __threadfence, atomicAdd) and polled with ld.acquire.gpu by one thread.
// Sites of one parity do not interact, so the result is bit-identical to two whole
// half-sweeps.  No deadlock: a ticket's dependencies all have smaller ticket numbers, and a CTA
// holds a ticket only while it is running.
// The lag L keeps the white front far enough behind the black front that in the steady state no
// CTA ever waits.  The last CTA to leave resets the control block for the next launch.
//
// MEASURED AND REJECTED (profiles/r2_fused_sweep.md): at 32^4 fp32-12 the schedule does what it was
// built for -- DRAM traffic per full sweep falls from 691 MB to 542 MB, L2 hit rate from 19 % to 66 % --
// but the sweep takes 127-136 us against 111 us for two launches, because the half-sweep is not
// bound by DRAM: the same kernel on an L2-RESIDENT 24^4 field runs at the same 6.9 TB/s per site
// update as on the 32^4 field streamed from HBM.  Compiled only with -DCULGT_MEASURE.
#ifdef CULGT_MEASURE
#include "staged.cuh"
#include "kernels.h"

namespace culgt {

__device__ __forceinline__ unsigned ld_acquire(const unsigned* p) {
  unsigned v;
  asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
  return v;
}

struct FusedPlan {
  int n3;            // time-slices
  int bps;           // site blocks per (slice, parity)
  FastDiv d_bps;
  int total;         // tickets per full sweep = 2 * n3 * bps
  int dir;           // 0 ascending, 1 descending
  int hints;         // L2 policies: bits 0-1 black loads, 2-3 black stores, 4-5 white loads, 6-7 white stores
                     // (0 evict_first, 1 evict_normal, 2 evict_last)
};

template <typename S, int BLOCK, int MINB, typename Power>
__global__ void __launch_bounds__(BLOCK, MINB)
or_full_sweep_fused_kernel(typename S::Vec* __restrict__ links, const Geom g, const Power omega,
                           FusedCtl* __restrict__ ctl, const FusedPlan plan, const int* __restrict__ stop_flag) {
  typedef typename S::Vec Vec;
  extern __shared__ __align__(16) unsigned char smem_raw[];
  Vec* const sm = reinterpret_cast<Vec*>(smem_raw) + threadIdx.x;
  const unsigned sm_addr = (unsigned)__cvta_generic_to_shared(sm);
  __shared__ int s_task[2][4];     // [buffer]{parity, site block (< 0: no more work), dependencies met, slice}
  L2Policies pols;
  pols.create();
  const uint64_t pol_ld_b = pols.pick(plan.hints & 3), pol_st_b = pols.pick((plan.hints >> 2) & 3);
  const uint64_t pol_ld_w = pols.pick((plan.hints >> 4) & 3), pol_st_w = pols.pick((plan.hints >> 6) & 3);

  // the black neighbours of a white slice t live in slices t-1, t, t+1
  auto deps_met = [&](int slice) {
    const int lo = slice > 0 ? slice - 1 : plan.n3 - 1;
    const int hi = slice + 1 < plan.n3 ? slice + 1 : 0;
    const unsigned a = ld_acquire(&ctl->done[0][lo]);
    const unsigned b = ld_acquire(&ctl->done[0][slice]);
    const unsigned c = ld_acquire(&ctl->done[0][hi]);
    const unsigned need = (unsigned)plan.bps;
    return a >= need && b >= need && c >= need;
  };
  // thread 0: draw the next ticket, decode it, probe its dependencies once
  auto draw = [&](int buf) {
    const unsigned k = atomicAdd(&ctl->ticket, 1u);
    if (k >= (unsigned)plan.total) {
      s_task[buf][1] = -1;
      return;
    }
    const unsigned u = plan.d_bps.div(k);
    const int b = (int)(k - u * (unsigned)plan.bps);
    const unsigned task = ctl->task[plan.dir][u];
    const int parity = (int)(task >> 31), slice = (int)(task & 0x7fffffffu);
    s_task[buf][0] = parity;
    s_task[buf][1] = slice * plan.bps + (plan.dir ? plan.bps - 1 - b : b);
    s_task[buf][2] = parity == 0 ? 1 : (int)deps_met(slice);
    s_task[buf][3] = slice;
  };

  // the next launch of the stream may be scheduled; the previous one is complete and visible
  pdl_prologue_done();
  if (stop_flag != nullptr && *stop_flag != 0) return;     // the driver loop has stopped (no ticket was drawn)
  if (threadIdx.x == 0) draw(0);
  __syncthreads();
  for (int it = 0;; ++it) {
    const int buf = it & 1;
    const int parity = s_task[buf][0], site_block = s_task[buf][1], met = s_task[buf][2], slice = s_task[buf][3];
    if (site_block < 0) break;
    const SiteRef<8> r = locate<BLOCK, 1>(g, parity, site_block, 0);
    if (!met) {            // uniform over the CTA; never taken in the steady state (the lag)
      if (threadIdx.x == 0)
        while (!deps_met(slice)) __nanosleep(100);
      __syncthreads();
    }
    issue_site_loads<S, BLOCK, true>(links, g, parity, r, sm, parity ? pol_ld_w : pol_ld_b);
    // while the loads are in flight: the next ticket (its latency hides behind them)
    if (threadIdx.x == 0) draw(buf ^ 1);
    cp_async_wait<0>();
    update_site<S, BLOCK, false, true>(links, g, parity, omega, r, sm_addr, parity ? pol_st_w : pol_st_b);
    __syncthreads();       // every thread's stores are issued; s_task[buf ^ 1] is written
    if (threadIdx.x == 0) {
      __threadfence();     // release: the block's stores are visible before the counter moves
      atomicAdd(&ctl->done[parity][slice], 1u);
    }
  }
  // the last CTA to leave puts the control block back to zero for the next launch
  if (threadIdx.x == 0) {
    const unsigned left = atomicAdd(&ctl->exited, 1u);
    if (left == gridDim.x - 1) {
      for (int t = 0; t < plan.n3; ++t) { ctl->done[0][t] = 0; ctl->done[1][t] = 0; }
      ctl->ticket = 0;
      ctl->exited = 0;
      __threadfence();
    }
  }
}

// ---------------------------------------------------------------------------------------------
// host side
// ---------------------------------------------------------------------------------------------

// Slice-task order of one full sweep (see the header comment).  out[u] = parity << 31 | slice.
void fused_schedule(int n3, int lag, int dir, unsigned* out) {
  if (lag < 1) lag = 1;                  // a white slice's last black neighbour slice must precede it
  if (lag > n3 - 2) lag = n3 - 2;
  if (lag < 0) lag = 0;                  // n3 = 2: both black slices first
  int u = 0;
  auto emit = [&](int parity, int t) { out[u++] = ((unsigned)parity << 31) | (unsigned)(dir ? n3 - 1 - t : t); };
  int next_black = 0;
  const int lead = lag + 2 < n3 ? lag + 2 : n3;
  for (; next_black < lead; ++next_black) emit(0, next_black);
  int next_white = 1;
  while (next_black < n3) {
    emit(1, next_white++);
    emit(0, next_black++);
  }
  for (; next_white <= n3 - 2; ++next_white) emit(1, next_white);
  if (n3 > 1) emit(1, n3 - 1);
  emit(1, 0);
}

int fused_default_lag(int grid, int bps) {
  // black leads white by enough slices that a white block's black neighbours were handed out at
  // least two grids of tickets earlier: every CTA that held one of them has long moved on
  int lag = (2 * grid + 2 * bps - 1) / (2 * bps);
  return lag < 1 ? 1 : lag;
}

template <typename S, int BLOCK, int MINB, typename Power>
static cudaError_t run_fused(void* links, const Geom& g, const Power& omega, FusedCtl* ctl, int n_sweeps,
                             int lag, int hints, bool alternate, const int* stop_flag, cudaStream_t st) {
  typedef typename S::Vec Vec;
  const int n3 = g.n[3];
  if (g.stride[3] % BLOCK != 0 || n3 > kFusedMaxSlices || g.pitch != g.vh) return cudaErrorNotSupported;
  auto kern = or_full_sweep_fused_kernel<S, BLOCK, MINB, Power>;
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
  FusedPlan plan;
  plan.n3 = n3;
  plan.bps = g.stride[3] / BLOCK;
  plan.d_bps.init((uint32_t)plan.bps);
  plan.total = 2 * n3 * plan.bps;
  plan.hints = hints;
  int grid = device_sm_count() * MINB;
  if (grid > plan.total) grid = plan.total;
  if (lag <= 0) lag = fused_default_lag(grid, plan.bps);
  // control block: counters to zero, the two slice-task lists (ascending, descending)
  static_assert(sizeof(FusedCtl) % 4 == 0, "");
  e = cudaMemsetAsync(ctl, 0, offsetof(FusedCtl, task), st);
  if (e != cudaSuccess) return e;
  unsigned sched[2][2 * kFusedMaxSlices];
  fused_schedule(n3, lag, 0, sched[0]);
  fused_schedule(n3, lag, 1, sched[1]);
  for (int d = 0; d < 2; ++d) {
    e = cudaMemcpyAsync(ctl->task[d], sched[d], 2 * (size_t)n3 * sizeof(unsigned), cudaMemcpyHostToDevice, st);
    if (e != cudaSuccess) return e;
  }
  for (int i = 0; i < n_sweeps; ++i) {
    plan.dir = alternate ? (i & 1) : 0;
    e = launch_pdl(kern, dim3((unsigned)grid), dim3(BLOCK), smem, st, (Vec*)links, g, omega, ctl, plan, stop_flag);
    if (e != cudaSuccess) return e;
  }
  return cudaSuccess;
}

cudaError_t launch_or_sweeps_fused(const LatticeDesc& d, void* links, double omega, void* ctl, int n_sweeps,
                                   int lag, int hints, bool alternate, const int* stop_flag, cudaStream_t st) {
  const Geom& g = d.geom;
  if (d.group != 3) return cudaErrorNotSupported;
  FusedCtl* c = (FusedCtl*)ctl;
  if (d.precision == 32 && d.params == 12)
    return run_fused<Storage<float, 3, 12>, 128, 4>(links, g, omega, c, n_sweeps, lag, hints, alternate, stop_flag, st);
  if (d.precision == 32)
    return run_fused<Storage<float, 3, 18>, 64, 5>(links, g, omega, c, n_sweeps, lag, hints, alternate, stop_flag, st);
  if (d.params == 12)
    return run_fused<Storage<double, 3, 12>, 64, 4>(links, g, omega, c, n_sweeps, lag, hints, alternate, stop_flag, st);
  return run_fused<Storage<double, 3, 18>, 64, 3>(links, g, omega, c, n_sweeps, lag, hints, alternate, stop_flag, st);
}

}  // namespace culgt
#endif  // CULGT_MEASURE
