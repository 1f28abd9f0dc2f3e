// slab.cu -- time-slab decomposition of the lattice over several GPUs (
// the paper's only hook is the title of its ref. [2], "... with Multi-GPUs").
//
// The lattice is cut along t into n_slabs slabs of T = N3 / n_slabs time-slices (T even, so that a
// site's parity is the same in the slab's and in the lattice's coordinates).  A slab is an internal-
// layout field of the LOCAL lattice (N0, N1, N2, T) whose planes [parity][mu][j] carry one extra GHOST
// slice behind the last one (pitch = vh + stride3):
//
//   * sites of one parity are independent, so a half-sweep of parity p runs on every slab at
//     once with the unchanged production kernel -- only the geometry differs: at x3 = 0 the neighbour
//     x - t_hat is not the slab's own last slice (periodic wrap) but the ghost slice, Geom::wrap3;
//   * the ghost slice of plane [1-p][3][j] holds the t-links U_t(y), y in the PREVIOUS slab's last
//     slice, parity 1-p.  The half-sweep of parity p READS AND WRITES them (U_t(x - t_hat) <- U_t(x - t_hat)
//     G(x)^dagger), so they go BACK to their owner after the half-sweep, and the owner's
//     t-links of parity p in its last slice (which its own sites have just updated as up links) go
//     FORWARD into the next slab's ghost slice for the half-sweep of parity 1-p.  Per half-sweep and
//     boundary exactly one message each way of N0 N1 N2 / 2 links (halo_bytes).
//   * theta and F: every slab reduces its own sites (the ghost slices supply U_t(x - t_hat) for its
//     first slice) to two raw sums; the n_slabs pairs are summed in slab order and normalised by one
//     tiny kernel, so the result is bit-reproducible for a given n_slabs.
//
// Transports: slabs of one process (same or peer devices) by one cudaMemcpy2DAsync per message;
// ranks by ncclSend / ncclRecv on the compute stream (NCCL is resolved at run time from the process,
// i.e. the libnccl torch has loaded; the library has no link-time dependency on it).
#include <dlfcn.h>
#include <nccl.h>
#include <stdio.h>
#include "kernels.h"

namespace culgt {

// ---- geometry ---------------------------------------------------------------------------------------
void make_slab_geom(Geom* g) {
  g->pitch = g->vh + g->stride[3];
  g->wrap3 = g->vh;                  // x3 = 0: h + vh = ghost slice, same position inside the slice
}

int slab_vectors_per_link(const LatticeDesc& d) {
  if (d.group == 2) return d.precision == 32 ? 1 : 2;
  if (d.precision == 32) return d.params == 12 ? 3 : 5;
  return d.params == 12 ? 6 : 9;
}

// Chunks of one halo message: vector j of the t-links of parity `parity` in the ghost slice
// (which = 0) or in the last slice (which = 1); offsets in bytes from the start of the slab's links.
void slab_halo_chunks(const LatticeDesc& d, int parity, int which, size_t* offsets, size_t* chunk_bytes, int* n_chunks) {
  const Geom& g = d.geom;
  const int nv = slab_vectors_per_link(d);
  for (int j = 0; j < nv; ++j) {
    const size_t plane = (size_t)((parity * 4 + 3) * nv + j) * (size_t)g.pitch;
    const size_t first = which == 0 ? (size_t)g.vh : (size_t)(g.vh - g.stride[3]);
    offsets[j] = (plane + first) * 16;
  }
  *chunk_bytes = (size_t)g.stride[3] * 16;
  *n_chunks = nv;
}

// One halo message between two slabs of this process: direction 0 = FORWARD (src's last slice ->
// dst's ghost slice), 1 = BACK (src's ghost slice -> dst's last slice).  The nv chunks are equally
// spaced (one plane pitch apart) on both sides: a single 2-D copy.
cudaError_t slab_halo_copy(const LatticeDesc& d, const void* src, void* dst, int parity, int direction, cudaStream_t st) {
  size_t so[9], dof[9], bytes;
  int n;
  slab_halo_chunks(d, parity, direction == 0 ? 1 : 0, so, &bytes, &n);
  slab_halo_chunks(d, parity, direction == 0 ? 0 : 1, dof, &bytes, &n);
  const size_t pitch_bytes = (size_t)d.geom.pitch * 16;
  return cudaMemcpy2DAsync((char*)dst + dof[0], pitch_bytes, (const char*)src + so[0], pitch_bytes, bytes, (size_t)n,
                           cudaMemcpyDeviceToDevice, st);
}

// ---- theta / F ------------------------------------------------------------------------------------------
// Slab k's two raw sums sit at sums[2k], sums[2k+1]; this kernel adds the n_slabs pairs in slab order
// (one thread: a fixed order, hence the same bits every time) and normalises with the GLOBAL volume.
__global__ void slab_combine_kernel(const double* __restrict__ sums, int n_slabs, double scale_theta, double scale_F,
                                    double* __restrict__ theta, double* __restrict__ F) {
  if (threadIdx.x != 0 || blockIdx.x != 0) return;
  double st = 0, sf = 0;
  for (int k = 0; k < n_slabs; ++k) {
    st += sums[2 * k];
    sf += sums[2 * k + 1];
  }
  *theta = st * scale_theta;
  *F = sf * scale_F;
}

cudaError_t slab_theta_F_combine(const LatticeDesc& global, const double* sums, int n_slabs, double* theta, double* F,
                                 cudaStream_t st) {
  const double nc = (double)global.group;
  slab_combine_kernel<<<1, 32, 0, st>>>(sums, n_slabs, 1.0 / (nc * (double)global.V), 1.0 / (4.0 * nc * (double)global.V),
                                        theta, F);
  return cudaGetLastError();
}

// ---- NCCL, resolved at run time -----------------------------------------------------------------------
struct Nccl {
  void* handle = nullptr;
  ncclResult_t (*GetUniqueId)(ncclUniqueId*) = nullptr;
  ncclResult_t (*CommInitRank)(ncclComm_t*, int, ncclUniqueId, int) = nullptr;
  ncclResult_t (*CommDestroy)(ncclComm_t) = nullptr;
  ncclResult_t (*Send)(const void*, size_t, ncclDataType_t, int, ncclComm_t, cudaStream_t) = nullptr;
  ncclResult_t (*Recv)(void*, size_t, ncclDataType_t, int, ncclComm_t, cudaStream_t) = nullptr;
  ncclResult_t (*AllGather)(const void*, void*, size_t, ncclDataType_t, ncclComm_t, cudaStream_t) = nullptr;
  ncclResult_t (*GroupStart)() = nullptr;
  ncclResult_t (*GroupEnd)() = nullptr;
  const char* (*GetErrorString)(ncclResult_t) = nullptr;
  bool ok = false;
};

static const Nccl& nccl() {
  static Nccl n = [] {
    Nccl r;
    // the copy already in the process (torch's) first; a fresh one otherwise
    r.handle = dlopen("libnccl.so.2", RTLD_NOW | RTLD_NOLOAD);
    if (!r.handle) r.handle = dlopen("libnccl.so.2", RTLD_NOW);
    if (!r.handle) r.handle = dlopen("libnccl.so", RTLD_NOW);
    if (!r.handle) return r;
    bool all = true;
    auto sym = [&](const char* name) {
      void* p = dlsym(r.handle, name);
      if (!p) all = false;
      return p;
    };
    r.GetUniqueId = (decltype(r.GetUniqueId))sym("ncclGetUniqueId");
    r.CommInitRank = (decltype(r.CommInitRank))sym("ncclCommInitRank");
    r.CommDestroy = (decltype(r.CommDestroy))sym("ncclCommDestroy");
    r.Send = (decltype(r.Send))sym("ncclSend");
    r.Recv = (decltype(r.Recv))sym("ncclRecv");
    r.AllGather = (decltype(r.AllGather))sym("ncclAllGather");
    r.GroupStart = (decltype(r.GroupStart))sym("ncclGroupStart");
    r.GroupEnd = (decltype(r.GroupEnd))sym("ncclGroupEnd");
    r.GetErrorString = (decltype(r.GetErrorString))sym("ncclGetErrorString");
    r.ok = all;
    return r;
  }();
  return n;
}

struct SlabComm {
  ncclComm_t comm;
  int rank, n_ranks;
};

bool slab_nccl_available() { return nccl().ok; }

const char* slab_nccl_error(int code) {
  return nccl().ok ? nccl().GetErrorString((ncclResult_t)code) : "libnccl.so.2 not found in the process";
}

int slab_comm_id(void* id128) {
  if (!nccl().ok) return -1;
  static_assert(sizeof(ncclUniqueId) == 128, "ncclUniqueId is 128 bytes");
  return (int)nccl().GetUniqueId((ncclUniqueId*)id128);
}

int slab_comm_create(const void* id128, int rank, int n_ranks, void** out) {
  if (!nccl().ok) return -1;
  ncclUniqueId id;
  memcpy(&id, id128, sizeof(id));
  SlabComm* c = new SlabComm;
  c->rank = rank;
  c->n_ranks = n_ranks;
  const ncclResult_t r = nccl().CommInitRank(&c->comm, n_ranks, id, rank);
  if (r != ncclSuccess) {
    delete c;
    return (int)r;
  }
  *out = c;
  return 0;
}

int slab_comm_destroy(void* comm) {
  if (!comm) return 0;
  SlabComm* c = (SlabComm*)comm;
  const int r = nccl().ok ? (int)nccl().CommDestroy(c->comm) : 0;
  delete c;
  return r;
}

void slab_comm_info(void* comm, int* rank, int* n_ranks) {
  SlabComm* c = (SlabComm*)comm;
  *rank = c->rank;
  *n_ranks = c->n_ranks;
}

// Ring neighbours of a halo message: FORWARD goes to the slab holding the later time-slices.
void slab_halo_peers(int rank, int n_ranks, int direction, int* send_to, int* recv_from) {
  const int next = (rank + 1) % n_ranks, prev = (rank + n_ranks - 1) % n_ranks;
  *send_to = direction == 0 ? next : prev;
  *recv_from = direction == 0 ? prev : next;
}

// One halo exchange around the ring of ranks (rank r owns slab r; r-1 holds the earlier time-slices):
// direction 0 = FORWARD: send my last slice to r+1, receive my ghost slice from r-1;
// direction 1 = BACK:    send my ghost slice to r-1, receive my last slice from r+1.
// All chunks of both messages in one NCCL group on `st`.
int slab_halo_exchange(void* comm, const LatticeDesc& d, void* links, int parity, int direction, cudaStream_t st) {
  if (!nccl().ok) return -1;
  SlabComm* c = (SlabComm*)comm;
  size_t ghost[9], last[9], bytes;
  int n;
  slab_halo_chunks(d, parity, 0, ghost, &bytes, &n);
  slab_halo_chunks(d, parity, 1, last, &bytes, &n);
  const size_t* send_off = direction == 0 ? last : ghost;
  const size_t* recv_off = direction == 0 ? ghost : last;
  int send_to, recv_from;
  slab_halo_peers(c->rank, c->n_ranks, direction, &send_to, &recv_from);
  ncclResult_t r = nccl().GroupStart();
  if (r != ncclSuccess) return (int)r;
  for (int j = 0; j < n && r == ncclSuccess; ++j) {
    r = nccl().Send((const char*)links + send_off[j], bytes, ncclChar, send_to, c->comm, st);
    if (r == ncclSuccess) r = nccl().Recv((char*)links + recv_off[j], bytes, ncclChar, recv_from, c->comm, st);
  }
  const ncclResult_t e = nccl().GroupEnd();
  return (int)(r != ncclSuccess ? r : e);
}

// every rank's two raw sums -> all[2 * n_ranks] on every rank, in rank (= slab) order
int slab_allgather_sums(void* comm, const double* sums2, double* all, cudaStream_t st) {
  if (!nccl().ok) return -1;
  SlabComm* c = (SlabComm*)comm;
  return (int)nccl().AllGather(sums2, all, 2, ncclDouble, c->comm, st);
}

}  // namespace culgt
