"""GPU parity of the time-slab decomposition (csrc/slab.cu) on ONE device:
n_slabs slabs, each its own internal-layout allocation with a ghost slice, swept by the unchanged
kernels with device-copy halo messages, must reproduce the undivided sweep BIT FOR BIT (sites of one
parity are independent; the halo carries exactly the links a boundary site reads and writes)
and match the oracle after one sweep; theta and F from per-slab sums must match the undivided
reduction and the oracle."""
import numpy as np
import pytest
import torch

import lattice_inputs as li
import oracle
import paper_1412_3655_b200 as culgt
from gpu_common import GpuField, TOL_LINK, np_dtype, storage_input, theta_close

pytestmark = pytest.mark.gpu

STORES = [(3, 64, 18), (3, 64, 12), (3, 32, 12), (3, 32, 18), (2, 64, 4), (2, 32, 4)]


class SlabbedField:
    """The field of `lat` cut into n_slabs time slabs on the current device."""

    def __init__(self, lat, n_slabs, uc):
        self.lat, self.n = lat, n_slabs
        self.local = culgt.culgt_slab_lattice(lat, n_slabs)
        self.nc = lat.group
        V = lat.volume
        self.v_loc = V // n_slabs
        can = torch.from_numpy(li.to_real(np.ascontiguousarray(uc), np_dtype(lat.precision))).cuda()
        self.slabs = [culgt.alloc_slab_links(self.local) for _ in range(n_slabs)]
        for k, s in enumerate(self.slabs):
            s.fill_(float("nan"))                       # ghost slices start as garbage: the exchange must fill them
            # the canonical field of slab k is a contiguous part of the global one (t is the slowest coordinate)
            culgt.culgt_slab_pack(self.local, can[k * self.v_loc:(k + 1) * self.v_loc], s)
        culgt.culgt_slab_exchange_all_local(self.local, self.slabs)
        self.ws = culgt.alloc_workspace(self.local)
        self.sums = torch.zeros(2 * n_slabs, dtype=torch.float64, device="cuda")
        self.scal = torch.zeros(2, dtype=torch.float64, device="cuda")
        torch.cuda.synchronize()

    def sweep(self, omega, n=1, boundary_first=False):
        culgt.culgt_slab_or_sweeps_local(self.local, self.slabs, n, omega, boundary_first)

    def download(self):
        can = torch.empty((self.lat.volume, 4, self.nc, self.nc, 2), dtype=self.lat.torch_dtype, device="cuda")
        for k, s in enumerate(self.slabs):
            culgt.culgt_slab_unpack(self.local, s, can[k * self.v_loc:(k + 1) * self.v_loc])
        torch.cuda.synchronize()
        return li.from_real(can.cpu().numpy())

    def theta_F(self):
        culgt.culgt_slab_theta_F_local(self.lat, self.local, self.slabs, self.ws, self.sums, self.scal[0:1], self.scal[1:2])
        return tuple(self.scal.cpu().tolist())


@pytest.mark.parametrize("group,precision,params", STORES)
@pytest.mark.parametrize("dims,n_slabs", [((8, 8, 8, 16), 1), ((8, 8, 8, 16), 2), ((8, 8, 8, 16), 4), ((8, 8, 8, 16), 8),
                                         ((4, 6, 2, 8), 2), ((4, 6, 2, 8), 4), ((6, 10, 12, 4), 2)])
def test_slabbed_sweeps_are_bit_identical_and_match_the_oracle(dims, n_slabs, group, precision, params):
    """(8,8,8,16): whole site blocks per time-slice, so boundary_first really sweeps slice windows;
    (4,6,2,8) and (6,10,12,4) do not and take the whole-slab launch; n_slabs = 1 is the periodic lattice
    talking to itself through its ghost slice."""
    omega = 1.7 if group == 3 else 1.5
    u = li.make_config(dims, group, "haar", 77) if group == 2 else \
        li.make_config(dims, group, "near_identity", 77, eps=0.5, scramble=True)
    lat = culgt.Lattice(dims, group, precision, params)
    whole = GpuField(dims, group, precision, params, u)
    ref = storage_input(u, precision, params)
    th_o, F_o = oracle.gauge_precision(dims, ref), oracle.functional(dims, ref)
    outs = {}
    for boundary_first in (False, True):
        f = SlabbedField(lat, n_slabs, u)
        th, F = f.theta_F()
        th_w, F_w = whole.theta_functional() if not outs else (th, F)
        assert abs(th - th_w) <= 1e-12 * th_w and abs(F - F_w) <= 1e-13 * abs(F_w)
        if precision == 64:
            assert theta_close(th, th_o) and abs(F - F_o) <= 1e-10 * abs(F_o)
        else:
            assert abs(th - th_o) <= 1e-9 * th_o and abs(F - F_o) <= 1e-10
        f.sweep(omega, 1, boundary_first)
        if not outs:
            oracle.full_sweep(dims, ref, omega)
        assert np.abs(f.download() - li.from_real(ref)).max() < TOL_LINK[precision]
        f.sweep(omega, 2, boundary_first)
        outs[boundary_first] = (f.download(), f.theta_F())
    whole.sweep(omega, 3)
    want = whole.download()
    th_w, F_w = whole.theta_functional()
    for out, (th, F) in outs.values():
        assert np.array_equal(out, want)
        assert abs(th - th_w) <= 1e-12 * th_w and abs(F - F_w) <= 1e-13 * abs(F_w)
    assert outs[False][1] == outs[True][1]              # per-slab sums in slab order: the same bits again


@pytest.mark.parametrize("name", ["cfg3_fp32", "cfg3_fp64"])
@pytest.mark.parametrize("n_slabs", [2, 8])
def test_slabbed_32x4_is_bit_identical(name, n_slabs):
    """The headline volume cut into 2 and 8 slabs (T = 16 and 4 slices: windows of 128 and 256 site
    blocks, halo messages of 786 KB / 2.36 MB): three full sweeps, all 4V links bit-identical."""
    c = li.CONFIGS[name]
    u = li.make_named(name)
    lat = culgt.Lattice(tuple(c["dims"]), c["group"], c["precision"], c["params"])
    f = SlabbedField(lat, n_slabs, u)
    local = f.local
    assert culgt.culgt_slab_halo_bytes(local) == 32 ** 3 // 2 * (48 if c["precision"] == 32 else 144)
    f.sweep(c["omega"], 3, boundary_first=True)
    got = f.download()
    th, F = f.theta_F()
    del f
    whole = GpuField(c["dims"], c["group"], c["precision"], c["params"], u)
    whole.sweep(c["omega"], 3)
    assert np.array_equal(got, whole.download())
    th_w, F_w = whole.theta_functional()
    assert abs(th - th_w) <= 1e-12 * th_w and abs(F - F_w) <= 1e-13 * abs(F_w)


def test_single_halo_messages_and_windows():
    """The pieces the drivers are made of, one at a time: a FORWARD copy fills exactly the ghost slice,
    window launches over [0,1), [T-1,T), [1,T-1) equal one whole-slab half-sweep."""
    dims, n_slabs = (8, 8, 8, 8), 2
    u = li.make_config(dims, 3, "near_identity", 78, eps=0.5, scramble=True)
    lat = culgt.Lattice(dims, 3, 64, 18)
    a, b = SlabbedField(lat, n_slabs, u), SlabbedField(lat, n_slabs, u)
    T = a.local.dims[3]
    for p in (0, 1):
        for k in range(n_slabs):
            culgt.culgt_slab_or_sweep(a.local, a.slabs[k], p, 1.7)
            for lo, hi in ((0, 1), (T - 1, T), (1, T - 1)):
                culgt.culgt_slab_or_sweep_window(b.local, b.slabs[k], p, 1.7, lo, hi)
        for f in (a, b):
            for k in range(n_slabs):
                culgt.culgt_slab_halo_copy(f.local, f.slabs[k], f.slabs[(k - 1) % n_slabs], 1 - p, 1)
                culgt.culgt_slab_halo_copy(f.local, f.slabs[k], f.slabs[(k + 1) % n_slabs], p, 0)
    torch.cuda.synchronize()
    for k in range(n_slabs):     # (the ghost slices of the spatial planes are never written: still NaN on both sides)
        assert torch.equal(torch.nan_to_num(a.slabs[k]), torch.nan_to_num(b.slabs[k]))
    whole = GpuField(dims, 3, 64, 18, u)
    whole.sweep(1.7, 1)
    assert np.array_equal(a.download(), whole.download())
    # error paths of the window call
    with pytest.raises(culgt.CulgtError):
        culgt.culgt_slab_or_sweep_window(a.local, a.slabs[0], 0, 1.7, 2, 1)
    with pytest.raises(culgt.CulgtError):
        culgt.culgt_slab_or_sweep_window(a.local, a.slabs[0], 0, 1.7, 0, T + 1)


@pytest.mark.parametrize("overlap", [False, True])
@pytest.mark.parametrize("precision,params", [(64, 18), (32, 12)])
def test_nccl_transport_with_one_rank(precision, params, overlap):
    """The one-slab-per-rank drivers (ncclSend / ncclRecv halo messages, all-gathered theta/F sums) with
    a communicator of ONE rank: every message is a send to self matched by a receive from self, i.e.
    the periodic lattice talking to itself through its ghost slice over the real NCCL code path.
    Three sweeps must be bit-identical to the undivided sweep, without and with the boundary-first
    schedule whose messages travel on a second stream.  (More ranks need more GPUs than this box has;
    the rank bookkeeping is covered by tests/test_slab_bookkeeping.py.)"""
    dims = (8, 8, 8, 8)
    u = li.make_config(dims, 3, "near_identity", 79, eps=0.5, scramble=True)
    lat = culgt.Lattice(dims, 3, precision, params)
    local = culgt.culgt_slab_lattice(lat, 1)
    comm = culgt.culgt_slab_comm_create(culgt.culgt_slab_comm_unique_id(), 0, 1)
    try:
        can = torch.from_numpy(li.to_real(np.ascontiguousarray(u), np_dtype(precision))).cuda()
        links = culgt.alloc_slab_links(local)
        links.fill_(float("nan"))
        culgt.culgt_slab_pack(local, can, links)
        culgt.culgt_slab_exchange_all_nccl(comm, local, links)
        ws = culgt.alloc_workspace(local)
        sums = torch.zeros(4, dtype=torch.float64, device="cuda")
        scal = torch.zeros(2, dtype=torch.float64, device="cuda")
        side = torch.cuda.Stream() if overlap else None
        culgt.culgt_slab_or_sweeps_nccl(comm, local, links, 3, 1.7, side)
        culgt.culgt_slab_theta_F_nccl(comm, lat, local, links, ws, sums, scal[0:1], scal[1:2])
        culgt.culgt_slab_unpack(local, links, can)
        torch.cuda.synchronize()
        got = li.from_real(can.cpu().numpy())
        th, F = scal.cpu().tolist()
    finally:
        culgt.culgt_slab_comm_destroy(comm)
    whole = GpuField(dims, 3, precision, params, u)
    whole.sweep(1.7, 3)
    assert np.array_equal(got, whole.download())
    th_w, F_w = whole.theta_functional()
    assert abs(th - th_w) <= 1e-12 * th_w and abs(F - F_w) <= 1e-13 * abs(F_w)
