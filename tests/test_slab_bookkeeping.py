"""Host-side logic of the time-slab decomposition (include/culgt_b200.h "Time-slab decomposition",
csrc/slab.cu), on CPU: slab descriptors and sizes, which byte ranges of a slab form a halo message,
which ranks exchange them -- checked against an independent numpy model of the parity-split
layout, in process for 1..8 slabs (wrap between the last and the first slab) and with two gloo
ranks that really send and receive the messages the library describes.  No GPU involved: the
"field" is an array of labels, one per 16-byte vector."""
import os
import socket
import sys

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import paper_1412_3655_b200 as culgt  # noqa: E402

NV = {(3, 32, 12): 3, (3, 32, 18): 5, (3, 64, 12): 6, (3, 64, 18): 9, (2, 32, 4): 1, (2, 64, 4): 2}


def global_labels(lat):
    """labels[parity][mu][j][h]: a distinct number for every 16-byte vector of the global internal field
    (h = canonical site >> 1; time-slice t is h in [t*stride3, (t+1)*stride3))."""
    n0, n1, n2, n3 = lat.dims
    vh = n0 * n1 * n2 * n3 // 2
    nv = NV[(lat.group, lat.precision, lat.params)]
    return np.arange(2 * 4 * nv * vh, dtype=np.int64).reshape(2, 4, nv, vh), nv, vh, n0 * n1 * n2 // 2


def slab_of(labels, local_lat, k, nv, stride3):
    """Slab k as the library lays it out: [parity][mu][j][pitch] with pitch = vh_loc + stride3 (ghost
    slice, here -1 = not yet received), as a flat array of one label per 16-byte vector."""
    T = local_lat.dims[3]
    vh_loc = stride3 * T
    out = np.full((2, 4, nv, vh_loc + stride3), -1, dtype=np.int64)
    out[..., :vh_loc] = labels[..., k * vh_loc:(k + 1) * vh_loc]
    return out.reshape(-1)


def chunks(local, parity, which):
    off, nbytes = culgt.culgt_slab_halo_chunks(local, parity, which)
    assert all(o % 16 == 0 for o in off) and nbytes % 16 == 0
    return [o // 16 for o in off], nbytes // 16


@pytest.mark.parametrize("desc", sorted(NV))
@pytest.mark.parametrize("dims,n_slabs", [((8, 8, 8, 16), 1), ((8, 8, 8, 16), 2), ((8, 8, 8, 16), 4), ((8, 8, 8, 16), 8),
                                         ((4, 6, 2, 8), 2), ((6, 10, 12, 4), 2), ((32, 32, 32, 32), 8)])
def test_descriptor_sizes_and_halo_ranges(desc, dims, n_slabs):
    group, precision, params = desc
    lat = culgt.Lattice(dims, group, precision, params)
    local = culgt.culgt_slab_lattice(lat, n_slabs)
    assert local.dims == (dims[0], dims[1], dims[2], dims[3] // n_slabs)
    nv = NV[desc]
    stride3 = dims[0] * dims[1] * dims[2] // 2
    vh_loc = stride3 * local.dims[3]
    assert culgt.culgt_slab_links_bytes(local) == 8 * nv * (vh_loc + stride3) * 16
    # one message = the t-links of one parity in one time-slice: N0 N1 N2 / 2 links
    link_bytes = nv * 16
    assert culgt.culgt_slab_halo_bytes(local) == stride3 * link_bytes
    for parity in (0, 1):
        for which in (0, 1):
            off, n = chunks(local, parity, which)
            assert n == stride3 and len(off) == nv
            for j, o in enumerate(off):
                plane = ((parity * 4 + 3) * nv + j) * (vh_loc + stride3)     # mu = 3: the t-links
                assert o == plane + (vh_loc if which == 0 else vh_loc - stride3)


def test_slab_lattice_errors():
    E = culgt.ERRORS
    lib = culgt.lib()
    import ctypes
    out = culgt.culgt_lattice()
    L = culgt.Lattice((8, 8, 8, 12), 3, 32, 12).c()
    for n, code in ((0, "CULGT_ERR_ARG"), (5, "CULGT_ERR_ARG"), (4, "CULGT_ERR_ARG"),     # 12/4 = 3 slices: odd
                    (12, "CULGT_ERR_ARG"), (-1, "CULGT_ERR_ARG")):
        assert lib.culgt_slab_lattice(ctypes.byref(L), n, ctypes.byref(out)) == E[code], n
    assert lib.culgt_slab_lattice(ctypes.byref(L), 2, None) == E["CULGT_ERR_NULL"]
    for n in (1, 2, 3, 6):
        assert lib.culgt_slab_lattice(ctypes.byref(L), n, ctypes.byref(out)) == 0 and out.dims[3] == 12 // n
    bad = culgt.Lattice((8, 8, 7, 12), 3, 32, 12).c()
    assert lib.culgt_slab_lattice(ctypes.byref(bad), 2, ctypes.byref(out)) == E["CULGT_ERR_DIMS"]
    assert culgt.culgt_slab_halo_peers(0, 4, 0) == (1, 3) and culgt.culgt_slab_halo_peers(0, 4, 1) == (3, 1)
    assert culgt.culgt_slab_halo_peers(3, 4, 0) == (0, 2) and culgt.culgt_slab_halo_peers(3, 4, 1) == (2, 0)
    assert culgt.culgt_slab_halo_peers(0, 1, 0) == (0, 0)


def exchange_in_process(slabs, local, parity, direction):
    """What one round of halo messages does, with the library's ranges and peers, on label arrays."""
    n = len(slabs)
    send_which, recv_which = (1, 0) if direction == 0 else (0, 1)
    s_off, m = chunks(local, parity, send_which)
    r_off, _ = chunks(local, parity, recv_which)
    msgs = [[slabs[k][o:o + m].copy() for o in s_off] for k in range(n)]
    for k in range(n):
        send_to, _ = culgt.culgt_slab_halo_peers(k, n, direction)
        for j, o in enumerate(r_off):
            slabs[send_to][o:o + m] = msgs[k][j]


@pytest.mark.parametrize("n_slabs", [1, 2, 4, 8])
@pytest.mark.parametrize("desc", [(3, 32, 12), (3, 64, 18), (2, 64, 4)])
def test_forward_and_back_messages_in_process(n_slabs, desc):
    """FORWARD fills every ghost slice with the previous slab's last-slice t-links (slab 0's from the
    LAST slab: the periodic wrap); BACK returns modified ghost links to exactly those places."""
    group, precision, params = desc
    lat = culgt.Lattice((4, 4, 6, 16), group, precision, params)
    local = culgt.culgt_slab_lattice(lat, n_slabs)
    labels, nv, vh, stride3 = global_labels(lat)
    T = local.dims[3]
    vh_loc = stride3 * T
    slabs = [slab_of(labels, local, k, nv, stride3) for k in range(n_slabs)]
    for parity in (0, 1):
        exchange_in_process(slabs, local, parity, 0)
    for k in range(n_slabs):
        s = slabs[k].reshape(2, 4, nv, vh_loc + stride3)
        t_prev = (k * T - 1) % lat.dims[3]                   # the global time-slice in front of slab k
        assert np.array_equal(s[:, 3, :, vh_loc:], labels[:, 3, :, t_prev * stride3:(t_prev + 1) * stride3])
        assert np.all(s[:, :3, :, vh_loc:] == -1)            # only t-links travel
        assert np.array_equal(s[..., :vh_loc], labels[..., k * vh_loc:(k + 1) * vh_loc])
    # the half-sweep of parity p rewrites the ghost t-links of parity 1-p; they go BACK to their owner
    p = 0
    for k in range(n_slabs):
        s = slabs[k].reshape(2, 4, nv, vh_loc + stride3)
        s[1 - p, 3, :, vh_loc:] += 10 ** 12
    exchange_in_process(slabs, local, 1 - p, 1)
    for k in range(n_slabs):
        s = slabs[k].reshape(2, 4, nv, vh_loc + stride3)
        want = labels[..., k * vh_loc:(k + 1) * vh_loc].copy()
        want[1 - p, 3, :, vh_loc - stride3:] += 10 ** 12     # my last slice's t-links of parity 1-p, and nothing else
        assert np.array_equal(s[..., :vh_loc], want)


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    port = s.getsockname()[1]
    s.close()
    return port


def _gloo_exchange(buf, local, parity, direction, rank, world):
    """The message pattern of culgt_slab_halo_exchange (csrc/slab.cu) with gloo send/recv in place of
    ncclSend/ncclRecv: same ranges, same peers, all chunks of one message back to back."""
    send_which, recv_which = (1, 0) if direction == 0 else (0, 1)
    s_off, m = chunks(local, parity, send_which)
    r_off, _ = chunks(local, parity, recv_which)
    send_to, recv_from = culgt.culgt_slab_halo_peers(rank, world, direction)
    ops = []
    for so, ro in zip(s_off, r_off):
        ops.append(dist.P2POp(dist.isend, buf[so:so + m].clone(), send_to))
        ops.append(dist.P2POp(dist.irecv, buf[ro:ro + m], recv_from))
    for req in dist.batch_isend_irecv(ops):
        req.wait()


def _worker(rank, world, port, out):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        lat = culgt.Lattice((4, 6, 2, 8), 3, 64, 18)
        local = culgt.culgt_slab_lattice(lat, world)
        labels, nv, vh, stride3 = global_labels(lat)
        T = local.dims[3]
        vh_loc = stride3 * T
        buf = torch.from_numpy(slab_of(labels, local, rank, nv, stride3))
        for parity in (0, 1):                                   # culgt_slab_exchange_all_nccl
            _gloo_exchange(buf, local, parity, 0, rank, world)
        s = buf.numpy().reshape(2, 4, nv, vh_loc + stride3)
        t_prev = (rank * T - 1) % lat.dims[3]
        ok_fwd = np.array_equal(s[:, 3, :, vh_loc:], labels[:, 3, :, t_prev * stride3:(t_prev + 1) * stride3])
        s[1, 3, :, vh_loc:] += 10 ** 12                         # half-sweep of parity 0 rewrote them
        _gloo_exchange(buf, local, 1, 1, rank, world)           # BACK, parity 1
        want = labels[..., rank * vh_loc:(rank + 1) * vh_loc].copy()
        want[1, 3, :, vh_loc - stride3:] += 10 ** 12
        ok_back = np.array_equal(buf.numpy().reshape(2, 4, nv, vh_loc + stride3)[..., :vh_loc], want)
        # theta / F: raw sums of every rank gathered in rank order, the same on every rank
        mine = torch.tensor([1.5 + rank, 10.0 * (rank + 1)], dtype=torch.float64)
        gathered = [torch.zeros(2, dtype=torch.float64) for _ in range(world)]
        dist.all_gather(gathered, mine)
        out[rank] = (bool(ok_fwd), bool(ok_back), [g.tolist() for g in gathered])
    finally:
        dist.destroy_process_group()


def test_two_gloo_ranks_exchange_the_halo_messages():
    world = 2
    with mp.Manager() as m:
        out = m.dict()
        mp.spawn(_worker, args=(world, _free_port(), out), nprocs=world, join=True)
        res = dict(out)
    assert res[0][:2] == (True, True) and res[1][:2] == (True, True)
    assert res[0][2] == res[1][2] == [[1.5, 10.0], [2.5, 20.0]]
