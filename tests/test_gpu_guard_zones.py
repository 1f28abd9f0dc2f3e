"""Out-of-bounds WRITE detection without compute-sanitizer (which is closed on this GPU pool): the
internal field sits between two guard zones filled with a sentinel; after every kernel of the path
has run on ragged, asymmetric lattices, for every sweep mapping, the guard zones must be intact
and the workspace must not be written past its declared size."""
import numpy as np
import pytest
import torch

import lattice_inputs as li
import paper_1412_3655_b200 as culgt
from test_gpu_parity_small import variants_for

pytestmark = pytest.mark.gpu

GUARD = 1 << 16          # elements on each side
SENT = 12345.678


def guarded(n, dtype):
    buf = torch.full((n + 2 * GUARD,), SENT, dtype=dtype, device="cuda")
    return buf, buf[GUARD:GUARD + n]


def intact(buf, n):
    return bool((buf[:GUARD] == SENT).all()) and bool((buf[GUARD + n:] == SENT).all())


@pytest.mark.parametrize("dims", [(4, 6, 2, 8), (6, 10, 12, 4), (2, 2, 2, 2), (12, 2, 6, 10)])
@pytest.mark.parametrize("group,precision,params", [(3, 64, 18), (3, 64, 12), (3, 32, 12), (3, 32, 18),
                                                    (2, 64, 4), (2, 32, 4)])
def test_guard_zones_survive_every_kernel(dims, group, precision, params):
    lat = culgt.Lattice(dims, group, precision, params)
    dt = lat.torch_dtype
    n_links = culgt.culgt_links_bytes(lat) // (precision // 8)
    n_can = culgt.culgt_canonical_bytes(lat) // (precision // 8)
    n_ws = culgt.culgt_workspace_bytes(lat) // 8
    lbuf, links = guarded(n_links, dt)
    cbuf, can = guarded(n_can, dt)
    wbuf, ws = guarded(n_ws, torch.float64)
    sbuf, scal = guarded(2 * dims[3], torch.float64)
    u = li.make_config(dims, group, "haar", 121)
    can.copy_(torch.from_numpy(li.to_real(u, np.float32 if precision == 32 else np.float64)).reshape(-1).cuda())
    culgt.culgt_pack(lat, can, links)
    variants = variants_for(precision, params) if group == 3 else [0]
    try:
        for v in variants:
            culgt.culgt_set_sweep_variant(v)
            culgt.culgt_or_sweeps(lat, links, 1, 1.7)
    finally:
        culgt.culgt_set_sweep_variant(0)
    culgt.culgt_or_sweeps_coulomb(lat, links, 1, 1.7)
    culgt.culgt_or_sweeps_series(lat, links, 1, 1.7, 4)
    culgt.culgt_sa_anneal(lat, links, 1.0, 0.1, 2, 9)
    culgt.culgt_sa_anneal_micro(lat, links, 1.0, 0.1, 2, 1, 9)
    culgt.culgt_micro_sweeps(lat, links, 1)
    culgt.culgt_reunitarize(lat, links)
    culgt.culgt_gauge_precision(lat, links, ws, scal[0:1])
    culgt.culgt_functional(lat, links, ws, scal[1:2])
    culgt.culgt_gauge_precision_functional(lat, links, ws, scal[0:1], scal[1:2])
    culgt.culgt_coulomb_precision_functional(lat, links, ws, scal[:dims[3]], scal[dims[3]:])
    culgt.culgt_landau_fix(lat, links, ws, 1.7, 1e-30, 3, 1)
    culgt.culgt_coulomb_fix(lat, links, ws, 1.7, 1e-30, 3, 1)
    g = li.haar_su3(li.volume(dims), 5) if group == 3 else li.haar_su2(li.volume(dims), 5)
    gt = torch.from_numpy(li.to_real(g, np.float32 if precision == 32 else np.float64)).cuda()
    culgt.culgt_gauge_transform(lat, links, gt)
    culgt.culgt_unpack(lat, links, can)
    torch.cuda.synchronize()
    assert intact(lbuf, n_links), "links"
    assert intact(cbuf, n_can), "canonical"
    assert intact(wbuf, n_ws), "workspace"
    assert intact(sbuf, 2 * dims[3]), "scalars"
    assert bool(torch.isfinite(links).all())
