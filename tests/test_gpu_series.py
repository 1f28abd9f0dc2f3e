"""GPU parity for the truncated-series overrelaxation (SURVEY.md 8(f) NEXT-2b; DESIGN.md reading
C-24) against the oracle's literal matrix-power implementation, through the C ABI."""
import numpy as np
import pytest

import lattice_inputs as li
import oracle
import paper_1412_3655_b200 as culgt
from gpu_common import GpuField, TOL_LINK, storage_input, theta_close

pytestmark = pytest.mark.gpu

STORES = [(3, 64, 18), (3, 64, 12), (3, 32, 12), (3, 32, 18), (2, 64, 4), (2, 32, 4)]


@pytest.mark.parametrize("dims", [(4, 4, 4, 4), (4, 6, 2, 8), (6, 10, 12, 4), (8, 8, 8, 8)])
@pytest.mark.parametrize("group,precision,params", STORES)
@pytest.mark.parametrize("order", [1, 4, 9])
def test_links_after_each_half_sweep(dims, group, precision, params, order):
    u = li.make_config(dims, group, "near_identity", 101, eps=0.5, scramble=True) if group == 3 \
        else li.make_config(dims, group, "haar", 101)
    ref = storage_input(u, precision, params)
    f = GpuField(dims, group, precision, params, u)
    for parity in (0, 1):
        oracle.or_sweep_series(dims, ref, parity, 1.7, order)
        culgt.culgt_or_sweep_series(f.lat, f.links, parity, 1.7, order)
        err = np.abs(f.download() - li.from_real(ref)).max()
        assert err < TOL_LINK[precision], (parity, err)


def test_trajectory_fp64_and_headline_size():
    dims = (8, 8, 8, 8)
    u = li.make_config(dims, 3, "near_identity", 102, eps=0.3, scramble=True)
    ref = storage_input(u, 64, 18)
    f = GpuField(dims, 3, 64, 18, u)
    for s in range(1, 41):
        oracle.full_sweep_series(dims, ref, 1.7, 4)
        culgt.culgt_or_sweeps_series(f.lat, f.links, 1, 1.7, 4)
        if s % 5 == 0:
            assert theta_close(f.theta(), oracle.gauge_precision(dims, ref)), s
            F_o = oracle.functional(dims, ref)
            assert abs(f.functional() - F_o) <= 1e-10 * abs(F_o), s
    c = li.CONFIGS["cfg3_fp32"]
    u = li.make_named("cfg3_fp32")
    ref = storage_input(u, 32, 12)
    f = GpuField(c["dims"], 3, 32, 12, u)
    del u
    oracle.set_threads(16)
    try:
        oracle.full_sweep_series(c["dims"], ref, 1.7, 4)
    finally:
        oracle.set_threads(1)
    culgt.culgt_or_sweeps_series(f.lat, f.links, 1, 1.7, 4)
    assert np.abs(f.download() - li.from_real(ref)).max() < TOL_LINK[32]


def test_argument_errors():
    lat = culgt.Lattice((4, 4, 4, 4), 3, 64, 18)
    links = culgt.alloc_links(lat)
    for bad in (-1, 17):
        with pytest.raises(culgt.CulgtError) as e:
            culgt.culgt_or_sweep_series(lat, links, 0, 1.7, bad)
        assert e.value.status == culgt.ERRORS["CULGT_ERR_ARG"]
