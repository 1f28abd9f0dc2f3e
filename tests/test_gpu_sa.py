"""GPU parity for simulated annealing (reading C-25): the same
counter-based random numbers on both sides, so the sampled sweep must reproduce the oracle's field
link by link."""
import numpy as np
import pytest

import lattice_inputs as li
import oracle
import paper_1412_3655_b200 as culgt
from gpu_common import GpuField, TOL_LINK, storage_input

pytestmark = pytest.mark.gpu

STORES = [(3, 64, 18), (3, 64, 12), (3, 32, 12), (3, 32, 18), (2, 64, 4), (2, 32, 4)]


@pytest.mark.parametrize("dims", [(4, 4, 4, 4), (4, 6, 2, 8), (6, 10, 12, 4), (8, 8, 8, 8)])
@pytest.mark.parametrize("group,precision,params", STORES)
@pytest.mark.parametrize("T", [3.0, 0.3, 0.01])
def test_links_after_each_half_sweep(dims, group, precision, params, T):
    u = li.make_config(dims, group, "haar", 111)
    ref = storage_input(u, precision, params)
    f = GpuField(dims, group, precision, params, u)
    for n in range(4):
        if precision == 32 and n > 0:
            # fp32 storage: the two fields differ by product rounding (~1e-7) after a half-sweep, and
            # an accept/reject decision of the heat bath within that margin would legitimately flip
            # (then the site draws a different sample).  Every half-sweep is therefore compared from
            # a COMMON stored state: the oracle restarts from what the GPU storage holds.
            ref = li.to_real(np.ascontiguousarray(f.download()))
        oracle.sa_sweep(dims, ref, n & 1, T, 2024, n)
        culgt.culgt_sa_sweep(f.lat, f.links, n & 1, T, 2024, n)
        err = np.abs(f.download() - li.from_real(ref)).max()
        assert err < TOL_LINK[precision], (n, err)


def test_anneal_schedule_and_overrelax_reaches_the_maximum():
    """culgt_sa_anneal runs the schedule T_i = T_max - (T_max - T_min) i/(n-1) with half-sweep counters
    0, 1, 2, ...: checked link by link against the oracle over the first sweeps (rounding differences
    grow along a sampled trajectory, so parity is a short-horizon statement, reading C-14), then the
    annealed pure-gauge field is overrelaxed to F = 1."""
    dims = (8, 8, 8, 8)
    u = li.make_config(dims, 3, "pure_gauge", 7)
    n_sweeps, T_max, T_min = 30, 2.0, 0.02
    ref = storage_input(u, 64, 18)
    g = GpuField(dims, 3, 64, 18, u)
    for i in range(3):
        T = T_max - (T_max - T_min) * i / (n_sweeps - 1)
        for parity in (0, 1):
            oracle.sa_sweep(dims, ref, parity, T, 5, 2 * i + parity)
            culgt.culgt_sa_sweep(g.lat, g.links, parity, T, 5, 2 * i + parity)
    assert np.abs(g.download() - li.from_real(ref)).max() < 1e-10
    # the driver's first three sweeps are exactly those calls
    f = GpuField(dims, 3, 64, 18, u)
    culgt.culgt_sa_anneal(f.lat, f.links, T_max, T_max - (T_max - T_min) * 2 / (n_sweeps - 1), 3, 5)
    assert np.array_equal(f.download(), g.download())
    f = GpuField(dims, 3, 64, 18, u)
    culgt.culgt_sa_anneal(f.lat, f.links, T_max, T_min, n_sweeps, 5)
    back = f.download()
    assert np.abs(back @ np.conj(np.swapaxes(back, -1, -2)) - np.eye(3)).max() < 1e-13
    done, theta, F = culgt.culgt_landau_fix(f.lat, f.links, f.ws, 1.7, 1e-22, 3000, 10)
    assert theta < 1e-22 and F > 0.999999


@pytest.mark.parametrize("name", ["cfg3_fp32", "cfg3_fp64"])
def test_headline_size_one_sweep(name):
    """32^4 in the launch configuration `bench.py --sa-temperature` times: all 4V links after a black and
    a white annealing half-sweep at T = 0.5, each from a common stored state."""
    c = li.CONFIGS[name]
    dims, prec = c["dims"], c["precision"]
    u = li.make_named(name)
    f = GpuField(dims, 3, prec, c["params"], u)
    del u
    oracle.set_threads(16)
    try:
        for n in range(2):
            ref = li.to_real(np.ascontiguousarray(f.download()))
            oracle.sa_sweep(dims, ref, n, 0.5, 31, n)
            culgt.culgt_sa_sweep(f.lat, f.links, n, 0.5, 31, n)
            err = np.abs(f.download() - li.from_real(ref)).max()
            assert err < TOL_LINK[prec], (n, err)
    finally:
        oracle.set_threads(1)


def test_argument_errors():
    lat = culgt.Lattice((4, 4, 4, 4), 3, 64, 18)
    links = culgt.alloc_links(lat)
    for T in (0.0, -1.0, float("nan")):
        with pytest.raises(culgt.CulgtError) as e:
            culgt.culgt_sa_sweep(lat, links, 0, T, 1, 0)
        assert e.value.status == culgt.ERRORS["CULGT_ERR_ARG"]
    with pytest.raises(culgt.CulgtError) as e:
        culgt.culgt_sa_anneal(lat, links, 0.1, 1.0, 10, 1)          # T_max < T_min
    assert e.value.status == culgt.ERRORS["CULGT_ERR_ARG"]
