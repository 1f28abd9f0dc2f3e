"""GPU parity for the Coulomb-gauge variant (reading C-22): the
half-sweep with K(x) from the spatial links only, and the per-time-slice theta_t / F_t, against
the oracle on the same seeded inputs, through the C ABI."""
import numpy as np
import pytest
import torch

import lattice_inputs as li
import oracle
import paper_1412_3655_b200 as culgt
from gpu_common import GpuField, TOL_LINK, storage_input, theta_close

pytestmark = pytest.mark.gpu

STORES = [(3, 64, 18), (3, 64, 12), (3, 32, 12), (3, 32, 18), (2, 64, 4), (2, 32, 4)]
DIMS = [(4, 4, 4, 4), (4, 6, 2, 8), (6, 10, 12, 4), (8, 8, 8, 8), (2, 2, 2, 2), (12, 2, 6, 10)]


def theta_F_gpu(f):
    n3 = f.lat.dims[3]
    out = torch.zeros(2 * n3, dtype=torch.float64, device="cuda")
    culgt.culgt_coulomb_precision_functional(f.lat, f.links, f.ws, out[:n3], out[n3:])
    r = out.cpu().numpy()
    return r[:n3], r[n3:]


def close_slices(th, th_o, F, F_o, precision):
    if precision == 64:
        return all(theta_close(a, b) for a, b in zip(th, th_o)) and np.all(np.abs(F - F_o) <= 1e-10 * np.abs(F_o) + 1e-15)
    return np.all(np.abs(th - th_o) <= 1e-9 * th_o + 1e-30) and np.all(np.abs(F - F_o) <= 1e-10)


@pytest.mark.parametrize("dims", DIMS)
@pytest.mark.parametrize("group,precision,params", STORES)
def test_links_theta_F_after_each_half_sweep(dims, group, precision, params):
    u = li.make_config(dims, group, "near_identity", 81, eps=0.5, scramble=True) if group == 3 \
        else li.make_config(dims, group, "haar", 81)
    omega = 1.7 if group == 3 else 1.5
    ref = storage_input(u, precision, params)
    f = GpuField(dims, group, precision, params, u)
    th, F = theta_F_gpu(f)
    th_o, F_o = oracle.coulomb_theta_F(dims, ref)
    assert close_slices(th, th_o, F, F_o, precision)
    for parity in (0, 1):
        oracle.or_sweep_coulomb(dims, ref, parity, omega)
        culgt.culgt_or_sweep_coulomb(f.lat, f.links, parity, omega)
        err = np.abs(f.download() - li.from_real(ref)).max()
        assert err < TOL_LINK[precision], (parity, err)
    th, F = theta_F_gpu(f)
    th_o, F_o = oracle.coulomb_theta_F(dims, ref)
    if precision == 64:
        assert close_slices(th, th_o, F, F_o, 64)
    else:
        assert np.all(np.abs(th - th_o) <= 1e-3 * th_o) and np.all(np.abs(F - F_o) <= 2e-6)
    assert theta_F_gpu(f)[0].tolist() == th.tolist()          # deterministic


def test_trajectory_and_driver_fp64():
    """8^4 SU(3) fp64: (theta_t, F_t) of every slice after every sweep, then the driver loop to
    max_t theta_t < 1e-20 against the oracle's own stop sweep."""
    dims = (8, 8, 8, 8)
    u = li.make_config(dims, 3, "near_identity", 82, eps=0.3, scramble=True)
    ref = storage_input(u, 64, 18)
    f = GpuField(dims, 3, 64, 18, u)
    for s in range(1, 31):
        oracle.full_sweep_coulomb(dims, ref, 1.7)
        culgt.culgt_or_sweeps_coulomb(f.lat, f.links, 1, 1.7)
        th, F = theta_F_gpu(f)
        th_o, F_o = oracle.coulomb_theta_F(dims, ref)
        assert close_slices(th, th_o, F, F_o, 64), s
    stop_o = 30
    while oracle.coulomb_theta_F(dims, ref)[0].max() >= 1e-20 and stop_o < 3000:
        oracle.full_sweep_coulomb(dims, ref, 1.7)
        stop_o += 1
    done, th, F = culgt.culgt_coulomb_fix(f.lat, f.links, f.ws, 1.7, 1e-20, 3000, 1)
    assert abs(30 + done - stop_o) <= 1 and max(th) < 1e-20
    assert np.abs(np.array(F) - oracle.coulomb_theta_F(dims, ref)[1]).max() < 1e-10
    back = f.download()
    assert np.abs(back @ np.conj(np.swapaxes(back, -1, -2)) - np.eye(3)).max() < 1e-13


@pytest.mark.parametrize("name", ["cfg3_fp32", "cfg3_fp64"])
def test_headline_size_links_after_one_sweep(name):
    """32^4 in the launch configuration bench.py --gauge coulomb times."""
    c = li.CONFIGS[name]
    dims, prec = c["dims"], c["precision"]
    u = li.make_named(name)
    ref = storage_input(u, prec, c["params"])
    f = GpuField(dims, 3, prec, c["params"], u)
    del u
    oracle.set_threads(16)
    try:
        oracle.full_sweep_coulomb(dims, ref, c["omega"])
        culgt.culgt_or_sweeps_coulomb(f.lat, f.links, 1, c["omega"])
        err = np.abs(f.download() - li.from_real(ref)).max()
        assert err < TOL_LINK[prec], err
        th, F = theta_F_gpu(f)
        th_o, F_o = oracle.coulomb_theta_F(dims, ref)
    finally:
        oracle.set_threads(1)
    if prec == 64:
        assert close_slices(th, th_o, F, F_o, 64)
    else:
        assert np.all(np.abs(th - th_o) <= 1e-3 * th_o) and np.all(np.abs(F - F_o) <= 2e-6)


def test_masked_sweep_and_per_slice_stopping():
    """Frozen slices keep their spatial links, active ones are swept exactly as by the oracle; the
    driver stops every slice at ITS theta_t like the same rule applied to
    the oracle."""
    dims = (6, 4, 4, 8)
    u = li.make_config(dims, 3, "near_identity", 83, eps=0.3, scramble=True)
    ref = storage_input(u, 64, 18)
    f = GpuField(dims, 3, 64, 18, u)
    active = np.array([1, 0, 1, 1, 0, 0, 1, 0], dtype=np.uint8)
    mask = torch.from_numpy(active).cuda()
    for parity in (0, 1):
        oracle.or_sweep_coulomb_masked(dims, ref, parity, 1.7, active)
        culgt.culgt_or_sweep_coulomb_masked(f.lat, f.links, parity, 1.7, mask)
    assert np.abs(f.download() - li.from_real(ref)).max() < TOL_LINK[64]
    # per-slice stopping, theta checked after every sweep
    target = 1e-16
    ref = storage_input(u, 64, 18)
    stop_o = np.zeros(dims[3], dtype=int)
    n = 0
    while True:
        th_o, F_o = oracle.coulomb_theta_F(dims, ref)
        act = (~(th_o < target)).astype(np.uint8)
        if act.sum() == 0 or n >= 3000:
            break
        for parity in (0, 1):
            oracle.or_sweep_coulomb_masked(dims, ref, parity, 1.7, act)
        n += 1
        stop_o[act == 1] = n
    f = GpuField(dims, 3, 64, 18, u)
    done, th, F = culgt.culgt_coulomb_fix(f.lat, f.links, f.ws, 1.7, target, 3000, 1)
    assert abs(done - n) <= 1 and max(th) < target
    assert len(set(stop_o)) > 1                              # the slices really stop at different sweeps
    assert np.abs(np.array(F) - F_o).max() < 1e-9
    assert np.abs(f.download() - li.from_real(ref)).max() < 1e-6   # same copy reached (a +-1 sweep near the target moves links by ~sqrt(target))


def test_argument_errors():
    lat = culgt.Lattice((4, 4, 4, 4), 3, 64, 18)
    links = culgt.alloc_links(lat)
    with pytest.raises(culgt.CulgtError) as e:
        culgt.culgt_or_sweep_coulomb(lat, links, 2, 1.7)
    assert e.value.status == culgt.ERRORS["CULGT_ERR_PARITY"]
    with pytest.raises(culgt.CulgtError) as e:
        culgt.culgt_or_sweep_coulomb(lat, links, 0, 2.0)
    assert e.value.status == culgt.ERRORS["CULGT_ERR_OMEGA"]
