"""GPU parity for culgt_reunitarize (reading C-23) against the oracle, and its use in a
long fp32 run: the stored rows drift off SU(3) (reading C-13), one call removes the drift."""
import numpy as np
import pytest
import torch

import lattice_inputs as li
import oracle
import paper_1412_3655_b200 as culgt
from gpu_common import GpuField

pytestmark = pytest.mark.gpu

STORES = [(3, 64, 18), (3, 64, 12), (3, 32, 12), (3, 32, 18), (2, 64, 4), (2, 32, 4)]


@pytest.mark.parametrize("dims", [(4, 4, 4, 4), (4, 6, 2, 8), (6, 10, 12, 4)])
@pytest.mark.parametrize("group,precision,params", STORES)
def test_matches_oracle_on_a_drifted_field(dims, group, precision, params):
    u = li.make_config(dims, group, "haar", 95)
    rng = np.random.default_rng(96)
    u = u + 1e-3 * (rng.standard_normal(u.shape) + 1j * rng.standard_normal(u.shape))
    if group == 2:   # keep the 4-parameter form: second row = (-conj(b), conj(a))
        u[..., 1, 0] = -np.conj(u[..., 0, 1])
        u[..., 1, 1] = np.conj(u[..., 0, 0])
    f = GpuField(dims, group, precision, params, u)
    stored = f.download()                        # what the storage really holds (rounded, row 2 rebuilt)
    ref = li.to_real(np.ascontiguousarray(stored))
    oracle.reunitarize(ref)
    culgt.culgt_reunitarize(f.lat, f.links)
    got = f.download()
    tol = 1e-14 if precision == 64 else 3e-7
    assert np.abs(got - li.from_real(ref)).max() < tol
    assert np.abs(got @ np.conj(np.swapaxes(got, -1, -2)) - np.eye(group)).max() < (1e-14 if precision == 64 else 5e-7)
    # idempotent to rounding
    culgt.culgt_reunitarize(f.lat, f.links)
    assert np.abs(f.download() - got).max() < (1e-15 if precision == 64 else 2e-7)


def test_long_fp32_run_drift_is_removed():
    """16^4 fp32-12, 600 sweeps: rows 0,1 drift (unitarity error grows), culgt_reunitarize brings the
    field back onto SU(3) without disturbing the gauge fixing (F unchanged to 1e-6)."""
    c = li.CONFIGS["cfg2"]
    f = GpuField(c["dims"], 3, 32, 12, li.make_named("cfg2"))
    f.sweep(c["omega"], 600)

    def unitarity():
        g = f.download()
        return np.abs(g @ np.conj(np.swapaxes(g, -1, -2)) - np.eye(3)).max()

    before, F0 = unitarity(), f.functional()
    culgt.culgt_reunitarize(f.lat, f.links)
    after, F1 = unitarity(), f.functional()
    assert after < 5e-7 and after <= before
    assert abs(F1 - F0) < 1e-6
    assert before < 1e-3          # the drift itself is slow (C-13) -- this records its size
    print(f"unitarity error after 600 fp32 sweeps: {before:.2e} -> {after:.2e}")
