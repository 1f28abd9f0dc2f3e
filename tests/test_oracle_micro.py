"""Pins for the oracle's microcanonical step (reading C-26; SURVEY.md 8(f) NEXT-3
"simulated annealing + microcanonical steps"): the per-subgroup reflection q = g^2 must leave the
local functional Re tr[G K] (hence F) unchanged while moving the links, is the exact omega = 2 power
(pinned separately), reduces for SU(2) to the textbook reflection G K = K^dagger (an involution), and
is a gauge transformation.  CPU only."""
import numpy as np
import pytest

import lattice_inputs as li
import oracle
from helpers import K_numpy, cplx, dag, real


def _to_c(m):
    return m[..., 0] + 1j * m[..., 1]


def _to_r(c):
    return np.ascontiguousarray(np.stack([c.real, c.imag], axis=-1))


@pytest.mark.parametrize("group", [2, 3])
def test_site_update_conserves_the_local_functional(group):
    """Re tr[G K] = Re tr[K] for arbitrary K of the form sum of 8 group elements (SU(3): after
    every subgroup step, so also for the product G), and G is in the group but far from 1."""
    dims = (4, 4, 4, 4)
    uc = li.make_config(dims, group, "haar", 21)
    K = K_numpy(uc, dims)
    far = 0.0
    for s in range(0, K.shape[0], 5):
        G = _to_c(oracle.site_G_micro(_to_r(K[s])))
        assert abs(np.trace(G @ K[s]).real - np.trace(K[s]).real) < 1e-13 * 8 * group
        assert np.abs(G @ dag(G) - np.eye(group)).max() < 1e-14
        assert abs(np.linalg.det(G) - 1) < 1e-14
        far = max(far, np.abs(G - np.eye(group)).max())
    assert far > 1.0


def test_su2_update_is_the_reflection_K_to_K_dagger():
    """SU(2): K = |k| h with h in SU(2), g = h^dagger, so G K = g^2 K = |k| h^dagger = K^dagger --
    the textbook overrelaxation reflection; applying the update to the reflected K undoes it."""
    dims = (4, 4, 4, 4)
    uc = li.make_config(dims, 2, "haar", 22)
    K = K_numpy(uc, dims)
    for s in range(0, K.shape[0], 7):
        G = _to_c(oracle.site_G_micro(_to_r(K[s])))
        assert np.abs(G @ K[s] - dag(K[s])).max() < 1e-14 * 8
        G2 = _to_c(oracle.site_G_micro(_to_r(G @ K[s])))
        assert np.abs(G2 @ G - np.eye(2)).max() < 1e-14


@pytest.mark.parametrize("group", [2, 3])
def test_site_update_is_the_exact_power_two(group):
    """q = g^2 written as a quaternion square equals the (separately pinned) exact group power at
    omega = 2, which goes through atan2 / sin / cos."""
    dims = (4, 4, 4, 4)
    uc = li.make_config(dims, group, "near_identity", 23, eps=0.7, scramble=True)
    K = K_numpy(uc, dims)
    for s in range(0, K.shape[0], 11):
        a = oracle.site_G_micro(_to_r(K[s]))
        b = oracle.site_G(_to_r(K[s]), 2.0)
        assert np.abs(a - b).max() < 5e-15


@pytest.mark.parametrize("group", [2, 3])
def test_sweep_conserves_F_and_moves_the_links(group):
    dims = (4, 6, 2, 8)
    u = li.make_config(dims, group, "near_identity", 24, eps=0.6, scramble=True)
    a = real(u)
    F0 = oracle.functional(dims, a)
    P0 = oracle.plaquette(dims, a)
    th0 = oracle.gauge_precision(dims, a)
    for n in range(40):
        before = a.copy()
        oracle.micro_sweep(dims, a, n & 1)
        assert abs(oracle.functional(dims, a) - F0) < 1e-13
        assert np.abs(a - before).max() > 0.05
    assert abs(oracle.plaquette(dims, a) - P0) < 1e-12          # a gauge transformation
    c = cplx(a)
    assert np.abs(c @ dag(c) - np.eye(group)).max() < 1e-13
    assert oracle.gauge_precision(dims, a) > 1e-3 * th0          # it does not fix the gauge
    # the literal definition at every site of one parity: U_mu(x) <- G U_mu(x), U_mu(x-mu) <- U_mu(x-mu) G^+
    b = real(u)
    oracle.micro_sweep(dims, b, 1)
    K = K_numpy(u, dims)
    par = li.parity_of_sites(dims)
    g = np.broadcast_to(np.eye(group, dtype=complex), (K.shape[0], group, group)).copy()
    for s in np.nonzero(par == 1)[0]:
        g[s] = _to_c(oracle.site_G_micro(_to_r(K[s])))
    want = li.gauge_scramble(u, g, dims)
    assert np.abs(cplx(b) - want).max() < 1e-13


def test_su2_half_sweep_twice_is_the_identity():
    """The SU(2) reflection is an involution site by site, and sites of one parity do not interact:
    two microcanonical half-sweeps of the same parity restore the field."""
    dims = (4, 4, 6, 2)
    u = real(li.make_config(dims, 2, "haar", 25))
    a = u.copy()
    oracle.micro_sweep(dims, a, 0)
    assert np.abs(a - u).max() > 0.1
    oracle.micro_sweep(dims, a, 0)
    assert np.abs(a - u).max() < 1e-13


def test_thread_count_does_not_matter_and_only_one_parity_moves():
    dims = (4, 4, 4, 6)
    u = real(li.make_config(dims, 3, "haar", 26))
    a, b = u.copy(), u.copy()
    oracle.micro_sweep(dims, a, 0)
    oracle.set_threads(4)
    try:
        oracle.micro_sweep(dims, b, 0)
    finally:
        oracle.set_threads(1)
    assert np.array_equal(a, b)


def test_annealing_with_microcanonical_steps_reaches_the_maximum():
    """The combined schedule (heat-bath sweep + n_micro reflections per temperature) on a pure-gauge
    field, followed by overrelaxation, ends at the global maximum F = 1."""
    dims = (4, 4, 4, 4)
    u = real(li.make_config(dims, 2, "pure_gauge", 5))
    oracle.sa_anneal_micro(dims, u, 2.0, 0.01, 60, 2, 9)
    assert oracle.functional(dims, u) > 0.95
    for _ in range(400):
        oracle.full_sweep(dims, u, 1.7)
    assert abs(oracle.functional(dims, u) - 1.0) < 1e-12
    assert oracle.gauge_precision(dims, u) < 1e-20
