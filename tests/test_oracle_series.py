"""Pins for the oracle's truncated-series overrelaxation (reading C-24; SURVEY.md 8(f)
NEXT-2b): g^omega ~ sum_{n<=N} binom(omega,n) (g-1)^n, projected back to SU(2).  CPU only."""
import numpy as np
import pytest
from scipy.special import binom

import lattice_inputs as li
import oracle
from helpers import cplx, dag, real


def unit_quaternion(alpha, axis):
    axis = np.asarray(axis, float) / np.linalg.norm(axis)
    return np.concatenate([[np.cos(alpha)], np.sin(alpha) * axis])


@pytest.mark.parametrize("omega", [1.3, 1.7, 1.95])
@pytest.mark.parametrize("order", [1, 2, 4, 7])
def test_is_the_normalised_complex_polynomial(omega, order):
    """(g-1)^n lives in span{1, i n.sigma}: with z = (c-1) + i|v| the series is the complex
    polynomial w = sum binom(omega,n) z^n and the result is (Re w, v/|v| Im w)/|w| -- written with
    scipy's binom and numpy complex powers, independent of the oracle's matrix loop."""
    rng = np.random.default_rng(5)
    for _ in range(50):
        q = unit_quaternion(rng.uniform(0, np.pi), rng.standard_normal(3))
        r = np.linalg.norm(q[1:])
        z = (q[0] - 1) + 1j * r
        w = sum(binom(omega, n) * z ** n for n in range(order + 1))
        want = np.concatenate([[w.real], q[1:] / r * w.imag]) / abs(w)
        got = oracle.su2_pow_series(q, omega, order)
        assert np.abs(got - want).max() < 1e-13
        assert abs(np.linalg.norm(got) - 1) < 1e-14


def test_converges_to_the_exact_power_inside_the_radius_of_convergence():
    """|g - 1| = 2 sin(alpha/2) < 1, i.e. alpha < pi/3: the series converges to the exact group
    power of reading C-8 (the oracle's pinned su2_pow)."""
    rng = np.random.default_rng(6)
    for _ in range(30):
        q = unit_quaternion(rng.uniform(0, 0.8), rng.standard_normal(3))
        exact = oracle.su2_pow(q, 1.7)
        assert np.abs(oracle.su2_pow_series(q, 1.7, 80) - exact).max() < 1e-12
        e4 = np.abs(oracle.su2_pow_series(q, 1.7, 4) - exact).max()
        e8 = np.abs(oracle.su2_pow_series(q, 1.7, 8) - exact).max()
        assert e8 <= e4 + 1e-15


def test_special_cases():
    rng = np.random.default_rng(7)
    q = unit_quaternion(1.1, rng.standard_normal(3))
    # omega = 1: binom(1, n) = 0 for n >= 2, so every order >= 1 returns g itself
    for order in (1, 3, 6):
        assert np.abs(oracle.su2_pow_series(q, 1.0, order) - q).max() < 1e-15
    # order 0: the identity; order 1: (1 - omega) + omega g, normalised
    assert np.abs(oracle.su2_pow_series(q, 1.7, 0) - [1, 0, 0, 0]).max() < 1e-15
    lin = 1.7 * q + np.array([1 - 1.7, 0, 0, 0])
    assert np.abs(oracle.su2_pow_series(q, 1.7, 1) - lin / np.linalg.norm(lin)).max() < 1e-15
    # g = 1 is a fixed point
    assert np.abs(oracle.su2_pow_series(np.array([1.0, 0, 0, 0]), 1.7, 5) - [1, 0, 0, 0]).max() < 1e-15


@pytest.mark.parametrize("group", [2, 3])
def test_sweep_is_the_literal_site_update_and_a_gauge_transformation(group):
    """or_sweep_series = gather K (pinned), site_G_series, apply -- restated with numpy; plaquette
    invariant; with omega = 1 it coincides with the exact-power sweep."""
    dims = (4, 6, 2, 8)
    u = li.make_config(dims, group, "near_identity", 8, eps=0.4, scramble=True)
    P0 = oracle.plaquette(dims, real(u))
    ur = real(u)
    oracle.or_sweep_series(dims, ur, 0, 1.7, 4)
    K = oracle.K_field(dims, real(u))
    par = li.parity_of_sites(dims)
    from helpers import shift
    G = np.tile(np.eye(group, dtype=np.complex128), (u.shape[0], 1, 1))
    for s in np.nonzero(par == 0)[0]:
        G[s] = cplx(oracle.site_G_series(K[s], 1.7, 4))
    want = np.empty_like(u)
    for mu in range(4):
        want[:, mu] = G @ u[:, mu] @ dag(shift(G, dims, mu, +1))
    assert np.abs(cplx(ur) - want).max() < 1e-14
    oracle.or_sweep_series(dims, ur, 1, 1.7, 4)
    assert abs(oracle.plaquette(dims, ur) - P0) < 1e-12
    a, b = real(u), real(u)
    oracle.full_sweep_series(dims, a, 1.0, 3)
    oracle.full_sweep(dims, b, 1.0)
    assert np.abs(a - b).max() < 1e-14


def test_fixes_the_gauge_on_a_smooth_field():
    """On a smooth (near-identity, scrambled then pre-relaxed) field all angles are inside the radius
    of convergence and the order-4 series drives theta down like the exact power does."""
    dims = (4, 4, 4, 4)
    u = real(li.make_config(dims, 3, "near_identity", 9, eps=0.3, scramble=True))
    for _ in range(5):
        oracle.full_sweep(dims, u, 1.0)
    F = oracle.functional(dims, u)
    for _ in range(150):
        oracle.full_sweep_series(dims, u, 1.7, 4)
        Fn = oracle.functional(dims, u)
        assert Fn >= F - 1e-13
        F = Fn
    assert oracle.gauge_precision(dims, u) < 1e-18
