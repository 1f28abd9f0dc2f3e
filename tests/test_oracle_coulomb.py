"""Pins for the oracle's Coulomb-gauge functions (reading C-22).

The paper names Coulomb gauge and defers its details to a reference that is
not available, so the definition is the Landau one (eqs. 1-3) restricted to the three spatial
directions, time-slice by time-slice.  Every pin below ties the Coulomb functions either to the
already-pinned Landau functions, to numpy restatements, or to invariants.  CPU only.
"""
import numpy as np
import pytest

import lattice_inputs as li
import oracle
from helpers import cplx, dag, expm_i_hermitian, plaquette_numpy, random_hermitian_traceless, real, shift

DIMS = (4, 6, 2, 8)       # all extents different; x3 = time has 8 slices
DIMS_B = (6, 4, 4, 4)


def scrambled(dims, group, seed, eps=0.4):
    return li.make_config(dims, group, "near_identity", seed, eps=eps, scramble=True)


def slice_of(dims):
    n0, n1, n2, n3 = dims
    return np.repeat(np.arange(n3), n0 * n1 * n2)


def K_spatial_numpy(uc, dims):
    K = np.zeros((uc.shape[0],) + uc.shape[2:], dtype=np.complex128)
    for mu in range(3):
        K += uc[:, mu] + dag(shift(uc[:, mu], dims, mu, -1))
    return K


@pytest.mark.parametrize("group", [2, 3])
def test_K_and_delta_match_numpy_and_each_other(group):
    u = scrambled(DIMS, group, 70)
    K = cplx(oracle.K_coulomb_field(DIMS, real(u)))
    assert np.abs(K - K_spatial_numpy(u, DIMS)).max() < 1e-14
    # Delta_C from the A_i form (oracle) equals the K_C form (reading C-11 restricted to i < 3)
    D = cplx(oracle.delta_coulomb_field(DIMS, real(u)))
    Dk = (K - dag(K)) / 2j
    Dk = Dk - (np.einsum("nii->n", Dk) / group)[:, None, None] * np.eye(group)
    assert np.abs(D - Dk).max() < 1e-14
    # and the Landau Delta is Delta_C plus the time-direction term
    A3 = (u[:, 3] - dag(u[:, 3])) / 2j
    A3 = A3 - (np.einsum("nii->n", A3) / group)[:, None, None] * np.eye(group)
    D4 = cplx(oracle.delta_field(DIMS, real(u)))
    assert np.abs(D4 - (D + A3 - shift(A3, DIMS, 3, -1))).max() < 1e-14


@pytest.mark.parametrize("group", [2, 3])
def test_theta_F_per_slice_match_numpy(group):
    u = scrambled(DIMS, group, 71)
    th, F = oracle.coulomb_theta_F(DIMS, real(u))
    t = slice_of(DIMS)
    D = cplx(oracle.delta_coulomb_field(DIMS, real(u)))
    term = np.einsum("nab,nab->n", D, np.conj(D)).real
    retr = np.einsum("nmii->n", u[:, :3]).real
    vs = DIMS[0] * DIMS[1] * DIMS[2]
    for k in range(DIMS[3]):
        assert abs(th[k] - term[t == k].sum() / (group * vs)) < 1e-13
        assert abs(F[k] - retr[t == k].sum() / (3 * group * vs)) < 1e-13
    # closed forms: unit field and pure gauge... F_t = 1 only for the unit field
    th1, F1 = oracle.coulomb_theta_F(DIMS, real(li.make_config(DIMS, group, "unit", 0)))
    assert np.all(np.abs(F1 - 1) < 1e-15) and np.all(th1 < 1e-30)


@pytest.mark.parametrize("group", [2, 3])
@pytest.mark.parametrize("omega", [1.0, 1.7])
def test_sweep_is_landau_sweep_with_time_links_removed(group, omega):
    """K_C = K with the time links set to zero matrices, so the spatial links after a Coulomb
    half-sweep are EXACTLY those of the (pinned) Landau half-sweep on that field; the time links
    follow the transformation law with the same G(x)."""
    u = scrambled(DIMS, group, 72)
    for parity in (0, 1):
        uc = real(u)
        oracle.or_sweep_coulomb(DIMS, uc, parity, omega)
        u0 = u.copy()
        u0[:, 3] = 0
        ul = real(u0)
        oracle.or_sweep(DIMS, ul, parity, omega)
        assert np.array_equal(uc[:, :3], ul[:, :3])
        # time links: U_3(x) <- G(x) U_3(x) G(x+t)^dagger with G = site_G(K_C) on this parity, 1 elsewhere
        Kc = oracle.K_coulomb_field(DIMS, real(u))
        par = li.parity_of_sites(DIMS)
        G = np.tile(np.eye(group, dtype=np.complex128), (u.shape[0], 1, 1))
        for s in np.nonzero(par == parity)[0]:
            G[s] = cplx(oracle.site_G(Kc[s], omega))
        want = G @ u[:, 3] @ dag(shift(G, DIMS, 3, +1))
        assert np.abs(cplx(uc)[:, 3] - want).max() < 1e-14


@pytest.mark.parametrize("group", [2, 3])
def test_slices_decouple(group):
    """The spatial links of slice t after a full Coulomb sweep depend only on the spatial links of
    slice t: changing every other slice (and all time links) leaves them bit-identical."""
    u = scrambled(DIMS, group, 73)
    v = li.make_config(DIMS, group, "haar", 74)
    t = slice_of(DIMS)
    keep = 3
    w = v.copy()
    w[t == keep, :3] = u[t == keep, :3]
    a, b = real(u), real(w)
    for _ in range(3):
        oracle.full_sweep_coulomb(DIMS, a, 1.7)
        oracle.full_sweep_coulomb(DIMS, b, 1.7)
    assert np.array_equal(a[t == keep, :3], b[t == keep, :3])
    assert not np.array_equal(a[t == keep + 1, :3], b[t == keep + 1, :3])


@pytest.mark.parametrize("group", [2, 3])
@pytest.mark.parametrize("omega", [1.0, 1.7])
def test_every_slice_functional_never_decreases_and_plaquette_is_invariant(group, omega):
    u = real(li.make_config(DIMS_B, group, "haar", 75))
    P0 = oracle.plaquette(DIMS_B, u)
    _, F = oracle.coulomb_theta_F(DIMS_B, u)
    for _ in range(25):
        for parity in (0, 1):
            oracle.or_sweep_coulomb(DIMS_B, u, parity, omega)
            _, Fn = oracle.coulomb_theta_F(DIMS_B, u)
            assert np.all(Fn >= F - 1e-14)
            F = Fn
    # a sweep is a gauge transformation: ALL plaquettes (temporal ones too) are unchanged
    assert abs(oracle.plaquette(DIMS_B, u) - P0) < 1e-12
    assert abs(plaquette_numpy(cplx(u), DIMS_B) - P0) < 1e-12


@pytest.mark.parametrize("group", [2, 3])
def test_gradient_of_F_t_is_minus_tr_X_delta_C(group):
    """d/de F_t(e^{ieX} o U) at e = 0 equals -(1/(3 N_c V_s)) sum_{x in t} tr[X(x) Delta_C(x)] for
    every slice t: pins Delta_C's sign, the 1/(2i), the traceless projection, the backward
    difference and the per-slice normalisations, from F_t and the transformation law alone."""
    V = li.volume(DIMS)
    u = scrambled(DIMS, group, 76)
    X = random_hermitian_traceless(V, group, np.random.default_rng(77))
    eps = 1e-5

    def F_of(e):
        ur = real(u)
        oracle.gauge_transform(DIMS, ur, real(expm_i_hermitian(e * X)))
        return oracle.coulomb_theta_F(DIMS, ur)[1]

    fd = (F_of(eps) - F_of(-eps)) / (2 * eps)
    D = cplx(oracle.delta_coulomb_field(DIMS, real(u)))
    per_site = np.einsum("nab,nba->n", X, D).real
    t = slice_of(DIMS)
    vs = DIMS[0] * DIMS[1] * DIMS[2]
    for k in range(DIMS[3]):
        want = -per_site[t == k].sum() / (3 * group * vs)
        assert abs(fd[k] - want) < 1e-8
    assert np.abs(fd).max() > 1e-4


@pytest.mark.parametrize("group,seed", [(2, 1), (3, 2)])
def test_pure_gauge_reaches_the_vacuum_in_every_slice(group, seed):
    """U = g(x) g(x+mu)^dagger: Coulomb fixing brings every slice to F_t = 1, theta_t -> 0, and
    the converged field is a fixed point of a further sweep."""
    dims = (4, 4, 4, 4)
    u = real(li.make_config(dims, group, "pure_gauge", seed))
    for _ in range(400):
        oracle.full_sweep_coulomb(dims, u, 1.7)
        th, F = oracle.coulomb_theta_F(dims, u)
        if th.max() < 1e-26:
            break
    assert th.max() < 1e-24 and np.abs(F - 1).max() < 1e-12
    before = u.copy()
    oracle.full_sweep_coulomb(dims, u, 1.7)
    assert np.abs(u - before).max() < 1e-11      # theta_t < 1e-24  =>  |g(x) - 1| <~ 1e-12
    c = cplx(u)
    assert np.abs(c @ dag(c) - np.eye(group)).max() < 1e-13


def test_masked_sweep_freezes_inactive_slices_and_matches_the_full_sweep_elsewhere():
    u = scrambled(DIMS, 3, 79)
    t = slice_of(DIMS)
    active = np.array([1, 0, 1, 1, 0, 0, 1, 0], dtype=np.uint8)
    a, b = real(u), real(u)
    for parity in (0, 1):
        oracle.or_sweep_coulomb_masked(DIMS, a, parity, 1.7, active)
        oracle.or_sweep_coulomb(DIMS, b, parity, 1.7)
    for k in range(DIMS[3]):
        if active[k]:      # spatial links of an active slice: exactly the unmasked sweep (slices decouple)
            assert np.array_equal(a[t == k, :3], b[t == k, :3])
        else:              # spatial links of a frozen slice: untouched
            assert np.array_equal(a[t == k, :3], real(u)[t == k, :3])
    assert abs(oracle.plaquette(DIMS, a) - oracle.plaquette(DIMS, real(u))) < 1e-12
    none = real(u)
    oracle.or_sweep_coulomb_masked(DIMS, none, 0, 1.7, np.zeros(DIMS[3], dtype=np.uint8))
    assert np.array_equal(none, real(u))


def test_threads_do_not_change_results():
    u = scrambled(DIMS, 3, 78)
    a, b = real(u), real(u)
    oracle.set_threads(1)
    oracle.full_sweep_coulomb(DIMS, a, 1.7)
    ta = oracle.coulomb_theta_F(DIMS, a)
    oracle.set_threads(4)
    oracle.full_sweep_coulomb(DIMS, b, 1.7)
    tb = oracle.coulomb_theta_F(DIMS, b)
    oracle.set_threads(1)
    assert np.array_equal(a, b) and np.array_equal(ta[0], tb[0]) and np.array_equal(ta[1], tb[1])
