"""Pins for the oracle's lattice-level functions: K gather, sweep, F, theta, gauge transform,
plaquette.  Invariants, closed forms, special cases and independent np.roll restatements
(SURVEY.md section 8(c) pins P-2 ... P-11).  CPU only.
"""
import numpy as np
import pytest

import lattice_inputs as li
import oracle
from helpers import (K_numpy, cplx, dag, delta_numpy, expm_i_hermitian, plaquette_numpy,
                     random_hermitian_traceless, real, shift)

DIMS_SYM = (4, 4, 4, 4)
DIMS_ASYM = (4, 6, 2, 8)   # all extents different, one extent 2 (x+mu == x-mu there)


def scrambled(dims, group, seed, eps=0.4):
    return li.make_config(dims, group, "near_identity", seed, eps=eps, scramble=True)


# ---------------------------------------------------------------- gather / identities (P-8)

@pytest.mark.parametrize("dims", [DIMS_SYM, DIMS_ASYM])
@pytest.mark.parametrize("group", [2, 3])
def test_K_matches_numpy_roll(dims, group):
    u = li.make_config(dims, group, "haar", 3)
    K = cplx(oracle.K_field(dims, real(u)))
    assert np.abs(K - K_numpy(u, dims)).max() < 1e-14


@pytest.mark.parametrize("group", [2, 3])
def test_functional_three_forms_agree(group):
    """eq. (2) link sum == 1/(2 N_d N_c V) sum_x Re tr K(x) == one parity's K sum."""
    dims = DIMS_ASYM
    u = scrambled(dims, group, 4)
    V = li.volume(dims)
    F = oracle.functional(dims, real(u))
    F_links = np.einsum("nmii->", u).real / (4 * group * V)
    assert abs(F - F_links) < 1e-14
    trK = np.einsum("nii->n", K_numpy(u, dims)).real
    assert abs(F - trK.sum() / (2 * 4 * group * V)) < 1e-14
    par = li.parity_of_sites(dims)
    for p in (0, 1):
        assert abs(F - trK[par == p].sum() / (4 * group * V)) < 1e-14


def test_functional_closed_forms():
    dims = DIMS_SYM
    assert oracle.functional(dims, real(li.make_config(dims, 3, "unit", 0))) == 1.0
    assert oracle.functional(dims, real(li.make_config(dims, 2, "unit", 0))) == 1.0
    # every link = diag(e^{ia}, e^{-ia}, 1): F = (2 cos a + 1)/3
    a = 0.37
    u = np.zeros((li.volume(dims), 4, 3, 3), dtype=np.complex128)
    u[..., 0, 0] = np.exp(1j * a)
    u[..., 1, 1] = np.exp(-1j * a)
    u[..., 2, 2] = 1
    assert abs(oracle.functional(dims, real(u)) - (2 * np.cos(a) + 1) / 3) < 1e-15


@pytest.mark.parametrize("dims", [DIMS_SYM, DIMS_ASYM])
@pytest.mark.parametrize("group", [2, 3])
def test_delta_and_theta_match_numpy_and_K_form(dims, group):
    """Delta from A_mu (eq. 1) == np.roll restatement == [(K - K^dagger)/(2i)]_traceless (C-11)."""
    u = scrambled(dims, group, 5)
    D = cplx(oracle.delta_field(dims, real(u)))
    Dn = delta_numpy(u, dims)
    assert np.abs(D - Dn).max() < 1e-14
    K = K_numpy(u, dims)
    Dk = (K - dag(K)) / 2j
    Dk = Dk - (np.einsum("nii->n", Dk) / group)[:, None, None] * np.eye(group)
    assert np.abs(D - Dk).max() < 1e-14
    theta = oracle.gauge_precision(dims, real(u))
    want = (np.abs(Dn) ** 2).sum() / (group * li.volume(dims))
    assert abs(theta - want) < 1e-13 * want
    # Delta is Hermitian and traceless
    assert np.abs(D - dag(D)).max() < 1e-14
    assert np.abs(np.einsum("nii->n", D)).max() < 1e-14


@pytest.mark.parametrize("group", [2, 3])
def test_gradient_of_F_is_minus_tr_X_delta(group):
    """P-7: d/de F(e^{ieX} o U) at e=0 equals -(1/(N_d N_c V)) sum_x tr[X(x) Delta(x)]: pins the
    sign, the 1/(2i), the traceless projection and the backward difference in Delta, using only
    eq. (2) and the transformation law."""
    dims = DIMS_ASYM
    V = li.volume(dims)
    u = scrambled(dims, group, 6)
    rng = np.random.default_rng(60)
    X = random_hermitian_traceless(V, group, rng)
    eps = 1e-5

    def F_of(e):
        ur = real(u)
        oracle.gauge_transform(dims, ur, real(expm_i_hermitian(e * X)))
        return oracle.functional(dims, ur)

    fd = (F_of(eps) - F_of(-eps)) / (2 * eps)
    D = cplx(oracle.delta_field(dims, real(u)))
    want = -np.einsum("nab,nba->", X, D).real / (4 * group * V)
    assert abs(fd - want) < 1e-9 * max(1.0, abs(want) / 1e-3)
    assert abs(want) > 1e-5   # the test is not vacuous


# ---------------------------------------------------------------- gauge transform / plaquette (P-5)

@pytest.mark.parametrize("group", [2, 3])
def test_gauge_transform_matches_numpy(group):
    dims = DIMS_ASYM
    V = li.volume(dims)
    u = li.make_config(dims, group, "haar", 8)
    g = (li.haar_su3 if group == 3 else li.haar_su2)(V, 9)
    ur = real(u)
    oracle.gauge_transform(dims, ur, real(g))
    want = np.empty_like(u)
    for mu in range(4):
        want[:, mu] = g @ u[:, mu] @ dag(shift(g, dims, mu, +1))
    assert np.abs(cplx(ur) - want).max() < 1e-14
    # the input generator's scramble is the same law
    assert np.abs(li.gauge_scramble(u, g, dims) - want).max() < 1e-14


@pytest.mark.parametrize("group", [2, 3])
def test_plaquette_pins(group):
    dims = DIMS_ASYM
    V = li.volume(dims)
    assert abs(oracle.plaquette(dims, real(li.make_config(dims, group, "unit", 0))) - 1) < 1e-15
    assert abs(oracle.plaquette(dims, real(li.make_config(dims, group, "pure_gauge", 3))) - 1) < 1e-14
    u = li.make_config(dims, group, "near_identity", 10, eps=0.7)
    P0 = oracle.plaquette(dims, real(u))
    assert abs(P0 - plaquette_numpy(u, dims)) < 1e-14
    assert 0.05 < P0 < 0.999
    # invariant under a random gauge transformation ...
    g = (li.haar_su3 if group == 3 else li.haar_su2)(V, 11)
    ur = real(u)
    oracle.gauge_transform(dims, ur, real(g))
    assert abs(oracle.plaquette(dims, ur) - P0) < 1e-12
    # ... and under overrelaxation sweeps (a sweep IS a gauge transformation)
    for _ in range(5):
        oracle.full_sweep(dims, ur, 1.7)
    assert abs(oracle.plaquette(dims, ur) - P0) < 1e-12


# ---------------------------------------------------------------- sweep pins

@pytest.mark.parametrize("omega", [1.0, 1.5])
def test_su2_half_sweep_gain_closed_form(omega):
    """P-2: one half-sweep changes F by (1/(N_d N_c V)) sum_{x in parity} 2|k|(cos((w-1)a) - cos a),
    k the quaternion of the np.roll K(x), cos a = k0/|k|."""
    dims = DIMS_ASYM
    V = li.volume(dims)
    u = li.make_config(dims, 2, "haar", 12)
    par = li.parity_of_sites(dims)
    ur = real(u)
    for p in (0, 1):
        uc = cplx(ur)
        K = K_numpy(uc, dims)
        nk = np.sqrt(np.linalg.det(K).real)
        alpha = np.arccos(np.clip(K[:, 0, 0].real / nk, -1, 1))
        gain = 2 * nk * (np.cos((omega - 1) * alpha) - np.cos(alpha))
        F0 = oracle.functional(dims, ur)
        oracle.or_sweep(dims, ur, p, omega)
        F1 = oracle.functional(dims, ur)
        assert abs((F1 - F0) - gain[par == p].sum() / (4 * 2 * V)) < 1e-13
        # links not touching the swept parity's sites do not exist: every link changed
        # exactly by G(x) on the side of the swept site
        G = np.zeros((V, 2, 2), dtype=np.complex128)
        g = dag(K) / nk[:, None, None]
        # g^omega via eigen-decomposition of the unitary g
        w, vec = np.linalg.eig(g)
        G = (vec * (w ** omega)[:, None, :]) @ np.linalg.inv(vec)
        G[par != p] = np.eye(2)
        want = li.gauge_scramble(uc, G, dims)
        assert np.abs(cplx(ur) - want).max() < 1e-12


@pytest.mark.parametrize("group,omega", [(2, 1.0), (2, 1.5), (3, 1.0), (3, 1.7)])
def test_F_never_decreases(group, omega):
    """P-3: F is non-decreasing after EVERY half-sweep (omega = 1 is the north-star pin; with
    the exact group power it holds for every omega in (0,2))."""
    dims = DIMS_SYM
    ur = real(scrambled(dims, group, 13))
    F = oracle.functional(dims, ur)
    for it in range(60):
        oracle.or_sweep(dims, ur, it & 1, omega)
        Fn = oracle.functional(dims, ur)
        assert Fn >= F - 1e-14
        F = Fn
    assert F > 0.5


def test_sweep_touches_only_its_parity():
    """omega = 1 maximises the local functional, so repeating a half-sweep on the SAME parity
    changes nothing (sites of one parity are independent), and at those sites the Landau
    condition (1) holds ("in each local maximum ... (1) is satisfied")."""
    dims = DIMS_ASYM
    for group in (2, 3):
        ur = real(scrambled(dims, group, 14))
        oracle.or_sweep(dims, ur, 0, 1.0)
        if group == 3:   # one pass over 3 subgroups is not the exact SU(3) maximum; iterate it
            for _ in range(300):
                oracle.or_sweep(dims, ur, 0, 1.0)
        before = ur.copy()
        oracle.or_sweep(dims, ur, 0, 1.0)
        assert np.abs(ur - before).max() < 1e-11
        # at the local maximum of a site, the Landau condition holds there
        D = cplx(oracle.delta_field(dims, ur))
        par = li.parity_of_sites(dims)
        assert np.abs(D[par == 0]).max() < 1e-10
        assert np.abs(D[par == 1]).max() > 1e-3


def test_cfg0_like_convergence_and_invariants():
    """P-4, P-11: run cfg0-like input to theta < 1e-20; unitarity / det to 1e-13; fixed point."""
    dims = DIMS_SYM
    u0 = li.make_named("cfg0")
    ur = real(u0)
    P0 = oracle.plaquette(dims, ur)
    theta = oracle.gauge_precision(dims, ur)
    sweeps = 0
    while theta >= 1e-20 and sweeps < 5000:
        oracle.full_sweep(dims, ur, 1.7)
        sweeps += 1
        theta = oracle.gauge_precision(dims, ur)
    assert theta < 1e-20 and 20 < sweeps < 1000
    uc = cplx(ur)
    assert np.abs(uc @ dag(uc) - np.eye(3)).max() < 1e-13
    assert np.abs(np.linalg.det(uc) - 1).max() < 1e-13
    assert abs(oracle.plaquette(dims, ur) - P0) < 1e-12
    # keep going: theta reaches the rounding floor, links stop moving (small-angle branch of su2_pow)
    for _ in range(40):
        oracle.full_sweep(dims, ur, 1.7)
    before = ur.copy()
    oracle.full_sweep(dims, ur, 1.7)
    assert np.abs(ur - before).max() < 1e-14
    assert oracle.gauge_precision(dims, ur) < 1e-26


@pytest.mark.parametrize("group,seed", [(3, 21), (2, 22)])
def test_pure_gauge_returns_to_vacuum(group, seed):
    """P-6: U_mu(x) = g(x) g(x+mu)^dagger is the unit configuration scrambled by a random gauge
    transformation: the sweep must bring it back to F = 1, theta < 1e-24 (north_star)."""
    dims = DIMS_SYM
    ur = real(li.make_config(dims, group, "pure_gauge", seed))
    assert oracle.functional(dims, ur) < 0.5
    omega = 1.7 if group == 3 else 1.5
    for it in range(1500):
        oracle.full_sweep(dims, ur, omega)
        if it % 10 == 9 and oracle.gauge_precision(dims, ur) < 1e-26:
            break
    assert abs(oracle.functional(dims, ur) - 1.0) < 1e-12
    assert oracle.gauge_precision(dims, ur) < 1e-24


def test_su3_code_reduces_to_su2_code_at_omega_1():
    """P-9: SU(3) links living in the (0,1) block, omega = 1: after the (0,1) step K's block is
    |k| 1, so steps (0,2),(1,2) are the identity and the SU(3) sweep equals the SU(2) sweep."""
    dims = DIMS_ASYM
    u2 = li.make_config(dims, 2, "haar", 23)
    u3 = np.zeros(u2.shape[:2] + (3, 3), dtype=np.complex128)
    u3[..., :2, :2] = u2
    u3[..., 2, 2] = 1
    r2, r3 = real(u2), real(u3)
    oracle.full_sweep(dims, r2, 1.0)
    oracle.full_sweep(dims, r3, 1.0)
    c3 = cplx(r3)
    assert np.abs(c3[..., :2, :2] - cplx(r2)).max() < 1e-13
    assert np.abs(c3[..., 2, 2] - 1).max() < 1e-13
    assert np.abs(c3[..., 2, :2]).max() < 1e-13 and np.abs(c3[..., :2, 2]).max() < 1e-13


@pytest.mark.parametrize("group", [2, 3])
def test_translation_covariance(group):
    """P-10: translating the field by an even vector commutes with a half-sweep; by an odd
    vector it swaps black and white.  Pins the index maps and parity logic on asymmetric dims."""
    dims = DIMS_ASYM
    u = scrambled(dims, group, 24)

    def translate(f, vec):
        for mu, step in enumerate(vec):
            f = shift(f, dims, mu, step)
        return f

    for vec, swap in (((2, 0, 0, 2), 0), ((0, 1, 0, 0), 1), ((1, 0, 1, 1), 1), ((1, 1, 0, 0), 0)):
        a = real(u)
        oracle.or_sweep(dims, a, 0, 1.7)
        a = translate(cplx(a), vec)
        b = real(translate(u, vec))
        oracle.or_sweep(dims, b, 0 ^ swap, 1.7)
        assert np.abs(a - cplx(b)).max() < 1e-13


def test_axis_permutation_covariance():
    """P-10: swapping two lattice axes together with the Lorentz index commutes with the sweep
    (up to summation order)."""
    dims = (4, 6, 2, 8)
    pdims = (6, 4, 2, 8)   # axes 0 and 1 swapped
    u = scrambled(dims, 3, 25)
    n0, n1, n2, n3 = dims

    def permute(f):
        g = f.reshape((n3, n2, n1, n0) + f.shape[1:])
        g = np.swapaxes(g, 2, 3)            # site axes
        g = g.reshape(f.shape)
        return g[:, [1, 0, 2, 3]]           # Lorentz index

    a = real(u)
    oracle.full_sweep(dims, a, 1.7)
    b = real(np.ascontiguousarray(permute(u)))
    oracle.full_sweep(pdims, b, 1.7)
    assert np.abs(permute(cplx(a)) - cplx(b)).max() < 1e-13


def test_global_rotation_covariance_su2():
    """P-10: U -> h U h^dagger with a constant h commutes with the SU(2) sweep."""
    dims = DIMS_SYM
    u = li.make_config(dims, 2, "haar", 26)
    h = li.haar_su2(1, 27)[0]
    a = real(u)
    oracle.full_sweep(dims, a, 1.5)
    b = real(h @ u @ dag(h))
    oracle.full_sweep(dims, b, 1.5)
    assert np.abs(h @ cplx(a) @ dag(h) - cplx(b)).max() < 1e-13


def test_threads_do_not_change_results():
    dims = DIMS_ASYM
    u = real(scrambled(dims, 3, 28))
    a, b = u.copy(), u.copy()
    oracle.set_threads(1)
    oracle.full_sweep(dims, a, 1.7)
    ta = oracle.gauge_precision(dims, a)
    oracle.set_threads(4)
    oracle.full_sweep(dims, b, 1.7)
    tb = oracle.gauge_precision(dims, b)
    oracle.set_threads(1)
    assert np.array_equal(a, b) and ta == tb
