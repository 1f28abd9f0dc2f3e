"""Pins for the oracle's single-site arithmetic (su2_pow, subgroup step, site_G).

Each pin compares the oracle with something fixed by the paper or by mathematics, not with the
oracle itself: brute force over the group manifold ("the local maximum at each
site can be found directly as g = K^dagger/sqrt(det K^dagger)"), the paper's formula evaluated
literally with numpy/scipy library routines, and closed forms.
"""
import numpy as np
import pytest
from scipy.linalg import fractional_matrix_power

import lattice_inputs as li
import oracle
from helpers import dag, real, cplx


def quat_to_mat(q):
    return li.su2_from_quaternion(np.asarray(q, dtype=np.float64)[None])[0]


def random_su2_K(rng):
    """A sum of 8 random SU(2) matrices (what K(x) is for SU(2)): a real multiple of SU(2)."""
    q = rng.standard_normal((8, 4))
    q /= np.linalg.norm(q, axis=1, keepdims=True)
    return li.su2_from_quaternion(q).sum(axis=0)


def random_su3_K(rng, seed):
    return li.haar_su3(8, seed).sum(axis=0)


# ---------------------------------------------------------------- su2_pow

@pytest.mark.parametrize("omega", [1.0, 1.3, 1.7, 1.99])
def test_su2_pow_matches_scipy_matrix_power(omega):
    """g^omega on the principal branch equals scipy's fractional_matrix_power of the 2x2 matrix."""
    rng = np.random.default_rng(7)
    for _ in range(25):
        q = rng.standard_normal(4)
        q /= np.linalg.norm(q)
        got = quat_to_mat(oracle.su2_pow(q, omega))
        want = fractional_matrix_power(quat_to_mat(q), omega)
        assert np.abs(got - want).max() < 1e-12


def test_su2_pow_group_laws():
    rng = np.random.default_rng(8)
    q = rng.standard_normal(4)
    q /= np.linalg.norm(q)
    g = quat_to_mat(q)
    assert np.abs(quat_to_mat(oracle.su2_pow(q, 1.0)) - g).max() < 1e-15
    assert np.abs(quat_to_mat(oracle.su2_pow(q, 2.0)) - g @ g).max() < 1e-14
    a = quat_to_mat(oracle.su2_pow(q, 0.6))
    b = quat_to_mat(oracle.su2_pow(q, 1.1))
    assert np.abs(a @ b - quat_to_mat(oracle.su2_pow(q, 1.7))).max() < 1e-14
    out = oracle.su2_pow(q, 1.7)
    assert abs(np.linalg.norm(out) - 1.0) < 1e-15


def test_su2_pow_small_angle_keeps_all_digits():
    """alpha via atan2, not acos: for a rotation angle 1e-9 the result is omega*v to ~1e-16
    relative (acos(c) would lose half the digits) -- SURVEY 7.4 item 5 / reading C-8."""
    v = np.array([3e-10, -4e-10, 12e-10])
    r = np.linalg.norm(v)
    q = np.array([np.sqrt(1.0 - r * r), *v])
    out = oracle.su2_pow(q, 1.7)
    assert np.allclose(out[1:], 1.7 * v, rtol=1e-12, atol=0)
    assert abs(out[0] - 1.0) < 1e-16
    # exactly the identity and exactly -1
    assert np.array_equal(oracle.su2_pow([1.0, 0, 0, 0], 1.7), [1.0, 0, 0, 0])
    m1 = oracle.su2_pow([-1.0, 0, 0, 0], 1.5)
    assert np.allclose(m1, [np.cos(1.5 * np.pi), 0, 0, np.sin(1.5 * np.pi)], atol=1e-15)


# ---------------------------------------------------------------- SU(2) site update

def test_su2_site_update_is_the_papers_formula():
    """omega = 1: G = K^dagger / sqrt(det K^dagger) literally, via np.linalg.det."""
    rng = np.random.default_rng(11)
    for _ in range(10):
        K = random_su2_K(rng)
        G = cplx(oracle.site_G(real(K), 1.0))
        want = dag(K) / np.sqrt(np.linalg.det(dag(K)))
        assert np.abs(G - want).max() < 1e-14


def test_su2_local_maximum_brute_force():
    """Re tr[g K] over 2e6 random points of S^3 approaches 2 sqrt(det K) from below and the
    arg-max approaches the oracle's g (P-1)."""
    rng = np.random.default_rng(12)
    K = random_su2_K(rng)
    G = cplx(oracle.site_G(real(K), 1.0))
    best_closed = np.trace(G @ K).real
    assert abs(best_closed - 2.0 * np.sqrt(np.linalg.det(K).real)) < 1e-12
    q = rng.standard_normal((2_000_000, 4))
    q /= np.linalg.norm(q, axis=1, keepdims=True)
    # Re tr[g K] for g = quaternion q, K = k0 + i k.sigma :  2 (q0 k0 - q.k)
    k = np.array([K[0, 0].real, K[0, 1].imag, K[0, 1].real, K[0, 0].imag])
    vals = 2.0 * (q[:, 0] * k[0] - q[:, 1:] @ k[1:])
    # spot-check that formula against an explicit matrix trace
    g7 = quat_to_mat(q[7])
    assert abs(np.trace(g7 @ K).real - vals[7]) < 1e-12
    i = int(np.argmax(vals))
    assert vals[i] <= best_closed + 1e-12
    assert vals[i] > best_closed * (1 - 2e-3)
    assert np.abs(quat_to_mat(q[i]) - G).max() < 0.08


@pytest.mark.parametrize("omega", [1.5, 1.7])
def test_su2_overrelaxed_update_is_matrix_power(omega):
    rng = np.random.default_rng(13)
    K = random_su2_K(rng)
    G = cplx(oracle.site_G(real(K), omega))
    g = dag(K) / np.sqrt(np.linalg.det(dag(K)))
    assert np.abs(G - fractional_matrix_power(g, omega)).max() < 1e-12
    # closed-form gain (P-2): Re tr[G K] = 2|k| cos((omega-1) alpha), cos(alpha) = k0/|k|
    nk = np.sqrt(np.linalg.det(K).real)
    alpha = np.arccos(K[0, 0].real / nk)
    assert abs(np.trace(G @ K).real - 2 * nk * np.cos((omega - 1) * alpha)) < 1e-12


def test_zero_K_is_skipped():
    G = oracle.site_G(np.zeros((2, 2, 2)), 1.7)
    assert np.array_equal(cplx(G), np.eye(2))
    G = oracle.site_G(np.zeros((3, 3, 2)), 1.7)
    assert np.array_equal(cplx(G), np.eye(3))


# ---------------------------------------------------------------- SU(3) subgroup steps

PAIRS = [(0, 1), (0, 2), (1, 2)]


def embed(g2, i, j):
    g = np.eye(3, dtype=np.complex128)
    g[np.ix_([i, j], [i, j])] = g2
    return g


def su2_part(B):
    """SU(2)-proportional part of a 2x2 complex block: (B + adj(B)^dagger)/2."""
    adj = np.array([[B[1, 1], -B[0, 1]], [-B[1, 0], B[0, 0]]])
    return 0.5 * (B + dag(adj))


@pytest.mark.parametrize("pair", PAIRS)
def test_su3_subgroup_step_brute_force(pair):
    """omega = 1: the embedded SU(2) element maximises Re tr[g_s K] over the (i,j) subgroup."""
    i, j = pair
    rng = np.random.default_rng(20 + i + 3 * j)
    K = random_su3_K(rng, 77 + i + 3 * j)
    gs, ok = oracle.subgroup_step(real(K), i, j, 1.0)
    assert ok
    gs = cplx(gs)
    # it is an embedded SU(2) element
    assert np.abs(gs @ dag(gs) - np.eye(3)).max() < 1e-14
    assert abs(np.linalg.det(gs) - 1) < 1e-14
    k = 3 - i - j
    assert gs[k, k] == 1.0 and np.count_nonzero(gs[k]) == 1 and np.count_nonzero(gs[:, k]) == 1
    best = np.trace(gs @ K).real
    q = rng.standard_normal((400_000, 4))
    q /= np.linalg.norm(q, axis=1, keepdims=True)
    g2 = li.su2_from_quaternion(q)
    B = K[np.ix_([i, j], [i, j])]
    vals = np.einsum("nab,ba->n", g2, B).real + K[k, k].real
    m = int(np.argmax(vals))
    assert abs(np.trace(embed(g2[m], i, j) @ K).real - vals[m]) < 1e-12
    assert vals[m] <= best + 1e-12
    assert vals[m] > best - 5e-3 * abs(best)
    assert np.abs(embed(g2[m], i, j) - gs).max() < 0.12


@pytest.mark.parametrize("omega", [1.0, 1.7])
def test_su3_site_G_is_three_literal_subgroup_updates(omega):
    """site_G = g_(1,2) g_(0,2) g_(0,1), each g = P^dagger/sqrt(det P^dagger) raised to omega
    with numpy det + scipy fractional_matrix_power, P the SU(2) part of the CURRENT K's block
    (readings C-6, C-10)."""
    rng = np.random.default_rng(31)
    for trial in range(5):
        K = random_su3_K(rng, 300 + trial)
        G = cplx(oracle.site_G(real(K), omega))
        Kc = K.copy()
        Gw = np.eye(3, dtype=np.complex128)
        for (i, j) in PAIRS:
            P = su2_part(Kc[np.ix_([i, j], [i, j])])
            g2 = dag(P) / np.sqrt(np.linalg.det(dag(P)))
            g2 = fractional_matrix_power(g2, omega)
            gs = embed(g2, i, j)
            Kc = gs @ Kc
            Gw = gs @ Gw
        assert np.abs(G - Gw).max() < 1e-12
        assert np.abs(G @ dag(G) - np.eye(3)).max() < 1e-14
        assert abs(np.linalg.det(G) - 1) < 1e-14


def test_su3_relaxation_never_lowers_local_functional():
    """omega = 1: Re tr[G K] >= Re tr[K] for every K (each subgroup step is a maximisation)."""
    rng = np.random.default_rng(32)
    for trial in range(20):
        K = random_su3_K(rng, 500 + trial)
        G = cplx(oracle.site_G(real(K), 1.0))
        assert np.trace(G @ K).real >= np.trace(K).real - 1e-13


def test_reconstruct12_round_trip():
    """12-parameter representation: rows 0,1 kept, row 2 = conj(row0 x row1)."""
    u = li.haar_su3(64, 5)
    r = real(u)
    r[:, 2] = 123.0  # destroy the third row
    oracle.reconstruct12(r)
    assert np.abs(cplx(r) - u).max() < 1e-15
    # and it is what np.cross gives
    assert np.abs(cplx(r)[:, 2] - np.conj(np.cross(u[:, 0], u[:, 1]))).max() < 1e-15
