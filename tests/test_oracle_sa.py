"""Pins for the oracle's simulated-annealing functions (reading C-25; SURVEY.md 8(f)
NEXT-3): the Philox generator against its published vectors, the heat-bath sample against the
closed-form moments and the density it must follow, the T -> 0 limit against the (pinned)
relaxation update, and the sweep's invariants.  CPU only."""
import os

import numpy as np
import pytest
from scipy.special import iv

import lattice_inputs as li
import oracle
from helpers import cplx, dag, real


def test_philox_known_answers():
    path = os.path.join(os.path.dirname(__file__), "golden", "philox4x32_10_kat.txt")
    rows = [l.split() for l in open(path) if l.strip() and not l.startswith("#")]
    assert len(rows) == 3
    for r in rows:
        v = [int(x, 16) for x in r]
        assert oracle.philox4x32_10(v[0:4], v[4:6]).tolist() == v[6:10]


def quat_mul(a, b):
    o = np.empty_like(a)
    o[..., 0] = a[..., 0] * b[..., 0] - np.sum(a[..., 1:] * b[..., 1:], axis=-1)
    o[..., 1:] = a[..., :1] * b[..., 1:] + b[..., :1] * a[..., 1:] - np.cross(a[..., 1:], b[..., 1:])
    return o


@pytest.mark.parametrize("alpha", [0.7, 3.0, 25.0])
def test_heatbath_density_and_moments(alpha):
    """h = q * p/|p| must have h_0 ~ sqrt(1-h_0^2) exp(alpha h_0) with alpha = |p|/T:
    <h_0> = I_2(alpha)/I_1(alpha) (closed form), a histogram chi-square against the density, and a
    vector part uniform on the sphere (zero mean, isotropic second moments)."""
    rng = np.random.default_rng(3)
    p = rng.standard_normal(4) * 2.0
    T = np.linalg.norm(p) / alpha
    n = 200000
    q = oracle.su2_heatbath_samples(p, T, 12345, n)
    assert np.abs(np.linalg.norm(q, axis=1) - 1).max() < 1e-14
    h = quat_mul(q, np.broadcast_to(p / np.linalg.norm(p), q.shape))
    h0 = h[:, 0]
    want = iv(2, alpha) / iv(1, alpha)
    sd = h0.std() / np.sqrt(n)
    assert abs(h0.mean() - want) < 5 * sd
    edges = np.linspace(-1, 1, 41)
    x = np.linspace(-1, 1, 400001)
    dens = np.sqrt(np.maximum(0, 1 - x * x)) * np.exp(alpha * (x - 1))
    cdf = np.concatenate([[0], np.cumsum((dens[1:] + dens[:-1]) / 2)])
    cdf /= cdf[-1]
    expect = n * np.diff(np.interp(edges, x, cdf))
    obs, _ = np.histogram(h0, edges)
    keep = expect > 20
    chi2 = np.sum((obs[keep] - expect[keep]) ** 2 / expect[keep])
    assert chi2 < keep.sum() + 6 * np.sqrt(2 * keep.sum())
    v = h[:, 1:] / np.linalg.norm(h[:, 1:], axis=1, keepdims=True)
    assert np.abs(v.mean(axis=0)).max() < 5 / np.sqrt(n)
    assert np.abs((v[:, :, None] * v[:, None, :]).mean(axis=0) - np.eye(3) / 3).max() < 5 / np.sqrt(n)


def test_zero_temperature_limit_is_the_relaxation_update():
    """T -> 0: the sample collapses onto the maximiser K^dagger/sqrt(det K^dagger), i.e.
    an SA half-sweep tends to the omega = 1 half-sweep of the pinned oracle; the distance shrinks
    like sqrt(T)."""
    dims = (4, 4, 4, 4)
    for group in (2, 3):
        u = li.make_config(dims, group, "near_identity", 11, eps=0.4, scramble=True)
        ref = real(u)
        oracle.or_sweep(dims, ref, 0, 1.0)
        errs = []
        for T in (1e-4, 1e-6, 1e-8):
            a = real(u)
            oracle.sa_sweep(dims, a, 0, T, 7, 0)
            errs.append(np.abs(a - ref).max())
        assert errs[0] < 0.2 and errs[1] < errs[0] / 5 and errs[2] < errs[1] / 5, errs


@pytest.mark.parametrize("group", [2, 3])
def test_sweep_is_a_gauge_transformation_and_counter_based(group):
    dims = (4, 6, 2, 8)
    u = li.make_config(dims, group, "haar", 12)
    P0 = oracle.plaquette(dims, real(u))
    a = real(u)
    for n in range(6):
        oracle.sa_sweep(dims, a, n & 1, 0.8, 99, n)
    assert abs(oracle.plaquette(dims, a) - P0) < 1e-12
    c = cplx(a)
    assert np.abs(c @ dag(c) - np.eye(group)).max() < 1e-13
    # same seed and counters -> same field, whatever the thread count; another counter -> another field
    b = real(u)
    oracle.set_threads(4)
    try:
        for n in range(6):
            oracle.sa_sweep(dims, b, n & 1, 0.8, 99, n)
    finally:
        oracle.set_threads(1)
    assert np.array_equal(a, b)
    d = real(u)
    oracle.sa_sweep(dims, d, 0, 0.8, 99, 1)
    e = real(u)
    oracle.sa_sweep(dims, e, 0, 0.8, 99, 0)
    assert not np.array_equal(d, e)
    # only links touching sites of the swept parity change (checkerboard)
    par = li.parity_of_sites(dims)
    changed = np.abs(e - real(u)).reshape(e.shape[0], 4, -1).max(axis=2) > 0
    assert changed[par == 0].all()


def test_annealing_raises_the_functional():
    """Lowering T towards 0 drives F up (the annealed field ends near a maximum of F); at high T the
    field stays disordered: <F>(T = 5) < <F>(T = 0.05) on a pure-gauge configuration whose global
    maximum is F = 1."""
    dims = (4, 4, 4, 4)
    u = real(li.make_config(dims, 2, "pure_gauge", 5))
    n = 0
    for T in (5.0,) * 20:
        for par in (0, 1):
            oracle.sa_sweep(dims, u, par, T, 1, n)
            n += 1
    F_hot = oracle.functional(dims, u)
    for T in np.linspace(2.0, 0.01, 150):
        for par in (0, 1):
            oracle.sa_sweep(dims, u, par, float(T), 1, n)
            n += 1
    F_cold = oracle.functional(dims, u)
    assert F_hot < 0.6 and F_cold > 0.97
