"""Pins for the oracle's re-unitarisation (reading C-23; SURVEY.md 8(f) NEXT-2c):
numpy/QR restatement, group properties, idempotence, stability.  CPU only."""
import numpy as np
import pytest

import lattice_inputs as li
import oracle
from helpers import cplx, dag, real


def perturbed(group, n, seed, size):
    u = (li.haar_su3 if group == 3 else li.haar_su2)(n, seed)
    rng = np.random.default_rng(seed + 1)
    return u + size * (rng.standard_normal(u.shape) + 1j * rng.standard_normal(u.shape))


@pytest.mark.parametrize("group", [2, 3])
def test_result_is_in_the_group_and_idempotent(group):
    m = real(perturbed(group, 500, 90, 1e-3))
    oracle.reunitarize(m)
    c = cplx(m)
    assert np.abs(c @ dag(c) - np.eye(group)).max() < 1e-14
    assert np.abs(np.linalg.det(c) - 1).max() < 1e-14
    again = m.copy()
    oracle.reunitarize(again)
    assert np.abs(again - m).max() < 4e-15


@pytest.mark.parametrize("group", [2, 3])
def test_group_elements_are_fixed_and_small_drift_is_removed_to_first_order(group):
    u = (li.haar_su3 if group == 3 else li.haar_su2)(300, 91)
    m = real(u)
    oracle.reunitarize(m)
    assert np.abs(cplx(m) - u).max() < 4e-15
    p = real(perturbed(group, 300, 91, 1e-6))
    oracle.reunitarize(p)
    assert np.abs(cplx(p) - u).max() < 1e-5          # stays next to the element it drifted from


def test_su3_rows_match_numpy_gram_schmidt_and_qr():
    a = perturbed(3, 200, 92, 1e-2)
    m = real(a)
    oracle.reunitarize(m)
    c = cplx(m)
    r0 = a[:, 0] / np.linalg.norm(a[:, 0], axis=1, keepdims=True)
    r1 = a[:, 1] - np.sum(np.conj(r0) * a[:, 1], axis=1, keepdims=True) * r0
    r1 /= np.linalg.norm(r1, axis=1, keepdims=True)
    assert np.abs(c[:, 0] - r0).max() < 1e-14 and np.abs(c[:, 1] - r1).max() < 1e-14
    assert np.abs(c[:, 2] - np.conj(np.cross(r0, r1))).max() < 1e-14
    # QR of the transposed first two rows spans the same flag: |<q_k, row_k>| = 1
    for k in range(20):
        q, _ = np.linalg.qr(a[k, :2].T)
        assert abs(abs(np.vdot(q[:, 0], c[k, 0])) - 1) < 1e-13
        assert abs(abs(np.vdot(q[:, 1], c[k, 1])) - 1) < 1e-13


def test_su2_is_quaternion_normalisation():
    a = perturbed(2, 200, 93, 1e-2)
    m = real(a)
    oracle.reunitarize(m)
    c = cplx(m)
    nrm = np.sqrt(np.abs(a[:, 0, 0]) ** 2 + np.abs(a[:, 0, 1]) ** 2)
    assert np.abs(c[:, 0, 0] - a[:, 0, 0] / nrm).max() < 1e-15
    assert np.abs(c[:, 1, 1] - np.conj(c[:, 0, 0])).max() < 1e-15
    assert np.abs(c[:, 1, 0] + np.conj(c[:, 0, 1])).max() < 1e-15
