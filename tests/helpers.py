"""Small numpy helpers for the tests: independent (np.roll / np.linalg) restatements of lattice
definitions used to PIN the oracle.  Nothing here is imported by the oracle or the CUDA path."""
import numpy as np

import lattice_inputs as li


def dag(m):
    return np.conj(np.swapaxes(m, -1, -2))


def shift(field, dims, mu, step):
    """field[x] -> field[x + step*mu_hat], periodic; field's first axis is the canonical site."""
    n0, n1, n2, n3 = dims
    f = field.reshape((n3, n2, n1, n0) + field.shape[1:])
    return np.roll(f, -step, axis=3 - mu).reshape(field.shape)


def K_numpy(uc, dims):
    """K(x) = sum_mu U_mu(x) + U_mu(x-mu)^dagger (eq. 3) with np.roll."""
    K = np.zeros((uc.shape[0],) + uc.shape[2:], dtype=np.complex128)
    for mu in range(4):
        K += uc[:, mu] + dag(shift(uc[:, mu], dims, mu, -1))
    return K


def plaquette_numpy(uc, dims):
    nc = uc.shape[-1]
    tot = 0.0
    for mu in range(4):
        for nu in range(mu + 1, 4):
            a = uc[:, mu]
            b = shift(uc[:, nu], dims, mu, +1)
            c = dag(shift(uc[:, mu], dims, nu, +1))
            d = dag(uc[:, nu])
            tot += np.einsum("nii->", a @ b @ c @ d).real
    return tot / (6.0 * nc * uc.shape[0])


def delta_numpy(uc, dims):
    """Delta(x) = sum_mu A_mu(x) - A_mu(x-mu), A = [(U-U^dag)/(2i)]_traceless (eq. 1)."""
    nc = uc.shape[-1]
    A = (uc - dag(uc)) / 2j
    tr = np.einsum("nmii->nm", A) / nc
    A = A - tr[..., None, None] * np.eye(nc)
    D = np.zeros((uc.shape[0], nc, nc), dtype=np.complex128)
    for mu in range(4):
        D += A[:, mu] - shift(A[:, mu], dims, mu, -1)
    return D


def real(uc):
    return li.to_real(np.ascontiguousarray(uc))


def cplx(ur):
    return li.from_real(ur)


def random_hermitian_traceless(n, nc, rng):
    z = rng.standard_normal((n, nc, nc)) + 1j * rng.standard_normal((n, nc, nc))
    h = (z + dag(z)) / 2
    tr = np.einsum("nii->n", h) / nc
    return h - tr[:, None, None] * np.eye(nc)


def expm_i_hermitian(h):
    w, v = np.linalg.eigh(h)
    return (v * np.exp(1j * w)[:, None, :]) @ dag(v)
