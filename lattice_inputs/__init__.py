"""Seeded synthetic gauge-field inputs (shared by the oracle tests, the GPU parity tests and bench.py).

This module only MAKES INPUTS.  It holds none of the method's arithmetic (no K(x), no
subgroup solve, no overrelaxation, no theta/F): the oracle (`oracle/`) and the CUDA path
(`paper_1412_3655_b200/`) are both handed the arrays made here and neither imports the
other.  It depends on numpy only.

Recipes follow BASELINE.json `configs[0..4]` (restated in DESIGN.md "Input recipe"):

* near-identity SU(3):  U = exp(i*eps*H),  H = sum_a c_a lambda_a/2 with c_a ~ N(0,1)
  (Gell-Mann basis), then re-unitarised (Gram-Schmidt rows 0,1; row 2 = conj(row0 x row1)).
* Haar SU(3): two complex Gaussian 3-vectors -> Gram-Schmidt -> row 2 = conj(row0 x row1).
* Haar SU(2): 4 Gaussians normalised to the unit 3-sphere -> (a0,a1,a2,a3).
* gauge scramble: U_mu(x) <- g(x) U_mu(x) g(x+mu)^dagger with Haar g(x)
  (the transformation law, used here only to SYNTHESISE an input).
* pure gauge: U_mu(x) = g(x) g(x+mu)^dagger.

Canonical layout: site index s = x0 + N0*(x1 + N1*(x2 + N2*x3)),
complex array U[s, mu, row, col]; the real view is real[V][4][Nc][Nc][2].

Random numbers: numpy Philox keyed by (seed, stream, chunk) and consumed in canonical order
chunk by chunk, so an array does not depend on how much memory the host has.
"""
from __future__ import annotations

import numpy as np

__all__ = [
    "volume", "site_coords", "parity_of_sites", "haar_su3", "haar_su2", "near_identity_su3",
    "gauge_scramble", "pure_gauge", "make_config", "to_real", "from_real", "round_to_fp32",
    "CONFIGS",
]

_CHUNK = 1 << 18  # matrices per RNG chunk (fixed: part of the recipe)

# Gell-Mann matrices lambda_1..lambda_8
_GM = np.zeros((8, 3, 3), dtype=np.complex128)
_GM[0][0, 1] = _GM[0][1, 0] = 1
_GM[1][0, 1] = -1j
_GM[1][1, 0] = 1j
_GM[2][0, 0] = 1
_GM[2][1, 1] = -1
_GM[3][0, 2] = _GM[3][2, 0] = 1
_GM[4][0, 2] = -1j
_GM[4][2, 0] = 1j
_GM[5][1, 2] = _GM[5][2, 1] = 1
_GM[6][1, 2] = -1j
_GM[6][2, 1] = 1j
_GM[7][0, 0] = _GM[7][1, 1] = 1 / np.sqrt(3.0)
_GM[7][2, 2] = -2 / np.sqrt(3.0)


def volume(dims) -> int:
    n0, n1, n2, n3 = (int(d) for d in dims)
    return n0 * n1 * n2 * n3


def site_coords(dims) -> np.ndarray:
    """int32 array [V,4] of (x0,x1,x2,x3) in canonical site order (x0 fastest)."""
    n0, n1, n2, n3 = (int(d) for d in dims)
    s = np.arange(n0 * n1 * n2 * n3, dtype=np.int64)
    out = np.empty((s.size, 4), dtype=np.int32)
    out[:, 0] = s % n0
    out[:, 1] = (s // n0) % n1
    out[:, 2] = (s // (n0 * n1)) % n2
    out[:, 3] = s // (n0 * n1 * n2)
    return out


def parity_of_sites(dims) -> np.ndarray:
    """uint8 array [V]: (x0+x1+x2+x3)&1; 0 = black (reading C-1)."""
    return (site_coords(dims).sum(axis=1) & 1).astype(np.uint8)


def _rng(seed: int, stream: int, chunk: int) -> np.random.Generator:
    return np.random.Generator(np.random.Philox(key=[(int(seed) << 20) ^ int(stream), int(chunk)]))


def _chunks(n: int):
    for c, lo in enumerate(range(0, n, _CHUNK)):
        yield c, lo, min(n, lo + _CHUNK)


def _fill_chunks(out: np.ndarray, make_chunk, threads: bool = True, first: int = 0) -> np.ndarray:
    """out = elements [first, first + len(out)) of the sequence whose RNG chunk c makes elements
    [c*_CHUNK, (c+1)*_CHUNK): out[...] = make_chunk(c, m)[...] for every chunk that overlaps the range
    (m = how many leading elements of the chunk are needed; a generator's first m elements do not depend
    on how many more are drawn).  Chunks are independent (each has its own Philox key), so they may be
    filled by a few threads -- the array does not depend on how many.  (threads=False for generators
    made of stacked 3x3 matmuls, which run slower side by side.)"""
    last = first + out.shape[0]

    def job(c):
        lo, hi = max(first, c * _CHUNK), min(last, (c + 1) * _CHUNK)
        out[lo - first:hi - first] = make_chunk(c, hi - c * _CHUNK)[lo - c * _CHUNK:]

    items = list(range(first // _CHUNK, (last + _CHUNK - 1) // _CHUNK)) if last > first else []
    if len(items) <= 1 or not threads:
        for item in items:
            job(item)
    else:
        import os
        from concurrent.futures import ThreadPoolExecutor
        with ThreadPoolExecutor(max_workers=min(len(items), os.cpu_count() or 1, 16)) as ex:
            list(ex.map(job, items))
    return out


def _cross_conj(a: np.ndarray, b: np.ndarray) -> np.ndarray:
    return np.conj(np.cross(a, b))


def _gram_schmidt_su3(a: np.ndarray, b: np.ndarray) -> np.ndarray:
    """Rows a, b ([n,3] complex) -> SU(3) matrices [n,3,3]: orthonormalise, third row closes det=1."""
    a = a / np.linalg.norm(a, axis=1, keepdims=True)
    b = b - a * np.sum(np.conj(a) * b, axis=1, keepdims=True)
    b = b / np.linalg.norm(b, axis=1, keepdims=True)
    out = np.empty((a.shape[0], 3, 3), dtype=np.complex128)
    out[:, 0] = a
    out[:, 1] = b
    out[:, 2] = _cross_conj(a, b)
    return out


def haar_su3(n: int, seed: int, stream: int = 0, first: int = 0) -> np.ndarray:
    """n Haar SU(3) matrices: elements [first, first + n) of the (seed, stream) sequence."""
    def chunk(c, m):
        z = _rng(seed, stream, c).standard_normal((m, 12))
        return _gram_schmidt_su3(z[:, 0:3] + 1j * z[:, 3:6], z[:, 6:9] + 1j * z[:, 9:12])

    return _fill_chunks(np.empty((n, 3, 3), dtype=np.complex128), chunk, first=first)


def su2_from_quaternion(a: np.ndarray) -> np.ndarray:
    """(a0,a1,a2,a3) [n,4] -> [[a0+i a3, a2+i a1], [-a2+i a1, a0-i a3]] (reading C-7)."""
    out = np.empty((a.shape[0], 2, 2), dtype=np.complex128)
    out[:, 0, 0] = a[:, 0] + 1j * a[:, 3]
    out[:, 0, 1] = a[:, 2] + 1j * a[:, 1]
    out[:, 1, 0] = -a[:, 2] + 1j * a[:, 1]
    out[:, 1, 1] = a[:, 0] - 1j * a[:, 3]
    return out


def haar_su2(n: int, seed: int, stream: int = 0, first: int = 0) -> np.ndarray:
    def chunk(c, m):
        z = _rng(seed, stream, c).standard_normal((m, 4))
        z /= np.linalg.norm(z, axis=1, keepdims=True)
        return su2_from_quaternion(z)

    return _fill_chunks(np.empty((n, 2, 2), dtype=np.complex128), chunk, first=first)


def _expm_i_hermitian(h: np.ndarray) -> np.ndarray:
    """exp(i h) for a stack of small Hermitian matrices: scaling-and-squaring Taylor series."""
    n = h.shape[-1]
    a = 1j * h / 64.0  # 2^-6
    eye = np.broadcast_to(np.eye(n, dtype=np.complex128), a.shape)
    term = eye.copy()
    acc = eye.copy()
    for k in range(1, 13):
        term = np.matmul(term, a) / k
        acc = acc + term
    for _ in range(6):
        acc = np.matmul(acc, acc)
    return acc


def near_identity_su3(n: int, eps: float, seed: int, stream: int = 0, first: int = 0) -> np.ndarray:
    def chunk(c, m):
        coef = _rng(seed, stream, c).standard_normal((m, 8))
        h = np.tensordot(coef, _GM, axes=(1, 0)) * 0.5
        u = _expm_i_hermitian(eps * h)
        return _gram_schmidt_su3(u[:, 0], u[:, 1])

    return _fill_chunks(np.empty((n, 3, 3), dtype=np.complex128), chunk, threads=False, first=first)


def near_identity_su2(n: int, eps: float, seed: int, stream: int = 0, first: int = 0) -> np.ndarray:
    """exp(i*eps*c.sigma/2), c ~ N(0,1)^3 (closed form on the 3-sphere)."""
    def chunk(c, m):
        v = _rng(seed, stream, c).standard_normal((m, 3)) * (0.5 * eps)
        r = np.linalg.norm(v, axis=1)
        q = np.empty((m, 4))
        q[:, 0] = np.cos(r)
        q[:, 1:] = v * (np.sinc(r / np.pi))[:, None]
        return su2_from_quaternion(q)

    return _fill_chunks(np.empty((n, 2, 2), dtype=np.complex128), chunk, first=first)


def _shift_sites(field: np.ndarray, dims, mu: int, step: int) -> np.ndarray:
    """field[x] -> field[x + step*mu_hat] (periodic), field indexed by canonical site first."""
    n0, n1, n2, n3 = (int(d) for d in dims)
    tail = field.shape[1:]
    f = field.reshape((n3, n2, n1, n0) + tail)
    f = np.roll(f, -step, axis=3 - mu)
    return f.reshape(field.shape)


def gauge_scramble(u: np.ndarray, g: np.ndarray, dims) -> np.ndarray:
    """U_mu(x) <- g(x) U_mu(x) g(x+mu)^dagger; u [V,4,nc,nc], g [V,nc,nc] (input synthesis only)."""
    out = np.empty_like(u)
    for mu in range(4):
        gf = _shift_sites(g, dims, mu, +1)
        out[:, mu] = np.matmul(np.matmul(g, u[:, mu]), np.conj(np.swapaxes(gf, 1, 2)))
    return out


def pure_gauge(g: np.ndarray, dims) -> np.ndarray:
    v, nc = g.shape[0], g.shape[1]
    out = np.empty((v, 4, nc, nc), dtype=np.complex128)
    for mu in range(4):
        gf = _shift_sites(g, dims, mu, +1)
        out[:, mu] = np.matmul(g, np.conj(np.swapaxes(gf, 1, 2)))
    return out


def make_config(dims, group: int, kind: str, seed: int, eps: float = 0.0,
                scramble: bool = False, t_range=None) -> np.ndarray:
    """Complex128 canonical field U[V,4,nc,nc].

    kind: "near_identity" (needs eps), "haar" (hot), "unit", "pure_gauge".
    scramble: apply a Haar random gauge transformation g(x) (stream 1 of the same seed).
    t_range = (t_lo, t_hi): only the sites of the time-slices [t_lo, t_hi) -- exactly the rows
    [t_lo*Vs, t_hi*Vs) of the full field (Vs = N0*N1*N2; t is the slowest coordinate), made without
    making the rest (one time slab per rank, bench.py --sharded).
    """
    if group not in (2, 3):
        raise ValueError("group must be 2 or 3")
    n0, n1, n2, n3 = (int(d) for d in dims)
    vs = n0 * n1 * n2
    t_lo, t_hi = (0, n3) if t_range is None else (int(t_range[0]), int(t_range[1]))
    if not 0 <= t_lo < t_hi <= n3:
        raise ValueError("t_range outside the lattice")
    v = vs * (t_hi - t_lo)
    haar = haar_su3 if group == 3 else haar_su2

    def g_field():
        """g(x) on the slices [t_lo, t_hi] (the slice behind the range is needed for g(x + t_hat); periodic)"""
        g = np.empty((v + vs, group, group), dtype=np.complex128)
        g[:v] = haar(v, seed, 1, first=vs * t_lo)
        g[v:] = haar(vs, seed, 1, first=vs * (t_hi % n3))
        return g

    if kind == "near_identity":
        near = near_identity_su3 if group == 3 else near_identity_su2
        u = near(4 * v, eps, seed, 0, first=4 * vs * t_lo).reshape(v, 4, group, group)
    elif kind == "haar":
        u = haar(4 * v, seed, 0, first=4 * vs * t_lo).reshape(v, 4, group, group)
    elif kind == "unit":
        u = np.broadcast_to(np.eye(group, dtype=np.complex128), (v, 4, group, group)).copy()
    elif kind == "pure_gauge":
        if t_range is None:
            return pure_gauge(haar(v, seed, 1), dims)
        u = np.broadcast_to(np.eye(group, dtype=np.complex128), (v, 4, group, group)).copy()
        return _scramble_slices(u, g_field(), (n0, n1, n2, t_hi - t_lo))
    else:
        raise ValueError(f"unknown kind {kind!r}")
    if scramble:
        if t_range is None:
            u = gauge_scramble(u, haar(v, seed, 1), dims)
        else:
            u = _scramble_slices(u, g_field(), (n0, n1, n2, t_hi - t_lo))
    return u


def _scramble_slices(u: np.ndarray, g: np.ndarray, dims_loc) -> np.ndarray:
    """gauge_scramble on a range of time-slices: g carries one extra slice (the one behind the range),
    spatial shifts are periodic inside a slice, the t shift reads the next slice of g."""
    n0, n1, n2, nt = dims_loc
    vs = n0 * n1 * n2
    v = vs * nt
    out = np.empty_like(u)
    gs = g[:v]
    for mu in range(3):
        gf = _shift_sites(gs, dims_loc, mu, +1)
        out[:, mu] = np.matmul(np.matmul(gs, u[:, mu]), np.conj(np.swapaxes(gf, 1, 2)))
    gf = g[vs:v + vs]                                   # g(x + t_hat): the same site one slice later
    out[:, 3] = np.matmul(np.matmul(gs, u[:, 3]), np.conj(np.swapaxes(gf, 1, 2)))
    return out


def to_real(uc: np.ndarray, dtype=np.float64) -> np.ndarray:
    """complex [...,nc,nc] -> real [...,nc,nc,2] (re, im interleaved), C-contiguous."""
    out = np.empty(uc.shape + (2,), dtype=dtype)
    out[..., 0] = uc.real
    out[..., 1] = uc.imag
    return out


def from_real(ur: np.ndarray) -> np.ndarray:
    return ur[..., 0].astype(np.float64) + 1j * ur[..., 1].astype(np.float64)


def round_to_fp32(uc: np.ndarray) -> np.ndarray:
    """Round every real component to the nearest fp32 value (returned as complex128)."""
    return uc.astype(np.complex64).astype(np.complex128)


# BASELINE.json configs[0..4].  Seeds are per-config constants.
CONFIGS = {
    "cfg0": dict(dims=(4, 4, 4, 4), group=3, precision=64, params=18, kind="near_identity",
                 eps=0.3, scramble=True, omega=1.7, seed=1000),
    "cfg1": dict(dims=(8, 8, 8, 8), group=2, precision=64, params=4, kind="haar",
                 eps=0.0, scramble=False, omega=1.5, seed=1001),
    "cfg2": dict(dims=(16, 16, 16, 16), group=3, precision=32, params=12, kind="near_identity",
                 eps=0.5, scramble=True, omega=1.7, seed=1002),
    "cfg3_fp32": dict(dims=(32, 32, 32, 32), group=3, precision=32, params=12,
                      kind="near_identity", eps=0.8, scramble=True, omega=1.7, seed=1003),
    "cfg3_fp64": dict(dims=(32, 32, 32, 32), group=3, precision=64, params=18,
                      kind="near_identity", eps=0.8, scramble=True, omega=1.7, seed=1003),
    # same lattice and input as cfg3 in the two remaining storage formats (SURVEY.md 8(f) NEXT-2d)
    "cfg3_fp32_18": dict(dims=(32, 32, 32, 32), group=3, precision=32, params=18,
                         kind="near_identity", eps=0.8, scramble=True, omega=1.7, seed=1003),
    "cfg3_fp64_12": dict(dims=(32, 32, 32, 32), group=3, precision=64, params=12,
                         kind="near_identity", eps=0.8, scramble=True, omega=1.7, seed=1003),
    # the SU(2) path of cfg1 at the headline volume (not a BASELINE.json config; measurement only)
    "su2_32_fp64": dict(dims=(32, 32, 32, 32), group=2, precision=64, params=4, kind="haar",
                        eps=0.0, scramble=False, omega=1.5, seed=1001),
    "su2_32_fp32": dict(dims=(32, 32, 32, 32), group=2, precision=32, params=4, kind="haar",
                        eps=0.0, scramble=False, omega=1.5, seed=1001),
    # L2-resident SU(3) volumes (measurement only: the SM-side limit of the sweep kernel)
    "l2_24_fp32": dict(dims=(24, 24, 24, 24), group=3, precision=32, params=12,
                       kind="near_identity", eps=0.8, scramble=True, omega=1.7, seed=1003),
    "l2_20_fp64": dict(dims=(20, 20, 20, 20), group=3, precision=64, params=18,
                       kind="near_identity", eps=0.8, scramble=True, omega=1.7, seed=1003),
    "cfg4_fp32": dict(dims=(48, 48, 48, 96), group=3, precision=32, params=12, kind="haar",
                      eps=0.0, scramble=False, omega=1.7, seed=1004),
    "cfg4_fp64": dict(dims=(64, 64, 64, 64), group=3, precision=64, params=18, kind="haar",
                      eps=0.0, scramble=False, omega=1.7, seed=1005),
}


def make_named(name: str) -> np.ndarray:
    c = CONFIGS[name]
    return make_config(c["dims"], c["group"], c["kind"], c["seed"], eps=c["eps"],
                       scramble=c["scramble"])
