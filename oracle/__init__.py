"""ctypes front end of the fp64 CPU oracle (oracle/oracle.cpp).  TEST INFRASTRUCTURE ONLY.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
import this.  It never imports the CUDA package and the CUDA package never imports it.

All fields are canonical real arrays: float64, C-contiguous, shape [V,4,nc,nc,2] (links) or
[V,nc,nc,2] (per-site matrices); site s = x0 + N0*(x1 + N1*(x2 + N2*x3)).
"""
from __future__ import annotations

import ctypes
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "oracle.cpp")
_LIB = os.path.join(_HERE, "liboracle.so")
_lib = None


def build(force: bool = False) -> str:
    """Compile oracle.cpp -> liboracle.so with g++ -O2 (no fast-math), OpenMP if available."""
    if not force and os.path.exists(_LIB) and os.path.getmtime(_LIB) >= os.path.getmtime(_SRC):
        return _LIB
    base = ["g++", "-O2", "-std=c++17", "-fPIC", "-shared", "-o", _LIB, _SRC]
    try:
        subprocess.run(base[:1] + ["-fopenmp"] + base[1:], check=True, capture_output=True)
    except subprocess.CalledProcessError:
        subprocess.run(base, check=True)
    return _LIB


def _load():
    global _lib
    if _lib is not None:
        return _lib
    build()
    lib = ctypes.CDLL(_LIB)
    i32p = ctypes.POINTER(ctypes.c_int32)
    dp = ctypes.POINTER(ctypes.c_double)
    lib.oracle_set_threads.argtypes = [ctypes.c_int]
    lib.oracle_set_threads.restype = ctypes.c_int
    lib.oracle_max_threads.restype = ctypes.c_int
    lib.oracle_su2_pow.argtypes = [dp, ctypes.c_double, dp]
    lib.oracle_K.argtypes = [i32p, ctypes.c_int, dp, dp]
    lib.oracle_site_G.argtypes = [ctypes.c_int, dp, ctypes.c_double, dp]
    lib.oracle_subgroup_step.argtypes = [ctypes.c_int, dp, ctypes.c_int, ctypes.c_int,
                                         ctypes.c_double, dp]
    lib.oracle_subgroup_step.restype = ctypes.c_int
    lib.oracle_or_sweep.argtypes = [i32p, ctypes.c_int, dp, ctypes.c_int, ctypes.c_double]
    lib.oracle_functional.argtypes = [i32p, ctypes.c_int, dp]
    lib.oracle_functional.restype = ctypes.c_double
    lib.oracle_delta.argtypes = [i32p, ctypes.c_int, dp, dp]
    lib.oracle_gauge_precision.argtypes = [i32p, ctypes.c_int, dp]
    lib.oracle_gauge_precision.restype = ctypes.c_double
    lib.oracle_gauge_transform.argtypes = [i32p, ctypes.c_int, dp, dp]
    lib.oracle_plaquette.argtypes = [i32p, ctypes.c_int, dp]
    lib.oracle_plaquette.restype = ctypes.c_double
    lib.oracle_reconstruct12.argtypes = [ctypes.c_int64, dp]
    lib.oracle_reunitarize.argtypes = [ctypes.c_int64, ctypes.c_int, dp]
    u32p = ctypes.POINTER(ctypes.c_uint32)
    lib.oracle_philox4x32_10.argtypes = [u32p, u32p, u32p]
    lib.oracle_su2_heatbath_samples.argtypes = [dp, ctypes.c_double, ctypes.c_uint64, ctypes.c_int64, dp]
    lib.oracle_sa_sweep.argtypes = [i32p, ctypes.c_int, dp, ctypes.c_int, ctypes.c_double, ctypes.c_uint64,
                                    ctypes.c_uint32]
    lib.oracle_site_G_micro.argtypes = [ctypes.c_int, dp, dp]
    lib.oracle_micro_sweep.argtypes = [i32p, ctypes.c_int, dp, ctypes.c_int]
    lib.oracle_su2_pow_series.argtypes = [dp, ctypes.c_double, ctypes.c_int, dp]
    lib.oracle_site_G_series.argtypes = [ctypes.c_int, dp, ctypes.c_double, ctypes.c_int, dp]
    lib.oracle_or_sweep_series.argtypes = [i32p, ctypes.c_int, dp, ctypes.c_int, ctypes.c_double, ctypes.c_int]
    lib.oracle_K_coulomb.argtypes = [i32p, ctypes.c_int, dp, dp]
    lib.oracle_delta_coulomb.argtypes = [i32p, ctypes.c_int, dp, dp]
    lib.oracle_or_sweep_coulomb.argtypes = [i32p, ctypes.c_int, dp, ctypes.c_int, ctypes.c_double]
    lib.oracle_coulomb_theta_F.argtypes = [i32p, ctypes.c_int, dp, dp, dp]
    lib.oracle_or_sweep_coulomb_masked.argtypes = [i32p, ctypes.c_int, dp, ctypes.c_int, ctypes.c_double,
                                                   ctypes.POINTER(ctypes.c_uint8)]
    _lib = lib
    return lib


def _dims(dims):
    arr = (ctypes.c_int32 * 4)(*[int(d) for d in dims])
    return arr


def _dp(a: np.ndarray):
    if a.dtype != np.float64 or not a.flags["C_CONTIGUOUS"]:
        raise TypeError("oracle arrays must be C-contiguous float64")
    return a.ctypes.data_as(ctypes.POINTER(ctypes.c_double))


def _check_links(dims, u: np.ndarray) -> int:
    v = int(np.prod([int(d) for d in dims]))
    if u.ndim != 5 or u.shape[0] != v or u.shape[1] != 4 or u.shape[2] != u.shape[3] or u.shape[4] != 2:
        raise ValueError(f"links must be [V,4,nc,nc,2], got {u.shape}")
    if u.shape[2] not in (2, 3):
        raise ValueError("nc must be 2 or 3")
    return u.shape[2]


def set_threads(n: int) -> int:
    return _load().oracle_set_threads(int(n))


def max_threads() -> int:
    return _load().oracle_max_threads()


def su2_pow(q, omega: float) -> np.ndarray:
    q = np.ascontiguousarray(q, dtype=np.float64)
    out = np.empty(4)
    _load().oracle_su2_pow(_dp(q), float(omega), _dp(out))
    return out


def K_field(dims, u: np.ndarray) -> np.ndarray:
    nc = _check_links(dims, u)
    out = np.empty((u.shape[0], nc, nc, 2))
    _load().oracle_K(_dims(dims), nc, _dp(u), _dp(out))
    return out


def site_G(K: np.ndarray, omega: float) -> np.ndarray:
    """K real [nc,nc,2] -> G real [nc,nc,2]."""
    K = np.ascontiguousarray(K, dtype=np.float64)
    out = np.empty_like(K)
    _load().oracle_site_G(K.shape[0], _dp(K), float(omega), _dp(out))
    return out


def subgroup_step(K: np.ndarray, i: int, j: int, omega: float):
    K = np.ascontiguousarray(K, dtype=np.float64)
    out = np.empty_like(K)
    ok = _load().oracle_subgroup_step(K.shape[0], _dp(K), int(i), int(j), float(omega), _dp(out))
    return out, bool(ok)


def or_sweep(dims, u: np.ndarray, parity: int, omega: float) -> None:
    """One half-sweep, in place."""
    nc = _check_links(dims, u)
    _load().oracle_or_sweep(_dims(dims), nc, _dp(u), int(parity), float(omega))


def full_sweep(dims, u: np.ndarray, omega: float) -> None:
    """Black (parity 0) then white (parity 1) half-sweep, in place."""
    or_sweep(dims, u, 0, omega)
    or_sweep(dims, u, 1, omega)


def functional(dims, u: np.ndarray) -> float:
    nc = _check_links(dims, u)
    return float(_load().oracle_functional(_dims(dims), nc, _dp(u)))


def delta_field(dims, u: np.ndarray) -> np.ndarray:
    nc = _check_links(dims, u)
    out = np.empty((u.shape[0], nc, nc, 2))
    _load().oracle_delta(_dims(dims), nc, _dp(u), _dp(out))
    return out


def gauge_precision(dims, u: np.ndarray) -> float:
    nc = _check_links(dims, u)
    return float(_load().oracle_gauge_precision(_dims(dims), nc, _dp(u)))


def gauge_transform(dims, u: np.ndarray, g: np.ndarray) -> None:
    nc = _check_links(dims, u)
    if g.shape != (u.shape[0], nc, nc, 2):
        raise ValueError("g must be [V,nc,nc,2]")
    _load().oracle_gauge_transform(_dims(dims), nc, _dp(u), _dp(g))


def plaquette(dims, u: np.ndarray) -> float:
    nc = _check_links(dims, u)
    return float(_load().oracle_plaquette(_dims(dims), nc, _dp(u)))


def reconstruct12(m: np.ndarray) -> None:
    """In place: rebuild row 2 = conj(row0 x row1) of every 3x3 matrix in real [...,3,3,2]."""
    if m.shape[-3:] != (3, 3, 2):
        raise ValueError("need [...,3,3,2]")
    _load().oracle_reconstruct12(int(m.size // 18), _dp(m))


# ---- Coulomb gauge (reading C-22): spatial directions only, per time-slice ----------

def K_coulomb_field(dims, u: np.ndarray) -> np.ndarray:
    nc = _check_links(dims, u)
    out = np.empty((u.shape[0], nc, nc, 2))
    _load().oracle_K_coulomb(_dims(dims), nc, _dp(u), _dp(out))
    return out


def delta_coulomb_field(dims, u: np.ndarray) -> np.ndarray:
    nc = _check_links(dims, u)
    out = np.empty((u.shape[0], nc, nc, 2))
    _load().oracle_delta_coulomb(_dims(dims), nc, _dp(u), _dp(out))
    return out


def or_sweep_coulomb(dims, u: np.ndarray, parity: int, omega: float) -> None:
    """One Coulomb-gauge half-sweep, in place."""
    nc = _check_links(dims, u)
    _load().oracle_or_sweep_coulomb(_dims(dims), nc, _dp(u), int(parity), float(omega))


def or_sweep_coulomb_masked(dims, u: np.ndarray, parity: int, omega: float, active) -> None:
    """Coulomb half-sweep over the time-slices t with active[t] != 0 only."""
    nc = _check_links(dims, u)
    a = np.ascontiguousarray(active, dtype=np.uint8)
    if a.shape != (int(dims[3]),):
        raise ValueError("active must have dims[3] entries")
    _load().oracle_or_sweep_coulomb_masked(_dims(dims), nc, _dp(u), int(parity), float(omega),
                                           a.ctypes.data_as(ctypes.POINTER(ctypes.c_uint8)))


def full_sweep_coulomb(dims, u: np.ndarray, omega: float) -> None:
    or_sweep_coulomb(dims, u, 0, omega)
    or_sweep_coulomb(dims, u, 1, omega)


def coulomb_theta_F(dims, u: np.ndarray):
    """(theta_t, F_t): float64 arrays of length N3, one value per time-slice."""
    nc = _check_links(dims, u)
    n3 = int(dims[3])
    th, f = np.empty(n3), np.empty(n3)
    _load().oracle_coulomb_theta_F(_dims(dims), nc, _dp(u), _dp(th), _dp(f))
    return th, f


def reunitarize(m: np.ndarray) -> None:
    """In place: project every nc x nc matrix of real [...,nc,nc,2] back onto SU(nc) by Gram-Schmidt
    on the first rows (reading C-23)."""
    nc = m.shape[-2]
    if m.shape[-3:] != (nc, nc, 2) or nc not in (2, 3):
        raise ValueError("need [...,nc,nc,2] with nc = 2 or 3")
    _load().oracle_reunitarize(int(m.size // (2 * nc * nc)), nc, _dp(m))


# ---- truncated-series overrelaxation (reading C-24) ------------------------------------

def su2_pow_series(q, omega: float, order: int) -> np.ndarray:
    q = np.ascontiguousarray(q, dtype=np.float64)
    out = np.empty(4)
    _load().oracle_su2_pow_series(_dp(q), float(omega), int(order), _dp(out))
    return out


def site_G_series(K: np.ndarray, omega: float, order: int) -> np.ndarray:
    K = np.ascontiguousarray(K, dtype=np.float64)
    out = np.empty_like(K)
    _load().oracle_site_G_series(K.shape[0], _dp(K), float(omega), int(order), _dp(out))
    return out


def or_sweep_series(dims, u: np.ndarray, parity: int, omega: float, order: int) -> None:
    nc = _check_links(dims, u)
    _load().oracle_or_sweep_series(_dims(dims), nc, _dp(u), int(parity), float(omega), int(order))


def full_sweep_series(dims, u: np.ndarray, omega: float, order: int) -> None:
    or_sweep_series(dims, u, 0, omega, order)
    or_sweep_series(dims, u, 1, omega, order)


# ---- simulated annealing (reading C-25) --------------------------------------------------

def philox4x32_10(ctr, key) -> np.ndarray:
    c = np.ascontiguousarray(ctr, dtype=np.uint32)
    k = np.ascontiguousarray(key, dtype=np.uint32)
    out = np.empty(4, dtype=np.uint32)
    u32p = ctypes.POINTER(ctypes.c_uint32)
    _load().oracle_philox4x32_10(c.ctypes.data_as(u32p), k.ctypes.data_as(u32p), out.ctypes.data_as(u32p))
    return out


def su2_heatbath_samples(p, T: float, seed: int, n: int) -> np.ndarray:
    p = np.ascontiguousarray(p, dtype=np.float64)
    out = np.empty((int(n), 4))
    _load().oracle_su2_heatbath_samples(_dp(p), float(T), int(seed), int(n), _dp(out))
    return out


def sa_sweep(dims, u: np.ndarray, parity: int, T: float, seed: int, counter: int) -> None:
    """One simulated-annealing half-sweep at temperature T, in place."""
    nc = _check_links(dims, u)
    _load().oracle_sa_sweep(_dims(dims), nc, _dp(u), int(parity), float(T), int(seed), int(counter))


# ---- microcanonical step (reading C-26) ---------------------------------------------------

def site_G_micro(K: np.ndarray) -> np.ndarray:
    K = np.ascontiguousarray(K, dtype=np.float64)
    out = np.empty_like(K)
    _load().oracle_site_G_micro(K.shape[0], _dp(K), _dp(out))
    return out


def micro_sweep(dims, u: np.ndarray, parity: int) -> None:
    """One microcanonical half-sweep (per-subgroup reflection g^2, F unchanged), in place."""
    nc = _check_links(dims, u)
    _load().oracle_micro_sweep(_dims(dims), nc, _dp(u), int(parity))


def sa_anneal_micro(dims, u: np.ndarray, T_max: float, T_min: float, n_sweeps: int, n_micro: int,
                    seed: int) -> None:
    """The schedule of culgt_sa_anneal_micro: annealing sweep i (T linear from T_max to T_min,
    half-sweep counters 2i, 2i+1) followed by n_micro microcanonical full sweeps."""
    for i in range(int(n_sweeps)):
        T = T_max - (T_max - T_min) * i / (n_sweeps - 1) if n_sweeps > 1 else T_min
        for parity in (0, 1):
            sa_sweep(dims, u, parity, T, seed, 2 * i + parity)
        for _ in range(int(n_micro)):
            for parity in (0, 1):
                micro_sweep(dims, u, parity)
