"""paper_1412_3655_b200 -- B200-native checkerboard overrelaxation for lattice Landau gauge fixing.

Thin Python binding of the C-ABI library libculgt_b200.so (include/culgt_b200.h): the functions
here have the same names as the C entry points and only marshal arguments (torch tensors ->
device pointers, the current torch stream -> cudaStream_t).  Every step of the method runs in
the CUDA kernels under csrc/.  PyTorch is used for device memory and streams only.

There is NO CPU fallback: importing works anywhere (so the ABI can be inspected), but the
library must have been built (python -m paper_1412_3655_b200.build) and every compute call
needs a CUDA device, else it raises.
"""
from __future__ import annotations

import ctypes
import os
from dataclasses import dataclass

_HERE = os.path.dirname(os.path.abspath(__file__))
# CULGT_MEASURE=1 selects the separately built measurement library (build.py --measure); default: the product
LIB_PATH = os.path.join(_HERE, "libculgt_b200_measure.so" if os.environ.get("CULGT_MEASURE", "") not in ("", "0")
                        else "libculgt_b200.so")

CULGT_OK = 0
ERRORS = {
    "CULGT_ERR_NULL": -1, "CULGT_ERR_DIMS": -2, "CULGT_ERR_DESC": -3, "CULGT_ERR_PARITY": -4,
    "CULGT_ERR_OMEGA": -5, "CULGT_ERR_ALIGN": -6, "CULGT_ERR_CUDA": -7, "CULGT_ERR_ARG": -8,
    "CULGT_ERR_NCCL": -9, "CULGT_ERR_TOO_LARGE": -10,
}
NOALLOC_MAX_SITES = 1 << 24   # CULGT_NOALLOC_MAX_SITES
FLOPS_PER_SITE = {3: 2304, 2: 278}   # fixed algorithmic counts, DESIGN.md "Measurement"


class CulgtError(RuntimeError):
    def __init__(self, status: int, where: str):
        self.status = status
        msg = lib().culgt_strerror(status).decode()
        if status in (ERRORS["CULGT_ERR_CUDA"], ERRORS["CULGT_ERR_NCCL"]):
            msg += ": " + lib().culgt_last_cuda_error().decode()
        super().__init__(f"{where}: {msg} ({status})")


class culgt_lattice(ctypes.Structure):
    _fields_ = [("dims", ctypes.c_int32 * 4), ("group", ctypes.c_int32),
                ("precision", ctypes.c_int32), ("params", ctypes.c_int32)]


_lib = None


def lib() -> ctypes.CDLL:
    """Load libculgt_b200.so (fails loudly if it has not been built)."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise ImportError(f"{LIB_PATH} is missing: build it with "
                          "`python -m paper_1412_3655_b200.build` (there is no CPU fallback)")
    L = ctypes.CDLL(LIB_PATH)
    latp = ctypes.POINTER(culgt_lattice)
    vp = ctypes.c_void_p
    dp = ctypes.POINTER(ctypes.c_double)
    for name in ("culgt_links_bytes", "culgt_canonical_bytes", "culgt_gfield_bytes", "culgt_workspace_bytes"):
        getattr(L, name).argtypes = [latp]
        getattr(L, name).restype = ctypes.c_size_t
    L.culgt_validate.argtypes = [latp]
    L.culgt_pack.argtypes = [latp, vp, vp, vp]
    L.culgt_unpack.argtypes = [latp, vp, vp, vp]
    L.culgt_reunitarize.argtypes = [latp, vp, vp]
    L.culgt_or_sweep.argtypes = [latp, vp, ctypes.c_int, ctypes.c_double, vp]
    L.culgt_or_sweeps.argtypes = [latp, vp, ctypes.c_int, ctypes.c_double, vp]
    if hasattr(L, "culgt_or_sweeps_ws"):       # measurement library only (csrc/measure_api.h)
        L.culgt_or_sweeps_ws.argtypes = [latp, vp, vp, ctypes.c_int, ctypes.c_double, vp]
    L.culgt_gauge_precision.argtypes = [latp, vp, vp, vp, vp]
    L.culgt_functional.argtypes = [latp, vp, vp, vp, vp]
    L.culgt_gauge_precision_functional.argtypes = [latp, vp, vp, vp, vp, vp]
    L.culgt_gauge_precision_functional_noalloc.argtypes = [latp, vp, vp, vp, vp]
    L.culgt_gauge_transform.argtypes = [latp, vp, vp, vp]
    L.culgt_landau_fix.argtypes = [latp, vp, vp, ctypes.c_double, ctypes.c_double, ctypes.c_int,
                                   ctypes.c_int, ctypes.POINTER(ctypes.c_int), dp, dp, vp]
    L.culgt_fix_host.argtypes = [latp, vp, vp, vp, vp, ctypes.c_int, ctypes.c_double, dp, dp, vp]
    L.culgt_or_sweep_series.argtypes = [latp, vp, ctypes.c_int, ctypes.c_double, ctypes.c_int, vp]
    L.culgt_or_sweeps_series.argtypes = [latp, vp, ctypes.c_int, ctypes.c_double, ctypes.c_int, vp]
    L.culgt_sa_sweep.argtypes = [latp, vp, ctypes.c_int, ctypes.c_double, ctypes.c_ulonglong, ctypes.c_uint, vp]
    L.culgt_sa_anneal.argtypes = [latp, vp, ctypes.c_double, ctypes.c_double, ctypes.c_int, ctypes.c_ulonglong, vp]
    L.culgt_micro_sweep.argtypes = [latp, vp, ctypes.c_int, vp]
    L.culgt_micro_sweeps.argtypes = [latp, vp, ctypes.c_int, vp]
    L.culgt_sa_anneal_micro.argtypes = [latp, vp, ctypes.c_double, ctypes.c_double, ctypes.c_int, ctypes.c_int,
                                        ctypes.c_ulonglong, vp]
    L.culgt_or_sweep_coulomb.argtypes = [latp, vp, ctypes.c_int, ctypes.c_double, vp]
    L.culgt_or_sweep_coulomb_masked.argtypes = [latp, vp, ctypes.c_int, ctypes.c_double, vp, vp]
    L.culgt_or_sweeps_coulomb.argtypes = [latp, vp, ctypes.c_int, ctypes.c_double, vp]
    L.culgt_coulomb_precision_functional.argtypes = [latp, vp, vp, vp, vp, vp]
    L.culgt_coulomb_fix.argtypes = [latp, vp, vp, ctypes.c_double, ctypes.c_double, ctypes.c_int, ctypes.c_int,
                                    ctypes.POINTER(ctypes.c_int), dp, dp, vp]
    L.culgt_set_sweep_variant.argtypes = [ctypes.c_int]
    L.culgt_autotune_sweep.argtypes = [latp, vp, vp, ctypes.c_double, ctypes.c_int, ctypes.POINTER(ctypes.c_int),
                                       ctypes.POINTER(ctypes.c_float), vp]
    szp = ctypes.POINTER(ctypes.c_size_t)
    ip = ctypes.POINTER(ctypes.c_int)
    L.culgt_slab_lattice.argtypes = [latp, ctypes.c_int, latp]
    for name in ("culgt_slab_links_bytes", "culgt_slab_halo_bytes"):
        getattr(L, name).argtypes = [latp]
        getattr(L, name).restype = ctypes.c_size_t
    L.culgt_slab_halo_chunks.argtypes = [latp, ctypes.c_int, ctypes.c_int, szp, szp, ip]
    L.culgt_slab_halo_peers.argtypes = [ctypes.c_int, ctypes.c_int, ctypes.c_int, ip, ip]
    L.culgt_slab_pack.argtypes = [latp, vp, vp, vp]
    L.culgt_slab_unpack.argtypes = [latp, vp, vp, vp]
    L.culgt_slab_or_sweep.argtypes = [latp, vp, ctypes.c_int, ctypes.c_double, vp]
    L.culgt_slab_or_sweep_window.argtypes = [latp, vp, ctypes.c_int, ctypes.c_double, ctypes.c_int, ctypes.c_int, vp]
    L.culgt_slab_halo_copy.argtypes = [latp, vp, vp, ctypes.c_int, ctypes.c_int, vp]
    L.culgt_slab_theta_F_sums.argtypes = [latp, vp, vp, vp, vp]
    L.culgt_slab_theta_F_combine.argtypes = [latp, vp, ctypes.c_int, vp, vp, vp]
    vpp = ctypes.POINTER(ctypes.c_void_p)
    L.culgt_slab_exchange_all_local.argtypes = [latp, vpp, ctypes.c_int, vp]
    L.culgt_slab_or_sweeps_local.argtypes = [latp, vpp, ctypes.c_int, ctypes.c_int, ctypes.c_double, ctypes.c_int, vp]
    L.culgt_slab_theta_F_local.argtypes = [latp, latp, vpp, ctypes.c_int, vp, vp, vp, vp, vp]
    L.culgt_slab_comm_unique_id.argtypes = [vp]
    L.culgt_slab_comm_create.argtypes = [vp, ctypes.c_int, ctypes.c_int, vpp]
    L.culgt_slab_comm_destroy.argtypes = [vp]
    L.culgt_slab_halo_exchange.argtypes = [vp, latp, vp, ctypes.c_int, ctypes.c_int, vp]
    L.culgt_slab_exchange_all_nccl.argtypes = [vp, latp, vp, vp]
    L.culgt_slab_or_sweeps_nccl.argtypes = [vp, latp, vp, ctypes.c_int, ctypes.c_double, vp, vp]
    L.culgt_slab_theta_F_nccl.argtypes = [vp, latp, latp, vp, vp, vp, vp, vp, vp]
    L.culgt_sweep_kernel_name.argtypes = [latp]
    L.culgt_sweep_kernel_name.restype = ctypes.c_char_p
    L.culgt_strerror.argtypes = [ctypes.c_int]
    L.culgt_strerror.restype = ctypes.c_char_p
    L.culgt_last_cuda_error.restype = ctypes.c_char_p
    _lib = L
    return L


@dataclass(frozen=True)
class Lattice:
    """Python mirror of the C `culgt_lattice` descriptor."""
    dims: tuple
    group: int = 3
    precision: int = 32
    params: int = 12

    def c(self) -> culgt_lattice:
        return culgt_lattice((ctypes.c_int32 * 4)(*[int(d) for d in self.dims]),
                             int(self.group), int(self.precision), int(self.params))

    @property
    def volume(self) -> int:
        v = 1
        for d in self.dims:
            v *= int(d)
        return v

    @property
    def torch_dtype(self):
        import torch
        return torch.float32 if self.precision == 32 else torch.float64


def _check(status: int, where: str) -> None:
    if status != CULGT_OK:
        raise CulgtError(status, where)


def _ptr(t) -> int:
    """Device (or host) address of a torch tensor / numpy array / raw int / None."""
    if t is None:
        return 0
    if isinstance(t, int):
        return t
    if hasattr(t, "data_ptr"):
        return t.data_ptr()
    if hasattr(t, "ctypes"):
        return t.ctypes.data
    raise TypeError(f"cannot take the address of {type(t)}")


def _stream(stream) -> int:
    if stream is None:
        import torch
        return torch.cuda.current_stream().cuda_stream
    if isinstance(stream, int):
        return stream
    return stream.cuda_stream


def _require_cuda():
    import torch
    if not torch.cuda.is_available():
        raise RuntimeError("paper_1412_3655_b200 needs a CUDA device; there is no CPU fallback")


# ---- sizes -----------------------------------------------------------------------------------

def culgt_validate(lat: Lattice) -> int:
    return lib().culgt_validate(ctypes.byref(lat.c()))


def culgt_links_bytes(lat: Lattice) -> int:
    return lib().culgt_links_bytes(ctypes.byref(lat.c()))


def culgt_canonical_bytes(lat: Lattice) -> int:
    return lib().culgt_canonical_bytes(ctypes.byref(lat.c()))


def culgt_gfield_bytes(lat: Lattice) -> int:
    return lib().culgt_gfield_bytes(ctypes.byref(lat.c()))


def culgt_workspace_bytes(lat: Lattice) -> int:
    return lib().culgt_workspace_bytes(ctypes.byref(lat.c()))


# ---- device-memory helpers (torch is the allocator) -------------------------------------------

def alloc_links(lat: Lattice, device="cuda"):
    import torch
    n = culgt_links_bytes(lat)
    if n == 0:
        _check(culgt_validate(lat), "alloc_links")
    return torch.empty(n // (lat.precision // 8), dtype=lat.torch_dtype, device=device)


def alloc_workspace(lat: Lattice, device="cuda"):
    import torch
    return torch.empty(culgt_workspace_bytes(lat) // 8, dtype=torch.float64, device=device)


# ---- the C entry points, same names ------------------------------------------------------------

def culgt_pack(lat: Lattice, canonical, links, stream=None) -> None:
    _require_cuda()
    _check(lib().culgt_pack(ctypes.byref(lat.c()), _ptr(canonical), _ptr(links), _stream(stream)), "culgt_pack")


def culgt_unpack(lat: Lattice, links, canonical, stream=None) -> None:
    _require_cuda()
    _check(lib().culgt_unpack(ctypes.byref(lat.c()), _ptr(links), _ptr(canonical), _stream(stream)), "culgt_unpack")


def culgt_reunitarize(lat: Lattice, links, stream=None) -> None:
    _require_cuda()
    _check(lib().culgt_reunitarize(ctypes.byref(lat.c()), _ptr(links), _stream(stream)), "culgt_reunitarize")


def culgt_or_sweep(lat: Lattice, links, parity: int, omega: float, stream=None) -> None:
    _require_cuda()
    _check(lib().culgt_or_sweep(ctypes.byref(lat.c()), _ptr(links), int(parity), float(omega),
                                _stream(stream)), "culgt_or_sweep")


def culgt_or_sweeps(lat: Lattice, links, n_sweeps: int, omega: float, stream=None) -> None:
    _require_cuda()
    _check(lib().culgt_or_sweeps(ctypes.byref(lat.c()), _ptr(links), int(n_sweeps), float(omega),
                                 _stream(stream)), "culgt_or_sweeps")


def culgt_or_sweeps_ws(lat: Lattice, links, workspace, n_sweeps: int, omega: float, stream=None) -> None:
    """Measurement library only (CULGT_MEASURE=1): full sweeps with a workspace, variant 60 = fused kernel."""
    _require_cuda()
    _check(lib().culgt_or_sweeps_ws(ctypes.byref(lat.c()), _ptr(links), _ptr(workspace), int(n_sweeps),
                                    float(omega), _stream(stream)), "culgt_or_sweeps_ws")


def culgt_gauge_precision(lat: Lattice, links, workspace, theta_dev, stream=None) -> None:
    _require_cuda()
    _check(lib().culgt_gauge_precision(ctypes.byref(lat.c()), _ptr(links), _ptr(workspace),
                                       _ptr(theta_dev), _stream(stream)), "culgt_gauge_precision")


def culgt_functional(lat: Lattice, links, workspace, F_dev, stream=None) -> None:
    _require_cuda()
    _check(lib().culgt_functional(ctypes.byref(lat.c()), _ptr(links), _ptr(workspace),
                                  _ptr(F_dev), _stream(stream)), "culgt_functional")


def culgt_gauge_precision_functional(lat: Lattice, links, workspace, theta_dev, F_dev, stream=None) -> None:
    _require_cuda()
    _check(lib().culgt_gauge_precision_functional(ctypes.byref(lat.c()), _ptr(links), _ptr(workspace),
                                                  _ptr(theta_dev), _ptr(F_dev), _stream(stream)),
           "culgt_gauge_precision_functional")


def culgt_gauge_precision_functional_noalloc(lat: Lattice, links, theta_dev, F_dev, stream=None) -> None:
    """theta and F without a workspace: the partials live in a 2 MiB device array of the library
    (at most NOALLOC_MAX_SITES sites); allocates nothing."""
    _require_cuda()
    _check(lib().culgt_gauge_precision_functional_noalloc(ctypes.byref(lat.c()), _ptr(links), _ptr(theta_dev),
                                                          _ptr(F_dev), _stream(stream)),
           "culgt_gauge_precision_functional_noalloc")


def culgt_gauge_transform(lat: Lattice, links, g, stream=None) -> None:
    _require_cuda()
    _check(lib().culgt_gauge_transform(ctypes.byref(lat.c()), _ptr(links), _ptr(g), _stream(stream)),
           "culgt_gauge_transform")


def culgt_landau_fix(lat: Lattice, links, workspace, omega: float, theta_target: float,
                     max_sweeps: int, check_every: int = 1, stream=None):
    """Returns (sweeps_done, theta, F)."""
    _require_cuda()
    done = ctypes.c_int(0)
    theta = ctypes.c_double(0.0)
    F = ctypes.c_double(0.0)
    _check(lib().culgt_landau_fix(ctypes.byref(lat.c()), _ptr(links), _ptr(workspace), float(omega),
                                  float(theta_target), int(max_sweeps), int(check_every),
                                  ctypes.byref(done), ctypes.byref(theta), ctypes.byref(F),
                                  _stream(stream)), "culgt_landau_fix")
    return done.value, theta.value, F.value


def culgt_fix_host(lat: Lattice, canonical_host, canonical_dev, links_dev, workspace,
                   n_sweeps: int, omega: float, stream=None):
    """Host-buffer end-to-end call; canonical_host is updated in place. Returns (theta, F)."""
    _require_cuda()
    theta = ctypes.c_double(0.0)
    F = ctypes.c_double(0.0)
    _check(lib().culgt_fix_host(ctypes.byref(lat.c()), _ptr(canonical_host), _ptr(canonical_dev),
                                _ptr(links_dev), _ptr(workspace), int(n_sweeps), float(omega),
                                ctypes.byref(theta), ctypes.byref(F), _stream(stream)), "culgt_fix_host")
    return theta.value, F.value


# ---- truncated-series overrelaxation (reading C-24) -----------------------------------

def culgt_or_sweep_series(lat: Lattice, links, parity: int, omega: float, order: int, stream=None) -> None:
    _require_cuda()
    _check(lib().culgt_or_sweep_series(ctypes.byref(lat.c()), _ptr(links), int(parity), float(omega),
                                       int(order), _stream(stream)), "culgt_or_sweep_series")


def culgt_or_sweeps_series(lat: Lattice, links, n_sweeps: int, omega: float, order: int, stream=None) -> None:
    _require_cuda()
    _check(lib().culgt_or_sweeps_series(ctypes.byref(lat.c()), _ptr(links), int(n_sweeps), float(omega),
                                        int(order), _stream(stream)), "culgt_or_sweeps_series")


# ---- simulated annealing (reading C-25) -----------------------------------------------

def culgt_sa_sweep(lat: Lattice, links, parity: int, T: float, seed: int, counter: int, stream=None) -> None:
    _require_cuda()
    _check(lib().culgt_sa_sweep(ctypes.byref(lat.c()), _ptr(links), int(parity), float(T), int(seed),
                                int(counter), _stream(stream)), "culgt_sa_sweep")


def culgt_sa_anneal(lat: Lattice, links, T_max: float, T_min: float, n_sweeps: int, seed: int, stream=None) -> None:
    _require_cuda()
    _check(lib().culgt_sa_anneal(ctypes.byref(lat.c()), _ptr(links), float(T_max), float(T_min),
                                 int(n_sweeps), int(seed), _stream(stream)), "culgt_sa_anneal")


# ---- microcanonical step (reading C-26) -----------------------------------------------

def culgt_micro_sweep(lat: Lattice, links, parity: int, stream=None) -> None:
    _require_cuda()
    _check(lib().culgt_micro_sweep(ctypes.byref(lat.c()), _ptr(links), int(parity), _stream(stream)),
           "culgt_micro_sweep")


def culgt_micro_sweeps(lat: Lattice, links, n_sweeps: int, stream=None) -> None:
    _require_cuda()
    _check(lib().culgt_micro_sweeps(ctypes.byref(lat.c()), _ptr(links), int(n_sweeps), _stream(stream)),
           "culgt_micro_sweeps")


def culgt_sa_anneal_micro(lat: Lattice, links, T_max: float, T_min: float, n_sweeps: int, n_micro: int,
                          seed: int, stream=None) -> None:
    _require_cuda()
    _check(lib().culgt_sa_anneal_micro(ctypes.byref(lat.c()), _ptr(links), float(T_max), float(T_min),
                                       int(n_sweeps), int(n_micro), int(seed), _stream(stream)),
           "culgt_sa_anneal_micro")


# ---- Coulomb gauge (reading C-22) ----------------------------------------------------

def culgt_or_sweep_coulomb(lat: Lattice, links, parity: int, omega: float, stream=None) -> None:
    _require_cuda()
    _check(lib().culgt_or_sweep_coulomb(ctypes.byref(lat.c()), _ptr(links), int(parity), float(omega),
                                        _stream(stream)), "culgt_or_sweep_coulomb")


def culgt_or_sweep_coulomb_masked(lat: Lattice, links, parity: int, omega: float, slice_active, stream=None) -> None:
    """slice_active: device uint8 tensor of dims[3] entries; slices with 0 are left untouched."""
    _require_cuda()
    _check(lib().culgt_or_sweep_coulomb_masked(ctypes.byref(lat.c()), _ptr(links), int(parity), float(omega),
                                               _ptr(slice_active), _stream(stream)), "culgt_or_sweep_coulomb_masked")


def culgt_or_sweeps_coulomb(lat: Lattice, links, n_sweeps: int, omega: float, stream=None) -> None:
    _require_cuda()
    _check(lib().culgt_or_sweeps_coulomb(ctypes.byref(lat.c()), _ptr(links), int(n_sweeps), float(omega),
                                         _stream(stream)), "culgt_or_sweeps_coulomb")


def culgt_coulomb_precision_functional(lat: Lattice, links, workspace, theta_t_dev, F_t_dev, stream=None) -> None:
    """theta_t_dev, F_t_dev: device float64 arrays of dims[3] elements."""
    _require_cuda()
    _check(lib().culgt_coulomb_precision_functional(ctypes.byref(lat.c()), _ptr(links), _ptr(workspace),
                                                    _ptr(theta_t_dev), _ptr(F_t_dev), _stream(stream)),
           "culgt_coulomb_precision_functional")


def culgt_coulomb_fix(lat: Lattice, links, workspace, omega: float, theta_target: float,
                      max_sweeps: int, check_every: int = 1, stream=None):
    """Returns (sweeps_done, theta_t, F_t) with theta_t, F_t lists of dims[3] floats."""
    _require_cuda()
    n3 = int(lat.dims[3])
    done = ctypes.c_int(0)
    th = (ctypes.c_double * n3)()
    F = (ctypes.c_double * n3)()
    _check(lib().culgt_coulomb_fix(ctypes.byref(lat.c()), _ptr(links), _ptr(workspace), float(omega),
                                   float(theta_target), int(max_sweeps), int(check_every),
                                   ctypes.byref(done), th, F, _stream(stream)), "culgt_coulomb_fix")
    return done.value, list(th), list(F)


# ---- time-slab decomposition over several GPUs (include/culgt_b200.h, csrc/slab.cu) -----------------

def culgt_slab_lattice(lat: Lattice, n_slabs: int) -> Lattice:
    """The local lattice (dims[3] = N3 / n_slabs) of one of n_slabs time slabs."""
    out = culgt_lattice()
    _check(lib().culgt_slab_lattice(ctypes.byref(lat.c()), int(n_slabs), ctypes.byref(out)), "culgt_slab_lattice")
    return Lattice(tuple(out.dims), out.group, out.precision, out.params)


def culgt_slab_links_bytes(local: Lattice) -> int:
    return lib().culgt_slab_links_bytes(ctypes.byref(local.c()))


def culgt_slab_halo_bytes(local: Lattice) -> int:
    return lib().culgt_slab_halo_bytes(ctypes.byref(local.c()))


def culgt_slab_halo_chunks(local: Lattice, parity: int, which: int):
    """(byte offsets, chunk_bytes) of one halo message: which = 0 ghost slice, 1 last slice (host only)."""
    off = (ctypes.c_size_t * 9)()
    nbytes = ctypes.c_size_t(0)
    n = ctypes.c_int(0)
    _check(lib().culgt_slab_halo_chunks(ctypes.byref(local.c()), int(parity), int(which), off, ctypes.byref(nbytes),
                                        ctypes.byref(n)), "culgt_slab_halo_chunks")
    return [int(off[j]) for j in range(n.value)], int(nbytes.value)


def culgt_slab_halo_peers(rank: int, n_ranks: int, direction: int):
    """(send_to, recv_from) of one halo message (host only)."""
    a, b = ctypes.c_int(0), ctypes.c_int(0)
    _check(lib().culgt_slab_halo_peers(int(rank), int(n_ranks), int(direction), ctypes.byref(a), ctypes.byref(b)),
           "culgt_slab_halo_peers")
    return a.value, b.value


def alloc_slab_links(local: Lattice, device="cuda"):
    import torch
    n = culgt_slab_links_bytes(local)
    if n == 0:
        _check(culgt_validate(local), "alloc_slab_links")
    return torch.empty(n // (local.precision // 8), dtype=local.torch_dtype, device=device)


def _ptr_array(tensors):
    return (ctypes.c_void_p * len(tensors))(*[_ptr(t) for t in tensors])


def culgt_slab_pack(local: Lattice, canonical_slab, links_slab, stream=None) -> None:
    _require_cuda()
    _check(lib().culgt_slab_pack(ctypes.byref(local.c()), _ptr(canonical_slab), _ptr(links_slab), _stream(stream)),
           "culgt_slab_pack")


def culgt_slab_unpack(local: Lattice, links_slab, canonical_slab, stream=None) -> None:
    _require_cuda()
    _check(lib().culgt_slab_unpack(ctypes.byref(local.c()), _ptr(links_slab), _ptr(canonical_slab), _stream(stream)),
           "culgt_slab_unpack")


def culgt_slab_or_sweep(local: Lattice, links_slab, parity: int, omega: float, stream=None) -> None:
    _require_cuda()
    _check(lib().culgt_slab_or_sweep(ctypes.byref(local.c()), _ptr(links_slab), int(parity), float(omega),
                                     _stream(stream)), "culgt_slab_or_sweep")


def culgt_slab_or_sweep_window(local: Lattice, links_slab, parity: int, omega: float, t_lo: int, t_hi: int,
                               stream=None) -> None:
    _require_cuda()
    _check(lib().culgt_slab_or_sweep_window(ctypes.byref(local.c()), _ptr(links_slab), int(parity), float(omega),
                                            int(t_lo), int(t_hi), _stream(stream)), "culgt_slab_or_sweep_window")


def culgt_slab_halo_copy(local: Lattice, src_links, dst_links, parity: int, direction: int, stream=None) -> None:
    _require_cuda()
    _check(lib().culgt_slab_halo_copy(ctypes.byref(local.c()), _ptr(src_links), _ptr(dst_links), int(parity),
                                      int(direction), _stream(stream)), "culgt_slab_halo_copy")


def culgt_slab_theta_F_sums(local: Lattice, links_slab, workspace, sums2_dev, stream=None) -> None:
    _require_cuda()
    _check(lib().culgt_slab_theta_F_sums(ctypes.byref(local.c()), _ptr(links_slab), _ptr(workspace), _ptr(sums2_dev),
                                         _stream(stream)), "culgt_slab_theta_F_sums")


def culgt_slab_theta_F_combine(lat: Lattice, sums_dev, n_slabs: int, theta_dev, F_dev, stream=None) -> None:
    _require_cuda()
    _check(lib().culgt_slab_theta_F_combine(ctypes.byref(lat.c()), _ptr(sums_dev), int(n_slabs), _ptr(theta_dev),
                                            _ptr(F_dev), _stream(stream)), "culgt_slab_theta_F_combine")


def culgt_slab_exchange_all_local(local: Lattice, links_slabs, stream=None) -> None:
    _require_cuda()
    _check(lib().culgt_slab_exchange_all_local(ctypes.byref(local.c()), _ptr_array(links_slabs), len(links_slabs),
                                               _stream(stream)), "culgt_slab_exchange_all_local")


def culgt_slab_or_sweeps_local(local: Lattice, links_slabs, n_sweeps: int, omega: float, boundary_first: bool = False,
                               stream=None) -> None:
    _require_cuda()
    _check(lib().culgt_slab_or_sweeps_local(ctypes.byref(local.c()), _ptr_array(links_slabs), len(links_slabs),
                                            int(n_sweeps), float(omega), int(bool(boundary_first)), _stream(stream)),
           "culgt_slab_or_sweeps_local")


def culgt_slab_theta_F_local(lat: Lattice, local: Lattice, links_slabs, workspace, sums_dev, theta_dev, F_dev,
                             stream=None) -> None:
    _require_cuda()
    _check(lib().culgt_slab_theta_F_local(ctypes.byref(lat.c()), ctypes.byref(local.c()), _ptr_array(links_slabs),
                                          len(links_slabs), _ptr(workspace), _ptr(sums_dev), _ptr(theta_dev),
                                          _ptr(F_dev), _stream(stream)), "culgt_slab_theta_F_local")


def culgt_slab_comm_unique_id() -> bytes:
    buf = ctypes.create_string_buffer(128)
    _check(lib().culgt_slab_comm_unique_id(buf), "culgt_slab_comm_unique_id")
    return buf.raw


def culgt_slab_comm_create(unique_id: bytes, rank: int, n_ranks: int) -> int:
    """Collective over the n_ranks ranks; returns the opaque communicator handle."""
    _require_cuda()
    comm = ctypes.c_void_p(0)
    _check(lib().culgt_slab_comm_create(ctypes.create_string_buffer(unique_id, 128), int(rank), int(n_ranks),
                                        ctypes.byref(comm)), "culgt_slab_comm_create")
    return comm.value


def culgt_slab_comm_destroy(comm: int) -> None:
    _check(lib().culgt_slab_comm_destroy(comm), "culgt_slab_comm_destroy")


def culgt_slab_halo_exchange(comm: int, local: Lattice, links_slab, parity: int, direction: int, stream=None) -> None:
    _require_cuda()
    _check(lib().culgt_slab_halo_exchange(comm, ctypes.byref(local.c()), _ptr(links_slab), int(parity), int(direction),
                                          _stream(stream)), "culgt_slab_halo_exchange")


def culgt_slab_exchange_all_nccl(comm: int, local: Lattice, links_slab, stream=None) -> None:
    _require_cuda()
    _check(lib().culgt_slab_exchange_all_nccl(comm, ctypes.byref(local.c()), _ptr(links_slab), _stream(stream)),
           "culgt_slab_exchange_all_nccl")


def culgt_slab_or_sweeps_nccl(comm: int, local: Lattice, links_slab, n_sweeps: int, omega: float, comm_stream=None,
                              stream=None) -> None:
    _require_cuda()
    _check(lib().culgt_slab_or_sweeps_nccl(comm, ctypes.byref(local.c()), _ptr(links_slab), int(n_sweeps), float(omega),
                                           None if comm_stream is None else _stream(comm_stream), _stream(stream)),
           "culgt_slab_or_sweeps_nccl")


def culgt_slab_theta_F_nccl(comm: int, lat: Lattice, local: Lattice, links_slab, workspace, sums_dev, theta_dev, F_dev,
                            stream=None) -> None:
    _require_cuda()
    _check(lib().culgt_slab_theta_F_nccl(comm, ctypes.byref(lat.c()), ctypes.byref(local.c()), _ptr(links_slab),
                                         _ptr(workspace), _ptr(sums_dev), _ptr(theta_dev), _ptr(F_dev),
                                         _stream(stream)), "culgt_slab_theta_F_nccl")


def culgt_set_sweep_variant(variant: int) -> None:
    _check(lib().culgt_set_sweep_variant(int(variant)), "culgt_set_sweep_variant")


def culgt_autotune_sweep(lat: Lattice, links, workspace, omega: float, sweeps_per_trial: int = 3, stream=None):
    """Times every result-equivalent sweep schedule on `links` (real sweeps), selects the fastest
    for the calling thread.  Returns (variant, microseconds per half-sweep)."""
    _require_cuda()
    v = ctypes.c_int(0)
    us = ctypes.c_float(0.0)
    _check(lib().culgt_autotune_sweep(ctypes.byref(lat.c()), _ptr(links), _ptr(workspace), float(omega),
                                      int(sweeps_per_trial),
                                      ctypes.byref(v), ctypes.byref(us), _stream(stream)), "culgt_autotune_sweep")
    return v.value, us.value


def culgt_get_sweep_variant() -> int:
    return lib().culgt_get_sweep_variant()


def culgt_fused_schedule(n_slices: int, lag: int, direction: int):
    """Measurement library only: [(parity, slice), ...] in the order the fused full sweep hands out
    its slice-tasks (host only)."""
    buf = (ctypes.c_uint * (2 * int(n_slices)))()
    _check(lib().culgt_fused_schedule(int(n_slices), int(lag), int(direction), buf), "culgt_fused_schedule")
    return [(w >> 31, w & 0x7FFFFFFF) for w in buf]


def culgt_sweep_kernel_name(lat: Lattice) -> str:
    return lib().culgt_sweep_kernel_name(ctypes.byref(lat.c())).decode()


def culgt_measure_build() -> bool:
    return bool(lib().culgt_measure_build())


def culgt_version() -> int:
    return lib().culgt_version()


def culgt_strerror(status: int) -> str:
    return lib().culgt_strerror(int(status)).decode()
