"""Helpers for the GPU parity tests: move seeded inputs to the device through the C ABI binding,
run the CUDA path, bring results back as canonical numpy arrays, and prepare the matching oracle
input.  The oracle and the CUDA package are both imported HERE (tests only), never by each other.
"""
import numpy as np
import torch

import lattice_inputs as li
import oracle
import paper_1412_3655_b200 as culgt

TOL_LINK = {64: 1e-12, 32: 2e-5}     # BASELINE.json north_star: per link component after one sweep


def np_dtype(precision):
    return np.float32 if precision == 32 else np.float64


def storage_input(uc, precision, params):
    """What a (precision, params) store holds, as the oracle's fp64 canonical real array:
    components rounded to the storage precision; for 12-parameter storage the third row is
    rebuilt in fp64 from the rounded rows (reading C-15)."""
    if precision == 32:
        uc = li.round_to_fp32(uc)
    ur = li.to_real(np.ascontiguousarray(uc))
    if params == 12:
        oracle.reconstruct12(ur)
    return ur


class GpuField:
    """A link field resident on the GPU in the internal layout."""

    def __init__(self, dims, group, precision, params, uc):
        self.lat = culgt.Lattice(tuple(int(d) for d in dims), group, precision, params)
        self.dims = self.lat.dims
        self.nc = group
        self.links = culgt.alloc_links(self.lat)
        self.ws = culgt.alloc_workspace(self.lat)
        self.scal = torch.zeros(2, dtype=torch.float64, device="cuda")
        self.upload(uc)

    def upload(self, uc):
        can = torch.from_numpy(li.to_real(np.ascontiguousarray(uc), np_dtype(self.lat.precision))).cuda()
        culgt.culgt_pack(self.lat, can, self.links)
        torch.cuda.synchronize()

    def download(self):
        """canonical complex128 [V,4,nc,nc]"""
        V = self.lat.volume
        can = torch.empty((V, 4, self.nc, self.nc, 2), dtype=self.lat.torch_dtype, device="cuda")
        culgt.culgt_unpack(self.lat, self.links, can)
        torch.cuda.synchronize()
        return li.from_real(can.cpu().numpy())

    def half_sweep(self, parity, omega):
        culgt.culgt_or_sweep(self.lat, self.links, parity, omega)

    def sweep(self, omega, n=1):
        culgt.culgt_or_sweeps(self.lat, self.links, n, omega)

    def sweep_ws(self, omega, n=1):
        """full sweeps through the workspace entry point (fused one-kernel schedule where it applies)"""
        culgt.culgt_or_sweeps_ws(self.lat, self.links, self.ws, n, omega)

    def theta(self):
        culgt.culgt_gauge_precision(self.lat, self.links, self.ws, self.scal[0:1])
        return float(self.scal[0].item())

    def functional(self):
        culgt.culgt_functional(self.lat, self.links, self.ws, self.scal[1:2])
        return float(self.scal[1].item())

    def theta_functional(self):
        """both scalars from the fused one-pass entry point"""
        culgt.culgt_gauge_precision_functional(self.lat, self.links, self.ws, self.scal[0:1], self.scal[1:2])
        th, F = self.scal.cpu().tolist()
        return th, F

    def transform(self, g):
        gt = torch.from_numpy(li.to_real(np.ascontiguousarray(g), np_dtype(self.lat.precision))).cuda()
        culgt.culgt_gauge_transform(self.lat, self.links, gt)
        torch.cuda.synchronize()


def theta_close(t_gpu, t_or):
    """DESIGN.md reading C-16: |dtheta| <= 1e-10 theta + 1e-16 sqrt(theta) + 1e-29."""
    return abs(t_gpu - t_or) <= 1e-10 * t_or + 1e-16 * np.sqrt(t_or) + 1e-29
