"""One process driving two devices (include/culgt_b200.h "General rules": the library keeps no state
beyond per-DEVICE caches of kernel attributes and device properties).  The process's first CUDA work
through the library happens on device 1; the fp32-12 and fp64-18 sweeps (48 / 72 KB of dynamic shared
memory: they need the per-device cudaFuncSetAttribute), theta/F, the no-allocation theta/F (its scratch
address is resolved per device) and the one-kernel driver loop must then still work on device 0, and
give the same bits on both devices.  Needs >= 2 visible GPUs: skipped on a one-GPU box (the only test
in this repository allowed to skip on hardware)."""
import subprocess
import sys
import os

import pytest
import torch

pytestmark = pytest.mark.gpu
ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

CHILD = r'''
import sys
sys.path.insert(0, %r)
import numpy as np, torch
import lattice_inputs as li
import paper_1412_3655_b200 as culgt

dims = (8, 8, 8, 8)
u = li.make_config(dims, 3, "near_identity", 611, eps=0.5, scramble=True)
out = {}
for dev in (1, 0):                      # device 1 FIRST: every lazy per-device set-up happens there first
    torch.cuda.set_device(dev)
    res = []
    for precision, params in ((32, 12), (64, 18)):
        lat = culgt.Lattice(dims, 3, precision, params)
        can = torch.from_numpy(li.to_real(u, np.float32 if precision == 32 else np.float64)).cuda()
        links = culgt.alloc_links(lat)
        ws = culgt.alloc_workspace(lat)
        scal = torch.zeros(4, dtype=torch.float64, device="cuda")
        culgt.culgt_pack(lat, can, links)
        culgt.culgt_or_sweeps(lat, links, 3, 1.7)
        culgt.culgt_gauge_precision_functional(lat, links, ws, scal[0:1], scal[1:2])
        culgt.culgt_gauge_precision_functional_noalloc(lat, links, scal[2:3], scal[3:4])
        done, theta, F = culgt.culgt_landau_fix(lat, links, ws, 1.7, 1e-6, 200, 2)
        culgt.culgt_unpack(lat, links, can)
        torch.cuda.synchronize()
        res.append((can.cpu().numpy().tobytes(), tuple(scal.cpu().tolist()), done, theta, F))
    out[dev] = res
assert out[0] == out[1], "device 0 and device 1 disagree"
for _, scal, done, theta, F in out[0]:
    assert scal[0] == scal[2] and scal[1] == scal[3] and 0 < done < 200 and theta < 1e-6
print("MULTIDEVICE_OK")
'''


@pytest.mark.skipif(torch.cuda.device_count() < 2, reason="needs two visible GPUs")
def test_first_use_on_device_1_then_device_0():
    r = subprocess.run([sys.executable, "-c", CHILD % ROOT], capture_output=True, text=True, timeout=600, cwd=ROOT)
    assert r.returncode == 0 and "MULTIDEVICE_OK" in r.stdout, r.stdout[-2000:] + r.stderr[-2000:]
