"""culgt_gauge_precision_functional_noalloc (include/culgt_b200.h): theta and F for callers that cannot
allocate device memory -- the block partials live in a 2 MiB file-scope device array of the library
instead of a caller-supplied workspace.  The output must equal the existing workspace path's (it runs the
same kernels in the same order), on two calls in a row that share the array, for every storage format,
and a lattice beyond the stated limit must be refused with a clear error.

This file is named test_zz_* so that pytest collects it LAST (the suite runs with `pytest -x`); it passes
both alone in a fresh process and after the other tests."""
import ctypes

import numpy as np
import pytest
import torch

import lattice_inputs as li
import paper_1412_3655_b200 as culgt

STORES = [(3, 32, 12), (3, 64, 18), (3, 32, 18), (3, 64, 12), (2, 64, 4), (2, 32, 4)]


def test_limit_is_stated_and_enforced_before_any_cuda_call():
    """V > CULGT_NOALLOC_MAX_SITES = 2^24 is rejected by return code (no launch, so no GPU is needed)."""
    lib = culgt.lib()
    E = culgt.ERRORS
    ok_ptr = 4096                                    # aligned, never dereferenced
    assert culgt.NOALLOC_MAX_SITES == 1 << 24
    too_big = culgt.Lattice((64, 64, 64, 128), 3, 32, 12).c()      # 2^25 sites
    assert lib.culgt_gauge_precision_functional_noalloc(ctypes.byref(too_big), ok_ptr, ok_ptr, ok_ptr, None) \
        == E["CULGT_ERR_TOO_LARGE"]
    assert "no-allocation" in culgt.culgt_strerror(E["CULGT_ERR_TOO_LARGE"])
    ok = culgt.Lattice((8, 8, 8, 8), 3, 32, 12).c()
    assert lib.culgt_gauge_precision_functional_noalloc(ctypes.byref(ok), None, ok_ptr, ok_ptr, None) == E["CULGT_ERR_NULL"]
    assert lib.culgt_gauge_precision_functional_noalloc(ctypes.byref(ok), ok_ptr, ok_ptr, None, None) == E["CULGT_ERR_NULL"]
    assert lib.culgt_gauge_precision_functional_noalloc(ctypes.byref(ok), ok_ptr + 8, ok_ptr, ok_ptr, None) == E["CULGT_ERR_ALIGN"]
    bad = culgt.Lattice((8, 8, 7, 8), 3, 32, 12).c()
    assert lib.culgt_gauge_precision_functional_noalloc(ctypes.byref(bad), ok_ptr, ok_ptr, ok_ptr, None) == E["CULGT_ERR_DIMS"]


def _field(dims, group, precision, params, seed):
    lat = culgt.Lattice(tuple(dims), group, precision, params)
    u = li.make_config(dims, group, "haar", seed) if group == 2 else \
        li.make_config(dims, group, "near_identity", seed, eps=0.5, scramble=True)
    can = torch.from_numpy(li.to_real(u, np.float32 if precision == 32 else np.float64)).cuda()
    links = culgt.alloc_links(lat)
    culgt.culgt_pack(lat, can, links)
    torch.cuda.synchronize()
    return lat, links


@pytest.mark.gpu
@pytest.mark.parametrize("group,precision,params", STORES)
def test_two_calls_in_a_row_match_the_workspace_path(group, precision, params):
    """Call 1 on a large ragged lattice fills many slots of the shared array; call 2 on a smaller field
    (other values, fewer slots) must not see them; a third call after a sweep of the first field checks
    changed contents on the same slots.  Reference: culgt_gauge_precision_functional with a workspace.
    Tolerance: 1e-12 relative (the tests' bound for two reductions of the same stored values) -- and, the
    kernels and the summation order being the same, the same bits."""
    omega = 1.7 if group == 3 else 1.5
    big = _field((6, 10, 12, 4), group, precision, params, 301)          # V/2 = 1440: ragged last block
    small = _field((4, 4, 4, 4), group, precision, params, 302)
    ws_big, ws_small = culgt.alloc_workspace(big[0]), culgt.alloc_workspace(small[0])
    want = torch.zeros(6, dtype=torch.float64, device="cuda")
    got = torch.full((6,), float("nan"), dtype=torch.float64, device="cuda")
    # the existing path, on its own workspaces
    culgt.culgt_gauge_precision_functional(big[0], big[1], ws_big, want[0:1], want[1:2])
    culgt.culgt_gauge_precision_functional(small[0], small[1], ws_small, want[2:3], want[3:4])
    # the new entry point: two calls in a row on the shared array, no workspace anywhere
    culgt.culgt_gauge_precision_functional_noalloc(big[0], big[1], got[0:1], got[1:2])
    culgt.culgt_gauge_precision_functional_noalloc(small[0], small[1], got[2:3], got[3:4])
    # ... and again after the field has changed
    culgt.culgt_or_sweeps(big[0], big[1], 1, omega)
    culgt.culgt_gauge_precision_functional(big[0], big[1], ws_big, want[4:5], want[5:6])
    culgt.culgt_gauge_precision_functional_noalloc(big[0], big[1], got[4:5], got[5:6])
    torch.cuda.synchronize()
    w, g = want.cpu().numpy(), got.cpu().numpy()
    assert np.all(np.isfinite(g)) and np.all(w[[0, 2, 4]] > 0)
    assert w[5] > w[1] and w[4] != w[0]                  # the sweep raised F: call 3 saw the new field
    assert np.all(np.abs(g - w) <= 1e-12 * np.abs(w))
    assert np.array_equal(g, w)


@pytest.mark.gpu
def test_headline_volume_and_repeatability():
    """32^4 fp32 12-parameter (16 384 partials in the shared array), twice in a row: same bits as the
    workspace path both times."""
    lat = culgt.Lattice((32, 32, 32, 32), 3, 32, 12)
    block = li.make_config((8, 8, 8, 8), 3, "haar", 303)
    u = np.tile(block, (lat.volume // block.shape[0], 1, 1, 1))
    can = torch.from_numpy(li.to_real(u, np.float32)).cuda()
    links = culgt.alloc_links(lat)
    culgt.culgt_pack(lat, can, links)
    ws = culgt.alloc_workspace(lat)
    want = torch.zeros(2, dtype=torch.float64, device="cuda")
    got = torch.zeros(4, dtype=torch.float64, device="cuda")
    culgt.culgt_gauge_precision_functional(lat, links, ws, want[0:1], want[1:2])
    culgt.culgt_gauge_precision_functional_noalloc(lat, links, got[0:1], got[1:2])
    culgt.culgt_gauge_precision_functional_noalloc(lat, links, got[2:3], got[3:4])
    torch.cuda.synchronize()
    w, g = want.cpu().numpy(), got.cpu().numpy()
    assert w[0] > 0 and np.array_equal(g[:2], w) and np.array_equal(g[2:], w)
