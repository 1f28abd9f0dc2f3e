"""CPU-side checks of the C-ABI boundary: the library loads, exports every symbol that
include/culgt_b200.h declares, sizes follow the formulas, and every argument error is reported
by return code BEFORE any CUDA call (so these run without a GPU)."""
import ctypes
import os
import re

import pytest

import paper_1412_3655_b200 as culgt

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
HEADER = os.path.join(ROOT, "include", "culgt_b200.h")


def declared_symbols():
    text = open(HEADER).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(culgt_[a-z0-9_]+)\s*\(", text)))


def test_library_exports_every_declared_symbol():
    lib = culgt.lib()
    names = declared_symbols()
    assert len(names) >= 19
    for n in names:
        assert hasattr(lib, n), f"{n} declared in culgt_b200.h but not exported"
    # and the Python binding offers the same names
    for n in names:
        if n in ("culgt_last_cuda_error",):
            continue
        assert hasattr(culgt, n), f"binding lacks {n}"


def test_sizes():
    L = culgt.Lattice((32, 32, 32, 32), 3, 32, 12)
    V = 32 ** 4
    assert culgt.culgt_links_bytes(L) == 4 * V * 48 == 201326592
    assert culgt.culgt_canonical_bytes(L) == 4 * V * 72
    assert culgt.culgt_gfield_bytes(L) == V * 72
    assert culgt.culgt_links_bytes(culgt.Lattice((32,) * 4, 3, 64, 18)) == 603979776
    assert culgt.culgt_links_bytes(culgt.Lattice((48, 48, 48, 96), 3, 32, 12)) == 2038431744
    assert culgt.culgt_links_bytes(culgt.Lattice((64,) * 4, 3, 64, 18)) == 9663676416
    assert culgt.culgt_links_bytes(culgt.Lattice((8,) * 4, 2, 64, 4)) == 524288
    assert culgt.culgt_workspace_bytes(L) >= 8 * 1024
    # the fused theta+F pass keeps two partials per 64 sites of a parity (the staged fp32 12-parameter
    # kernel; the other formats use every other slot's worth, 128 sites per partial), plus the 2 scalars
    # + 2 * N3 result slots (theta_t, F_t of the Coulomb driver; the Landau scalars use two) + N3 mask bytes
    # ... rounded up to 16 doubles, + the driver loop's control block (16 doubles) + the fused sweep's
    # (32 words of counters, 2 x 512 slice counters, 2 x 1024 slice-task words)
    ctl = 16 * 8 + (32 + 2 * 512 + 2 * 1024) * 4

    def ws_bytes(partials, n3):
        red = partials + 2 * n3 + (n3 + 7) // 8
        return (red + 15) // 16 * 16 * 8 + ctl
    assert culgt.culgt_workspace_bytes(culgt.Lattice((64,) * 4, 3, 64, 18)) == ws_bytes(2 * (64 ** 4 // 2 // 64) + 8, 64)
    assert culgt.culgt_workspace_bytes(culgt.Lattice((4,) * 4, 3, 64, 18)) == ws_bytes(4096, 4)


@pytest.mark.parametrize("lat,code", [
    (culgt.Lattice((3, 4, 4, 4)), "CULGT_ERR_DIMS"),
    (culgt.Lattice((4, 4, 0, 4)), "CULGT_ERR_DIMS"),
    (culgt.Lattice((4, 4, 4, -2)), "CULGT_ERR_DIMS"),
    (culgt.Lattice((1024, 1024, 1024, 4)), "CULGT_ERR_DIMS"),
    (culgt.Lattice((4, 4, 4, 4), 4, 32, 12), "CULGT_ERR_DESC"),
    (culgt.Lattice((4, 4, 4, 4), 3, 16, 12), "CULGT_ERR_DESC"),
    (culgt.Lattice((4, 4, 4, 4), 3, 32, 8), "CULGT_ERR_DESC"),
    (culgt.Lattice((4, 4, 4, 4), 2, 32, 12), "CULGT_ERR_DESC"),
])
def test_descriptor_errors(lat, code):
    assert culgt.culgt_validate(lat) == culgt.ERRORS[code]
    assert culgt.culgt_links_bytes(lat) == 0
    assert culgt.culgt_canonical_bytes(lat) == 0


def test_argument_errors_by_return_code():
    lib = culgt.lib()
    L = culgt.Lattice((4, 4, 4, 4), 3, 64, 18).c()
    ref = ctypes.byref(L)
    E = culgt.ERRORS
    ok_ptr = 4096       # aligned, never dereferenced: validation fails first
    assert lib.culgt_or_sweep(None, ok_ptr, 0, 1.7, None) == E["CULGT_ERR_NULL"]
    assert lib.culgt_or_sweep(ref, None, 0, 1.7, None) == E["CULGT_ERR_NULL"]
    assert lib.culgt_or_sweep(ref, ok_ptr + 8, 0, 1.7, None) == E["CULGT_ERR_ALIGN"]
    assert lib.culgt_or_sweep(ref, ok_ptr, 2, 1.7, None) == E["CULGT_ERR_PARITY"]
    assert lib.culgt_or_sweep(ref, ok_ptr, -1, 1.7, None) == E["CULGT_ERR_PARITY"]
    for bad in (0.99, 2.0, float("nan"), float("inf"), -1.5):
        assert lib.culgt_or_sweep(ref, ok_ptr, 0, bad, None) == E["CULGT_ERR_OMEGA"]
        assert lib.culgt_or_sweeps(ref, ok_ptr, 1, bad, None) == E["CULGT_ERR_OMEGA"]
    assert lib.culgt_or_sweeps(ref, ok_ptr, -1, 1.7, None) == E["CULGT_ERR_ARG"]
    assert lib.culgt_pack(ref, None, ok_ptr, None) == E["CULGT_ERR_NULL"]
    assert lib.culgt_unpack(ref, ok_ptr, None, None) == E["CULGT_ERR_NULL"]
    assert lib.culgt_gauge_precision(ref, ok_ptr, None, ok_ptr, None) == E["CULGT_ERR_NULL"]
    assert lib.culgt_functional(ref, ok_ptr, ok_ptr, None, None) == E["CULGT_ERR_NULL"]
    assert lib.culgt_gauge_transform(ref, ok_ptr, None, None) == E["CULGT_ERR_NULL"]
    assert lib.culgt_landau_fix(ref, ok_ptr, ok_ptr, 1.7, 1e-10, 10, 0, None, None, None, None) == E["CULGT_ERR_ARG"]
    assert lib.culgt_fix_host(ref, None, ok_ptr, ok_ptr, ok_ptr, 1, 1.7, None, None, None) == E["CULGT_ERR_NULL"]
    assert lib.culgt_set_sweep_variant(-3) == E["CULGT_ERR_ARG"]
    # the widened entry points (Coulomb gauge, series power, annealing, re-unitarisation, autotuner)
    assert lib.culgt_or_sweep_coulomb(ref, None, 0, 1.7, None) == E["CULGT_ERR_NULL"]
    assert lib.culgt_or_sweep_coulomb(ref, ok_ptr, 3, 1.7, None) == E["CULGT_ERR_PARITY"]
    assert lib.culgt_or_sweeps_coulomb(ref, ok_ptr, -1, 1.7, None) == E["CULGT_ERR_ARG"]
    assert lib.culgt_coulomb_precision_functional(ref, ok_ptr, ok_ptr, None, ok_ptr, None) == E["CULGT_ERR_NULL"]
    assert lib.culgt_coulomb_fix(ref, ok_ptr, ok_ptr, 1.7, 1e-10, 10, 0, None, None, None, None) == E["CULGT_ERR_ARG"]
    assert lib.culgt_or_sweep_series(ref, ok_ptr, 0, 1.7, 17, None) == E["CULGT_ERR_ARG"]
    assert lib.culgt_or_sweep_series(ref, ok_ptr, 0, 2.5, 4, None) == E["CULGT_ERR_OMEGA"]
    assert lib.culgt_or_sweeps_series(ref, ok_ptr + 8, 1, 1.7, 4, None) == E["CULGT_ERR_ALIGN"]
    assert lib.culgt_sa_sweep(ref, ok_ptr, 0, 0.0, 1, 0, None) == E["CULGT_ERR_ARG"]
    assert lib.culgt_sa_sweep(ref, ok_ptr, 2, 1.0, 1, 0, None) == E["CULGT_ERR_PARITY"]
    assert lib.culgt_sa_anneal(ref, ok_ptr, 0.1, 1.0, 5, 1, None) == E["CULGT_ERR_ARG"]
    assert lib.culgt_micro_sweep(ref, ok_ptr, 2, None) == E["CULGT_ERR_PARITY"]
    assert lib.culgt_micro_sweeps(ref, None, 1, None) == E["CULGT_ERR_NULL"]
    assert lib.culgt_sa_anneal_micro(ref, ok_ptr, 1.0, 0.1, 5, -1, 1, None) == E["CULGT_ERR_ARG"]
    assert lib.culgt_reunitarize(ref, None, None) == E["CULGT_ERR_NULL"]
    assert lib.culgt_autotune_sweep(ref, ok_ptr, ok_ptr, 1.7, 0, None, None, None) == E["CULGT_ERR_ARG"]
    assert lib.culgt_autotune_sweep(ref, ok_ptr, None, 1.7, 1, None, None, None) == E["CULGT_ERR_NULL"]
    assert lib.culgt_gauge_precision_functional(ref, ok_ptr, ok_ptr, ok_ptr, None, None) == E["CULGT_ERR_NULL"]
    for code in E.values():
        assert culgt.culgt_strerror(code) != "unknown status"
    assert culgt.culgt_strerror(-99) == "unknown status"


def test_product_build_rejects_measurement_variants():
    """The product library accepts only schedules that compute the method, bit-identically: the
    all-fp32 kernels (11, 14, 25), the G = 1 / no-solve measurement kernels (28, 32) and the rejected
    mappings exist only in a -DCULGT_MEASURE build (include/culgt_b200.h, culgt_set_sweep_variant)."""
    lib = culgt.lib()
    E = culgt.ERRORS
    assert culgt.culgt_measure_build() is False, "the committed build step must produce the product library"
    assert not hasattr(lib, "culgt_or_sweeps_ws") and not hasattr(lib, "culgt_fused_schedule")
    for v in (0, 20, 24, 33, 34):
        assert lib.culgt_set_sweep_variant(v) == culgt.CULGT_OK
        assert culgt.culgt_get_sweep_variant() == v
    lib.culgt_set_sweep_variant(0)
    for v in (11, 14, 25, 28, 32, 1, 2, 4, 8, 21, 22, 23, 26, 27, 29, 30, 31, 41, 44, 51, 54, 60, 61, 99, 100, 100000, 150123):
        assert lib.culgt_set_sweep_variant(v) == E["CULGT_ERR_ARG"], v
        assert culgt.culgt_get_sweep_variant() == 0


def test_sweep_variant_is_per_thread():
    """The selection is a per-host-thread setting (no process-global mutable state)."""
    import threading
    lib = culgt.lib()
    assert lib.culgt_set_sweep_variant(33) == culgt.CULGT_OK
    seen = []
    t = threading.Thread(target=lambda: seen.append(culgt.culgt_get_sweep_variant()))
    t.start()
    t.join()
    assert seen == [0] and culgt.culgt_get_sweep_variant() == 33
    lib.culgt_set_sweep_variant(0)


def test_no_cpu_fallback():
    """Without a CUDA device the binding refuses to compute (it never routes to the oracle)."""
    import torch
    if torch.cuda.is_available():
        pytest.skip("CUDA device present")
    L = culgt.Lattice((4, 4, 4, 4), 3, 64, 18)
    with pytest.raises(RuntimeError, match="no CPU fallback"):
        culgt.culgt_or_sweep(L, 4096, 0, 1.7)
    src = open(os.path.join(ROOT, "paper_1412_3655_b200", "__init__.py")).read()
    assert "import oracle" not in src and "from oracle" not in src
