"""GPU parity tests on small lattices: every storage layout, every thread-to-site mapping, all
entry points, element by element against the oracle on the same seeded inputs.  Sizes span
several 128-thread tiles and a ragged tail (V/2 not a multiple of 128) and asymmetric extents
that are not powers of two (exercise the multiply-shift index decode)."""
import numpy as np
import pytest
import torch

import lattice_inputs as li
import oracle
import paper_1412_3655_b200 as culgt
from gpu_common import GpuField, TOL_LINK, storage_input, theta_close

pytestmark = pytest.mark.gpu

SU3_STORES = [(64, 18), (64, 12), (32, 12), (32, 18)]
DIMS = [(4, 4, 4, 4), (4, 6, 2, 8), (6, 10, 12, 4), (8, 8, 8, 8), (2, 2, 2, 2), (12, 2, 6, 10)]


def make(dims, group, seed, kind="near_identity"):
    if kind == "haar":
        return li.make_config(dims, group, "haar", seed)
    return li.make_config(dims, group, "near_identity", seed, eps=0.5, scramble=True)


@pytest.mark.parametrize("dims", DIMS)
@pytest.mark.parametrize("precision,params", SU3_STORES)
def test_pack_unpack_round_trip_su3(dims, precision, params):
    u = make(dims, 3, 41, "haar")
    f = GpuField(dims, 3, precision, params, u)
    back = f.download()
    want = li.from_real(storage_input(u, precision, params))
    tol = 1e-15 if precision == 64 else 3e-7     # fp32 reconstruction of the third row
    assert np.abs(back - want).max() < tol
    if params == 18:
        assert np.array_equal(back, want)        # pure data movement: bit exact


@pytest.mark.parametrize("dims", DIMS)
@pytest.mark.parametrize("precision", [64, 32])
def test_pack_unpack_round_trip_su2(dims, precision):
    u = make(dims, 2, 42, "haar")
    f = GpuField(dims, 2, precision, 4, u)
    want = li.round_to_fp32(u) if precision == 32 else u
    assert np.array_equal(f.download(), want)


PRODUCT_VARIANTS = [0, 24, 33, 34]


def variants_for(precision, params):
    """Product build: 0 = the production mapping; 24 / 33 / 34 = the same kernel without the reversed
    odd-parity traversal / programmatic dependent launch / L2 eviction hints.  A library built with
    -DCULGT_MEASURE (culgt_measure_build()) also carries the measured alternatives of
    csrc/or_sweep_measure.cu that compute the same update: 1..8 = direct register kernels with that
    many threads per site; 21+ = staged mappings (flat / persistent grids, 1-2 stages, 1/2/4 threads
    per site, prefetch, chunked, stream stores)."""
    if not culgt.culgt_measure_build():
        return list(PRODUCT_VARIANTS)
    if precision == 32 and params == 12:
        return PRODUCT_VARIANTS + [1, 2, 4, 21, 22, 23, 26, 27, 29, 30, 31]
    if precision == 32:
        return PRODUCT_VARIANTS + [2, 4, 21, 22, 23, 30]
    if params == 12:
        return PRODUCT_VARIANTS + [2, 4, 8, 21, 22, 23, 30]
    return PRODUCT_VARIANTS + [4, 8, 21, 22, 23, 26, 27, 30, 31, 32]


@pytest.mark.parametrize("dims", DIMS)
@pytest.mark.parametrize("precision,params", SU3_STORES)
def test_su3_links_after_one_sweep(dims, precision, params):
    """North-star link parity: after one black+white sweep every link component agrees with the
    oracle within 1e-12 (fp64) / 2e-5 (fp32); also after each half-sweep separately."""
    u = make(dims, 3, 43)
    ref = storage_input(u, precision, params)
    oracle.or_sweep(dims, ref, 0, 1.7)
    ref_black = li.from_real(ref)
    oracle.or_sweep(dims, ref, 1, 1.7)
    ref_full = li.from_real(ref)
    for variant in variants_for(precision, params):
        culgt.culgt_set_sweep_variant(variant)
        try:
            f = GpuField(dims, 3, precision, params, u)
            f.half_sweep(0, 1.7)
            err_b = np.abs(f.download() - ref_black).max()
            f.half_sweep(1, 1.7)
            err_f = np.abs(f.download() - ref_full).max()
        finally:
            culgt.culgt_set_sweep_variant(0)
        assert err_b < TOL_LINK[precision], (variant, err_b)
        assert err_f < TOL_LINK[precision], (variant, err_f)


@pytest.mark.parametrize("dims", DIMS)
@pytest.mark.parametrize("precision", [64, 32])
def test_su2_links_after_one_sweep(dims, precision):
    u = make(dims, 2, 44, "haar")
    ref = storage_input(u, precision, 4)
    oracle.full_sweep(dims, ref, 1.5)
    f = GpuField(dims, 2, precision, 4, u)
    f.sweep(1.5)
    assert np.abs(f.download() - li.from_real(ref)).max() < TOL_LINK[precision]


@pytest.mark.parametrize("dims", DIMS)
@pytest.mark.parametrize("group,precision,params", [(3, 64, 18), (3, 64, 12), (3, 32, 12), (3, 32, 18),
                                                    (2, 64, 4), (2, 32, 4)])
def test_theta_and_F_match_oracle(dims, group, precision, params):
    u = make(dims, group, 45)
    ref = storage_input(u, precision, params)
    f = GpuField(dims, group, precision, params, u)
    th, F = f.theta(), f.functional()
    th_o, F_o = oracle.gauge_precision(dims, ref), oracle.functional(dims, ref)
    if precision == 64:
        assert theta_close(th, th_o)
        assert abs(F - F_o) <= 1e-10 * abs(F_o) + 1e-15
    else:   # fp32 storage: fp64 arithmetic on identical inputs (12-param: row 2 rebuilt in fp64)
        assert abs(th - th_o) <= 1e-9 * th_o
        assert abs(F - F_o) <= 1e-10
    # deterministic: same bits when repeated
    assert f.theta() == th and f.functional() == F
    # the fused one-pass entry point gives the same two scalars (it IS the same pass)
    th2, F2 = f.theta_functional()
    assert th2 == th and F2 == F
    assert f.theta_functional() == (th2, F2)
    if precision == 64:
        assert theta_close(th2, th_o) and abs(F2 - F_o) <= 1e-10 * abs(F_o) + 1e-15


@pytest.mark.parametrize("dims", DIMS[:4])
@pytest.mark.parametrize("group,precision,params", [(3, 64, 18), (3, 64, 12), (3, 32, 12), (3, 32, 18),
                                                    (2, 64, 4), (2, 32, 4)])
def test_gauge_transform_matches_oracle(dims, group, precision, params):
    u = make(dims, group, 46, "haar")
    g = (li.haar_su3 if group == 3 else li.haar_su2)(li.volume(dims), 47)
    if precision == 32:
        g = li.round_to_fp32(g)
    ref = storage_input(u, precision, params)
    oracle.gauge_transform(dims, ref, li.to_real(g))
    f = GpuField(dims, group, precision, params, u)
    f.transform(g)
    tol = 1e-13 if precision == 64 else 2e-6
    assert np.abs(f.download() - li.from_real(ref)).max() < tol


def test_unit_and_converged_fields_are_fixed_points():
    """Degenerate cases: unit field (every g = 1, |v| = 0 branch of su2_pow) stays exactly unit."""
    dims = (4, 4, 4, 4)
    for group, precision, params in [(3, 64, 18), (3, 32, 12), (2, 64, 4)]:
        u = li.make_config(dims, group, "unit", 0)
        f = GpuField(dims, group, precision, params, u)
        f.sweep(1.7, 3)
        assert np.array_equal(f.download(), u)
        assert f.theta() == 0.0 and abs(f.functional() - 1.0) < 1e-15


def test_pure_gauge_returns_to_vacuum_on_gpu():
    """North star: a unit configuration scrambled by a random gauge transformation returns to
    F = 1, theta < 1e-24 (fp64)."""
    dims = (4, 4, 4, 4)
    u = li.make_config(dims, 3, "pure_gauge", 21)
    f = GpuField(dims, 3, 64, 18, u)
    done, theta, F = culgt.culgt_landau_fix(f.lat, f.links, f.ws, 1.7, 1e-26, 3000, 10)
    assert theta < 1e-24 and abs(F - 1.0) < 1e-12, (done, theta, F)
    back = f.download()
    assert np.abs(back @ np.conj(np.swapaxes(back, -1, -2)) - np.eye(3)).max() < 1e-13
    assert np.abs(np.linalg.det(back) - 1).max() < 1e-13


def test_omega_1_monotone_F_and_plaquette_invariance():
    dims = (4, 6, 2, 8)
    u = make(dims, 3, 48)
    f = GpuField(dims, 3, 64, 18, u)
    P0 = oracle.plaquette(dims, li.to_real(u))
    F = f.functional()
    for it in range(40):
        f.half_sweep(it & 1, 1.0)
        Fn = f.functional()
        assert Fn >= F - 1e-14
        F = Fn
    assert abs(oracle.plaquette(dims, li.to_real(f.download())) - P0) < 1e-12


def test_sweep_is_asynchronous():
    """The sweep call only enqueues: many launches return before the device has finished."""
    dims = (16, 16, 16, 16)
    u = li.make_config(dims, 3, "unit", 0)
    f = GpuField(dims, 3, 32, 12, u)
    torch.cuda.synchronize()
    ev = torch.cuda.Event()
    f.sweep(1.7, 200)
    ev.record()
    assert not ev.query()          # work still in flight when the calls have returned
    torch.cuda.synchronize()


def test_autotuner_picks_a_result_equivalent_mapping():
    """culgt_autotune_sweep (PAPER.md L89 (d), L134): returns one of the built schedules with a
    positive time, leaves it selected, and sweeps with it still match the oracle."""
    dims = (8, 8, 8, 8)
    u = make(dims, 3, 47)
    for precision, params in SU3_STORES:
        scratch = GpuField(dims, 3, precision, params, u)
        try:
            v, us = culgt.culgt_autotune_sweep(scratch.lat, scratch.links, scratch.ws, 1.7, 2)
            assert v in variants_for(precision, params) + ([41, 42, 43, 44, 60] if culgt.culgt_measure_build() else []) and us > 0
            assert culgt.culgt_get_sweep_variant() == v
            ref = storage_input(u, precision, params)
            oracle.full_sweep(dims, ref, 1.7)
            f = GpuField(dims, 3, precision, params, u)
            f.sweep(1.7)
            assert np.abs(f.download() - li.from_real(ref)).max() < TOL_LINK[precision]
        finally:
            culgt.culgt_set_sweep_variant(0)


@pytest.mark.parametrize("dims", [(4, 4, 4, 4), (8, 8, 8, 8), (4, 6, 2, 8), (2, 2, 2, 2)])
@pytest.mark.parametrize("precision,params", SU3_STORES)
def test_one_kernel_driver_loop_is_the_same_loop(dims, precision, params):
    """culgt_landau_fix on a small SU(3) lattice runs the whole loop as one cooperative kernel
    (csrc/fix_persistent.cu: grid barriers between half-sweeps, theta/F reduced inside).  Against the
    launch-per-half-sweep path (any non-zero product variant selects it): the same number of sweeps, the
    same links bit for bit, theta and F to rounding -- when it stops on theta and when it runs to
    max_sweeps, with theta checked every sweep and every third."""
    u = make(dims, 3, 50)
    for target, max_sweeps, every in ((1e-6, 300, 1), (1e-6, 300, 3), (0.0, 7, 3)):
        res = {}
        for variant in (34, 0):
            culgt.culgt_set_sweep_variant(variant)
            try:
                f = GpuField(dims, 3, precision, params, u)
                res[variant] = culgt.culgt_landau_fix(f.lat, f.links, f.ws, 1.7, target, max_sweeps, every) + (f.links.clone(),)
            finally:
                culgt.culgt_set_sweep_variant(0)
        (d0, th0, F0, l0), (d1, th1, F1, l1) = res[34], res[0]
        assert d0 == d1 and (d0 == 7 if target == 0.0 else 0 < d0 < 300), (d0, d1)
        assert torch.equal(l0, l1)
        assert abs(th0 - th1) <= 1e-12 * th0 and abs(F0 - F1) <= 1e-13 * abs(F0)
        if target > 0:
            assert th1 < target and d1 % every == 0
