"""Tests of the fused one-kernel full sweep (csrc/or_sweep_fused.cu), which exists only in the
measurement library (python -m paper_1412_3655_b200.build --measure; run the tests with
CULGT_MEASURE=1).  With the product library this module defines no tests: the kernel was measured and
rejected (profiles/r2_fused_sweep.md) and is not part of the product build."""
import numpy as np
import pytest

import paper_1412_3655_b200 as culgt

if culgt.culgt_measure_build():
    import torch

    import lattice_inputs as li
    import oracle
    from gpu_common import GpuField, TOL_LINK, storage_input
    from test_gpu_parity_small import SU3_STORES, make

    def test_fused_schedule_order_and_dependencies():
        """The slice-task order: every slice of both parities exactly once, and every white slice t
        after the black slices t-1, t, t+1 (periodic) -- what makes the ticket scheme deadlock-free."""
        for n3 in (2, 4, 6, 8, 12, 32, 96, 512):
            for lag in (0, 1, 2, 5, 40, 1000):
                for direction in (0, 1):
                    tasks = culgt.culgt_fused_schedule(n3, lag, direction)
                    assert sorted(tasks) == sorted((p, t) for p in (0, 1) for t in range(n3))
                    pos = {task: i for i, task in enumerate(tasks)}
                    for t in range(n3):
                        for nb in ((t - 1) % n3, t, (t + 1) % n3):
                            assert pos[(0, nb)] < pos[(1, t)], (n3, lag, direction, t, nb)
                    assert tasks[0] == ((0, 0) if direction == 0 else (0, n3 - 1))

    FUSED_DIMS = [(8, 8, 8, 8), (8, 8, 8, 12), (16, 8, 8, 6), (8, 8, 4, 2), (8, 8, 8, 4), (8, 4, 8, 16), (4, 6, 2, 8)]
    
    
    @pytest.mark.gpu
    @pytest.mark.parametrize("dims", FUSED_DIMS)
    @pytest.mark.parametrize("precision,params", SU3_STORES)
    def test_fused_full_sweep_is_the_same_sweep(dims, precision, params):
        """culgt_or_sweeps_ws with variant 60 (csrc/or_sweep_fused.cu: black and white half-sweeps
        interleaved slice by slice inside ONE persistent kernel, tickets + per-slice completion counters,
        every other sweep descending) only reorders independent site updates: one sweep must agree with
        the oracle, and three more must be bit-identical to the two-launch schedule (variant 0).  Covers
        N3 = 2 (both black slices first), N3 = 4 (lag clamped), long time extents, and (4,6,2,8), which
        does not hold whole site blocks per slice and takes the two-launch fallback.  With -DCULGT_MEASURE
        also the launch-level slab schedules 41-43."""
        u = make(dims, 3, 46)
        ref = storage_input(u, precision, params)
        oracle.full_sweep(dims, ref, 1.7)
        outs = {}
        for variant in [0, 60, 41, 42, 43]:
            culgt.culgt_set_sweep_variant(variant)
            try:
                f = GpuField(dims, 3, precision, params, u)
                f.sweep_ws(1.7, 1)
                assert np.abs(f.download() - li.from_real(ref)).max() < TOL_LINK[precision], variant
                f.sweep_ws(1.7, 3)
                f.sweep_ws(1.7, 2)          # a second call: the control block is set up again
                torch.cuda.synchronize()
                outs[variant] = f.download()
            finally:
                culgt.culgt_set_sweep_variant(0)
        for variant, out in outs.items():
            assert np.array_equal(out, outs[0]), variant
    
    
    @pytest.mark.gpu
    def test_fused_sweep_in_the_driver_loop_and_host_call():
        """culgt_landau_fix and culgt_fix_host hand their workspace to the sweeps: with the fused schedule
        forced on they must stop at the same sweep with the same theta and F, bit for bit, as the
        launch-per-half-sweep path (variant 34; variant 0 would take the one-kernel loop on this small lattice)."""
        dims = (8, 8, 8, 8)
        u = make(dims, 3, 49)
        res = {}
        for variant in (34, 60):
            culgt.culgt_set_sweep_variant(variant)
            try:
                f = GpuField(dims, 3, 64, 18, u)
                res[variant] = culgt.culgt_landau_fix(f.lat, f.links, f.ws, 1.7, 1e-12, 400, 3)
                host = torch.from_numpy(li.to_real(u)).pin_memory()
                can = torch.empty_like(host, device="cuda")
                res[variant] += culgt.culgt_fix_host(f.lat, host, can, f.links, f.ws, 5, 1.7)
                res[variant] += (host.numpy().tobytes(),)
            finally:
                culgt.culgt_set_sweep_variant(0)
        assert res[60] == res[34]
        assert res[60][1] < 1e-12 and res[60][0] % 3 == 0

    from test_gpu_configs import field_and_ref, max_abs_diff, named_input

    @pytest.mark.gpu
    @pytest.mark.parametrize("name", ["cfg3_fp32", "cfg3_fp64", "cfg3_fp32_18", "cfg3_fp64_12"])
    def test_cfg3_fused_sweep_bit_identical_and_matches_oracle(name):
        """The fused one-kernel full sweep (culgt_or_sweeps_ws, csrc/or_sweep_fused.cu) at the headline
        volume, where its dependency counters and the lag between the black and the white front are really
        exercised (thousands of tickets per resident CTA): all 4V links after sweep 1 against the oracle,
        and bit-identical to the two-launch schedule after 6 sweeps (ascending and descending passes)."""
        c, f, ref = field_and_ref(name)
        dims, om, prec = c["dims"], c["omega"], c["precision"]
        u = named_input(name)
        oracle.full_sweep(dims, ref, om)
        culgt.culgt_set_sweep_variant(60)
        try:
            f.sweep_ws(om, 1)
            err = max_abs_diff(f.download(), ref)
            assert err < TOL_LINK[prec], err
            f.sweep_ws(om, 5)
            fused = f.links.clone()
        finally:
            culgt.culgt_set_sweep_variant(0)
        f.upload(u)
        f.sweep(om, 6)
        torch.cuda.synchronize()
        assert torch.equal(fused, f.links)
