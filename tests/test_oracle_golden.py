"""Regression of the pinned oracle against its own committed cfg0 trajectory
(tests/golden/cfg0_trajectory.txt, written by tests/golden/make_golden.py from oracle/ only)."""
import os

import numpy as np

import lattice_inputs as li
import oracle

GOLD = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden", "cfg0_trajectory.txt")


def test_cfg0_trajectory_regression():
    rows = np.loadtxt(GOLD)
    cfg = li.CONFIGS["cfg0"]
    dims = cfg["dims"]
    u = li.to_real(li.make_named("cfg0"))
    for s, F, th in rows:
        if s > 0:
            oracle.full_sweep(dims, u, cfg["omega"])
        assert abs(oracle.functional(dims, u) - F) <= 1e-13
        got = oracle.gauge_precision(dims, u)
        assert abs(got - th) <= 1e-9 * th + 1e-15 * np.sqrt(th) + 1e-29
    assert rows[-1][2] < 1e-20 <= rows[-2][2]
    # orders of magnitude the survey's throw-away probe saw: ~120 sweeps
    assert 60 < rows[-1][0] < 400
