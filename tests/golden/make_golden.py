"""Writes tests/golden/cfg0_trajectory.txt by calling ONLY oracle/ and lattice_inputs/.

The paper (arXiv:1412.3655) prints no numeric F, theta or link value for any configuration
(SURVEY.md section 4), so there is no paper fixture to store.  This file is a regression
fixture of the pinned oracle on BASELINE.json configs[0] (4^4 SU(3), eps=0.3, scrambled,
omega=1.7): F and theta after every full sweep until theta < 1e-20.  It guards the oracle against
accidental change; it is not evidence of the oracle's correctness (the pins are).

    python tests/golden/make_golden.py
"""
import os
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
sys.path.insert(0, ROOT)

import lattice_inputs as li  # noqa: E402
import oracle  # noqa: E402


def main():
    cfg = li.CONFIGS["cfg0"]
    dims = cfg["dims"]
    u = li.to_real(li.make_named("cfg0"))
    rows = [(0, oracle.functional(dims, u), oracle.gauge_precision(dims, u))]
    sweeps = 0
    while rows[-1][2] >= 1e-20 and sweeps < 5000:
        oracle.full_sweep(dims, u, cfg["omega"])
        sweeps += 1
        rows.append((sweeps, oracle.functional(dims, u), oracle.gauge_precision(dims, u)))
    out = os.path.join(os.path.dirname(os.path.abspath(__file__)), "cfg0_trajectory.txt")
    with open(out, "w") as f:
        f.write("# written by tests/golden/make_golden.py (oracle only); cfg0 = BASELINE.json configs[0]\n")
        f.write("# sweep  F  theta\n")
        for s, F, th in rows:
            f.write(f"{s} {F!r} {th!r}\n")
    print(f"{out}: {len(rows)} rows, final theta {rows[-1][2]:.3e}, F {rows[-1][1]:.6f}")


if __name__ == "__main__":
    main()
