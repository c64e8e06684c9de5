"""Writes tests/golden/oracle_cycle_4x4x4.txt.  Calls ONLY oracle/ (never the
CUDA path).  Purpose: a regression pin -- a later change to the oracle's
arithmetic shows up as a diff of this file and must be justified in the commit
message (the paper prints no worked example, so there is
no paper-given value to store).

Run:  python tests/golden/make_golden.py
"""
import os
import sys

import numpy as np

sys.path.insert(0, os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__)))))
from oracle import ora  # noqa: E402

QE, ME = -1.602176634e-19, 9.1093837015e-31
HERE = os.path.dirname(os.path.abspath(__file__))


def case(order):
    """Six hand-picked electrons on a 4x4x4 anisotropic grid, 2 steps."""
    dx, dy, dz = 0.5e-6, 0.4e-6, 0.25e-6
    g = ora.make_grid(4, 4, 4, dx, dy, dz)
    dt = 0.99 * ora.courant_dt(g)
    sim = ora.OracleSim(4, 4, 4, dx, dy, dz, 0.0, 0.0, 0.0, dt, order, 1)
    frac = np.array([[0.10, 0.20, 0.30], [1.50, 2.25, 3.75], [3.95, 0.05, 1.50],
                     [2.00, 2.00, 2.00], [0.01, 3.99, 0.50], [3.30, 1.70, 2.60]])
    u = 299792458.0 * np.array([[0.5, -0.2, 0.1], [-0.9, 0.3, 0.4], [0.8, -0.8, 0.0],
                                [0.0, 0.0, 0.0], [-0.7, 0.6, -0.5], [0.05, 0.02, -0.03]])
    w = np.array([1.0e5, 2.0e5, 1.5e5, 1.0e5, 3.0e5, 0.5e5])
    sim.load_particles(0, QE, ME, frac[:, 0] * dx, frac[:, 1] * dy, frac[:, 2] * dz, u[:, 0], u[:, 1], u[:, 2], w)
    sim.step(2)
    return sim


def main():
    lines = ["# oracle regression fixture: 4x4x4 cells (0.5,0.4,0.25 um), 6 electrons, dt=0.99 Courant, 2 steps",
             "# written by tests/golden/make_golden.py from oracle/ only; %.17e round-trips fp64",
             "# columns: order name index value"]
    for order in (1, 2, 3):
        sim = case(order)
        f = sim.get_fields(); p = sim.get_particles(0)
        for name in ("Ex", "Ey", "Ez", "Bx", "By", "Bz", "Jx", "Jy", "Jz"):
            for i in (0, 21, 42, 63):
                lines.append("%d %s %d %.17e" % (order, name, i, f[name][i]))
        for name in ("x", "y", "z", "ux", "uy", "uz"):
            for i in range(6):
                lines.append("%d %s %d %.17e" % (order, name, i, p[name][i]))
    with open(os.path.join(HERE, "oracle_cycle_4x4x4.txt"), "w") as fh:
        fh.write("\n".join(lines) + "\n")


if __name__ == "__main__":
    main()
