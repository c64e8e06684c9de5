"""Writes tests/golden/config1_32cube_100steps.npz: the ORACLE's state after 100
steps of BASELINE.json configs[1] at its parity size (SURVEY.md 8(d) table,
last column: 32^3 cells, 262,144 electrons + 262,144 protons, order 3).  The
oracle needs about 11 minutes of one host core for this run, too long for the
GPU test session, so its result is stored; tests/test_gpu_slow.py regenerates
the same seeded inputs, runs the CUDA path (sort every 4 steps) and compares.

Calls ONLY oracle/ and the seeded input generator (never the CUDA path).
Stored: the six E, B components after 1, 10 and 100 steps (fp64), the state of
2,048 sampled particles per species after 100 steps, the Gauss residual
max|div E - rho/eps0| at steps 0 and 100 (its constancy is the oracle's own
whole-cycle pin), and a checksum of the inputs so that a change of the
generator cannot go unnoticed.

Run:  python tests/golden/make_golden_slow.py        (about 11 minutes)
"""
import hashlib
import os
import sys

import numpy as np

sys.path.insert(0, os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__)))))
from oracle import ora  # noqa: E402
from paper_2303_12873_b200 import workloads as W  # noqa: E402  (seeded inputs only, no method arithmetic)

HERE = os.path.dirname(os.path.abspath(__file__))
OUT = os.path.join(HERE, "config1_32cube_100steps.npz")
NSAMPLE = 2048
EPS0 = 8.8541878128e-12


def input_digest(wl):
    h = hashlib.sha256()
    for sp in wl.species:
        for a in sp.arrays():
            h.update(np.ascontiguousarray(a, dtype=np.float64).tobytes())
    return h.hexdigest()


def gauss_residual(sim, wl):
    """max |div E - rho_total/eps0| at the nodes (backward differences of E), reading R19."""
    f = sim.get_fields()
    sh = (wl.nz, wl.ny, wl.nx)
    ex, ey, ez = (f[n].reshape(sh) for n in ("Ex", "Ey", "Ez"))
    div = ((ex - np.roll(ex, 1, axis=2)) / wl.dx + (ey - np.roll(ey, 1, axis=1)) / wl.dy
           + (ez - np.roll(ez, 1, axis=0)) / wl.dz)
    rho = sim.deposit_rho(-1).reshape(sh)
    # scale: ONE species' rho / eps0 (the two co-located species cancel to roundoff in the total)
    return float(np.abs(div - rho / EPS0).max()), float(np.abs(sim.deposit_rho(0)).max() / EPS0)


def main():
    wl = W.config(1, parity=True)              # 32^3, 8 + 8 ppc, order 3, sort_every 4, 100 steps
    assert (wl.nx, wl.ny, wl.nz) == (32, 32, 32) and wl.order == 3 and wl.nsteps == 100
    sim = ora.OracleSim(*wl.grid_args(), wl.dt, wl.order, len(wl.species))
    for s, sp in enumerate(wl.species):
        sim.load_particles(s, sp.q, sp.m, *sp.arrays())
    out = {"digest": np.array(input_digest(wl)), "dt": np.array(wl.dt)}
    g0, scale = gauss_residual(sim, wl)
    out["gauss0"] = np.array(g0)
    out["gauss_scale"] = np.array(scale)
    done = 0
    for upto in (1, 10, 100):
        sim.step(upto - done)
        done = upto
        f = sim.get_fields()
        for n in ("Ex", "Ey", "Ez", "Bx", "By", "Bz"):
            out["%s_%d" % (n, upto)] = f[n]
        print("step %d done" % upto, flush=True)
    out["gauss100"] = np.array(gauss_residual(sim, wl)[0])
    rng = np.random.default_rng(20230312)
    for s, sp in enumerate(wl.species):
        ids = np.sort(rng.choice(sp.n, NSAMPLE, replace=False)).astype(np.int64)
        p = sim.get_particles(s)
        inv = np.empty(sp.n, dtype=np.int64)
        inv[p["id"].astype(np.int64)] = np.arange(sp.n)
        out["sp%d_ids" % s] = ids
        for n in ("x", "y", "z", "ux", "uy", "uz"):
            out["sp%d_%s" % (s, n)] = p[n][inv[ids]]
    np.savez_compressed(OUT, **out)
    print("wrote", OUT, os.path.getsize(OUT), "bytes; gauss residual", g0, "->", float(out["gauss100"]),
          "of scale", scale)


if __name__ == "__main__":
    main()
