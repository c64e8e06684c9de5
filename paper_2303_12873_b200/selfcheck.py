"""Installation self-check: a small uniform plasma stepped through every
particle path of the library (global-atomic kernel, fused per-tile kernel in
its fresh and drift variants, deferred and immediate sort) at orders 1-3,
checked against what must hold without any reference: finite state, particle
count and ids conserved, every particle counted by exactly one path, total
charge conserved, and total current equal to sum q w v (SURVEY.md 8(c.3)
Esirkepov pin (ii)) to roundoff.

    python -m paper_2303_12873_b200.selfcheck [--n 16] [--orders 1,2,3]

This is also the workload put under ``compute-sanitizer`` (racecheck, memcheck,
initcheck; profiles/r02_sanitizer.md).  It never touches oracle/.
"""
from __future__ import annotations

import argparse
import sys

import numpy as np

from . import workloads as W
from .binding import Sim


def _total_current(sim, wl):
    f = sim.get_fields()
    dv = wl.dx * wl.dy * wl.dz
    return np.array([f["Jx"].sum(), f["Jy"].sum(), f["Jz"].sum()]) * dv


def run_case(n, order, mode, verbose=True):
    """mode: 'global' | 'fresh' | 'drift' | 'fresh_immediate'"""
    wl = W.uniform_plasma(n, n, n, ppc=8, u_th=0.05, order=order, seed=4242 + order, shuffle=(mode == "global"))
    sim = Sim.from_workload(wl)
    if mode == "global":
        sim.set_option("force_path", 1)
    if mode == "fresh_immediate":
        sim.set_option("sort_deferred", 0)
    npart = wl.nparticles
    q0 = sim.deposit_rho(-1).sum()
    nsteps = 3
    if mode != "global":
        sim.sort()
    for it in range(nsteps):
        if mode in ("fresh", "fresh_immediate") and it > 0:
            sim.sort()
        before = sim.get_particles(0)
        sim.step(1)
        after = sim.get_particles(0)
        # total current of the step = sum q w (x1 - x0) / dt with the periodic image nearest to x0
        o0, o1 = np.argsort(before["id"]), np.argsort(after["id"])
        tot = np.zeros(3)
        for d, (name, Ld) in enumerate(zip("xyz", (wl.nx * wl.dx, wl.ny * wl.dy, wl.nz * wl.dz))):
            dlt = after[name][o1] - before[name][o0]
            dlt -= Ld * np.round(dlt / Ld)
            tot[d] = float(np.sum(wl.species[0].q * before["w"][o0] * dlt)) / wl.dt
        jt = _total_current(sim, wl)
        scale = float(np.sum(np.abs(wl.species[0].q) * before["w"])) * 0.05 * W.C_LIGHT
        err = float(np.abs(jt - tot).max()) / scale
        assert err < 1e-12, "total current mismatch %.3e (%s order %d step %d)" % (err, mode, order, it)
        assert np.array_equal(np.sort(after["id"]), np.arange(npart, dtype=after["id"].dtype)), "ids lost"
        for k in ("x", "y", "z", "ux", "uy", "uz"):
            assert np.isfinite(after[k]).all(), "non-finite " + k
    f = sim.get_fields()
    for k, v in f.items():
        assert np.isfinite(v).all(), "non-finite " + k
    q1 = sim.deposit_rho(-1).sum()
    assert abs(q1 - q0) <= 1e-12 * abs(q0), "total charge changed: %r -> %r" % (q0, q1)
    c = sim.counters()
    assert c["fast"] + c["slow"] + c["global"] == npart * nsteps, c
    if mode == "global":
        assert c["fast"] + c["slow"] == 0, c
    else:
        assert c["global"] == 0 and c["fast"] > 0.5 * npart * nsteps, c
    if verbose:
        print("selfcheck ok: n=%d order=%d mode=%-15s counters=%s current err %.1e" % (n, order, mode, c, err), flush=True)
    sim.close()


def main(argv=None):
    ap = argparse.ArgumentParser()
    ap.add_argument("--n", type=int, default=16)
    ap.add_argument("--orders", default="1,2,3")
    ap.add_argument("--modes", default="global,fresh,drift,fresh_immediate")
    a = ap.parse_args(argv)
    import torch
    torch.cuda.set_device(0)
    for order in [int(v) for v in a.orders.split(",")]:
        for mode in a.modes.split(","):
            run_case(a.n, order, mode)
    print("selfcheck: all cases passed")
    return 0


if __name__ == "__main__":
    sys.exit(main())
