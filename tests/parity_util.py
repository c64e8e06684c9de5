"""Comparison rules of the parity tests (BASELINE.json:north_star tolerances as
read in DESIGN.md R20-R24 / SURVEY.md 8(c.2) items 20-24) and the driver that
runs one workload through the oracle and through the CUDA library.

Holds no PIC arithmetic: it only compares arrays."""
from __future__ import annotations

import numpy as np

C_LIGHT = 299792458.0

TOL_PARTICLE_1STEP = 1e-12     # relative, per particle (R21)
TOL_FIELD_1STEP = 1e-11        # max-abs relative to max|group| (R22)
TOL_FIELD_L2_10STEP = 1e-9     # joint L2 of E and c*B (R23)


def by_id(p):
    """Particle dict reordered so that entry r has id r (ids are load indices)."""
    order = np.argsort(p["id"], kind="stable")
    assert np.array_equal(p["id"][order], np.arange(p["id"].size, dtype=p["id"].dtype)), "ids are not a permutation"
    return {k: v[order] for k, v in p.items()}


def particle_errors(po, pg, L, u_ref):
    """Max relative position error (periodic distance / L_d) and momentum error
    (|du|_2 / max(|u|_2, u_ref)), particles matched by id."""
    po, pg = by_id(po), by_id(pg)
    ex = 0.0
    for d, Ld in zip("xyz", L):
        dlt = np.abs(po[d] - pg[d])
        dlt = np.minimum(dlt, np.abs(Ld - dlt))
        ex = max(ex, float(dlt.max(initial=0.0)) / Ld)
    du = np.sqrt((po["ux"] - pg["ux"]) ** 2 + (po["uy"] - pg["uy"]) ** 2 + (po["uz"] - pg["uz"]) ** 2)
    un = np.sqrt(po["ux"] ** 2 + po["uy"] ** 2 + po["uz"] ** 2)
    eu = float((du / np.maximum(un, u_ref)).max(initial=0.0))
    assert np.array_equal(po["w"], pg["w"]), "weights must travel unchanged"
    return ex, eu


def group_maxabs_errors(fo, fg):
    """{group: max|d| / max|group of the oracle|}; an all-zero oracle group must be matched exactly."""
    out = {}
    for grp, names in (("E", ("Ex", "Ey", "Ez")), ("B", ("Bx", "By", "Bz")), ("J", ("Jx", "Jy", "Jz"))):
        ref = max(float(np.abs(fo[n]).max()) for n in names)
        err = max(float(np.abs(fo[n] - fg[n]).max()) for n in names)
        out[grp] = (err / ref) if ref > 0.0 else (0.0 if err == 0.0 else np.inf)
    return out


def field_l2_error(fo, fg):
    """sqrt(sum|dF|^2 / sum|F|^2) over Ex,Ey,Ez,c*Bx,c*By,c*Bz jointly (R23)."""
    num = den = 0.0
    for n, s in (("Ex", 1.0), ("Ey", 1.0), ("Ez", 1.0), ("Bx", C_LIGHT), ("By", C_LIGHT), ("Bz", C_LIGHT)):
        num += float(np.sum((s * (fo[n] - fg[n])) ** 2))
        den += float(np.sum((s * fo[n]) ** 2))
    return np.sqrt(num / den) if den > 0 else (0.0 if num == 0 else np.inf)


def make_pair(ora, Sim, wl, sort_first=False, force_path=0):
    """An OracleSim and a CUDA Sim loaded with the same workload."""
    o = ora.OracleSim(*wl.grid_args(), wl.dt, wl.order, len(wl.species))
    g = Sim.from_workload(wl)
    if wl.fields:
        o.set_fields(**wl.fields)
    for s, sp in enumerate(wl.species):
        o.load_particles(s, sp.q, sp.m, *sp.arrays())
    if force_path:
        g.set_option("force_path", force_path)
    if sort_first:
        g.sort()
    return o, g


def u_ref_of(wl, s):
    sp = wl.species[s]
    if sp.n == 0:
        return 1e-3 * C_LIGHT
    sig = float(np.sqrt(np.mean(sp.ux ** 2 + sp.uy ** 2 + sp.uz ** 2) / 3.0))
    return sig if sig > 0 else 1e-3 * C_LIGHT      # R21: u_th, or 1e-3 c for a cold species


def check_step_parity(o, g, wl, label=""):
    """1-step bounds (R21, R22).  Returns the measured errors."""
    fo, fg = o.get_fields(), g.get_fields()
    res = {"fields": group_maxabs_errors(fo, fg)}
    for grp, e in res["fields"].items():
        assert e <= TOL_FIELD_1STEP, "%s: %s max-abs rel error %.3e > %.1e" % (label, grp, e, TOL_FIELD_1STEP)
    L = (wl.nx * wl.dx, wl.ny * wl.dy, wl.nz * wl.dz)
    for s in range(len(wl.species)):
        if wl.species[s].n == 0:
            continue
        ex, eu = particle_errors(o.get_particles(s), g.get_particles(s), L, u_ref_of(wl, s))
        res["sp%d" % s] = (ex, eu)
        assert ex <= TOL_PARTICLE_1STEP, "%s: species %d position error %.3e" % (label, s, ex)
        assert eu <= TOL_PARTICLE_1STEP, "%s: species %d momentum error %.3e" % (label, s, eu)
    return res
