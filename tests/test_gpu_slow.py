"""Parity at the sizes SURVEY.md 8(d) lists in its "parity size" column, and sampled
element-wise parity at BASELINE.json's full sizes for configs 1, 3 and 4 (config 2's
is in test_gpu_tile_kernel.py).  ``-m "gpu and slow"``; part of ``-m gpu``.

  config 1  32^3 x 100 steps, sort every 4: against the ORACLE's stored result
            (tests/golden/config1_32cube_100steps.npz, written by
            tests/golden/make_golden_slow.py from oracle/ only: the oracle needs 11 minutes
            of one core for it) after 1, 10 and 100 steps, plus the Gauss residual
  config 2  32^3 x 10 steps, sort every step            (live oracle)
  config 3  the true 16 x 16 x 1024 crop x 20 steps      (live oracle; z profile NOT rescaled)
  config 4  8 x 8 x 512 x 20 steps                        (live oracle)

The three live oracle runs are started together in threads (the oracle is single-threaded
C called through ctypes, which releases the GIL), so they cost the wall time of the longest.
"""
import hashlib
import os
from concurrent.futures import ThreadPoolExecutor

import numpy as np
import pytest

from paper_2303_12873_b200 import workloads as W

from parity_util import (TOL_FIELD_1STEP, TOL_FIELD_L2_10STEP, TOL_PARTICLE_1STEP, check_step_parity, field_l2_error,
                         group_maxabs_errors, particle_errors, u_ref_of)

pytestmark = [pytest.mark.gpu, pytest.mark.slow]

HERE = os.path.dirname(os.path.abspath(__file__))
EPS0 = 8.8541878128e-12
FNAMES = ("Ex", "Ey", "Ez", "Bx", "By", "Bz")


@pytest.fixture(scope="module")
def Sim():
    from paper_2303_12873_b200.binding import Sim as S
    return S


# ------------------------------------------------------------------ live oracle runs, in threads
class _OracleRun:
    """State of the oracle after 1 step and after wl.nsteps steps (particles of every species, all nine fields)."""

    def __init__(self, ora, wl):
        o = ora.OracleSim(*wl.grid_args(), wl.dt, wl.order, len(wl.species))
        if wl.fields:
            o.set_fields(**wl.fields)
        for s, sp in enumerate(wl.species):
            o.load_particles(s, sp.q, sp.m, *sp.arrays())
        o.step(1)
        self.f1 = o.get_fields()
        self.p1 = [o.get_particles(s) for s in range(len(wl.species))]
        o.step(wl.nsteps - 1)
        self.fN = o.get_fields()
        self.pN = [o.get_particles(s) for s in range(len(wl.species))]


class _FakeOracle:
    """Presents a stored oracle state through the two calls check_step_parity makes."""

    def __init__(self, f, p):
        self._f, self._p = f, p

    def get_fields(self):
        return self._f

    def get_particles(self, s):
        return self._p[s]


@pytest.fixture(scope="module")
def live(ora):
    wls = {2: W.config(2, parity=True), 3: W.config(3, parity=True), 4: W.config(4, parity=True)}
    assert (wls[2].nx, wls[2].nsteps, wls[2].sort_every) == (32, 10, 1)
    assert (wls[3].nx, wls[3].ny, wls[3].nz, wls[3].nsteps) == (16, 16, 1024, 20)
    assert (wls[4].nx, wls[4].ny, wls[4].nz, wls[4].nsteps) == (8, 8, 512, 20)
    pool = ThreadPoolExecutor(max_workers=3)
    fut = {k: pool.submit(_OracleRun, ora, wl) for k, wl in wls.items()}
    pool.shutdown(wait=False)
    return wls, fut


def _run_gpu_against(Sim, wl, run, label):
    g = Sim.from_workload(wl)
    g.sort()
    g.step(1)
    res = check_step_parity(_FakeOracle(run.f1, run.p1), g, wl, label + " step 1")
    for it in range(1, wl.nsteps):
        if wl.sort_every and it % wl.sort_every == 0:
            g.sort()
        g.step(1)
    fg = g.get_fields()
    e = field_l2_error(run.fN, fg)
    assert e <= TOL_FIELD_L2_10STEP, "%s: %d-step field L2 error %.3e" % (label, wl.nsteps, e)
    L = (wl.nx * wl.dx, wl.ny * wl.dy, wl.nz * wl.dz)
    for s in range(len(wl.species)):
        ex, eu = particle_errors(run.pN[s], g.get_particles(s), L, u_ref_of(wl, s))
        assert ex <= 1e-9 and eu <= 1e-8, (label, s, ex, eu)
    c = g.counters()
    assert c["steps"] == wl.nsteps and c["fast"] + c["slow"] + c["global"] == wl.nsteps * wl.nparticles
    g.close()
    return res, e


def test_config2_32cube_10_steps(Sim, live):
    wls, fut = live
    _run_gpu_against(Sim, wls[2], fut[2].result(), "config2 32^3")


def test_config3_true_crop_16x16x1024_20_steps(Sim, live):
    wls, fut = live
    wl = wls[3]
    # the crop keeps the config's own z profile: ramp over cells 600-700, flat to 1000, pulse centred at cell 400
    zc = wl.species[0].z / wl.dz
    assert zc.min() >= 600 and zc.max() < 1000 and abs(wl.dz - 0.8e-6 / 32) < 1e-20
    _run_gpu_against(Sim, wl, fut[3].result(), "config3 16x16x1024")


def test_config4_crop_8x8x512_20_steps(Sim, live):
    wls, fut = live
    _run_gpu_against(Sim, wls[4], fut[4].result(), "config4 8x8x512")


# ------------------------------------------------------------------ config 1: stored oracle result
def _digest(wl):
    h = hashlib.sha256()
    for sp in wl.species:
        for a in sp.arrays():
            h.update(np.ascontiguousarray(a, dtype=np.float64).tobytes())
    return h.hexdigest()


def _gauss(g, wl):
    f = g.get_fields(names=("Ex", "Ey", "Ez"))
    sh = (wl.nz, wl.ny, wl.nx)
    ex, ey, ez = (f[n].reshape(sh) for n in ("Ex", "Ey", "Ez"))
    div = ((ex - np.roll(ex, 1, axis=2)) / wl.dx + (ey - np.roll(ey, 1, axis=1)) / wl.dy
           + (ez - np.roll(ez, 1, axis=0)) / wl.dz)
    return div - g.deposit_rho(-1).reshape(sh) / EPS0


def test_config1_32cube_100_steps_sort_every_4_against_stored_oracle(Sim):
    path = os.path.join(HERE, "golden", "config1_32cube_100steps.npz")
    gold = np.load(path)
    wl = W.config(1, parity=True)
    assert (wl.nx, wl.order, wl.sort_every, wl.nsteps) == (32, 3, 4, 100)
    assert _digest(wl) == str(gold["digest"]), "seeded inputs differ from the ones the stored oracle result was made from"
    assert float(gold["dt"]) == wl.dt
    g = Sim.from_workload(wl)
    g0 = _gauss(g, wl)
    g.sort()
    done = 0
    for upto in (1, 10, 100):
        for it in range(done, upto):
            if it and it % wl.sort_every == 0:
                g.sort()
            g.step(1)
        done = upto
        fg = g.get_fields(names=FNAMES)
        fo = {n: gold["%s_%d" % (n, upto)] for n in FNAMES}
        if upto == 1:
            fo1 = dict(fo, Jx=np.ones(1), Jy=np.ones(1), Jz=np.ones(1))
            fg1 = dict(fg, Jx=np.ones(1), Jy=np.ones(1), Jz=np.ones(1))
            for grp, e in group_maxabs_errors(fo1, fg1).items():
                assert e <= TOL_FIELD_1STEP, (grp, e)
        e = field_l2_error(fo, fg)
        assert e <= TOL_FIELD_L2_10STEP, "config1 32^3: %d-step field L2 error %.3e" % (upto, e)
    # Gauss residual unchanged over the 100 steps (R19), in units of one species' rho/eps0; the oracle's own
    # residual (stored) moved by no more than that either
    scale = float(gold["gauss_scale"])
    drift = float(np.abs(_gauss(g, wl) - g0).max())
    assert drift <= 1e-9 * scale, (drift, scale)
    assert abs(float(gold["gauss100"]) - float(gold["gauss0"])) <= 1e-9 * scale
    # sampled particles after 100 steps
    L = (wl.nx * wl.dx,) * 3
    for s, sp in enumerate(wl.species):
        p = g.get_particles(s)
        inv = np.empty(sp.n, dtype=np.int64)
        inv[p["id"].astype(np.int64)] = np.arange(sp.n)
        pos = inv[gold["sp%d_ids" % s]]
        for d, nm in enumerate("xyz"):
            dlt = np.abs(p[nm][pos] - gold["sp%d_%s" % (s, nm)])
            dlt = np.minimum(dlt, L[d] - dlt)
            assert dlt.max() <= 1e-9 * L[d], (s, nm, dlt.max())
        du = np.sqrt(sum((p[nm][pos] - gold["sp%d_%s" % (s, nm)]) ** 2 for nm in ("ux", "uy", "uz")))
        un = np.sqrt(sum(gold["sp%d_%s" % (s, nm)] ** 2 for nm in ("ux", "uy", "uz")))
        assert np.all(du <= 1e-8 * np.maximum(un, 0.01 * W.C_LIGHT)), (s, du.max())
    c = g.counters()
    assert c["sorts"] == 25 and c["steps"] == 100
    g.close()


# ------------------------------------------------------------------ full size, sampled element-wise
def _smooth_fields(wl, seed):
    """A few Fourier modes per component: a non-trivial gather everywhere (configs whose own fields are zero)."""
    rng = np.random.default_rng(seed)
    k, j, i = np.meshgrid(np.arange(wl.nz), np.arange(wl.ny), np.arange(wl.nx), indexing="ij")
    out = {}
    for nm, amp in (("Ex", 3e9), ("Ey", 3e9), ("Ez", 3e9), ("Bx", 10.0), ("By", 10.0), ("Bz", 10.0)):
        m = rng.integers(1, 4, size=3)
        ph = rng.uniform(0, 2 * np.pi, size=3)
        out[nm] = (amp * np.sin(2 * np.pi * m[0] * i / wl.nx + ph[0]) * np.sin(2 * np.pi * m[1] * j / wl.ny + ph[1])
                   * np.cos(2 * np.pi * m[2] * k / wl.nz + ph[2])).reshape(-1)
    return out


def _full_size_sampled(ora, Sim, wl, fields, block0, nsample=2048, bw=10, mg=3):
    """One step of the fused kernel on the whole workload; nsample particles per species against the oracle's
    gather + Boris + move + wrap, and J on a bw^3 block against the oracle's Esirkepov deposition of every
    particle that can reach it."""
    import torch
    g = Sim.from_workload(wl)
    if fields is not wl.fields:
        g.set_fields(**fields)
    g.sort()
    g.step(1)
    J = g.get_fields(names=("Jx", "Jy", "Jz"), device=True)
    og = ora.make_grid(wl.nx, wl.ny, wl.nz, wl.dx, wl.dy, wl.dz)
    zero = np.zeros(wl.ncell)                          # a laser config sets only some of the components
    E = tuple(fields.get(n, zero) for n in ("Ex", "Ey", "Ez"))
    B = tuple(fields.get(n, zero) for n in ("Bx", "By", "Bz"))
    Ld = (wl.nx * wl.dx, wl.ny * wl.dy, wl.nz * wl.dz)
    rng = np.random.default_rng(1234)
    Jo = [np.zeros(wl.ncell) for _ in range(3)]
    for s, sp in enumerate(wl.species):

        def oracle_push(sel):
            x, y, z = sp.x[sel].copy(), sp.y[sel].copy(), sp.z[sel].copy()
            ux, uy, uz = sp.ux[sel].copy(), sp.uy[sel].copy(), sp.uz[sel].copy()
            f = ora.gather(og, wl.order, x, y, z, E, B)
            ora.boris(sp.q, sp.m, wl.dt, ux, uy, uz, f[:3], f[3:])
            x1, y1, z1 = ora.move(wl.dt, x, y, z, ux, uy, uz)
            return (x, y, z), (x1, y1, z1), (ux, uy, uz)

        pg = g.get_particles(s, device=True)
        inv = torch.empty(sp.n, dtype=torch.int64, device=pg["id"].device)
        inv[pg["id"]] = torch.arange(sp.n, device=inv.device)
        ids = rng.choice(sp.n, size=nsample, replace=False)
        pos = inv[torch.from_numpy(ids).to(inv.device)]
        _, p1, u1 = oracle_push(ids)
        xw, yw, zw = (a.copy() for a in p1)
        ora.wrap(og, xw, yw, zw)
        for nm, ref, L in zip("xyz", (xw, yw, zw), Ld):
            d = np.abs(pg[nm][pos].cpu().numpy() - ref)
            d = np.minimum(d, L - d)
            assert d.max() <= TOL_PARTICLE_1STEP * L, (s, nm, d.max())
        du = np.sqrt(sum((pg[nm][pos].cpu().numpy() - ref) ** 2 for nm, ref in zip(("ux", "uy", "uz"), u1)))
        un = np.sqrt(sum(r ** 2 for r in u1))
        assert np.all(du <= TOL_PARTICLE_1STEP * np.maximum(un, u_ref_of(wl, s))), (s, du.max())
        del pg, inv
        ci = np.floor(sp.x / wl.dx).astype(np.int32)
        cj = np.floor(sp.y / wl.dy).astype(np.int32)
        ck = np.floor(sp.z / wl.dz).astype(np.int32)
        b = block0
        sel = np.nonzero((ci >= b[0] - mg) & (ci < b[0] + bw + mg) & (cj >= b[1] - mg) & (cj < b[1] + bw + mg)
                         & (ck >= b[2] - mg) & (ck < b[2] + bw + mg))[0]
        del ci, cj, ck
        assert sel.size > 0, "the J block holds no particle of species %d" % s
        q0, q1, _ = oracle_push(sel)
        ora.deposit_esirkepov(og, wl.order, sp.q, wl.dt, sp.w[sel], q0, q1, Jo)
    blk = (slice(block0[2], block0[2] + bw), slice(block0[1], block0[1] + bw), slice(block0[0], block0[0] + bw))
    jmax = max(float(J[c].abs().max()) for c in ("Jx", "Jy", "Jz"))
    assert jmax > 0
    for c, ref in zip(("Jx", "Jy", "Jz"), Jo):
        got = J[c].view(wl.nz, wl.ny, wl.nx)[blk].cpu().numpy()
        err = np.abs(got - ref.reshape(wl.nz, wl.ny, wl.nx)[blk]).max()
        assert err <= TOL_FIELD_1STEP * jmax, (c, err, jmax)
    cnt = g.counters()
    assert cnt["global"] == 0 and cnt["fast"] + cnt["slow"] == wl.nparticles
    g.close()


def test_full_size_config1_sampled_parity(ora, Sim):
    wl = W.config(1)                                   # 128^3, 16.8 M e- + 16.8 M p+, order 3
    _full_size_sampled(ora, Sim, wl, _smooth_fields(wl, 41), block0=(60, 50, 70))


def test_full_size_config3_sampled_parity(ora, Sim):
    wl = W.config(3)                                   # 128 x 128 x 1024, laser pulse in E, B; 2 ppc behind a ramp
    _full_size_sampled(ora, Sim, wl, wl.fields, block0=(60, 50, 695))      # block straddles the end of the ramp


def test_full_size_config4_sampled_parity(ora, Sim):
    wl = W.config(4)                                   # 256 x 256 x 512, slab at 16 + 4 ppc, a0 = 10
    _full_size_sampled(ora, Sim, wl, wl.fields, block0=(120, 130, 395), nsample=1024)   # pre-plasma / slab front
