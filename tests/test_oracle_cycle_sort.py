"""Pins for the whole oracle cycle and the sort (SURVEY.md 8(c.3) rows "Whole
cycle" and "Sort"): Gauss's law residual constant over 100 steps, q = 0 species
leaves fields untouched, cold-plasma oscillation at omega_p, wrap rule,
sort = stable permutation with a brute-force histogram prefix."""
import numpy as np
import pytest

from paper_2303_12873_b200 import workloads as W

EPS0 = 8.8541878128e-12


def _sim(ora, wl, order=None):
    sim = ora.OracleSim(*wl.grid_args(), wl.dt, order or wl.order, len(wl.species))
    if wl.fields:
        sim.set_fields(**wl.fields)
    for s, sp in enumerate(wl.species):
        sim.load_particles(s, sp.q, sp.m, *sp.arrays())
    return sim


def _gauss_residual(sim, wl):
    f = sim.get_fields()
    Ex, Ey, Ez = (f[k].reshape(wl.nz, wl.ny, wl.nx) for k in ("Ex", "Ey", "Ez"))
    div = ((Ex - np.roll(Ex, 1, 2)) / wl.dx + (Ey - np.roll(Ey, 1, 1)) / wl.dy + (Ez - np.roll(Ez, 1, 0)) / wl.dz)
    return div - sim.deposit_rho(-1).reshape(wl.nz, wl.ny, wl.nx) / EPS0


@pytest.mark.parametrize("order", (1, 2, 3))
def test_gauss_law_preserved_100_steps(ora, order):
    """G = div E - rho/eps0 is constant in time (R19): couples push, wrap,
    deposition and the E update.  8^3 cells x 4 ppc, warm (0.05c) so that
    particles cross cells and the periodic seam."""
    wl = W.uniform_plasma(8, 8, 8, ppc=4, u_th=0.05, order=order, seed=5)
    sim = _sim(ora, wl)
    G0 = _gauss_residual(sim, wl)
    rho_scale = np.abs(sim.deposit_rho(-1)).max() / EPS0
    assert np.abs(G0).max() > 1e-3 * rho_scale            # E(0)=0, rho non-uniform: G != 0 (R19)
    for _ in range(4):
        sim.step(25)
        G = _gauss_residual(sim, wl)
        assert np.abs(G - G0).max() <= 1e-12 * rho_scale
    p = sim.get_particles(0)
    assert p["x"].min() >= 0.0 and p["x"].max() < wl.nx * wl.dx
    assert np.abs(sim.get_fields()["Ex"]).max() > 0


def test_gauss_zero_for_colocated_pairs(ora):
    wl = W.uniform_plasma(6, 6, 6, ppc=4, u_th=0.02, order=3, seed=6, protons=True)
    sim = _sim(ora, wl)
    rho_e = np.abs(sim.deposit_rho(0)).max() / EPS0
    assert np.abs(_gauss_residual(sim, wl)).max() <= 1e-13 * rho_e
    sim.step(30)
    assert np.abs(_gauss_residual(sim, wl)).max() <= 1e-12 * rho_e


def test_neutral_species_leaves_fields_untouched(ora):
    wl = W.uniform_plasma(6, 6, 6, ppc=2, u_th=0.05, order=2, seed=7)
    wl.species[0].q = 0.0
    sim = _sim(ora, wl)
    x0 = sim.get_particles(0)["x"]
    sim.step(5)
    f = sim.get_fields()
    assert all(np.all(f[k] == 0.0) for k in f)
    assert not np.array_equal(sim.get_particles(0)["x"], x0)   # but it streams


def test_cold_plasma_oscillates_at_omega_p(ora):
    """Cold uniform electrons on a lattice + small sinusoidal velocity
    perturbation: Ex oscillates at omega_p (36.9 steps per period at config-0
    parameters) -- sanity of units and signs, not roundoff."""
    nx = 16
    wl = W.uniform_plasma(nx, 4, 4, ppc=1, u_th=0.0, order=1, seed=8)
    sp = wl.species[0]
    # regular lattice (one particle at each cell centre) -> rho uniform, E stays 0 without perturbation
    k, j, i = np.meshgrid(np.arange(4), np.arange(4), np.arange(nx), indexing="ij")
    sp.x = ((i + 0.5) * wl.dx).reshape(-1); sp.y = ((j + 0.5) * wl.dy).reshape(-1); sp.z = ((k + 0.5) * wl.dz).reshape(-1)
    v0 = 1e-4 * W.C_LIGHT
    sp.ux = v0 * np.sin(2 * np.pi * sp.x / (nx * wl.dx)); sp.uy = np.zeros(sp.n); sp.uz = np.zeros(sp.n)
    sim = _sim(ora, wl)
    n0 = 1e25
    wp = np.sqrt(n0 * W.Q_E ** 2 / (EPS0 * W.M_E))
    period_steps = 2 * np.pi / (wp * wl.dt)
    assert 36 < period_steps < 38
    amp = []
    for _ in range(int(2.5 * period_steps)):
        sim.step(1)
        Ex = sim.get_fields()["Ex"].reshape(4, 4, nx)
        amp.append(Ex[0, 0, 3])
    amp = np.array(amp)
    # zero crossings of Ex(t) at a fixed point give the period
    zc = np.nonzero(np.signbit(amp[1:]) != np.signbit(amp[:-1]))[0]
    t = zc + amp[zc] / (amp[zc] - amp[zc + 1])          # linear interpolation of the crossing
    half = np.diff(t).mean()
    assert abs(2 * half - period_steps) < 0.06 * period_steps
    assert np.abs(amp).max() > 0


def test_wrap_rule(ora):
    g = ora.make_grid(4, 4, 4, 0.5, 0.5, 0.5, -1.0, 0.0, 0.0)
    x = np.array([-1.0, 0.999, 1.0, 1.2, -1.3, -1.0 - 1e-17, np.nextafter(1.0, 0)])
    y = np.full(7, 0.5); z = np.full(7, 0.5)
    ora.wrap(g, x, y, z)
    np.testing.assert_array_equal(x, [-1.0, 0.999, -1.0, 1.2 - 2.0, -1.3 + 2.0, -1.0, np.nextafter(1.0, 0)])
    assert np.all((x >= -1.0) & (x < 1.0))
    # a position a hair below xmin must not land ON xmax
    x = np.array([np.nextafter(-1.0, -2.0)]); y = np.array([0.5]); z = np.array([0.5])
    ora.wrap(g, x, y, z)
    assert -1.0 <= x[0] < 1.0


def test_sort_is_stable_permutation_with_bruteforce_offsets(ora):
    wl = W.uniform_plasma(5, 4, 3, ppc=6, u_th=0.01, order=1, seed=9, shuffle=True)
    sim = _sim(ora, wl)
    before = sim.get_particles(0)
    sim.sort()
    after = sim.get_particles(0)
    g = sim.g
    key = (np.clip(np.floor(after["x"] / wl.dx), 0, wl.nx - 1)
           + wl.nx * (np.clip(np.floor(after["y"] / wl.dy), 0, wl.ny - 1)
                      + wl.ny * np.clip(np.floor(after["z"] / wl.dz), 0, wl.nz - 1))).astype(np.int64)
    assert np.all(np.diff(key) >= 0)                                           # keys non-decreasing
    assert np.array_equal(np.sort(after["id"]), np.arange(wl.nparticles, dtype=np.uint64))   # id multiset
    for name in ("x", "y", "z", "ux", "uy", "uz", "w"):                        # attributes travel with ids
        assert np.array_equal(after[name], before[name][after["id"].astype(np.int64)])
    hist = np.bincount(key, minlength=wl.ncell)
    assert np.array_equal(sim.cell_offset[0], np.concatenate([[0], np.cumsum(hist)]))
    # stability: inside a cell, ids keep their input order
    for c in range(wl.ncell):
        ids = after["id"][sim.cell_offset[0][c]:sim.cell_offset[0][c + 1]]
        assert np.all(np.diff(ids.astype(np.int64)) > 0)
    # and it matches numpy's stable argsort on the keys of the input
    key_in = ora.cell_keys(g, before["x"], before["y"], before["z"])
    assert np.array_equal(after["id"].astype(np.int64), np.argsort(key_in, kind="stable"))


def test_step_after_sort_equals_step_without_sort(ora):
    wl = W.uniform_plasma(6, 5, 4, ppc=5, u_th=0.03, order=3, seed=10, shuffle=True)
    a, b = _sim(ora, wl), _sim(ora, wl)
    b.sort()
    a.step(2); b.step(2)
    fa, fb = a.get_fields(), b.get_fields()
    for k in fa:
        scale = np.abs(fa[k]).max()
        assert np.abs(fa[k] - fb[k]).max() <= 1e-12 * scale       # summation order only
    pa, pb = a.get_particles(0), b.get_particles(0)
    inv = np.argsort(pb["id"])
    for name in ("x", "ux"):
        np.testing.assert_allclose(pb[name][inv], pa[name], rtol=1e-12, atol=1e-12 * wl.nx * wl.dx if name == "x" else 0)
