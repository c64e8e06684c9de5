"""Parity of the CUDA path (through the C ABI) against the oracle, element by
element on the same seeded inputs (BASELINE.json:north_star tolerances; readings
R20-R24 in DESIGN.md).  All tests here need a B200: ``-m gpu``."""
import numpy as np
import pytest

from paper_2303_12873_b200 import workloads as W

from parity_util import (TOL_FIELD_L2_10STEP, check_step_parity, field_l2_error, make_pair,
                         particle_errors, u_ref_of)

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def Sim():
    from paper_2303_12873_b200.binding import Sim as S
    return S


def _rand_fields(wl, seed, e_amp=1e9):
    """Smooth-ish random E and B on every component so the gather sees all six staggerings."""
    rng = np.random.default_rng(seed)
    f = {}
    for n in ("Ex", "Ey", "Ez"):
        f[n] = e_amp * rng.standard_normal(wl.ncell)
    for n in ("Bx", "By", "Bz"):
        f[n] = (e_amp / W.C_LIGHT) * rng.standard_normal(wl.ncell)
    return f


# path: 1 = global-atomic kernel, 2 = fused per-tile kernel (needs a sort first)
@pytest.mark.parametrize("path", [1, 2])
@pytest.mark.parametrize("order", [1, 2, 3])
def test_one_step_every_order_random_fields(ora, Sim, order, path):
    # anisotropic cells, extents that are not multiples of the tile, 5 ppc, hot (0.3 c) electrons
    wl = W.uniform_plasma(19, 13, 11, ppc=5, u_th=0.3, order=order, seed=100 + order, dx=0.5e-6, dy=0.3e-6,
                          dz=0.7e-6, shuffle=(path == 1))
    wl.fields = _rand_fields(wl, 7 + order)
    o, g = make_pair(ora, Sim, wl, sort_first=(path == 2), force_path=path)
    o.step(1)
    g.step(1)
    check_step_parity(o, g, wl, "order %d path %d" % (order, path))
    c = g.counters()
    if path == 1:
        assert c["global"] == wl.nparticles and c["fast"] + c["slow"] == 0
    else:
        assert c["fast"] + c["slow"] + c["global"] == wl.nparticles and c["fast"] + c["slow"] > 0


def test_config0_full_size_1_and_10_steps(ora, Sim):
    wl = W.config(0)                                   # 32^3, 262,144 electrons, CIC
    o, g = make_pair(ora, Sim, wl)
    g.sort()
    o.step(1); g.step(1)
    check_step_parity(o, g, wl, "config0 step 1")
    o.step(9); g.step(9)
    e = field_l2_error(o.get_fields(), g.get_fields())
    assert e <= TOL_FIELD_L2_10STEP, "10-step field L2 error %.3e" % e
    L = (wl.nx * wl.dx,) * 3
    ex, eu = particle_errors(o.get_particles(0), g.get_particles(0), L, u_ref_of(wl, 0))
    assert ex <= 1e-10 and eu <= 1e-9, (ex, eu)


def test_config1_parity_two_species_sort_every_4(ora, Sim):
    wl = W.config(1, parity=True, n=16)                # 16^3 x (8+8) ppc, order 3
    o, g = make_pair(ora, Sim, wl)
    g.sort()
    o.step(1); g.step(1)
    check_step_parity(o, g, wl, "config1 step 1")
    for it in range(1, 12):
        if it % wl.sort_every == 0:
            g.sort()
        o.step(1); g.step(1)
    e = field_l2_error(o.get_fields(), g.get_fields())
    assert e <= TOL_FIELD_L2_10STEP, "12-step field L2 error %.3e" % e
    c = g.counters()
    assert c["sorts"] == 3 and c["steps"] == 12


def test_config2_parity_hot_order3(ora, Sim):
    wl = W.config(2, parity=True, n=24)                # 0.05 c, order 3, 10 steps, sort every 4
    o, g = make_pair(ora, Sim, wl)
    g.sort()
    o.step(1); g.step(1)
    check_step_parity(o, g, wl, "config2 step 1")
    for it in range(1, 10):
        if it % wl.sort_every == 0:
            g.sort()
        o.step(1); g.step(1)
    e = field_l2_error(o.get_fields(), g.get_fields())
    assert e <= TOL_FIELD_L2_10STEP, "10-step field L2 error %.3e" % e


def test_config3_lwfa_crop(ora, Sim):
    wl = W.config(3, parity=True, nx=8, ny=8, nz=256)  # laser pulse in the fields, cold 2 ppc, ramp
    o, g = make_pair(ora, Sim, wl)
    g.sort()
    o.step(1); g.step(1)
    check_step_parity(o, g, wl, "config3 step 1")
    o.step(9); g.step(9)
    e = field_l2_error(o.get_fields(), g.get_fields())
    assert e <= TOL_FIELD_L2_10STEP, "10-step field L2 error %.3e" % e


def test_config4_plasma_mirror_crop(ora, Sim):
    wl = W.config(4, parity=True, nx=8, ny=8, nz=128)  # 0 vs 20 particles per cell, two species, a0 = 10
    o, g = make_pair(ora, Sim, wl)
    g.sort()
    o.step(1); g.step(1)
    check_step_parity(o, g, wl, "config4 step 1")
    o.step(9); g.step(9)
    e = field_l2_error(o.get_fields(), g.get_fields())
    assert e <= TOL_FIELD_L2_10STEP, "10-step field L2 error %.3e" % e


def test_sorted_vs_unsorted_vs_shuffled_same_physics(ora, Sim):
    """pic_sort never changes the physics beyond summation order; pic_step is correct for any order."""
    wl = W.uniform_plasma(12, 12, 12, ppc=6, u_th=0.1, order=3, seed=5, shuffle=True)
    wl.fields = _rand_fields(wl, 11, e_amp=1e8)
    o, g1 = make_pair(ora, Sim, wl)                    # shuffled, never sorted -> global path
    _, g2 = make_pair(ora, Sim, wl, sort_first=True)   # sorted -> tile path
    o.step(3); g1.step(3); g2.step(3)
    fo = o.get_fields()
    assert field_l2_error(fo, g1.get_fields()) <= TOL_FIELD_L2_10STEP
    assert field_l2_error(fo, g2.get_fields()) <= TOL_FIELD_L2_10STEP
    assert g1.counters()["global"] == 3 * wl.nparticles
    assert g2.counters()["global"] < 3 * wl.nparticles


def test_boundary_straddling_particles(ora, Sim):
    """Particles within a fraction of a cell of every face and corner, moving outwards at ~0.9 c."""
    nx, ny, nz, d = 8, 6, 5, 0.5e-6
    rng = np.random.default_rng(3)
    n = 4096
    L = np.array([nx, ny, nz]) * d
    side = rng.integers(0, 2, size=(3, n))
    eps = rng.random((3, n)) * 0.3 * d
    pos = np.where(side == 0, eps, L[:, None] - eps)
    pos = np.minimum(pos, np.nextafter(L, 0)[:, None])
    u = (np.where(side == 0, -1.0, 1.0)) * 2.0 * W.C_LIGHT * rng.random((3, n))
    for order in (1, 2, 3):
        wl = W.Workload("straddle", nx, ny, nz, d, d, d, W.courant_dt(d, d, d), order, 1, 0,
                        [W.Species("e", -W.Q_E, W.M_E, pos[0].copy(), pos[1].copy(), pos[2].copy(),
                                   u[0].copy(), u[1].copy(), u[2].copy(), np.full(n, 1e5))])
        for path in (1, 2):
            o, g = make_pair(ora, Sim, wl, sort_first=(path == 2), force_path=path)
            o.step(2); g.step(2)
            check_step_parity(o, g, wl, "straddle order %d path %d" % (order, path))
            p = g.get_particles(0)
            for dd, Ld in zip("xyz", L):
                assert (p[dd] >= 0).all() and (p[dd] < Ld).all()


@pytest.mark.parametrize("dims", [(1, 1, 1), (2, 3, 1), (3, 3, 3), (4, 5, 6), (130, 3, 2)])
def test_tiny_and_ragged_grids(ora, Sim, dims):
    """Grids smaller than the guard width (several periodic images per cell) and a pitch > one block."""
    nx, ny, nz = dims
    wl = W.uniform_plasma(nx, ny, nz, ppc=3, u_th=0.2, order=3, seed=17)
    wl.fields = _rand_fields(wl, 19, e_amp=1e8)
    for path in (1, 2):
        o, g = make_pair(ora, Sim, wl, sort_first=(path == 2), force_path=path)
        o.step(2); g.step(2)
        check_step_parity(o, g, wl, "grid %s path %d" % (dims, path))


def test_empty_species_and_q0_species(ora, Sim):
    """n = 0 species is a no-op; a q = 0 species streams freely and leaves the fields untouched."""
    wl = W.uniform_plasma(8, 8, 8, ppc=2, u_th=0.1, order=2, seed=23, protons=True)
    wl.species[1].q = 0.0
    z = np.zeros(0)
    wl.species.append(W.Species("none", W.Q_E, W.M_P, z, z, z, z, z, z, z))
    o, g = make_pair(ora, Sim, wl)
    g.sort()
    o.step(2); g.step(2)
    check_step_parity(o, g, wl, "empty+q0")
    assert g.num_particles(2) == 0


def test_yee_vacuum_and_source_exact(ora, Sim):
    """No particles that matter (one q = 0 particle): the Yee update alone, random E, B; the two sides
    evaluate the same expression tree up to FMA contraction -> 1e-14 relative."""
    wl = W.uniform_plasma(21, 10, 7, ppc=1, u_th=0.0, order=1, seed=2, dx=0.4e-6, dy=0.5e-6, dz=0.3e-6)
    wl.species[0].q = 0.0
    wl.fields = _rand_fields(wl, 5)
    o, g = make_pair(ora, Sim, wl)
    o.step(5); g.step(5)
    fo, fg = o.get_fields(), g.get_fields()
    for grp in (("Ex", "Ey", "Ez"), ("Bx", "By", "Bz")):
        ref = max(np.abs(fo[n]).max() for n in grp)
        for n in grp:
            assert np.abs(fo[n] - fg[n]).max() <= 1e-13 * ref
    for n in ("Jx", "Jy", "Jz"):
        assert not fg[n].any()


@pytest.mark.parametrize("dims", [(21, 10, 7), (32, 8, 8), (33, 9, 17), (70, 5, 3), (2, 1, 40), (96, 24, 13)])
def test_yee_tma_and_plain_kernels_agree(ora, Sim, dims):
    """The TMA-staged tile kernels (default) and the plain one-thread-per-cell kernels evaluate the same expression
    tree: bit-identical E, B after 4 steps on grids that are smaller than, equal to and ragged against the
    32 x 8 x 4 / 32 x 8 x 8 Yee tiles; all within 1e-13 of the oracle
    (J = 0: one q = 0 particle)."""
    nx, ny, nz = dims
    wl = W.uniform_plasma(nx, ny, nz, ppc=1, u_th=0.0, order=1, seed=2, dx=0.4e-6, dy=0.5e-6, dz=0.3e-6)
    wl.species[0].q = 0.0
    wl.fields = _rand_fields(wl, 7)
    out = []
    for mode in (3, 0, 1, 2):   # per-tile TMA, plain, B only, E only
        o, g = make_pair(ora, Sim, wl)
        g.set_option("yee_tma", mode)
        assert g.counters()["yee_tma"] == 1
        g.step(4)
        out.append(g.get_fields())
    o.step(4)
    fo = o.get_fields()
    for n in ("Ex", "Ey", "Ez", "Bx", "By", "Bz"):
        for other in out[1:]:
            assert np.array_equal(out[0][n], other[n]), n
    for grp in (("Ex", "Ey", "Ez"), ("Bx", "By", "Bz")):
        ref = max(np.abs(fo[n]).max() for n in grp)
        for n in grp:
            assert np.abs(fo[n] - out[0][n]).max() <= 1e-13 * ref
