"""Parity of the NEXT-3 options against the oracle's variants:
``pic_set_option("gather_variant", 1)`` (order n-1 along each component's staggered directions) on both
particle paths and every order, and ``pic_set_option("smooth_passes", k)`` (binomial smoothing of J).
Same tolerances as the plain path (BASELINE.json:north_star)."""
import numpy as np
import pytest

from paper_2303_12873_b200 import workloads as W

from parity_util import TOL_FIELD_L2_10STEP, check_step_parity, field_l2_error

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def Sim():
    from paper_2303_12873_b200.binding import Sim as S
    return S


def _rand_fields(wl, seed, e_amp=1e9):
    rng = np.random.default_rng(seed)
    f = {}
    for n in ("Ex", "Ey", "Ez"):
        f[n] = e_amp * rng.standard_normal(wl.ncell)
    for n in ("Bx", "By", "Bz"):
        f[n] = (e_amp / W.C_LIGHT) * rng.standard_normal(wl.ncell)
    return f


def _pair(ora, Sim, wl, gather_variant=0, smooth_passes=0, sort_first=False, force_path=0, deposit_variant=0):
    o = ora.OracleSim(*wl.grid_args(), wl.dt, wl.order, len(wl.species), gather_variant=gather_variant,
                      smooth_passes=smooth_passes, deposit_variant=deposit_variant)
    g = Sim.from_workload(wl)
    if wl.fields:
        o.set_fields(**wl.fields)
    for s, sp in enumerate(wl.species):
        o.load_particles(s, sp.q, sp.m, *sp.arrays())
    g.set_option("gather_variant", gather_variant)
    g.set_option("smooth_passes", smooth_passes)
    g.set_option("deposit_variant", deposit_variant)
    if force_path:
        g.set_option("force_path", force_path)
    if sort_first:
        g.sort()
    return o, g


# path: 1 = global-atomic kernel, 2 = fused per-tile kernel (needs a sort first)
@pytest.mark.parametrize("path", [1, 2])
@pytest.mark.parametrize("order", [1, 2, 3])
def test_energy_conserving_gather_one_step_random_fields(ora, Sim, order, path):
    wl = W.uniform_plasma(19, 13, 11, ppc=5, u_th=0.3, order=order, seed=300 + order, dx=0.5e-6, dy=0.3e-6,
                          dz=0.7e-6, shuffle=(path == 1))
    wl.fields = _rand_fields(wl, 17 + order)
    o, g = _pair(ora, Sim, wl, gather_variant=1, sort_first=(path == 2), force_path=path)
    o.step(1)
    g.step(1)
    check_step_parity(o, g, wl, "variant 1 order %d path %d" % (order, path))
    # and the variant really is a different gather: the plain oracle differs by far more than the tolerance
    o0 = ora.OracleSim(*wl.grid_args(), wl.dt, wl.order, 1)
    o0.set_fields(**wl.fields)
    sp = wl.species[0]
    o0.load_particles(0, sp.q, sp.m, *sp.arrays())
    o0.step(1)
    pu = np.sort(o0.get_particles(0)["ux"]); gu = np.sort(g.get_particles(0)["ux"])
    assert np.abs(pu - gu).max() > 1e-6 * np.abs(pu).max()
    g.close()


@pytest.mark.parametrize("order", [1, 2, 3])
def test_energy_conserving_gather_10_steps_sort_and_drift(ora, Sim, order):
    """Fresh-sort and drift instantiations of the tile kernel, deferred sort, two species."""
    wl = W.uniform_plasma(16, 12, 16, ppc=6, u_th=0.05, order=order, seed=320 + order, protons=True)
    o, g = _pair(ora, Sim, wl, gather_variant=1)
    g.sort()
    o.step(1); g.step(1)
    check_step_parity(o, g, wl, "variant 1 order %d step 1" % order)
    for it in range(1, 10):
        if it % 4 == 0:
            g.sort()
        o.step(1); g.step(1)
    e = field_l2_error(o.get_fields(), g.get_fields())
    assert e <= TOL_FIELD_L2_10STEP, e
    c = g.counters()
    assert c["fast"] + c["slow"] + c["global"] == 10 * wl.nparticles and c["fast"] > 0
    g.close()


@pytest.mark.parametrize("passes", [1, 2])
def test_binomial_smoothing_of_J(ora, Sim, passes):
    """Grids smaller than the guard width included (periodic images of images)."""
    for dims in ((12, 9, 10), (3, 5, 2)):
        wl = W.uniform_plasma(*dims, ppc=6, u_th=0.1, order=3, seed=340 + passes)
        wl.fields = _rand_fields(wl, 41, e_amp=1e8)
        o, g = _pair(ora, Sim, wl, smooth_passes=passes, sort_first=True)
        o.step(1); g.step(1)
        check_step_parity(o, g, wl, "smoothing %d passes %s" % (passes, dims))
        # the filter conserves the total current: compare with an unsmoothed step from the same state
        o2, g2 = _pair(ora, Sim, wl, smooth_passes=0, sort_first=True)
        g2.step(1)
        js, j0 = g.get_fields(names=("Jx", "Jy", "Jz")), g2.get_fields(names=("Jx", "Jy", "Jz"))
        for n in ("Jx", "Jy", "Jz"):
            assert abs(js[n].sum() - j0[n].sum()) <= 1e-10 * np.abs(j0[n]).sum()
            assert np.abs(js[n] - j0[n]).max() > 1e-3 * np.abs(j0[n]).max()      # and it did smooth
        g2.close()
        o.step(3); g.step(3)
        assert field_l2_error(o.get_fields(), g.get_fields()) <= TOL_FIELD_L2_10STEP
        g.close()


@pytest.mark.parametrize("order", [1, 2, 3])
def test_direct_deposition(ora, Sim, order):
    """deposit_variant = 1 against ora_deposit_direct: 1 step and 10 steps, sorted or not (a sorted species leaves the
    fused kernel while the option is set: every update is counted as 'global'), with the energy-conserving gather too."""
    wl = W.uniform_plasma(11, 9, 10, ppc=5, u_th=0.2, order=order, seed=360 + order, protons=True, dy=0.4e-6)
    wl.fields = _rand_fields(wl, 43, e_amp=3e8)
    o, g = _pair(ora, Sim, wl, deposit_variant=1, gather_variant=order % 2, sort_first=True)
    o.step(1); g.step(1)
    check_step_parity(o, g, wl, "direct deposition order %d" % order)
    o.step(9); g.step(9)
    assert field_l2_error(o.get_fields(), g.get_fields()) <= TOL_FIELD_L2_10STEP
    c = g.counters()
    assert c["global"] == 10 * wl.nparticles and c["fast"] + c["slow"] == 0
    g.close()


def test_option_validation(Sim):
    from paper_2303_12873_b200.binding import PicError
    wl = W.uniform_plasma(8, 8, 8, ppc=1, u_th=0.0, order=1, seed=1)
    g = Sim.from_workload(wl)
    for name, bad in (("gather_variant", 2), ("gather_variant", -1), ("smooth_passes", -1), ("smooth_passes", 17),
                      ("deposit_variant", 2)):
        with pytest.raises(PicError):
            g.set_option(name, bad)
    g.close()
