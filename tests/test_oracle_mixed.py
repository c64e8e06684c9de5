"""Pins for the oracle's NEXT-4 functions: the gather and the Boris push in single
precision with everything that touches a position kept in double.  They are pinned to the fp64 functions (themselves
pinned by closed forms) through the standard forward error bounds of float products and sums, from above AND from
below (the result must really carry float roundoff), to the invariants that survive rounding, and, for the whole
cycle, to the one invariant mixed precision must not touch: Gauss's law, which the fp64 deposition alone upholds."""
import numpy as np
import pytest

EPS32 = float(np.finfo(np.float32).eps) / 2        # unit roundoff 2^-24
C_LIGHT, EPS0 = 299792458.0, 8.8541878128e-12
QE, ME = -1.602176634e-19, 9.1093837015e-31
ORDERS = (1, 2, 3)


def _grid(ora, nx=11, ny=9, nz=10):
    return ora.make_grid(nx, ny, nz, 0.5e-6, 0.8e-6, 0.3e-6, -1e-6, 2e-6, 0.5e-6)


def _rand_particles(g, rng, n):
    return (g.xmin + rng.random(n) * g.nx * g.dx, g.ymin + rng.random(n) * g.ny * g.dy, g.zmin + rng.random(n) * g.nz * g.dz)


def _is_float(a):
    return np.array_equal(a.astype(np.float32).astype(np.float64), a)


@pytest.mark.parametrize("variant", (0, 1))
@pytest.mark.parametrize("n", ORDERS)
def test_gather_f32_is_the_fp64_gather_within_the_float_error_bound(ora, n, variant):
    g = _grid(ora); rng = np.random.default_rng(30 + n)
    x, y, z = _rand_particles(g, rng, 300)
    nc = g.nx * g.ny * g.nz
    # positive fields: sum |terms| is the result itself, so the bound is relative
    F = [rng.random(nc) * a + a for a in (1e9, 2e9, 3e9, 1.0, 2.0, 3.0)]
    ref = ora.gather_variant(g, n, variant, x, y, z, F[:3], F[3:])
    got = ora.gather_f32(g, n, variant, x, y, z, F[:3], F[3:])
    nterms = (n + 1) ** 3
    for r, o in zip(ref, got):
        assert _is_float(o)
        err = np.abs(o - r) / r
        assert err.max() <= (8 + nterms) * EPS32, err.max()          # 7 roundings per term + the running sum + the last cast
        assert err.max() >= 0.05 * EPS32, "no float roundoff in the result: it was not computed in single precision"
    # any sign: the bound is relative to max |F| (the shapes sum to one)
    F = [rng.standard_normal(nc) * a for a in (1e9, 2e9, 3e9, 1.0, 2.0, 3.0)]
    ref = ora.gather_variant(g, n, variant, x, y, z, F[:3], F[3:])
    got = ora.gather_f32(g, n, variant, x, y, z, F[:3], F[3:])
    for r, o, f in zip(ref, got, F):
        assert np.abs(o - r).max() <= (8 + nterms) * EPS32 * np.abs(f).max()
    # a constant field comes back to within the bound, and as a float
    F = [np.full(nc, v) for v in (1.5e9, -2.0e9, 3.25e9, 1e-3, -7.0, 0.125)]
    got = ora.gather_f32(g, n, variant, x, y, z, F[:3], F[3:])
    for o, f in zip(got, F):
        assert np.abs(o / f[0] - 1).max() <= (8 + nterms) * EPS32


def test_boris_f32_against_fp64_boris_and_its_invariants(ora):
    rng = np.random.default_rng(40)
    n = 400
    dt = 1e-16
    u = rng.standard_normal((3, n)) * 0.5 * C_LIGHT
    u32 = u.astype(np.float32).astype(np.float64)
    E = rng.standard_normal((3, n)) * 1e11
    B = rng.standard_normal((3, n)) * 1e3
    a = [c.copy() for c in u32]; b = [c.copy() for c in u32]
    ora.boris(QE, ME, dt, *a, E, B)
    ora.boris_f32(QE, ME, dt, *b, E, B)
    scale = np.sqrt(sum(c ** 2 for c in a))
    for ca, cb in zip(a, b):
        assert _is_float(cb)
        d = np.abs(ca - cb) / scale
        assert d.max() <= 40 * EPS32 and d.max() >= 0.05 * EPS32
    # pure rotation: |u| kept to a few float roundings; u parallel to B untouched beyond that
    Bz = np.zeros((3, n)); Bz[2] = 2e3
    Z = np.zeros((3, n))
    c = [v.copy() for v in u32]
    ora.boris_f32(QE, ME, dt, *c, Z, Bz)
    n0 = np.sqrt(sum(v ** 2 for v in u32)); n1 = np.sqrt(sum(v ** 2 for v in c))
    assert np.abs(n1 / n0 - 1).max() <= 12 * EPS32
    assert np.abs(c[2] - u32[2]).max() <= 4 * EPS32 * n0.max()
    # uniform E, no B: the exact kick q E dt / m to float roundoff
    Ex = np.zeros((3, n)); Ex[0] = 3e10
    d = [v.copy() for v in u32]
    ora.boris_f32(QE, ME, dt, *d, Ex, Z)
    kick = QE * 3e10 * dt / ME
    assert np.abs(d[0] - (u32[0] + kick)).max() <= 6 * EPS32 * (np.abs(u32[0]).max() + abs(kick))
    assert np.array_equal(d[1], u32[1]) and np.array_equal(d[2], u32[2])


@pytest.mark.parametrize("order", (1, 3))
def test_mixed_precision_cycle_keeps_gauss_and_stays_close_to_fp64(ora, order):
    rng = np.random.default_rng(50)
    n, dx, ppc = 8, 0.5e-6, 6
    g = ora.make_grid(n, n, n, dx, dx, dx)
    dt = 0.99 * ora.courant_dt(g)
    npart = n ** 3 * ppc
    cells = np.repeat(np.arange(n ** 3), ppc)
    x = ((cells % n) + rng.random(npart)) * dx
    y = (((cells // n) % n) + rng.random(npart)) * dx
    z = ((cells // (n * n)) + rng.random(npart)) * dx
    u = rng.standard_normal((3, npart)) * 0.05 * C_LIGHT
    w = np.full(npart, 1e25 * dx ** 3 / ppc)
    sims = []
    for prec in (0, 1):
        sim = ora.OracleSim(n, n, n, dx, dx, dx, 0, 0, 0, dt, order, 1, precision=prec)
        sim.load_particles(0, QE, ME, x, y, z, u[0], u[1], u[2], w)
        rho0 = sim.deposit_rho()
        sim.step(20)
        f = sim.get_fields()
        sh = (n, n, n)
        div = sum((f[k].reshape(sh) - np.roll(f[k].reshape(sh), 1, axis=ax)) / dx for k, ax in (("Ex", 2), ("Ey", 1), ("Ez", 0)))
        res = div - (sim.deposit_rho() - rho0).reshape(sh) / EPS0
        assert np.abs(res).max() <= 1e-9 * np.abs(rho0).max() / EPS0, prec        # fp64 deposition: exact in both modes
        sims.append(sim)
    p0, p1 = sims[0].get_particles(0), sims[1].get_particles(0)
    assert _is_float(p1["ux"]) and not _is_float(p0["ux"])
    dpos = max(np.abs(((p0[k] - p1[k] + 0.5 * n * dx) % (n * dx)) - 0.5 * n * dx).max() for k in "xyz")
    assert 1e-12 * dx < dpos <= 1e-4 * dx
    f0, f1 = sims[0].get_fields(), sims[1].get_fields()
    num = sum(np.sum((f0[k] - f1[k]) ** 2) for k in ("Ex", "Ey", "Ez"))
    den = sum(np.sum(f0[k] ** 2) for k in ("Ex", "Ey", "Ez"))
    assert 1e-12 < np.sqrt(num / den) <= 1e-3
