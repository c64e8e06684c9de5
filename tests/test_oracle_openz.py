"""Pins for the oracle's NEXT-2 mode (the wakefield science case): a z boundary
beyond which every field is zero and particles are deleted (``open_z``), the moving window and the plane current
source (antenna).  The mode is composed of the pinned periodic functions plus zeroing and relabelling, so the pins
check exactly those additions: the interior must not notice them (to roundoff, inside the light cone), the boundary
planes must match a Yee step written independently with numpy on zero-padded arrays, a moving window must be a pure
relabelling of a larger fixed box, the antenna must obey Ampere's law exactly, and charge that leaves is the only charge
that goes missing."""
import numpy as np
import pytest

C_LIGHT = 299792458.0
EPS0 = 8.8541878128e-12
QE, ME = -1.602176634e-19, 9.1093837015e-31


def _sim(ora, nz, open_z, nx=6, ny=5, order=3, nsp=1, dx=0.5e-6, dz=0.25e-6):
    g = ora.make_grid(nx, ny, nz, dx, dx, dz)
    dt = 0.99 * ora.courant_dt(g)
    return ora.OracleSim(nx, ny, nz, dx, dx, dz, 0.0, 0.0, 0.0, dt, order, nsp, open_z=open_z), dt


def _blob(rng, nx, ny, nz, k0, k1, amp):
    f = np.zeros((nz, ny, nx))
    f[k0:k1] = amp * rng.standard_normal((k1 - k0, ny, nx))
    return f.reshape(-1)


def _particles(rng, n, nx, ny, zlo, zhi, dx, dz, u_th=0.1):
    x = rng.random(n) * nx * dx; y = rng.random(n) * ny * dx; z = (zlo + rng.random(n) * (zhi - zlo)) * dz
    u = rng.standard_normal((3, n)) * u_th * C_LIGHT
    return x, y, z, u[0], u[1], u[2], np.full(n, 1e3)


@pytest.mark.parametrize("order", (1, 2, 3))
def test_interior_does_not_notice_the_open_boundary(ora, order):
    """Fields and particles confined to the middle third: for as many steps as light needs to reach a z face the open
    box and the periodic box of the same size agree to roundoff everywhere."""
    rng = np.random.default_rng(1)
    nx, ny, nz = 6, 5, 36
    fields = {n: _blob(rng, nx, ny, nz, 14, 22, a) for n, a in (("Ex", 1e9), ("Ey", 1e9), ("Ez", 1e9), ("Bx", 3.0), ("By", 3.0), ("Bz", 3.0))}
    parts = _particles(rng, 40, nx, ny, 15, 21, 0.5e-6, 0.25e-6)
    out = []
    for open_z in (False, True):
        sim, dt = _sim(ora, nz, open_z, order=order)
        sim.set_fields(**fields)
        sim.load_particles(0, QE, ME, *parts)
        sim.step(8)                 # the blob's edge is 14 planes from a face; it moves at most one plane per step
        out.append((sim.get_fields(), sim.get_particles(0)))
    # not bit for bit: the padded grid's origin is 4 cells lower, so (z - zmin) / dz rounds differently (reading R30)
    for n in out[0][0]:
        ref = np.abs(out[0][0][n]).max()
        assert ref > 0
        assert np.abs(out[0][0][n] - out[1][0][n]).max() <= 1e-11 * ref, n
    for n in ("x", "y", "z", "ux", "uy", "uz"):
        np.testing.assert_allclose(out[0][1][n], out[1][1][n], rtol=1e-12, atol=1e-20)


def _yee_step_numpy(E, B, J, dt, d):
    """One B half / E / B half step with every value outside the z range equal to zero and x, y periodic: an independent
    numpy statement of SURVEY 8(c.1) steps 6-8 (arrays [k, j, i])."""
    dx, dy, dz = d
    c2 = C_LIGHT ** 2

    def up(a, axis):        # a[index + 1]
        if axis == 0:
            return np.concatenate([a[1:], np.zeros_like(a[:1])], axis=0)
        return np.roll(a, -1, axis=axis)

    def dn(a, axis):        # a[index - 1]
        if axis == 0:
            return np.concatenate([np.zeros_like(a[:1]), a[:-1]], axis=0)
        return np.roll(a, 1, axis=axis)

    Ex, Ey, Ez = (a.copy() for a in E); Bx, By, Bz = (a.copy() for a in B)

    def push_B(h):
        nonlocal Bx, By, Bz
        Bx = Bx - h * ((up(Ez, 1) - Ez) / dy - (up(Ey, 0) - Ey) / dz)
        By = By - h * ((up(Ex, 0) - Ex) / dz - (up(Ez, 2) - Ez) / dx)
        Bz = Bz - h * ((up(Ey, 2) - Ey) / dx - (up(Ex, 1) - Ex) / dy)

    push_B(0.5 * dt)
    Ex = Ex + dt * (c2 * ((Bz - dn(Bz, 1)) / dy - (By - dn(By, 0)) / dz) - J[0] / EPS0)
    Ey = Ey + dt * (c2 * ((Bx - dn(Bx, 0)) / dz - (Bz - dn(Bz, 2)) / dx) - J[1] / EPS0)
    Ez = Ez + dt * (c2 * ((By - dn(By, 2)) / dx - (Bx - dn(Bx, 1)) / dy) - J[2] / EPS0)
    push_B(0.5 * dt)
    return (Ex, Ey, Ez), (Bx, By, Bz)


def test_boundary_planes_against_numpy_yee_with_zero_exterior(ora):
    rng = np.random.default_rng(2)
    nx, ny, nz = 6, 5, 9
    sim, dt = _sim(ora, nz, True, nsp=1)
    names = ("Ex", "Ey", "Ez", "Bx", "By", "Bz")
    f = {n: rng.standard_normal(nx * ny * nz) * (1e9 if n[0] == "E" else 3.0) for n in names}     # non-zero right up to both faces
    sim.set_fields(**f)
    E = tuple(f[n].reshape(nz, ny, nx) for n in names[:3]); B = tuple(f[n].reshape(nz, ny, nx) for n in names[3:])
    zero = np.zeros((nz, ny, nx))
    for step in range(3):
        sim.step(1)
        E, B = _yee_step_numpy(E, B, (zero, zero, zero), dt, (0.5e-6, 0.5e-6, 0.25e-6))
        got = sim.get_fields()
        for n, ref in zip(names, E + B):
            np.testing.assert_allclose(got[n].reshape(nz, ny, nx), ref, rtol=0, atol=4e-15 * np.abs(ref).max())
    # and the periodic box differs at the faces (the wrap is really gone)
    per, _ = _sim(ora, nz, False)
    per.set_fields(**f)
    per.step(1)
    assert np.abs(per.get_fields()["Bx"].reshape(nz, ny, nx)[-1] - _yee_step_numpy(
        tuple(f[n].reshape(nz, ny, nx) for n in names[:3]), tuple(f[n].reshape(nz, ny, nx) for n in names[3:]),
        (zero, zero, zero), dt, (0.5e-6, 0.5e-6, 0.25e-6))[1][0][-1]).max() > 1e-3


def test_moving_window_is_a_relabelling_of_a_larger_fixed_box(ora):
    """A window of 30 planes that moves up one cell per step sees exactly what planes m .. m + 29 of a fixed 48-plane box
    hold, particles included, as long as nothing has reached a face of either."""
    rng = np.random.default_rng(3)
    nx, ny = 6, 5
    big, _ = _sim(ora, 48, True)
    win, _ = _sim(ora, 30, True)
    fb = {n: _blob(rng, nx, ny, 48, 16, 20, a) for n, a in (("Ex", 1e9), ("By", 3.0), ("Ez", 1e9), ("Bx", 3.0))}
    parts = _particles(rng, 30, nx, ny, 16.5, 19.5, 0.5e-6, 0.25e-6)
    big.set_fields(**fb)
    win.set_fields(**{n: v.reshape(48, ny, nx)[:30].reshape(-1) for n, v in fb.items()})
    big.load_particles(0, QE, ME, *parts)
    win.load_particles(0, QE, ME, *parts)
    for m in range(1, 7):
        big.step(1)
        win.step(1)
        win.shift_window(1)
        a, b = big.get_fields(), win.get_fields()
        for n in a:         # to roundoff: the window's origin moves, so (z - zmin) / dz rounds differently (R30)
            ref = max(np.abs(a[n]).max(), 1e-300)
            assert np.abs(a[n].reshape(48, ny, nx)[m:m + 30] - b[n].reshape(30, ny, nx)).max() <= 1e-11 * ref, (n, m)
            assert not a[n].reshape(48, ny, nx)[:m].any() and not a[n].reshape(48, ny, nx)[m + 30:].any()
        assert abs(win.zmin - m * 0.25e-6) < 1e-20
    pa, pb = big.get_particles(0), win.get_particles(0)
    assert np.array_equal(pa["id"], pb["id"]) and np.array_equal(pa["w"], pb["w"])
    for n in ("x", "y", "z", "ux", "uy", "uz"):
        np.testing.assert_allclose(pa[n], pb[n], rtol=1e-12, atol=1e-20)
    # a window that has moved past a particle deletes it
    win.shift_window(20)
    assert win.get_particles(0)["x"].size == 0 and win.deleted == 30


def test_antenna_obeys_ampere_exactly_and_is_used_once(ora):
    rng = np.random.default_rng(4)
    nx, ny, nz = 6, 5, 16
    sim, dt = _sim(ora, nz, True)
    S = rng.standard_normal((ny, nx)) * 1e12
    sim.add_plane_source(0, 7, S)                   # Jx on plane 7
    sim.step(1)
    f = sim.get_fields()
    ex = f["Ex"].reshape(nz, ny, nx); by = f["By"].reshape(nz, ny, nx)
    np.testing.assert_allclose(ex[7], -dt * (S / EPS0), rtol=4e-16)
    assert np.count_nonzero(ex) == nx * ny and np.array_equal(f["Jx"].reshape(nz, ny, nx)[7], S)
    # By sits at k + 1/2: the second half push gives By[k] -= (dt/2) (Ex[k+1] - Ex[k]) / dz
    np.testing.assert_allclose(by[6], -0.5 * dt * ex[7] / 0.25e-6, rtol=4e-16)
    np.testing.assert_allclose(by[7], +0.5 * dt * ex[7] / 0.25e-6, rtol=4e-16)
    assert np.count_nonzero(by) == 2 * nx * ny
    sim.step(1)
    assert not sim.get_fields()["Jx"].any()         # the source was for one step


@pytest.mark.parametrize("order", (1, 3))
def test_only_charge_that_leaves_goes_missing(ora, order):
    """Particles streaming towards the upper face: continuity holds to roundoff at every node at least three planes
    inside the face, deleted particles are counted, and once everybody has left the interior J is zero."""
    rng = np.random.default_rng(5)
    nx, ny, nz = 6, 5, 12
    sim, dt = _sim(ora, nz, True, order=order)
    n = 50
    x, y, z, ux, uy, uz, w = _particles(rng, n, nx, ny, 8.0, 11.5, 0.5e-6, 0.25e-6, u_th=0.0)
    uz = np.full(n, 2.0 * C_LIGHT)                   # gamma ~ 2.2, v_z ~ 0.89 c: 0.44 cells per step at this dt/dz
    sim.load_particles(0, QE, ME, x, y, z, ux, uy, uz, w)
    g = sim.g
    for step in range(12):
        rho0 = sim.deposit_rho(0).reshape(nz, ny, nx)
        alive = sim.get_particles(0)["x"].size
        sim.step(1)
        rho1 = sim.deposit_rho(0).reshape(nz, ny, nx)
        f = sim.get_fields()
        jx, jy, jz = (f[c].reshape(nz, ny, nx) for c in ("Jx", "Jy", "Jz"))
        div = ((jx - np.roll(jx, 1, 2)) / g.dx + (jy - np.roll(jy, 1, 1)) / g.dy)
        div[1:] += (jz[1:] - jz[:-1]) / g.dz
        div[0] += jz[0] / g.dz
        res = (rho1 - rho0) / dt + div
        scale = max(np.abs(rho0).max(), np.abs(rho1).max(), 1e-300) / dt
        assert np.abs(res[:nz - 3]).max() <= 1e-12 * scale, (step, np.abs(res[:nz - 3]).max() / scale)
        assert sim.get_particles(0)["x"].size + sim.deleted == n and sim.get_particles(0)["x"].size <= alive
    assert sim.get_particles(0)["x"].size == 0 and sim.deleted == n
    sim.step(1)
    assert not any(sim.get_fields()[c].any() for c in ("Jx", "Jy", "Jz"))


def test_damping_layer_absorbs_what_the_bare_open_end_reflects(ora):
    """A plane pulse sent at the upper end: the bare open end (zero exterior) reflects all of its energy, a 12-cell
    damping layer with a smooth profile sends back less than 2 %; factors of 1 change nothing; one step multiplies the
    layer's planes by exactly the given factors."""
    nx, ny, nz = 4, 4, 96
    dz = 0.25e-6
    k, _, _ = np.meshgrid(np.arange(nz), np.arange(ny), np.arange(nx), indexing="ij")
    env = np.exp(-((k - 40.0) / 6.0) ** 2) * np.cos(2 * np.pi * (k - 40.0) / 12.0)
    envb = np.exp(-((k + 0.5 - 40.0) / 6.0) ** 2) * np.cos(2 * np.pi * (k + 0.5 - 40.0) / 12.0)
    fields = {"Ex": (1e9 * env).reshape(-1), "By": (1e9 / C_LIGHT * envb).reshape(-1)}      # travels towards +z

    def energy(sim, lo, hi):
        f = sim.get_fields()
        e = sum(np.sum(f[n].reshape(nz, ny, nx)[lo:hi] ** 2) for n in ("Ex", "Ey", "Ez"))
        b = sum(np.sum(f[n].reshape(nz, ny, nx)[lo:hi] ** 2) for n in ("Bx", "By", "Bz"))
        return EPS0 * (e + C_LIGHT ** 2 * b)

    nd = 12
    prof = np.exp(-0.35 * ((nd - np.arange(nd)) / nd) ** 2)
    back = {}
    for name, factors in (("bare", None), ("ones", np.ones(nd)), ("layer", prof)):
        sim, dt = _sim(ora, nz, True, nx=nx, ny=ny)
        sim.set_fields(**fields)
        if factors is not None:
            sim.set_damping(factors)
        e0 = energy(sim, 0, nz)
        nsteps = int(2 * (nz - 40) * dz / (C_LIGHT * dt)) + 10          # to the end and back to the middle
        sim.step(nsteps)
        back[name] = energy(sim, 0, nz - nd - 4) / e0
    assert back["bare"] > 0.9 and abs(back["bare"] - back["ones"]) < 1e-12
    assert back["layer"] < 0.02, back
    # where it acts: factors of zero leave exactly zero on the layer's planes at both ends, and one step changes nothing
    # further than its stencils reach (3 pushes, one plane each)
    rng = np.random.default_rng(6)
    f = {n: rng.standard_normal(nx * ny * nz) * (1e9 if n[0] == "E" else 3.0) for n in ("Ex", "Ey", "Ez", "Bx", "By", "Bz")}
    a, _ = _sim(ora, nz, True, nx=nx, ny=ny)
    b, _ = _sim(ora, nz, True, nx=nx, ny=ny)
    a.set_fields(**f)
    b.set_fields(**f)
    b.set_damping(np.zeros(2))
    a.step(1)
    b.step(1)
    fa, fb = a.get_fields(), b.get_fields()
    for n in ("Ex", "Ey", "Ez", "Bx", "By", "Bz"):
        va, vb = fa[n].reshape(nz, ny, nx), fb[n].reshape(nz, ny, nx)
        assert np.array_equal(va[5:nz - 5], vb[5:nz - 5]), n
        assert not vb[:2].any() and not vb[nz - 2:].any(), n
        assert va[:2].any(), n
    assert any(not np.array_equal(fa[n].reshape(nz, ny, nx)[2:5], fb[n].reshape(nz, ny, nx)[2:5]) for n in ("Ex", "Ey", "Bx", "By"))
    with pytest.raises(ValueError):
        b.set_damping(np.ones(nz))
