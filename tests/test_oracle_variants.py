"""Pins for the oracle's NEXT-3 functions: the
"energy-conserving" gather (shape order n-1 along the directions in which a component is
staggered) and binomial smoothing.  None of these re-types the oracle's loops: they use
B-spline identities (partition of unity, reproduction of linear functions, the derivative
identity d/dxi S^n(xi - i) = S^{n-1}(xi - i + 1/2) - S^{n-1}(xi - i - 1/2)), closed-form values,
the discrete work-energy identity that gives the variant its name, and Fourier symbols."""
import numpy as np
import pytest

ORDERS = (1, 2, 3)
STAG = {0: (0.5, 0, 0), 1: (0, 0.5, 0), 2: (0, 0, 0.5), 3: (0, 0.5, 0.5), 4: (0.5, 0, 0.5), 5: (0.5, 0.5, 0)}


def _grid(ora, nx=12, ny=10, nz=9):
    return ora.make_grid(nx, ny, nz, 0.5e-6, 0.8e-6, 0.3e-6, -1e-6, 2e-6, 0.5e-6)


def _rand_particles(g, rng, n, margin=0.0):
    x = g.xmin + (margin + rng.random(n) * (g.nx - 2 * margin)) * g.dx
    y = g.ymin + (margin + rng.random(n) * (g.ny - 2 * margin)) * g.dy
    z = g.zmin + (margin + rng.random(n) * (g.nz - 2 * margin)) * g.dz
    return x, y, z


def _S(ora, n, r):
    if n == 0:
        return np.array([ora.shape0(float(v)) for v in np.atleast_1d(r)])
    return np.array([ora.shape(n, float(v)) for v in np.atleast_1d(r)])


def test_top_hat_is_half_open_and_sums_to_one(ora):
    assert ora.shape0(-0.5) == 1.0 and ora.shape0(0.5) == 0.0 and ora.shape0(0.0) == 1.0
    assert ora.shape0(0.5000001) == 0.0 and ora.shape0(-0.5000001) == 0.0
    rng = np.random.default_rng(0)
    for xi in np.concatenate([rng.random(50) * 9, [3.0, 3.5, 4.0]]):
        assert sum(ora.shape0(xi - i - 0.5) for i in range(-2, 12)) == 1.0       # partition of unity
        assert sum(ora.shape0(xi - i - 0.5) * i for i in range(-2, 12)) == np.floor(xi)   # the cell floor() names


@pytest.mark.parametrize("n", ORDERS)
def test_variant0_is_the_plain_gather(ora, n):
    g = _grid(ora); rng = np.random.default_rng(1)
    x, y, z = _rand_particles(g, rng, 100)
    F = [rng.standard_normal(g.nx * g.ny * g.nz) for _ in range(6)]
    a = ora.gather(g, n, x, y, z, F[:3], F[3:])
    b = ora.gather_variant(g, n, 0, x, y, z, F[:3], F[3:])
    for u, v in zip(a, b):
        assert np.array_equal(u, v)


@pytest.mark.parametrize("n", ORDERS)
def test_constant_field(ora, n):
    g = _grid(ora); rng = np.random.default_rng(3)
    x, y, z = _rand_particles(g, rng, 300)
    nc = g.nx * g.ny * g.nz
    vals = [1.5, -2.0, 3.25, 1e-3, -7.0, 0.125]
    F = [np.full(nc, v) for v in vals]
    out = ora.gather_variant(g, n, 1, x, y, z, F[:3], F[3:])
    for o, v in zip(out, vals):
        np.testing.assert_allclose(o, v, rtol=2e-15, atol=0)


@pytest.mark.parametrize("n", (2, 3))
def test_linear_field_every_staggering(ora, n):
    """Orders n and n-1 >= 1 both reproduce linear functions, each at its own (staggered) nodes."""
    g = _grid(ora); rng = np.random.default_rng(4)
    x, y, z = _rand_particles(g, rng, 400, margin=3.0)
    I, J, K = np.meshgrid(np.arange(g.nx), np.arange(g.ny), np.arange(g.nz), indexing="ij")
    a, b = 0.7, np.array([2.0e5, -3.0e5, 1.1e6])
    F = []
    for c in range(6):
        ox, oy, oz = STAG[c]
        f = a * (c + 1) + b[0] * (g.xmin + (I + ox) * g.dx) + b[1] * (g.ymin + (J + oy) * g.dy) + b[2] * (g.zmin + (K + oz) * g.dz)
        F.append(np.ascontiguousarray(f.transpose(2, 1, 0)).reshape(-1))
    out = ora.gather_variant(g, n, 1, x, y, z, F[:3], F[3:])
    for c in range(6):
        ref = a * (c + 1) + b[0] * x + b[1] * y + b[2] * z
        np.testing.assert_allclose(out[c], ref, rtol=0, atol=2e-15 * np.abs(ref).max())


def test_order1_takes_the_value_of_the_staggered_node_in_the_particles_cell(ora):
    """n = 1: order 0 along x for Ex means Ex_p = sum_jk S1 S1 Ex[floor(xi), j, k] (nearest staggered node),
    linear in y and z: for a field that depends on x only it is exactly the value at cell floor(xi)."""
    g = _grid(ora); rng = np.random.default_rng(5)
    x, y, z = _rand_particles(g, rng, 300)
    prof = rng.standard_normal(g.nx)
    I, J, K = np.meshgrid(np.arange(g.nx), np.arange(g.ny), np.arange(g.nz), indexing="ij")
    fx = np.ascontiguousarray((prof[I] + 0 * J).transpose(2, 1, 0)).reshape(-1)
    Z = np.zeros_like(fx)
    out = ora.gather_variant(g, 1, 1, x, y, z, (fx, Z, Z), (Z, Z, Z))
    ci = np.floor((x - g.xmin) / g.dx).astype(int)
    np.testing.assert_allclose(out[0], prof[ci], rtol=4e-16, atol=0)


@pytest.mark.parametrize("n", ORDERS)
def test_unit_impulse_is_product_of_mixed_order_shapes(ora, n):
    g = _grid(ora); rng = np.random.default_rng(6)
    nc = g.nx * g.ny * g.nz
    for c in range(6):
        ox, oy, oz = STAG[c]
        nx_, ny_, nz_ = (n - 1 if ox else n), (n - 1 if oy else n), (n - 1 if oz else n)
        i, j, k = 5, 4, 3
        F = [np.zeros(nc) for _ in range(6)]
        F[c][i + g.nx * (j + g.ny * k)] = 1.0
        x = g.xmin + (i + ox + (rng.random(60) - 0.5) * (n + 1.5)) * g.dx
        y = g.ymin + (j + oy + (rng.random(60) - 0.5) * (n + 1.5)) * g.dy
        z = g.zmin + (k + oz + (rng.random(60) - 0.5) * (n + 1.5)) * g.dz
        out = ora.gather_variant(g, n, 1, x, y, z, F[:3], F[3:])
        xi = (x - g.xmin) / g.dx; eta = (y - g.ymin) / g.dy; zeta = (z - g.zmin) / g.dz
        ref = _S(ora, nx_, xi - i - ox) * _S(ora, ny_, eta - j - oy) * _S(ora, nz_, zeta - k - oz)
        np.testing.assert_allclose(out[c], ref, rtol=0, atol=1e-15)
        assert ref.max() > 0.05
        # and it differs from the same-order gather (a swapped variant flag would pass nothing else)
        same = ora.gather(g, n, x, y, z, F[:3], F[3:])[c]
        assert np.abs(same - out[c]).max() > 1e-3
        for o in range(6):
            if o != c:
                assert np.all(out[o] == 0.0)


@pytest.mark.parametrize("n", ORDERS)
def test_gradient_of_a_nodal_potential_is_gathered_exactly(ora, n):
    """The identity behind the variant: with E_x[i+1/2,j,k] = -(phi[i+1,j,k] - phi[i,j,k]) / dx on the
    Yee grid, the variant-1 gather returns exactly -d/dx of the order-n interpolant of phi, because
    d/dxi S^n(xi - i) = S^{n-1}(xi - i + 1/2) - S^{n-1}(xi - i - 1/2).  Checked against a centred
    finite difference of the oracle's own order-n nodal interpolation (rho-deposit adjoint is not
    needed: Bx.. are zero, phi is gathered as the nodal-in-every-direction part of no component, so the
    interpolant is evaluated here from ora.shape directly)."""
    g = _grid(ora, 10, 9, 8); rng = np.random.default_rng(7)
    phi = rng.standard_normal((g.nx, g.ny, g.nz))
    ex = -(np.roll(phi, -1, 0) - phi) / g.dx
    ey = -(np.roll(phi, -1, 1) - phi) / g.dy
    ez = -(np.roll(phi, -1, 2) - phi) / g.dz
    flat = lambda a: np.ascontiguousarray(a.transpose(2, 1, 0)).reshape(-1)
    x, y, z = _rand_particles(g, rng, 40, margin=3.0)
    Z = np.zeros(g.nx * g.ny * g.nz)
    out = ora.gather_variant(g, n, 1, x, y, z, (flat(ex), flat(ey), flat(ez)), (Z, Z, Z))

    def interp(xi, eta, zeta):
        s = 0.0
        for i in range(int(np.floor(xi)) - 2, int(np.floor(xi)) + 4):
            for j in range(int(np.floor(eta)) - 2, int(np.floor(eta)) + 4):
                for k in range(int(np.floor(zeta)) - 2, int(np.floor(zeta)) + 4):
                    s += ora.shape(n, xi - i) * ora.shape(n, eta - j) * ora.shape(n, zeta - k) * phi[i % g.nx, j % g.ny, k % g.nz]
        return s

    def dshape(m, r):      # analytic derivative of S^m through the identity above (m >= 1)
        lo = ora.shape0(r + 0.5) if m == 1 else ora.shape(m - 1, r + 0.5)
        hi = ora.shape0(r - 0.5) if m == 1 else ora.shape(m - 1, r - 0.5)
        return lo - hi

    for p in range(x.size):
        xi = (x[p] - g.xmin) / g.dx; eta = (y[p] - g.ymin) / g.dy; zeta = (z[p] - g.zmin) / g.dz
        gx = gy = gz = 0.0
        for i in range(int(np.floor(xi)) - 2, int(np.floor(xi)) + 4):
            for j in range(int(np.floor(eta)) - 2, int(np.floor(eta)) + 4):
                for k in range(int(np.floor(zeta)) - 2, int(np.floor(zeta)) + 4):
                    v = phi[i % g.nx, j % g.ny, k % g.nz]
                    sx, sy, sz = ora.shape(n, xi - i), ora.shape(n, eta - j), ora.shape(n, zeta - k)
                    gx += dshape(n, xi - i) * sy * sz * v
                    gy += sx * dshape(n, eta - j) * sz * v
                    gz += sx * sy * dshape(n, zeta - k) * v
        ref = np.array([-gx / g.dx, -gy / g.dy, -gz / g.dz])
        got = np.array([out[0][p], out[1][p], out[2][p]])
        np.testing.assert_allclose(got, ref, rtol=0, atol=5e-15 * np.abs(ref).max() + 1e-9)
        if n >= 2:      # and the derivative identity itself against a centred difference of the interpolant
            h = 1e-5
            fd = -(interp(xi + h, eta, zeta) - interp(xi - h, eta, zeta)) / (2 * h * g.dx)
            assert abs(fd - got[0]) <= 1e-8 * max(1.0, abs(got[0])) * 1e3


@pytest.mark.parametrize("n", ORDERS)
def test_work_energy_identity_with_esirkepov_for_motion_along_one_axis(ora, n):
    """Why the variant is called energy-conserving: for a straight move along x,
    sum_grid Jx Ex dV dt = q w int_{x0}^{x1} Ex_p(x) dx with Ex_p the VARIANT-1 gather (Esirkepov's
    Jx for such a move is (q w/(dt dy dz)) Sy Sz int S^{n-1}(xi - i - 1/2) dxi, SURVEY 8(c.3) pin iv).
    The path integral is done by Gauss-Legendre on every sub-interval between shape breakpoints, where
    the integrand is a polynomial of degree n-1 (exact quadrature).  The same-order gather does not
    satisfy it."""
    g = _grid(ora, 9, 8, 7); rng = np.random.default_rng(8)
    nc = g.nx * g.ny * g.nz
    Ex = rng.standard_normal(nc)
    Z = np.zeros(nc)
    q, w, dt = -1.602176634e-19, 3.0e4, 1.0e-16
    gl_x, gl_w = np.polynomial.legendre.leggauss(4)
    for trial in range(6):
        xi0 = 3.0 + rng.random() * 2; dxi = (rng.random() - 0.5) * 1.8
        eta, zeta = 2.0 + rng.random() * 3, 2.0 + rng.random() * 2
        x0 = np.array([g.xmin + xi0 * g.dx]); x1 = np.array([g.xmin + (xi0 + dxi) * g.dx])
        y = np.array([g.ymin + eta * g.dy]); z = np.array([g.zmin + zeta * g.dz])
        J = [np.zeros(nc) for _ in range(3)]
        ora.deposit_esirkepov(g, n, q, dt, np.array([w]), (x0, y, z), (x1, y, z), J)
        lhs = float(np.dot(J[0], Ex)) * g.dx * g.dy * g.dz * dt
        # breakpoints of S^{n-1}(xi - i - 1/2): integers (n-1 even -> half-integers shifted by 1/2 = integers) or
        # half-integers; split at both to be safe
        a, b = (x0[0], x1[0]) if dxi >= 0 else (x1[0], x0[0])
        xa, xb = (a - g.xmin) / g.dx, (b - g.xmin) / g.dx
        cuts = [xa] + [c for c in np.arange(np.floor(xa * 2) / 2, xb + 1, 0.5) if xa < c < xb] + [xb]
        integral = {0: 0.0, 1: 0.0}
        for lo, hi in zip(cuts[:-1], cuts[1:]):
            xs = g.xmin + (0.5 * (hi + lo) + 0.5 * (hi - lo) * gl_x) * g.dx
            for variant in (0, 1):
                e = ora.gather_variant(g, n, variant, xs, np.full(4, y[0]), np.full(4, z[0]), (Ex, Z, Z), (Z, Z, Z))[0]
                integral[variant] += 0.5 * (hi - lo) * g.dx * float(np.dot(gl_w, e))
        sign = 1.0 if dxi >= 0 else -1.0
        rhs = {v: q * w * sign * integral[v] for v in (0, 1)}
        assert abs(lhs - rhs[1]) <= 2e-13 * abs(lhs) + 1e-40, (trial, lhs, rhs)
        assert abs(lhs - rhs[0]) >= 1e-4 * abs(lhs), "same-order gather unexpectedly satisfies the identity"


# ---------------------------------------------------------------- binomial smoothing ---
def test_binomial_smoothing_fourier_symbol_and_constants(ora):
    """One pass multiplies a Fourier mode exp(i k.x) by prod_d cos^2(k_d/2); constants are untouched;
    the sum over the grid is conserved; the Nyquist mode along any axis is annihilated."""
    g = _grid(ora, 12, 10, 8)
    I, J, K = np.meshgrid(np.arange(g.nx), np.arange(g.ny), np.arange(g.nz), indexing="ij")
    flat = lambda a: np.ascontiguousarray(a.transpose(2, 1, 0)).reshape(-1)
    for (mx, my, mz) in ((1, 0, 0), (2, 3, 1), (0, 5, 0), (3, 2, 4)):
        kx, ky, kz = 2 * np.pi * mx / g.nx, 2 * np.pi * my / g.ny, 2 * np.pi * mz / g.nz
        f = np.cos(kx * I + ky * J + kz * K + 0.3)
        F = flat(f).copy()
        ora.smooth_binomial(g, 2, F)
        sym = (np.cos(kx / 2) ** 2 * np.cos(ky / 2) ** 2 * np.cos(kz / 2) ** 2) ** 2
        np.testing.assert_allclose(F, sym * flat(f), rtol=0, atol=2e-15)      # six 3-term passes of roundoff
    F = np.full(g.nx * g.ny * g.nz, 2.5); ora.smooth_binomial(g, 3, F)
    np.testing.assert_allclose(F, 2.5, rtol=4e-16)
    rng = np.random.default_rng(9)
    F = rng.standard_normal(g.nx * g.ny * g.nz); s0 = F.sum()
    ora.smooth_binomial(g, 1, F)
    assert abs(F.sum() - s0) < 1e-12
    F = flat(((-1.0) ** I) * (1 + 0 * J)).copy(); ora.smooth_binomial(g, 1, F)
    assert np.abs(F).max() == 0.0
    # an impulse spreads to the 27 neighbours with weights (1/4, 1/2, 1/4)^3, periodic at the seam
    F = np.zeros(g.nx * g.ny * g.nz); F[0] = 1.0
    ora.smooth_binomial(g, 1, F)
    f3 = F.reshape(g.nz, g.ny, g.nx)
    assert f3[0, 0, 0] == 0.125 and f3[0, 0, 1] == 0.0625 and f3[0, 0, g.nx - 1] == 0.0625
    assert f3[g.nz - 1, g.ny - 1, g.nx - 1] == 1.0 / 64 and np.count_nonzero(F) == 27
    F0 = rng.standard_normal(g.nx * g.ny * g.nz); F = F0.copy(); ora.smooth_binomial(g, 0, F)
    assert np.array_equal(F, F0)


def test_cycle_with_variant_keeps_gauss_and_conserves_energy_better(ora):
    """Whole cycle with gather_variant = 1: Gauss's law residual stays constant (deposit untouched), and over
    60 steps of a thermal plasma the total (field + kinetic) energy drifts less than with the same-order gather
    (the property the variant is chosen for); smoothing J keeps Gauss only up to the smoothed rho, so it is
    checked for charge conservation of the smoothed pair instead."""
    rng = np.random.default_rng(10)
    n = 8; dx = 0.5e-6
    EPS0, C, QE, ME = 8.8541878128e-12, 299792458.0, -1.602176634e-19, 9.1093837015e-31
    g = ora.make_grid(n, n, n, dx, dx, dx)
    dt = 0.99 * ora.courant_dt(g)
    ppc = 8; npart = n ** 3 * ppc
    cells = np.repeat(np.arange(n ** 3), ppc)
    x = ((cells % n) + rng.random(npart)) * dx
    y = (((cells // n) % n) + rng.random(npart)) * dx
    z = ((cells // (n * n)) + rng.random(npart)) * dx
    u = rng.standard_normal((3, npart)) * 0.05 * C
    w = np.full(npart, 1e25 * dx ** 3 / ppc)

    def energy(sim):
        f = sim.get_fields()
        fe = 0.5 * EPS0 * sum(np.sum(f[k] ** 2) for k in ("Ex", "Ey", "Ez")) * dx ** 3
        fb = 0.5 * EPS0 * C * C * sum(np.sum(f[k] ** 2) for k in ("Bx", "By", "Bz")) * dx ** 3
        p = sim.get_particles(0)
        gam = np.sqrt(1 + (p["ux"] ** 2 + p["uy"] ** 2 + p["uz"] ** 2) / C ** 2)
        return fe + fb + np.sum(p["w"] * ME * C * C * (gam - 1))

    drift = {}
    for variant in (0, 1):
        sim = ora.OracleSim(n, n, n, dx, dx, dx, 0, 0, 0, dt, 2, 1, gather_variant=variant)
        sim.load_particles(0, QE, ME, x, y, z, u[0], u[1], u[2], w)
        rho0 = sim.deposit_rho()
        e0 = energy(sim)
        sim.step(60)
        f = sim.get_fields()
        sh = (n, n, n)
        div = sum((f[k].reshape(sh) - np.roll(f[k].reshape(sh), 1, axis=ax)) / dx for k, ax in (("Ex", 2), ("Ey", 1), ("Ez", 0)))
        res = div - (sim.deposit_rho() - rho0).reshape(sh) / EPS0        # E(0) = 0, so the residual is -rho0/eps0 at all times
        assert np.abs(res).max() <= 1e-9 * np.abs(rho0).max() / EPS0
        drift[variant] = abs(energy(sim) - e0) / e0
    assert drift[1] < drift[0], drift


# ---------------------------------------------------------------- direct deposition ---
@pytest.mark.parametrize("n", ORDERS)
def test_direct_deposition_moments_impulse_and_zero_move(ora, n):
    """ora_deposit_direct: total current = sum q w v exactly (partition of unity at each staggering); its first moment
    along the staggered axis puts the current at the mid-point of the move (B-splines reproduce linear functions);
    one particle = product of shapes at the mid-point (checked against ora_shape at every grid point); no move, no
    current; linear in q w; and, unlike Esirkepov, it does NOT satisfy discrete continuity."""
    g = _grid(ora, 10, 9, 8); rng = np.random.default_rng(20 + n)
    nc = g.nx * g.ny * g.nz
    dt, q = 1.3e-16, -1.602176634e-19
    npart = 30
    x0, y0, z0 = _rand_particles(g, rng, npart, margin=3.0)
    d = (rng.random((3, npart)) - 0.5) * 1.6
    x1, y1, z1 = x0 + d[0] * g.dx, y0 + d[1] * g.dy, z0 + d[2] * g.dz
    w = rng.random(npart) * 1e4 + 1.0
    J = [np.zeros(nc) for _ in range(3)]
    ora.deposit_direct(g, n, q, dt, w, (x0, y0, z0), (x1, y1, z1), J)
    dv = g.dx * g.dy * g.dz
    for c, (a0, a1) in enumerate(((x0, x1), (y0, y1), (z0, z1))):
        tot = np.sum(q * w * (a1 - a0) / dt)
        assert abs(J[c].sum() * dv - tot) <= 2e-14 * np.sum(np.abs(q * w * (a1 - a0) / dt))
    # first moment of Jx along x: sum Jx[i+1/2,..] (i + 1/2) dV = sum q w vx xi_half
    I = np.arange(g.nx)
    jx = J[0].reshape(g.nz, g.ny, g.nx)
    lhs = np.sum(jx.sum(axis=(0, 1)) * (I + 0.5)) * dv
    xi_h = (0.5 * (x0 + x1) - g.xmin) / g.dx
    rhs = np.sum(q * w * (x1 - x0) / dt * xi_h)
    assert abs(lhs - rhs) <= 1e-13 * np.sum(np.abs(q * w * (x1 - x0) / dt * xi_h))
    # one particle, every grid point
    J1 = [np.zeros(nc) for _ in range(3)]
    ora.deposit_direct(g, n, q, dt, w[:1], (x0[:1], y0[:1], z0[:1]), (x1[:1], y1[:1], z1[:1]), J1)
    xi = (0.5 * (x0[0] + x1[0]) - g.xmin) / g.dx; et = (0.5 * (y0[0] + y1[0]) - g.ymin) / g.dy
    ze = (0.5 * (z0[0] + z1[0]) - g.zmin) / g.dz
    v = ((x1[0] - x0[0]) / dt, (y1[0] - y0[0]) / dt, (z1[0] - z0[0]) / dt)
    for c in range(3):
        ox, oy, oz = STAG[c]
        ref = np.zeros((g.nz, g.ny, g.nx))
        for k in range(g.nz):
            for j in range(g.ny):
                for i in range(g.nx):
                    ref[k, j, i] = ora.shape(n, xi - i - ox) * ora.shape(n, et - j - oy) * ora.shape(n, ze - k - oz)
        ref *= q * w[0] * v[c] / dv
        np.testing.assert_allclose(J1[c].reshape(g.nz, g.ny, g.nx), ref, rtol=0, atol=1e-13 * np.abs(ref).max())   # xi is (x - xmin) * (1/dx) in the oracle
    # no move, no current; linear in the weight
    J0 = [np.zeros(nc) for _ in range(3)]
    ora.deposit_direct(g, n, q, dt, w, (x0, y0, z0), (x0, y0, z0), J0)
    assert not any(a.any() for a in J0)
    J2 = [np.zeros(nc) for _ in range(3)]
    ora.deposit_direct(g, n, q, dt, 2.0 * w, (x0, y0, z0), (x1, y1, z1), J2)
    for a, b in zip(J, J2):
        np.testing.assert_allclose(b, 2.0 * a, rtol=4e-16)
    # continuity is violated (that is what "direct" gives up), Esirkepov on the same moves satisfies it
    def residual(Jc):
        rho0 = np.zeros(nc); rho1 = np.zeros(nc)
        ora.deposit_rho(g, n, q, w, x0, y0, z0, rho0); ora.deposit_rho(g, n, q, w, x1, y1, z1, rho1)
        sh = (g.nz, g.ny, g.nx)
        jx_, jy_, jz_ = (a.reshape(sh) for a in Jc)
        div = ((jx_ - np.roll(jx_, 1, 2)) / g.dx + (jy_ - np.roll(jy_, 1, 1)) / g.dy + (jz_ - np.roll(jz_, 1, 0)) / g.dz)
        return np.abs((rho1 - rho0).reshape(sh) / dt + div).max() / (np.abs(rho0).max() / dt)
    Je = [np.zeros(nc) for _ in range(3)]
    ora.deposit_esirkepov(g, n, q, dt, w, (x0, y0, z0), (x1, y1, z1), Je)
    assert residual(Je) < 1e-13 and residual(J) > 1e-4
