"""Pins for the oracle's Boris push and position update (SURVEY.md 8(c.3) row
"Boris"): closed forms for pure B (exact rotation), pure E (exact momentum,
hyperbolic trajectory to O(dt^2)), E x B drift, q = 0."""
import numpy as np

QE, ME, C0 = -1.602176634e-19, 9.1093837015e-31, 299792458.0


def _arr(v, n=1):
    return np.full(n, float(v))


def test_pure_B_preserves_norm_and_parallel_component(ora):
    rng = np.random.default_rng(11)
    n = 2000
    u = rng.normal(size=(3, n)) * 0.5 * C0            # relativistic too
    B = rng.normal(size=(3, n)) * 50.0                 # tesla
    ux, uy, uz = (u[i].copy() for i in range(3))
    zero = np.zeros(n)
    ora.boris(QE, ME, 3e-13, ux, uy, uz, (zero, zero, zero), (B[0].copy(), B[1].copy(), B[2].copy()))
    n0 = np.sqrt((u ** 2).sum(0)); n1 = np.sqrt(ux ** 2 + uy ** 2 + uz ** 2)
    assert np.max(np.abs(n1 - n0) / n0) < 2e-15        # |u| preserved to roundoff (a few ulp)
    bhat = B / np.sqrt((B ** 2).sum(0))
    par0 = (u * bhat).sum(0); par1 = ux * bhat[0] + uy * bhat[1] + uz * bhat[2]
    assert np.max(np.abs(par1 - par0) / n0) < 2e-15    # u.B unchanged


def test_pure_B_rotation_angle_closed_form(ora):
    """theta = -sign(q) * 2 atan(|q| B dt / (2 m gamma)) about B: exact for one step."""
    for q in (QE, -QE, 3 * QE):
        for Bz, dt, u0 in ((1.0, 1e-12, 0.1 * C0), (200.0, 5e-13, 2.0 * C0), (5e3, 1e-13, 0.01 * C0)):
            ux, uy, uz = _arr(u0), _arr(0.0), _arr(0.3 * u0)
            ora.boris(q, ME, dt, ux, uy, uz, (_arr(0), _arr(0), _arr(0)), (_arr(0), _arr(0), _arr(Bz)))
            gam = np.sqrt(1 + (u0 ** 2 + (0.3 * u0) ** 2) / C0 ** 2)
            theta = -np.sign(q) * 2 * np.arctan(abs(q) * Bz * dt / (2 * ME * gam))
            assert abs(ux[0] - u0 * np.cos(theta)) < 4e-16 * u0
            assert abs(uy[0] - u0 * np.sin(theta)) < 4e-16 * u0
            assert uz[0] == 0.3 * u0


def test_uniform_E_momentum_exact_and_trajectory_second_order(ora):
    E0 = 5e11
    qm = QE / ME
    T = 2e-14                                           # q E T / (m c) ~ 5.9: strongly relativistic

    def run(nsteps):
        dt = T / nsteps
        # leap-frog start: u^{-1/2} = exact u(-dt/2) for a particle at rest at t=0
        ux = _arr(qm * E0 * (-dt / 2)); uy, uz = _arr(0.0), _arr(0.0)
        x, y, z = _arr(0.0), _arr(0.0), _arr(0.0)
        for k in range(nsteps):
            ora.boris(QE, ME, dt, ux, uy, uz, (_arr(E0), _arr(0), _arr(0)), (_arr(0), _arr(0), _arr(0)))
            assert abs(ux[0] - qm * E0 * (k + 0.5) * dt) <= 1e-14 * abs(qm * E0 * T)   # exact momentum
            x, y, z = ora.move(dt, x, y, z, ux, uy, uz)
        return x[0]

    a = qm * E0 / C0
    exact = C0 / a * (np.sqrt(1 + (a * T) ** 2) - 1)     # (m c^2/qE)(sqrt(1+(qEt/mc)^2)-1)
    e1, e2 = abs(run(50) - exact), abs(run(100) - exact)
    assert e1 < 1e-3 * abs(exact)
    assert 3.5 < e1 / e2 < 4.5                           # second order


def test_ExB_drift(ora):
    Ey, Bz = 1e5, 1.0                                    # E/B = 1e5 m/s << c
    dt = 1e-13                                           # omega_c dt = 0.0176
    ux, uy, uz = _arr(0.0), _arr(0.0), _arr(0.0)
    x, y, z = _arr(0.0), _arr(0.0), _arr(0.0)
    nsteps = 357 * 20                                    # ~20 gyro-periods (T_c = 3.57e-11 s)
    for _ in range(nsteps):
        ora.boris(QE, ME, dt, ux, uy, uz, (_arr(0), _arr(Ey), _arr(0)), (_arr(0), _arr(0), _arr(Bz)))
        x, y, z = ora.move(dt, x, y, z, ux, uy, uz)
    vd = x[0] / (nsteps * dt)
    assert abs(vd - Ey / Bz) < 0.02 * Ey / Bz            # E x B / B^2 = +x, independent of q
    assert abs(y[0]) < 2.5 * (ME * (Ey / Bz) / (abs(QE) * Bz))   # bounded by the gyro-diameter


def test_q_zero_free_streaming(ora):
    rng = np.random.default_rng(12)
    n = 100
    u = rng.normal(size=(3, n)) * C0
    ux, uy, uz = (u[i].copy() for i in range(3))
    F = [rng.normal(size=n) * 1e12 for _ in range(6)]
    ora.boris(0.0, ME, 1e-15, ux, uy, uz, F[:3], F[3:])
    assert np.array_equal(ux, u[0]) and np.array_equal(uy, u[1]) and np.array_equal(uz, u[2])
    x0 = rng.random(n); y0 = rng.random(n); z0 = rng.random(n)
    x1, y1, z1 = ora.move(1e-9, x0, y0, z0, ux, uy, uz)
    gam = np.sqrt(1 + (u ** 2).sum(0) / C0 ** 2)
    np.testing.assert_allclose(x1, x0 + 1e-9 * u[0] / gam, rtol=1e-15)
    v = np.sqrt(((np.array([x1 - x0, y1 - y0, z1 - z0]) / 1e-9) ** 2).sum(0))
    assert np.all(v < C0)
