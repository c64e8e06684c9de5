"""Pins for the oracle's Yee update (SURVEY.md 8(c.3) row "Yee"): the analytic
vacuum dispersion relation as a roundoff-exact three-level recurrence for a
discretely transverse plane wave at Courant number 0.99, div B and div E
preservation, equivalence of the split B push with the leap-frog B push."""
import numpy as np

C0 = 299792458.0


def _grid(ora, nx=12, ny=10, nz=8):
    return ora.make_grid(nx, ny, nz, 0.5e-6, 0.7e-6, 0.4e-6, 0.0, 0.0, 0.0)


def _idx(g):
    K, J, I = np.meshgrid(np.arange(g.nz), np.arange(g.ny), np.arange(g.nx), indexing="ij")
    return I, J, K


def _plane_wave_E(g, modes, e_pol, phase0=0.3):
    """E components of one Fourier mode sampled at their own Yee locations."""
    I, J, K = _idx(g)
    kx = 2 * np.pi * modes[0] / (g.nx * g.dx); ky = 2 * np.pi * modes[1] / (g.ny * g.dy)
    kz = 2 * np.pi * modes[2] / (g.nz * g.dz)
    out = []
    for c, (ox, oy, oz) in enumerate(((0.5, 0, 0), (0, 0.5, 0), (0, 0, 0.5))):
        ph = kx * (I + ox) * g.dx + ky * (J + oy) * g.dy + kz * (K + oz) * g.dz + phase0
        out.append((e_pol[c] * np.cos(ph)).reshape(-1).copy())
    return out, (kx, ky, kz)


def _step(ora, g, dt, E, B, J=None):
    nc = g.nx * g.ny * g.nz
    J = J or [np.zeros(nc) for _ in range(3)]
    ora.yee_push_B(g, 0.5 * dt, E, B)
    ora.yee_push_E(g, dt, E, B, J)
    ora.yee_push_B(g, 0.5 * dt, E, B)


def test_vacuum_dispersion_recurrence(ora):
    """E^{n+1} + E^{n-1} = 2 cos(w dt) E^n with cos(w dt) = 1 - c^2 dt^2 sum K_d^2 / 2,
    K_d = 2 sin(k_d D_d/2)/D_d, i.e. sin^2(w dt/2)/(c dt)^2 = sum sin^2(k_d D_d/2)/D_d^2."""
    g = _grid(ora)
    dt = 0.99 * ora.courant_dt(g)
    modes = (2, -1, 3)                                   # oblique k
    kvec = [2 * np.pi * m / (N * d) for m, N, d in zip(modes, (g.nx, g.ny, g.nz), (g.dx, g.dy, g.dz))]
    Kd = np.array([2 * np.sin(k * d / 2) / d for k, d in zip(kvec, (g.dx, g.dy, g.dz))])
    a = np.array([1.0, 0.4, -0.7])
    e_pol = a - Kd * (a @ Kd) / (Kd @ Kd)                # discretely transverse: e.K = 0
    E, _ = _plane_wave_E(g, modes, e_pol * 1e9)
    nc = g.nx * g.ny * g.nz
    B = [np.zeros(nc) for _ in range(3)]                 # B^0 = 0: standing-wave start
    hist = [np.concatenate(E)]
    for _ in range(12):
        _step(ora, g, dt, E, B)
        hist.append(np.concatenate(E))
    cosw = 1.0 - 0.5 * C0 ** 2 * dt ** 2 * (Kd @ Kd)
    assert -1.0 < cosw < 1.0
    scale = np.abs(hist[0]).max()
    for n in range(1, 12):
        res = hist[n + 1] + hist[n - 1] - 2 * cosw * hist[n]
        assert np.abs(res).max() <= 2e-14 * scale
    # and it is not trivially satisfied: the field really oscillates
    assert np.abs(hist[6] - hist[0]).max() > 0.1 * scale


def _divB(g, B):
    Bx, By, Bz = (a.reshape(g.nz, g.ny, g.nx) for a in B)
    return ((np.roll(Bx, -1, 2) - Bx) / g.dx + (np.roll(By, -1, 1) - By) / g.dy + (np.roll(Bz, -1, 0) - Bz) / g.dz)


def _divE(g, E):
    Ex, Ey, Ez = (a.reshape(g.nz, g.ny, g.nx) for a in E)
    return ((Ex - np.roll(Ex, 1, 2)) / g.dx + (Ey - np.roll(Ey, 1, 1)) / g.dy + (Ez - np.roll(Ez, 1, 0)) / g.dz)


def test_divB_and_divE_preserved(ora):
    g = _grid(ora); rng = np.random.default_rng(71)
    nc = g.nx * g.ny * g.nz
    dt = 0.99 * ora.courant_dt(g)
    E = [rng.normal(size=nc) * 1e9 for _ in range(3)]    # arbitrary E (not divergence-free)
    B = [np.zeros(nc) for _ in range(3)]                 # div B = 0 start
    dE0 = _divE(g, E)
    for _ in range(20):
        _step(ora, g, dt, E, B)
    bscale = max(np.abs(b).max() for b in B) / min(g.dx, g.dy, g.dz)
    assert np.abs(_divB(g, B)).max() <= 1e-13 * bscale
    escale = max(np.abs(e).max() for e in E) / min(g.dx, g.dy, g.dz)
    assert np.abs(_divE(g, E) - dE0).max() <= 1e-13 * escale


def test_split_B_equals_leapfrog_B(ora):
    """B^{n+1/2} of the textbook leap-frog equals our B after the first half
    push; two half pushes with the same E equal one full push."""
    g = _grid(ora); rng = np.random.default_rng(72)
    nc = g.nx * g.ny * g.nz
    dt = 0.9 * ora.courant_dt(g)
    E = [rng.normal(size=nc) for _ in range(3)]
    B1 = [rng.normal(size=nc) / C0 for _ in range(3)]
    B2 = [b.copy() for b in B1]
    ora.yee_push_B(g, 0.5 * dt, E, B1); ora.yee_push_B(g, 0.5 * dt, E, B1)
    ora.yee_push_B(g, dt, E, B2)
    for a, b in zip(B1, B2):
        assert np.abs(a - b).max() <= 4e-16 * np.abs(b).max() + 1e-30


def test_uniform_current_drives_uniform_E(ora):
    """Ampere with a uniform J and no curl: E -= dt J / eps0 exactly."""
    g = _grid(ora); nc = g.nx * g.ny * g.nz
    E = [np.zeros(nc) for _ in range(3)]; B = [np.zeros(nc) for _ in range(3)]
    J = [np.full(nc, 3.0), np.full(nc, -1.0), np.full(nc, 0.5)]
    dt = 1e-16
    ora.yee_push_E(g, dt, E, B, J)
    for e, j in zip(E, (3.0, -1.0, 0.5)):
        np.testing.assert_allclose(e, -dt * j / 8.8541878128e-12, rtol=1e-15)


def test_single_impulse_curl_signs(ora):
    """A unit Ez impulse at (i,j,k+1/2) must produce, after a B push,
    Bx[i,j,k] = -dth/dy (from +dEz/dy at j-1... i.e. Bx(i,j-1) = -dth/dy, Bx(i,j) = +dth/dy)
    and By(i-1,j) = +dth/dx, By(i,j) = -dth/dx  (Faraday: dB/dt = -curl E)."""
    g = _grid(ora); nc = g.nx * g.ny * g.nz
    i, j, k = 5, 4, 3
    E = [np.zeros(nc) for _ in range(3)]; B = [np.zeros(nc) for _ in range(3)]
    E[2][i + g.nx * (j + g.ny * k)] = 1.0
    dth = 1e-16
    ora.yee_push_B(g, dth, E, B)
    Bx, By, Bz = (a.reshape(g.nz, g.ny, g.nx) for a in B)
    # (curl E)_x = dEz/dy - dEy/dz ; Bx at (i, j+1/2, k+1/2) uses Ez[j+1]-Ez[j]
    assert np.isclose(Bx[k, j, i], +dth / g.dy) and np.isclose(Bx[k, j - 1, i], -dth / g.dy)
    # (curl E)_y = dEx/dz - dEz/dx ; By at (i+1/2, j, k+1/2) uses Ez[i+1]-Ez[i]
    assert np.isclose(By[k, j, i], -dth / g.dx) and np.isclose(By[k, j, i - 1], +dth / g.dx)
    assert np.all(Bz == 0.0)
    assert np.count_nonzero(Bx) == 2 and np.count_nonzero(By) == 2
