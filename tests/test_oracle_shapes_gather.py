"""Pins for the oracle's shape functions, gather and rho deposit (SURVEY.md
8(c.3) rows "Shapes" and "Gather").  None of these re-types the oracle's
formula: they use B-spline identities, the per-interval polynomial form, the
convolution definition, closed-form values and brute force."""
import numpy as np
import pytest

ORDERS = (1, 2, 3)


def _S(ora, n, r):
    return np.array([ora.shape(n, float(v)) for v in np.atleast_1d(r)])


@pytest.mark.parametrize("n", ORDERS)
def test_partition_of_unity_and_first_moment(ora, n):
    rng = np.random.default_rng(1)
    m = np.arange(-4, 6)
    for xi in rng.random(200) * 3.0 - 1.0:
        s = _S(ora, n, xi - m)
        assert abs(s.sum() - 1.0) <= 4e-16
        assert abs((m * s).sum() - xi) <= 4e-15          # linear reproduction


@pytest.mark.parametrize("n", ORDERS)
def test_symmetry_support_positivity(ora, n):
    r = np.linspace(-3, 3, 1201)
    s = _S(ora, n, r)
    assert np.array_equal(s, _S(ora, n, -r))
    half = 0.5 * (n + 1)
    assert np.all(s[np.abs(r) >= half] == 0.0)
    assert np.all(s[np.abs(r) < half - 1e-12] > 0.0)


def test_values_at_nodes(ora):
    # cardinal B-spline values at the knots/centres: textbook numbers
    assert _S(ora, 1, [0, 1, -1, 0.5]).tolist() == [1.0, 0.0, 0.0, 0.5]
    np.testing.assert_allclose(_S(ora, 2, [-1, 0, 1]), [1 / 8, 3 / 4, 1 / 8], rtol=0, atol=1e-16)
    np.testing.assert_allclose(_S(ora, 3, [-1, 0, 1, 2]), [1 / 6, 2 / 3, 1 / 6, 0], rtol=0, atol=1e-16)
    np.testing.assert_allclose(_S(ora, 2, [0.5, 1.5]), [0.5, 0.0], rtol=0, atol=1e-16)
    np.testing.assert_allclose(_S(ora, 3, [0.5, 1.5]), [23 / 48, 1 / 48], rtol=0, atol=1e-16)


@pytest.mark.parametrize("n", ORDERS)
def test_continuity_across_breakpoints(ora, n):
    # a floor/round tie must change nothing: S^n is C^{n-1}
    brk = np.arange(-(n + 1), n + 2) * 0.5
    eps = 1e-9
    for b in brk:
        lo, mid, hi = ora.shape(n, b - eps), ora.shape(n, b), ora.shape(n, b + eps)
        assert abs(lo - mid) < 2e-9 and abs(hi - mid) < 2e-9


@pytest.mark.parametrize("n", ORDERS)
def test_convolution_definition(ora, n):
    """S^n = S^{n-1} * top-hat (S^0 = 1 on [-1/2,1/2)): the definition of the
    cardinal B-spline, integrated here with composite Gauss-Legendre per piece."""
    gx, gw = np.polynomial.legendre.leggauss(8)

    def S_prev(r):
        if n == 1:
            return np.where((r >= -0.5) & (r < 0.5), 1.0, 0.0)
        return _S(ora, n - 1, r)

    for r in np.linspace(-2.4, 2.4, 41):
        # integral over t in [r-1/2, r+1/2] of S^{n-1}(t), split at breakpoints of S^{n-1}
        a, b = r - 0.5, r + 0.5
        cuts = [a] + [c for c in np.arange(-3, 3.01, 0.5) if a < c < b] + [b]
        val = 0.0
        for lo, hi in zip(cuts[:-1], cuts[1:]):
            t = 0.5 * (hi - lo) * gx + 0.5 * (hi + lo)
            val += 0.5 * (hi - lo) * np.dot(gw, S_prev(t))
        assert abs(val - ora.shape(n, r)) < 5e-15


def test_interval_polynomial_form(ora):
    """delta-polynomial form: a genuinely different evaluation."""
    rng = np.random.default_rng(2)
    for xi in rng.random(100) * 8 + 1:
        i0 = np.floor(xi); d = xi - i0
        np.testing.assert_allclose(_S(ora, 1, xi - np.array([i0, i0 + 1])), [1 - d, d], atol=2.3e-16)
        b = np.floor(xi + 0.5); e = xi - b
        np.testing.assert_allclose(_S(ora, 2, xi - np.array([b - 1, b, b + 1])),
                                   [0.5 * (0.5 - e) ** 2, 0.75 - e * e, 0.5 * (0.5 + e) ** 2], atol=2.3e-16)
        np.testing.assert_allclose(
            _S(ora, 3, xi - np.array([i0 - 1, i0, i0 + 1, i0 + 2])),
            [(1 - d) ** 3 / 6, (4 - 6 * d * d + 3 * d ** 3) / 6, (1 + 3 * d + 3 * d * d - 3 * d ** 3) / 6,
             d ** 3 / 6], atol=2.3e-16)


# ---------------------------------------------------------------- gather ---
STAG = {  # component -> (ox, oy, oz) Yee staggering (SURVEY 8(c.1) "Yee layout")
    0: (0.5, 0, 0), 1: (0, 0.5, 0), 2: (0, 0, 0.5), 3: (0, 0.5, 0.5), 4: (0.5, 0, 0.5), 5: (0.5, 0.5, 0)}


def _grid(ora, nx=12, ny=10, nz=9):
    return ora.make_grid(nx, ny, nz, 0.5e-6, 0.8e-6, 0.3e-6, -1e-6, 2e-6, 0.5e-6)


def _rand_particles(g, rng, n, margin=0.0):
    x = g.xmin + (margin + rng.random(n) * (g.nx - 2 * margin)) * g.dx
    y = g.ymin + (margin + rng.random(n) * (g.ny - 2 * margin)) * g.dy
    z = g.zmin + (margin + rng.random(n) * (g.nz - 2 * margin)) * g.dz
    return x, y, z


@pytest.mark.parametrize("n", ORDERS)
def test_gather_constant_field(ora, n):
    g = _grid(ora); rng = np.random.default_rng(3)
    x, y, z = _rand_particles(g, rng, 300)
    nc = g.nx * g.ny * g.nz
    vals = [1.5, -2.0, 3.25, 1e-3, -7.0, 0.125]
    F = [np.full(nc, v) for v in vals]
    out = ora.gather(g, n, x, y, z, F[:3], F[3:])
    for o, v in zip(out, vals):
        np.testing.assert_allclose(o, v, rtol=2e-15, atol=0)   # a few ulp of a 64..216-term sum


@pytest.mark.parametrize("n", ORDERS)
def test_gather_linear_field_every_staggering(ora, n):
    """A field a + b.x sampled at each component's own Yee location must be
    returned as a + b.x_p (B-splines reproduce linear functions)."""
    g = _grid(ora); rng = np.random.default_rng(4)
    x, y, z = _rand_particles(g, rng, 400, margin=3.0)     # keep away from the periodic seam
    I, J, K = np.meshgrid(np.arange(g.nx), np.arange(g.ny), np.arange(g.nz), indexing="ij")
    a, b = 0.7, np.array([2.0e5, -3.0e5, 1.1e6])
    F = []
    for c in range(6):
        ox, oy, oz = STAG[c]
        xs = g.xmin + (I + ox) * g.dx; ys = g.ymin + (J + oy) * g.dy; zs = g.zmin + (K + oz) * g.dz
        f = a * (c + 1) + b[0] * xs + b[1] * ys + b[2] * zs
        F.append(np.ascontiguousarray(f.transpose(2, 1, 0)).reshape(-1))      # x fastest
    out = ora.gather(g, n, x, y, z, F[:3], F[3:])
    for c in range(6):
        ref = a * (c + 1) + b[0] * x + b[1] * y + b[2] * z
        np.testing.assert_allclose(out[c], ref, rtol=0, atol=2e-15 * np.abs(ref).max())


@pytest.mark.parametrize("n", ORDERS)
def test_gather_unit_impulse_is_product_of_shapes(ora, n):
    g = _grid(ora); rng = np.random.default_rng(5)
    nc = g.nx * g.ny * g.nz
    for c in range(6):
        ox, oy, oz = STAG[c]
        i, j, k = 5, 4, 3
        F = [np.zeros(nc) for _ in range(6)]
        F[c][i + g.nx * (j + g.ny * k)] = 1.0
        # particles around the impulse
        x = g.xmin + (i + ox + (rng.random(50) - 0.5) * (n + 1.5)) * g.dx
        y = g.ymin + (j + oy + (rng.random(50) - 0.5) * (n + 1.5)) * g.dy
        z = g.zmin + (k + oz + (rng.random(50) - 0.5) * (n + 1.5)) * g.dz
        out = ora.gather(g, n, x, y, z, F[:3], F[3:])
        xi = (x - g.xmin) / g.dx; eta = (y - g.ymin) / g.dy; zeta = (z - g.zmin) / g.dz
        ref = _S(ora, n, xi - i - ox) * _S(ora, n, eta - j - oy) * _S(ora, n, zeta - k - oz)
        np.testing.assert_allclose(out[c], ref, rtol=0, atol=1e-15)
        assert ref.max() > 0.05
        for o in range(6):
            if o != c:
                assert np.all(out[o] == 0.0)


@pytest.mark.parametrize("n", ORDERS)
def test_gather_periodic_images(ora, n):
    """Shifting a particle by one period changes nothing but roundoff; and a
    particle next to the seam sees the wrapped field (impulse at index 0)."""
    g = _grid(ora); nc = g.nx * g.ny * g.nz
    F = [np.zeros(nc) for _ in range(6)]
    F[1][0 + g.nx * (2 + g.ny * 2)] = 1.0                       # Ey impulse at i=0
    x = np.array([g.xmin + (g.nx - 0.3) * g.dx]); y = np.array([g.ymin + 2.4 * g.dy]); z = np.array([g.zmin + 2.1 * g.dz])
    out = ora.gather(g, n, x, y, z, F[:3], F[3:])
    ref = ora.shape(n, -0.3) * ora.shape(n, 2.4 - 2 - 0.5) * ora.shape(n, 0.1)
    assert abs(out[1][0] - ref) < 2e-14 and ref > 0.1        # ulp(xi ~ 12) = 1.8e-15


@pytest.mark.parametrize("n", ORDERS)
def test_rho_brute_force_and_total_charge(ora, n):
    g = _grid(ora); rng = np.random.default_rng(6)
    x, y, z = _rand_particles(g, rng, 40)
    w = rng.random(40) + 0.5
    q = -1.6e-19
    rho = np.zeros(g.nx * g.ny * g.nz)
    ora.deposit_rho(g, n, q, w, x, y, z, rho)
    dV = g.dx * g.dy * g.dz
    assert abs(rho.sum() * dV - q * w.sum()) <= 1e-14 * abs(q * w.sum())
    # brute force over ALL nodes and the nearest periodic images
    xi = (x - g.xmin) / g.dx; eta = (y - g.ymin) / g.dy; zeta = (z - g.zmin) / g.dz
    ref = np.zeros((g.nz, g.ny, g.nx))
    for p in range(40):
        sx = sum(_S(ora, n, xi[p] - (np.arange(g.nx) + s * g.nx)) for s in (-1, 0, 1))
        sy = sum(_S(ora, n, eta[p] - (np.arange(g.ny) + s * g.ny)) for s in (-1, 0, 1))
        sz = sum(_S(ora, n, zeta[p] - (np.arange(g.nz) + s * g.nz)) for s in (-1, 0, 1))
        ref += q * w[p] / dV * sz[:, None, None] * sy[None, :, None] * sx[None, None, :]
    np.testing.assert_allclose(rho, ref.reshape(-1), rtol=0, atol=1e-14 * np.abs(ref).max())


@pytest.mark.parametrize("n", ORDERS)
def test_gather_adjoint_of_rho_deposit(ora, n):
    """sum_p q w phi(x_p) = sum_grid phi rho dV for a nodal phi.  The oracle
    has no nodal gather, so phi is gathered through the nodal directions of
    three components: Ex is nodal in (y,z), so use a phi that depends on (y,z)
    only, etc.  Here: Bx is nodal in x only, Ex in (y,z).  Use Ex with phi(y,z)."""
    g = _grid(ora); rng = np.random.default_rng(7)
    x, y, z = _rand_particles(g, rng, 60)
    w = rng.random(60) + 0.5; q = 2.0
    nc = g.nx * g.ny * g.nz
    phi_jk = rng.normal(size=(g.nz, g.ny))
    phi = np.broadcast_to(phi_jk[:, :, None], (g.nz, g.ny, g.nx)).reshape(-1).copy()
    F = [phi] + [np.zeros(nc) for _ in range(5)]
    out = ora.gather(g, n, x, y, z, F[:3], F[3:])       # x-dependence sums to 1 at any staggering
    rho = np.zeros(nc); ora.deposit_rho(g, n, q, w, x, y, z, rho)
    lhs = (q * w * out[0]).sum(); rhs = (phi * rho).sum() * g.dx * g.dy * g.dz
    assert abs(lhs - rhs) <= 1e-13 * max(abs(lhs), np.abs(q * w * out[0]).sum())
