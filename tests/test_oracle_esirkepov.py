"""Pins for the oracle's Esirkepov deposition (SURVEY.md 8(c.3) row
"Esirkepov"): discrete continuity against independent nodal rho deposits,
total current, the Villasenor-Buneman closed form (order 1, one cell), the
1-D closed form (integral of the order n-1 spline), zero move, reversal
antisymmetry and a brute-force solve of the difference equation."""
import numpy as np
import pytest

ORDERS = (1, 2, 3)
Q = -1.602176634e-19


def _grid(ora, nx=9, ny=8, nz=7):
    return ora.make_grid(nx, ny, nz, 0.5e-6, 0.8e-6, 0.3e-6, -1e-6, 2e-6, 0.5e-6)   # anisotropic


def _pos(g, xi, eta, zeta):
    return (g.xmin + np.asarray(xi) * g.dx, g.ymin + np.asarray(eta) * g.dy, g.zmin + np.asarray(zeta) * g.dz)


def _J(ora, g, n, q, dt, w, p0, p1):
    nc = g.nx * g.ny * g.nz
    J = [np.zeros(nc) for _ in range(3)]
    ora.deposit_esirkepov(g, n, q, dt, w, p0, p1, J)
    return [a.reshape(g.nz, g.ny, g.nx) for a in J]


def _div_backward(g, J):
    return ((J[0] - np.roll(J[0], 1, axis=2)) / g.dx + (J[1] - np.roll(J[1], 1, axis=1)) / g.dy
            + (J[2] - np.roll(J[2], 1, axis=0)) / g.dz)


def _moves(g, rng, n, amp=0.999):
    xi0 = rng.random(n) * g.nx; et0 = rng.random(n) * g.ny; ze0 = rng.random(n) * g.nz
    d = (rng.random((3, n)) * 2 - 1) * amp
    return (xi0, et0, ze0), (xi0 + d[0], et0 + d[1], ze0 + d[2])


@pytest.mark.parametrize("n", ORDERS)
def test_discrete_continuity(ora, n):
    """(rho1 - rho0)/dt + div J = 0 at every node, to roundoff, with random
    moves up to +-0.999 cell including moves across the periodic seam."""
    g = _grid(ora); rng = np.random.default_rng(21 + n)
    c0, c1 = _moves(g, rng, 300)
    p0, p1 = _pos(g, *c0), _pos(g, *c1)
    w = rng.random(300) + 0.5; dt = 1e-16
    J = _J(ora, g, n, Q, dt, w, p0, p1)
    nc = g.nx * g.ny * g.nz
    rho0 = np.zeros(nc); rho1 = np.zeros(nc)
    ora.deposit_rho(g, n, Q, w, *p0, rho0)
    x1w, y1w, z1w = (a.copy() for a in p1)
    ora.wrap(g, x1w, y1w, z1w)
    ora.deposit_rho(g, n, Q, w, x1w, y1w, z1w, rho1)
    res = (rho1 - rho0).reshape(g.nz, g.ny, g.nx) / dt + _div_backward(g, J)
    assert np.abs(res).max() <= 1e-13 * np.abs(rho0).max() / dt
    assert np.abs(J[0]).max() > 0


@pytest.mark.parametrize("n", ORDERS)
def test_total_current(ora, n):
    g = _grid(ora); rng = np.random.default_rng(31)
    c0, c1 = _moves(g, rng, 50)
    p0, p1 = _pos(g, *c0), _pos(g, *c1)
    w = rng.random(50) + 0.5; dt = 2e-16
    J = _J(ora, g, n, Q, dt, w, p0, p1)
    dV = g.dx * g.dy * g.dz
    for d in range(3):
        ref = (Q * w * (p1[d] - p0[d]) / dt).sum()
        scale = np.abs(Q * w * (p1[d] - p0[d]) / dt).sum()
        assert abs(J[d].sum() * dV - ref) <= 1e-13 * scale


def test_villasenor_buneman_closed_form(ora):
    """Order 1, both positions in one cell: the four Jx values are
    dx*[(1-ybar)(1-zbar)+dy dz/12], dx*[ybar(1-zbar)-dy dz/12],
    dx*[(1-ybar)zbar-dy dz/12], dx*[ybar zbar+dy dz/12] (cell units) times
    q w/(dt dy dz); same by cyclic permutation for Jy, Jz."""
    g = _grid(ora); rng = np.random.default_rng(41)
    dt, w = 1e-16, np.array([1.7])
    for _ in range(20):
        cell = np.array([rng.integers(0, g.nx), rng.integers(0, g.ny), rng.integers(0, g.nz)])
        f0 = 0.05 + 0.9 * rng.random(3); f1 = 0.05 + 0.9 * rng.random(3)
        J = _J(ora, g, 1, Q, dt, w, _pos(g, *[[v] for v in cell + f0]), _pos(g, *[[v] for v in cell + f1]))
        d = f1 - f0; bar = 0.5 * (f0 + f1)
        h = [g.dx, g.dy, g.dz]
        for a in range(3):                               # a: direction of the current
            b, c = (a + 1) % 3, (a + 2) % 3
            coef = Q * w[0] / dt * h[a] / (g.dx * g.dy * g.dz)       # q w/(dt * transverse area)
            exp = np.zeros((2, 2))                        # [db, dc]
            exp[0, 0] = d[a] * ((1 - bar[b]) * (1 - bar[c]) + d[b] * d[c] / 12)
            exp[1, 0] = d[a] * (bar[b] * (1 - bar[c]) - d[b] * d[c] / 12)
            exp[0, 1] = d[a] * ((1 - bar[b]) * bar[c] - d[b] * d[c] / 12)
            exp[1, 1] = d[a] * (bar[b] * bar[c] + d[b] * d[c] / 12)
            got = np.zeros((2, 2)); N = [g.nx, g.ny, g.nz]
            for db in range(2):
                for dc in range(2):
                    idx = cell.copy(); idx[b] = (idx[b] + db) % N[b]; idx[c] = (idx[c] + dc) % N[c]
                    got[db, dc] = J[a][idx[2], idx[1], idx[0]]
            np.testing.assert_allclose(got, coef * exp, rtol=0, atol=4e-15 * abs(coef))
            assert abs(np.abs(J[a]).sum() - np.abs(got).sum()) <= 1e-14 * abs(coef)   # nothing elsewhere


def _S_prev(n, r):
    """S^{n-1}; S^0 is the top-hat on [-1/2, 1/2)."""
    r = np.asarray(r, dtype=float); a = np.abs(r)
    if n == 1:
        return np.where(a < 0.5, 1.0, 0.0)
    if n == 2:
        return np.maximum(0.0, 1.0 - a)
    return np.where(a <= 0.5, 0.75 - a * a, np.where(a <= 1.5, 0.5 * (1.5 - a) ** 2, 0.0))


@pytest.mark.parametrize("n", ORDERS)
def test_motion_along_x_only_closed_form(ora, n):
    """Jx[i+1/2,j,k] = (q w/(dt dy dz)) Sy[j] Sz[k] int_{xi0}^{xi1} S^{n-1}(xi-i-1/2) dxi."""
    g = _grid(ora); gx, gw = np.polynomial.legendre.leggauss(6)
    dt, w = 1e-16, np.array([2.5])
    for xi0, xi1 in ((3.2, 3.9), (3.7, 4.4), (4.1, 3.3), (0.2, -0.5), (8.6, 9.3)):
        eta, zeta = 4.37, 2.81
        J = _J(ora, g, n, Q, dt, w, _pos(g, [xi0], [eta], [zeta]), _pos(g, [xi1], [eta], [zeta]))
        assert np.all(J[1] == 0.0) and np.all(J[2] == 0.0)
        coef = Q * w[0] / (dt * g.dy * g.dz)
        ref = np.zeros((g.nz, g.ny, g.nx))
        for i in range(-4, g.nx + 4):
            lo, hi = min(xi0, xi1), max(xi0, xi1)
            cuts = [lo] + [c for c in i + np.arange(-2, 3.01, 0.5) if lo < c < hi] + [hi]
            val = 0.0
            for a, b in zip(cuts[:-1], cuts[1:]):
                t = 0.5 * (b - a) * gx + 0.5 * (b + a)
                val += 0.5 * (b - a) * np.dot(gw, _S_prev(n, t - i - 0.5))
            val *= np.sign(xi1 - xi0)
            for j in range(g.ny):
                for k in range(g.nz):
                    ref[k, j, i % g.nx] += coef * val * ora.shape(n, eta - j) * ora.shape(n, zeta - k)
        np.testing.assert_allclose(J[0], ref, rtol=0, atol=4e-15 * abs(coef))


@pytest.mark.parametrize("n", ORDERS)
def test_zero_move_and_reversal(ora, n):
    g = _grid(ora); rng = np.random.default_rng(51)
    c0, c1 = _moves(g, rng, 30)
    p0, p1 = _pos(g, *c0), _pos(g, *c1)
    w = rng.random(30) + 0.5; dt = 1e-16
    J0 = _J(ora, g, n, Q, dt, w, p0, p0)
    assert all(np.all(a == 0.0) for a in J0)                          # x1 = x0 -> J == 0 exactly
    Jf = _J(ora, g, n, Q, dt, w, p0, p1)
    Jb = _J(ora, g, n, Q, dt, w, p1, p0)                               # unwrapped start is fine
    for a, b in zip(Jf, Jb):
        assert np.abs(a + b).max() <= 2e-14 * np.abs(a).max()


# ---- brute force: own shapes, oversized window, difference equation from 0 --
def _S_np(n, r):
    a = abs(r)
    if n == 1:
        return max(0.0, 1.0 - a)
    if n == 2:
        return 0.75 - a * a if a <= 0.5 else (0.5 * (1.5 - a) ** 2 if a <= 1.5 else 0.0)
    return (2 / 3 - a * a + a ** 3 / 2) if a <= 1 else ((2 - a) ** 3 / 6 if a <= 2 else 0.0)


def _brute(g, n, q, dt, w, c0, c1):
    """For each particle: W on a 12^3 window straight from Esirkepov's
    definition, then J[i+1/2] = J[i-1/2] - coef*W[i] marching from zero."""
    N = (g.nx, g.ny, g.nz); h = (g.dx, g.dy, g.dz)
    J = [np.zeros((g.nz, g.ny, g.nx)) for _ in range(3)]
    M = 12
    for p in range(len(w)):
        base = [int(np.floor(c0[d][p])) - 5 for d in range(3)]
        S0 = [[_S_np(n, c0[d][p] - (base[d] + m)) for m in range(M)] for d in range(3)]
        S1 = [[_S_np(n, c1[d][p] - (base[d] + m)) for m in range(M)] for d in range(3)]
        for a in range(3):
            b, c = (a + 1) % 3, (a + 2) % 3
            coef = q * w[p] * h[a] / (dt * h[0] * h[1] * h[2])
            for mb in range(M):
                for mc in range(M):
                    cur = 0.0
                    for ma in range(M):
                        DSa = S1[a][ma] - S0[a][ma]; DSb = S1[b][mb] - S0[b][mb]; DSc = S1[c][mc] - S0[c][mc]
                        W = DSa * (S0[b][mb] * S0[c][mc] + DSb * S0[c][mc] / 2 + S0[b][mb] * DSc / 2
                                   + DSb * DSc / 3)
                        cur = cur - coef * W
                        idx = [0, 0, 0]
                        idx[a] = (base[a] + ma) % N[a]; idx[b] = (base[b] + mb) % N[b]; idx[c] = (base[c] + mc) % N[c]
                        J[a][idx[2], idx[1], idx[0]] += cur
    return J


@pytest.mark.parametrize("n", ORDERS)
@pytest.mark.parametrize("npart", (1, 2, 3))
def test_brute_force_small_inputs(ora, n, npart):
    g = _grid(ora); rng = np.random.default_rng(60 + 10 * n + npart)
    c0, c1 = _moves(g, rng, npart)
    if npart == 3:                                  # force one particle across the seam and one cell change
        c0[0][0], c1[0][0] = g.nx - 0.2, g.nx + 0.6
        c0[1][1], c1[1][1] = 0.3, -0.4
    w = rng.random(npart) + 0.5; dt = 1e-16
    J = _J(ora, g, n, Q, dt, w, _pos(g, *c0), _pos(g, *c1))
    # the brute force works in cell units: feed it the xi the oracle itself forms
    xi0 = [(p - o) * (1.0 / hh) for p, o, hh in zip(_pos(g, *c0), (g.xmin, g.ymin, g.zmin), (g.dx, g.dy, g.dz))]
    xi1 = [(p - o) * (1.0 / hh) for p, o, hh in zip(_pos(g, *c1), (g.xmin, g.ymin, g.zmin), (g.dx, g.dy, g.dz))]
    ref = _brute(g, n, Q, dt, w, xi0, xi1)
    for a, b in zip(J, ref):
        assert np.abs(a - b).max() <= 1e-13 * np.abs(b).max()


def test_move_of_one_cell_or_more_is_rejected(ora):
    g = _grid(ora)
    J = [np.zeros(g.nx * g.ny * g.nz) for _ in range(3)]
    with pytest.raises(RuntimeError):
        ora.deposit_esirkepov(g, 1, Q, 1e-16, np.ones(1), _pos(g, [2.0], [2.0], [2.0]),
                              _pos(g, [3.0], [2.0], [2.0]), J)
