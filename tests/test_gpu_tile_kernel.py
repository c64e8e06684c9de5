"""Edge cases of the fused per-tile kernel (phase A / slow path / phase B / flush) and parity at
BASELINE.json's full size in the launch configuration bench.py times, on sampled outputs the oracle
computes one by one plus whole-grid properties.  All tests need a B200: ``-m gpu``."""
import numpy as np
import pytest

from paper_2303_12873_b200 import workloads as W

from parity_util import TOL_FIELD_L2_10STEP, check_step_parity, field_l2_error, make_pair
from test_gpu_parity import _rand_fields

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def Sim():
    from paper_2303_12873_b200.binding import Sim as S
    return S


@pytest.mark.parametrize("order", [1, 2, 3])
def test_dense_cells_rows_longer_than_a_chunk(ora, Sim, order):
    """40 particles per cell: a row of 8 cells holds 320 particles = 5 staging chunks, every cell spans
    chunk boundaries, phase B accumulators persist across chunks; 0.2 c gives ~25 % cell crossers."""
    wl = W.uniform_plasma(10, 6, 5, ppc=40, u_th=0.2, order=order, seed=300 + order, dx=0.4e-6, dy=0.5e-6,
                          dz=0.3e-6)
    wl.fields = _rand_fields(wl, 17 + order)
    o, g = make_pair(ora, Sim, wl, sort_first=True, force_path=2)
    o.step(1)
    g.step(1)
    check_step_parity(o, g, wl, "dense order %d" % order)
    c = g.counters()
    assert c["fast"] > 0 and c["slow"] > 0 and c["fast"] + c["slow"] + c["global"] == wl.nparticles


def test_drift_between_sorts_uses_slow_and_global_paths(ora, Sim):
    """One sort, then 6 steps at 0.3 c without sorting: particles leave their listed cell (slow path) and
    some leave the tile's halo (global gather); the result must not depend on it (R39)."""
    wl = W.uniform_plasma(24, 9, 9, ppc=6, u_th=0.3, order=3, seed=77)
    wl.fields = _rand_fields(wl, 5, e_amp=1e8)
    o, g = make_pair(ora, Sim, wl, sort_first=True, force_path=2)
    o.step(1)
    g.step(1)
    check_step_parity(o, g, wl, "drift step 1")
    o.step(5)
    g.step(5)
    e = field_l2_error(o.get_fields(), g.get_fields())
    assert e <= TOL_FIELD_L2_10STEP, e
    c = g.counters()
    assert c["slow"] > 0.2 * wl.nparticles and c["global"] > 0
    assert c["fast"] + c["slow"] + c["global"] == 6 * wl.nparticles


def test_sort_every_step_ten_steps(ora, Sim):
    """The cadence bench.py times for configs[2]: pic_sort before every pic_step."""
    wl = W.config(2, parity=True, n=16)
    assert wl.sort_every == 1
    o, g = make_pair(ora, Sim, wl)
    for _ in range(10):
        g.sort()
        o.step(1)
        g.step(1)
    e = field_l2_error(o.get_fields(), g.get_fields())
    assert e <= TOL_FIELD_L2_10STEP, e
    c = g.counters()
    assert c["global"] == 0 and c["slow"] < 0.15 * 10 * wl.nparticles


def test_single_row_and_single_cell_grids(ora, Sim):
    """Grids thinner than a tile in y and z, and a 1-cell-wide x: every window wraps onto itself."""
    for dims in ((17, 1, 1), (1, 5, 3), (8, 4, 4)):
        wl = W.uniform_plasma(*dims, ppc=9, u_th=0.1, order=3, seed=sum(dims))
        wl.fields = _rand_fields(wl, 3, e_amp=1e8)
        o, g = make_pair(ora, Sim, wl, sort_first=True, force_path=2)
        o.step(2)
        g.step(2)
        e = field_l2_error(o.get_fields(), g.get_fields())
        assert e <= TOL_FIELD_L2_10STEP, (dims, e)


def test_full_size_config2_sampled_parity_and_continuity(ora, Sim):
    """BASELINE.json configs[2] at full size (256^3 cells, 134,217,728 electrons, order 3), sorted, one step
    with non-zero E and B: (a) 4,096 sampled particles against the oracle's gather + Boris + move + wrap,
    (b) J on a 12^3 block against the oracle's Esirkepov deposition of every particle that can reach it,
    (c) discrete continuity div J + (rho1 - rho0)/dt = 0 on the whole grid (R20), (d) path counters."""
    import torch
    wl = W.config(2)
    n, N = wl.nx, wl.nparticles
    sp = wl.species[0]
    rng = np.random.default_rng(99)
    # smooth random fields (a few Fourier modes per component) so the gather is non-trivial everywhere
    k, j, i = np.meshgrid(np.arange(n), np.arange(n), np.arange(n), indexing="ij")
    fields = {}
    for nm, amp in (("Ex", 3e9), ("Ey", 3e9), ("Ez", 3e9), ("Bx", 10.0), ("By", 10.0), ("Bz", 10.0)):
        m = rng.integers(1, 4, size=3)
        ph = rng.uniform(0, 2 * np.pi, size=3)
        fields[nm] = (amp * np.sin(2 * np.pi * m[0] * i / n + ph[0]) * np.sin(2 * np.pi * m[1] * j / n + ph[1])
                      * np.cos(2 * np.pi * m[2] * k / n + ph[2])).reshape(-1)
    del i, j, k
    g = Sim.from_workload(wl)
    g.set_fields(**fields)
    g.sort()
    rho0 = g.deposit_rho(device=True)
    g.step(1)
    rho1 = g.deposit_rho(device=True)
    J = g.get_fields(names=("Jx", "Jy", "Jz"), device=True)
    # (c) continuity on the whole grid, on the device (torch is plumbing here, not the product)
    Jx, Jy, Jz = (J[c].view(n, n, n) for c in ("Jx", "Jy", "Jz"))     # [k, j, i]
    div = ((Jx - torch.roll(Jx, 1, 2)) / wl.dx + (Jy - torch.roll(Jy, 1, 1)) / wl.dy
           + (Jz - torch.roll(Jz, 1, 0)) / wl.dz)
    res = div + (rho1 - rho0).view(n, n, n) / wl.dt
    bound = 1e-13 * float(rho0.abs().max()) / wl.dt
    assert float(res.abs().max()) <= bound, (float(res.abs().max()), bound)
    del div, res, rho1
    # (a) sampled particles
    pg = g.get_particles(0, device=True)
    inv = torch.empty(N, dtype=torch.int64, device=pg["id"].device)
    inv[pg["id"]] = torch.arange(N, device=inv.device)
    ids = rng.choice(N, size=4096, replace=False)
    pos = inv[torch.from_numpy(ids).to(inv.device)]
    og = ora.make_grid(n, n, n, wl.dx, wl.dy, wl.dz)
    E = (fields["Ex"], fields["Ey"], fields["Ez"]); B = (fields["Bx"], fields["By"], fields["Bz"])

    def oracle_push(sel):
        x, y, z = sp.x[sel].copy(), sp.y[sel].copy(), sp.z[sel].copy()
        ux, uy, uz = sp.ux[sel].copy(), sp.uy[sel].copy(), sp.uz[sel].copy()
        f = ora.gather(og, wl.order, x, y, z, E, B)
        ora.boris(sp.q, sp.m, wl.dt, ux, uy, uz, f[:3], f[3:])
        x1, y1, z1 = ora.move(wl.dt, x, y, z, ux, uy, uz)
        return (x, y, z), (x1, y1, z1), (ux, uy, uz)

    p0, p1, u1 = oracle_push(ids)
    xw, yw, zw = (a.copy() for a in p1)
    ora.wrap(og, xw, yw, zw)
    L = n * wl.dx
    for nm, ref in (("x", xw), ("y", yw), ("z", zw)):
        d = np.abs(pg[nm][pos].cpu().numpy() - ref)
        d = np.minimum(d, L - d)
        assert d.max() <= 1e-12 * L, (nm, d.max())
    du = np.sqrt(sum((pg[nm][pos].cpu().numpy() - ref) ** 2 for nm, ref in zip(("ux", "uy", "uz"), u1)))
    un = np.sqrt(sum(r ** 2 for r in u1))
    assert np.all(du <= 1e-12 * np.maximum(un, 0.05 * W.C_LIGHT)), du.max()
    # (b) J on a block: every particle whose old cell lies within 3 cells of the block can reach it
    b0, bw, mg = 100, 12, 3
    ci, cj, ck = (np.floor(a / wl.dx).astype(np.int32) for a in (sp.x, sp.y, sp.z))
    sel = np.nonzero((ci >= b0 - mg) & (ci < b0 + bw + mg) & (cj >= b0 - mg) & (cj < b0 + bw + mg)
                     & (ck >= b0 - mg) & (ck < b0 + bw + mg))[0]
    del ci, cj, ck
    q0, q1, _ = oracle_push(sel)
    Jo = [np.zeros(n * n * n) for _ in range(3)]
    ora.deposit_esirkepov(og, wl.order, sp.q, wl.dt, sp.w[sel], q0, q1, Jo)
    blk = (slice(b0, b0 + bw),) * 3
    jmax = max(float(J[c].abs().max()) for c in ("Jx", "Jy", "Jz"))
    for c, ref in zip(("Jx", "Jy", "Jz"), Jo):
        got = J[c].view(n, n, n)[blk].cpu().numpy()
        err = np.abs(got - ref.reshape(n, n, n)[blk]).max()
        assert err <= 1e-11 * jmax, (c, err, jmax)
    # (d) everything went through the fused kernel; only cell crossers took its slow path
    c = g.counters()
    assert c["global"] == 0 and c["fast"] + c["slow"] == N and c["slow"] < 0.12 * N


@pytest.mark.parametrize("order", [1, 2, 3])
@pytest.mark.parametrize("fresh", [0, 1])
def test_fresh_and_drift_variants_of_the_tile_kernel(ora, Sim, order, fresh):
    """Right after pic_sort the tile kernel runs its small-stencil, two-blocks-per-SM variant (option
    tile_fresh = 1, the default); tile_fresh = 0 forces the drift-tolerant variant.  Same arithmetic per
    particle, so both meet the 1-step bounds; grid sizes ragged against the 8 x 4 x 4 tile, 0.15 c so that
    every face of a tile is crossed, random fields on all six staggerings."""
    wl = W.uniform_plasma(19, 10, 7, ppc=9, u_th=0.15, order=order, seed=500 + order, dx=0.4e-6, dy=0.5e-6,
                          dz=0.3e-6)
    wl.fields = _rand_fields(wl, 23 + order)
    o, g = make_pair(ora, Sim, wl, sort_first=True, force_path=2)
    g.set_option("tile_fresh", fresh)
    o.step(1)
    g.step(1)
    check_step_parity(o, g, wl, "fresh=%d order %d" % (fresh, order))
    c = g.counters()
    assert c["global"] == 0 and c["fast"] + c["slow"] == wl.nparticles
    g.sort()
    o.step(1)
    g.step(1)
    check_step_parity(o, g, wl, "fresh=%d order %d step 2" % (fresh, order))


def test_full_size_config1_drift_step_continuity_and_gauss(ora, Sim):
    """BASELINE.json configs[1] at full size (128^3 cells, 16.8 M electrons + 16.8 M protons, order 3, sort every
    4 steps): properties that hold at any size, on the launch sequence bench.py --config 1 times.  Step 1 runs
    the fresh-sort variant through the deferred permutation, steps 2-4 the drift-tolerant variant in place.
    (a) discrete continuity of the total current on the whole grid for step 4 (R20), (b) Gauss's law residual
    div E - rho/eps0 unchanged from t = 0 (R19; it is zero here: electrons and protons start co-located),
    (c) every particle took the fused kernel, and only drifted / multi-face crossers its slow path."""
    import torch
    eps0 = 8.8541878128e-12
    wl = W.config(1)
    n = wl.nx
    g = Sim.from_workload(wl)
    g.sort()
    g.step(3)
    rho3 = g.deposit_rho(-1, device=True)
    g.step(1)
    rho4 = g.deposit_rho(-1, device=True)
    F = g.get_fields(names=("Ex", "Ey", "Ez", "Jx", "Jy", "Jz"), device=True)

    def div_back(a, b, c):
        a, b, c = (t.view(n, n, n) for t in (a, b, c))
        return ((a - torch.roll(a, 1, 2)) / wl.dx + (b - torch.roll(b, 1, 1)) / wl.dy + (c - torch.roll(c, 1, 0)) / wl.dz)

    # scale of one species' charge density (the total cancels to roundoff at t = 0)
    sp = wl.species[0]
    rho_scale = abs(sp.q) * float(sp.w[0]) * 8 / (wl.dx * wl.dy * wl.dz)
    res = div_back(F["Jx"], F["Jy"], F["Jz"]) + (rho4 - rho3).view(n, n, n) / wl.dt
    assert float(res.abs().max()) <= 1e-12 * rho_scale / wl.dt, float(res.abs().max())
    gauss = div_back(F["Ex"], F["Ey"], F["Ez"]) - rho4.view(n, n, n) / eps0
    assert float(gauss.abs().max()) <= 1e-10 * rho_scale / eps0, float(gauss.abs().max())
    c = g.counters()
    N = wl.nparticles
    assert c["global"] == 0 and c["fast"] + c["slow"] == 4 * N and c["slow"] < 0.05 * 4 * N
    assert c["sorts"] == 1 and c["steps"] == 4


@pytest.mark.parametrize("cfg", [3, 4])
def test_full_size_laser_configs_continuity_and_gauss(ora, Sim, cfg):
    """BASELINE.json configs[3] (laser-wakefield box, 128 x 128 x 1024, 13 M electrons behind a density ramp)
    and configs[4] (plasma mirror, 256 x 256 x 512, 101 M electrons at 16 ppc + 25 M protons at 4 ppc in a slab:
    empty tiles next to rows several chunks long) at full size, laser pulse in E and B: sort, two steps (the
    fresh-sort variant, then the drift variant), and the properties that hold at any size: continuity of the
    total current for step 2 on the whole grid (R20) and a Gauss residual div E - rho/eps0 that stays what it
    was at t = 0 (R19)."""
    import torch
    eps0 = 8.8541878128e-12
    wl = W.config(cfg)
    nx, ny, nz = wl.nx, wl.ny, wl.nz
    g = Sim.from_workload(wl)

    def div_back(a, b, c):
        a, b, c = (t.view(nz, ny, nx) for t in (a, b, c))
        return ((a - torch.roll(a, 1, 2)) / wl.dx + (b - torch.roll(b, 1, 1)) / wl.dy + (c - torch.roll(c, 1, 0)) / wl.dz)

    def gauss_residual():
        F = g.get_fields(names=("Ex", "Ey", "Ez"), device=True)
        return div_back(F["Ex"], F["Ey"], F["Ez"]) - g.deposit_rho(-1, device=True).view(nz, ny, nx) / eps0

    g0 = gauss_residual()
    g.sort()
    g.step(1)
    rho1 = g.deposit_rho(-1, device=True)
    g.step(1)
    rho2 = g.deposit_rho(-1, device=True)
    J = g.get_fields(names=("Jx", "Jy", "Jz"), device=True)
    rho_scale = float(rho1.abs().max())
    assert rho_scale > 0
    res = div_back(J["Jx"], J["Jy"], J["Jz"]) + (rho2 - rho1).view(nz, ny, nx) / wl.dt
    assert float(res.abs().max()) <= 1e-12 * rho_scale / wl.dt, float(res.abs().max())
    del res, J, rho1
    drift = gauss_residual() - g0
    assert float(drift.abs().max()) <= 1e-10 * rho_scale / eps0, float(drift.abs().max())
    c = g.counters()
    N = wl.nparticles
    assert c["global"] == 0 and c["fast"] + c["slow"] == 2 * N
