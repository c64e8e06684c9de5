"""NEXT-2: open ends along z (zero exterior, particles deleted), the moving window and
the plane current source of a laser antenna, CUDA path against the oracle's ``open_z`` mode on the same seeded inputs;
BASELINE.json:north_star tolerances (1 step: 1e-12 / 1e-11; many steps: field L2 1e-9)."""
import numpy as np
import pytest

from paper_2303_12873_b200 import workloads as W

from parity_util import TOL_FIELD_1STEP, TOL_FIELD_L2_10STEP, TOL_PARTICLE_1STEP, field_l2_error, group_maxabs_errors

pytestmark = pytest.mark.gpu

C_LIGHT = 299792458.0


@pytest.fixture(scope="module")
def Sim():
    from paper_2303_12873_b200.binding import Sim as S
    return S


def _match_particles(po, pg, Lxy, u_ref, tol):
    """Same survivors (by id) and the same state, x and y compared as periodic distances."""
    io, ig = np.argsort(po["id"]), np.argsort(pg["id"])
    assert np.array_equal(po["id"][io], pg["id"][ig]), "different particles survived"
    for nm, L in (("x", Lxy[0]), ("y", Lxy[1]), ("z", None)):
        d = np.abs(po[nm][io] - pg[nm][ig])
        if L is not None:
            d = np.minimum(d, np.abs(L - d))
        assert d.max(initial=0.0) <= tol * (L if L is not None else Lxy[2]), (nm, d.max())
    du = np.sqrt(sum((po[k][io] - pg[k][ig]) ** 2 for k in ("ux", "uy", "uz")))
    un = np.sqrt(sum(po[k][io] ** 2 for k in ("ux", "uy", "uz")))
    assert np.all(du <= tol * np.maximum(un, u_ref)), du.max(initial=0.0)
    assert np.array_equal(po["w"][io], pg["w"][ig])


def _rand_fields(ncell, seed, e_amp=3e8):
    rng = np.random.default_rng(seed)
    f = {n: e_amp * rng.standard_normal(ncell) for n in ("Ex", "Ey", "Ez")}
    f.update({n: (e_amp / C_LIGHT) * rng.standard_normal(ncell) for n in ("Bx", "By", "Bz")})
    return f


@pytest.mark.parametrize("order", [1, 2, 3])
def test_open_ends_along_z_match_the_oracle(ora, Sim, order):
    """Hot electrons and protons, random E and B right up to the faces; particles do leave and are deleted on both sides."""
    wl = W.uniform_plasma(9, 8, 20, ppc=4, u_th=0.3, order=order, seed=700 + order, protons=True, dz=0.3e-6)
    wl.fields = _rand_fields(wl.ncell, 71)
    o = ora.OracleSim(*wl.grid_args(), wl.dt, wl.order, 2, open_z=True)
    g = Sim.from_workload(wl)
    g.set_option("absorb_mask", 4)
    g.set_fields(**wl.fields)                     # (re)loads the fields: the z guards are zero now
    o.set_fields(**wl.fields)
    for s, sp in enumerate(wl.species):
        o.load_particles(s, sp.q, sp.m, *sp.arrays())
    L = (wl.nx * wl.dx, wl.ny * wl.dy, wl.nz * wl.dz)
    g.sort()
    o.step(1); g.step(1)
    for grp, e in group_maxabs_errors(o.get_fields(), g.get_fields()).items():
        assert e <= TOL_FIELD_1STEP, (grp, e)
    for s in range(2):
        _match_particles(o.get_particles(s), g.get_particles(s), L, 0.3 * C_LIGHT if s == 0 else 1e-3 * C_LIGHT, TOL_PARTICLE_1STEP)
    for it in range(1, 10):
        g.sort()
        o.step(1); g.step(1)
    assert field_l2_error(o.get_fields(), g.get_fields()) <= TOL_FIELD_L2_10STEP
    n_left = o.get_particles(0)["x"].size
    assert n_left < wl.species[0].n, "nobody left through the open ends: the test does not test them"
    for s in range(2):
        _match_particles(o.get_particles(s), g.get_particles(s), L, 0.3 * C_LIGHT if s == 0 else 1e-3 * C_LIGHT, 1e-9)
    g.close()


def test_moving_window_with_antenna_and_fresh_plasma(ora, Sim):
    """A wakefield-shaped run in miniature (config 3's geometry: dx = dy = 4 dz, 2 ppc cold electrons behind a vacuum gap):
    an antenna plane radiates a few-cycle pulse, the window follows it at c (one cell whenever c t passes a cell), plasma
    enters through the top plane.  Fields, deleted counts and the surviving particles must match the oracle after 36
    steps; the CUDA side sorts every step."""
    nx, ny, nz, order = 8, 8, 48, 3
    dz = 25e-9; dx = 4 * dz
    dt = 0.99 * W.courant_dt(dx, dx, dz)
    rng = np.random.default_rng(77)
    ppc, n0 = 2, 5e24
    wgt = n0 * dx * dx * dz / ppc

    def plasma_planes(k0, k1, zmin):
        """ppc cold electrons per cell in planes k0 .. k1-1 of the box whose lowest node is at zmin."""
        n = (k1 - k0) * ny * nx * ppc
        k, j, i, _ = np.meshgrid(np.arange(k0, k1), np.arange(ny), np.arange(nx), np.arange(ppc), indexing="ij")
        x = (i.reshape(-1) + rng.random(n)) * dx; y = (j.reshape(-1) + rng.random(n)) * dx
        z = zmin + (k.reshape(-1) + rng.random(n)) * dz
        z = np.minimum(z, np.nextafter(zmin + k1 * dz, 0.0))          # keep the rounding of zmin + ... inside the box
        zero = np.zeros(n)
        return x, y, z, zero, zero.copy(), zero.copy(), np.full(n, wgt)

    first = plasma_planes(28, nz, 0.0)
    n_first = first[0].size
    o = ora.OracleSim(nx, ny, nz, dx, dx, dz, 0.0, 0.0, 0.0, dt, order, 1, open_z=True)
    g = Sim(nx, ny, nz, dx, dx, dz, 0.0, 0.0, 0.0, dt, order, [4 * n_first])
    g.set_option("absorb_mask", 4)
    o.load_particles(0, W.Q_E * -1.0, W.M_E, *first)
    g.load_particles(0, W.Q_E * -1.0, W.M_E, *first)
    next_id = n_first
    lam = 0.8e-6
    omega = 2 * np.pi * C_LIGHT / lam
    jj, ii = np.meshgrid(np.arange(ny), np.arange(nx), indexing="ij")
    profile = np.exp(-(((ii + 0.5) - nx / 2) ** 2 + (jj - ny / 2) ** 2) / 9.0)       # Jx sits at (i + 1/2, j)
    k_ant, shifted, deleted_o, deleted_g = 5, 0, 0, 0
    for it in range(36):
        g.sort()
        t_half = (it + 0.5) * dt
        amp = 4e19 * np.sin(omega * t_half) * np.sin(np.pi * min(t_half / (6 * lam / C_LIGHT), 1.0)) ** 2
        src = amp * profile
        ka = k_ant - shifted                        # the antenna stays where it is while the window moves on
        if ka >= 0 and it < 24:
            o.add_plane_source(0, ka, src)
        o.step(1)
        g.step_stage(0)
        if ka >= 0 and it < 24:
            g.add_plane("Jx", ka, np.ascontiguousarray(src))
        for st in (1, 2, 3):
            g.step_stage(st)
        if it == 0:
            for grp, e in group_maxabs_errors(o.get_fields(), g.get_fields()).items():
                assert e <= TOL_FIELD_1STEP, (grp, e)
        want = int(np.floor(C_LIGHT * (it + 1) * dt / dz))
        if want > shifted:
            n = want - shifted
            before = o.deleted
            o.shift_window(n)
            deleted_o += o.deleted - before
            deleted_g += g.shift_window(n)
            shifted = want
            fresh = plasma_planes(nz - n, nz, shifted * dz)
            ids = np.arange(next_id, next_id + fresh[0].size, dtype=np.uint64)
            next_id += fresh[0].size
            o.append_particles(0, *fresh, ids)
            g.append_particles(0, *fresh, ids)
    assert shifted >= 30 and deleted_o == deleted_g and deleted_o > 0
    fo, fg = o.get_fields(), g.get_fields()
    assert max(np.abs(fo[n]).max() for n in ("Ex", "By")) > 0 and np.abs(fo["Jz"]).max() > 0      # the pulse drives the plasma
    assert field_l2_error(fo, fg) <= TOL_FIELD_L2_10STEP
    po, pg = o.get_particles(0), g.get_particles(0)
    u_ref = max(1e-3 * C_LIGHT, float(np.sqrt(np.mean(po["ux"] ** 2 + po["uy"] ** 2 + po["uz"] ** 2))))
    _match_particles(po, pg, (nx * dx, ny * dx, nz * dz), u_ref, 1e-9)
    c = g.counters()
    assert c["steps"] == 36
    g.close()


def test_open_end_calls_reject_bad_arguments(Sim):
    from paper_2303_12873_b200.binding import PicError
    wl = W.uniform_plasma(8, 8, 8, ppc=1, u_th=0.0, order=1, seed=5)
    g = Sim.from_workload(wl)
    with pytest.raises(PicError):
        g.shift_window(1)                          # no open ends along z
    with pytest.raises(PicError):
        g.set_option("absorb_mask", 8)
    with pytest.raises(PicError):
        g.add_plane("Jx", 8, np.zeros(64))
    g.set_option("absorb_mask", 4)
    g.step(1)                                      # pic_step stays available: every open dimension is absorbing
    assert g.shift_window(0) == 0
    with pytest.raises(PicError):
        g.shift_window(9)
    g.close()
    wl2 = W.uniform_plasma(8, 8, 2, ppc=1, u_th=0.0, order=1, seed=5)
    g2 = Sim.from_workload(wl2)
    with pytest.raises(PicError):
        g2.set_option("absorb_mask", 4)            # fewer than NG cells along z
    g2.close()


def test_damping_layers_match_the_oracle_and_absorb(ora, Sim):
    """pic_set_damping against OracleSim.set_damping: random fields and hot plasma for 10 steps (1-step and 10-step
    tolerances), then a vacuum pulse sent into the upper layer: what comes back is the oracle's small remainder, not the
    full reflection of the bare open end.  Validation of the arguments too."""
    from paper_2303_12873_b200.binding import PicError
    wl = W.uniform_plasma(9, 7, 40, ppc=3, u_th=0.2, order=2, seed=731, dz=0.3e-6)
    wl.fields = _rand_fields(wl.ncell, 73)
    nd = 9
    prof = np.exp(-0.35 * ((nd - np.arange(nd)) / nd) ** 2)
    o = ora.OracleSim(*wl.grid_args(), wl.dt, wl.order, 1, open_z=True)
    g = Sim.from_workload(wl)
    with pytest.raises(PicError):
        g.set_damping(prof)                        # no open ends yet
    g.set_option("absorb_mask", 4)
    with pytest.raises(PicError):
        g.set_damping(np.ones(21))                 # 2 x 21 > nz
    with pytest.raises(PicError):
        g.set_damping(np.array([1.0, np.nan]))
    g.set_damping(prof)
    o.set_damping(prof)
    g.set_fields(**wl.fields); o.set_fields(**wl.fields)
    sp = wl.species[0]
    o.load_particles(0, sp.q, sp.m, *sp.arrays())
    g.sort()
    o.step(1); g.step(1)
    for grp, e in group_maxabs_errors(o.get_fields(), g.get_fields()).items():
        assert e <= TOL_FIELD_1STEP, (grp, e)
    o.step(9); g.step(9)
    assert field_l2_error(o.get_fields(), g.get_fields()) <= TOL_FIELD_L2_10STEP
    g.close()

    # vacuum pulse into the layer (no particles that matter: one cold particle at rest, weight 0)
    nx, ny, nz = 4, 4, 96
    wl = W.uniform_plasma(nx, ny, nz, ppc=1, u_th=0.0, order=1, seed=5, dx=1e-6, dy=1e-6, dz=0.25e-6)
    wl.species[0].w[:] = 0.0
    k, _, _ = np.meshgrid(np.arange(nz), np.arange(ny), np.arange(nx), indexing="ij")
    env = np.exp(-((k - 40.0) / 6.0) ** 2) * np.cos(2 * np.pi * (k - 40.0) / 12.0)
    envb = np.exp(-((k + 0.5 - 40.0) / 6.0) ** 2) * np.cos(2 * np.pi * (k + 0.5 - 40.0) / 12.0)
    zero = np.zeros(wl.ncell)
    f = {n: zero for n in ("Ex", "Ey", "Ez", "Bx", "By", "Bz")}
    f["Ex"] = (1e9 * env).reshape(-1); f["By"] = (1e9 / C_LIGHT * envb).reshape(-1)
    nd = 12
    prof = np.exp(-0.35 * ((nd - np.arange(nd)) / nd) ** 2)
    nsteps = int(2 * (nz - 40) * 0.25e-6 / (C_LIGHT * wl.dt)) + 10
    back = {}
    for name in ("bare", "layer"):
        g = Sim.from_workload(wl)
        g.set_option("absorb_mask", 4)
        g.set_fields(**f)
        if name == "layer":
            g.set_damping(prof)
        g.step(nsteps)
        out = g.get_fields()
        back[name] = sum(np.sum(out[n].reshape(nz, ny, nx)[:nz - nd - 4] ** 2) for n in ("Ex", "Ey", "Ez")) / np.sum(f["Ex"] ** 2)
        if name == "layer":
            o = ora.OracleSim(*wl.grid_args(), wl.dt, 1, 1, open_z=True)
            o.set_fields(**f); o.set_damping(prof)
            sp = wl.species[0]
            o.load_particles(0, sp.q, sp.m, *sp.arrays())
            o.step(nsteps)
            fo = o.get_fields()
            ref = max(np.abs(f["Ex"]).max(), 1.0)
            assert np.abs(fo["Ex"] - out["Ex"]).max() <= 1e-9 * ref
        g.set_damping([])                           # and the layers can be removed again
        g.close()
    assert back["bare"] > 0.4 and back["layer"] < 0.02 * back["bare"], back


def test_window_shift_deletes_more_than_a_third_of_the_container(Sim):
    """The index scratch behind the deletion holds np_max / 3 entries; a shift that drops more than that used to
    fail with PIC_ENOMEM after the fields and the box had already moved.  It now deletes in batches."""
    nx, ny, nz, d = 8, 8, 16, 0.5e-6
    rng = np.random.default_rng(77)
    n = 3001
    x, y, z = rng.random(n) * nx * d, rng.random(n) * ny * d, rng.random(n) * nz * d
    zero = np.zeros(n)
    g = Sim(nx, ny, nz, d, d, d, 0.0, 0.0, 0.0, W.courant_dt(d, d, d), 1, [n])      # np_max = n: batches of 1,000
    g.set_option("absorb_mask", 4)
    g.load_particles(0, -W.Q_E, W.M_E, x, y, z, zero, zero, zero, np.ones(n))
    survivors = np.nonzero(z >= 0.0 + 11 * d)[0]
    assert n - survivors.size > 2 * (n // 3)                        # needs three batches
    assert g.shift_window(11) == n - survivors.size
    p = g.get_particles(0)
    assert np.array_equal(np.sort(p["id"]), survivors.astype(np.uint64))
    order = np.argsort(p["id"])
    assert np.array_equal(p["z"][order], z[survivors]) and np.array_equal(p["x"][order], x[survivors])
    assert g.counters()["deleted"] == n - survivors.size
    # and the same through a step: everything flies out of the top face at once
    g2 = Sim(nx, ny, nz, d, d, d, 0.0, 0.0, 0.0, W.courant_dt(d, d, d), 1, [n])
    g2.set_option("absorb_mask", 4)
    ztop = (nz - 1e-3 * rng.random(n)) * d
    g2.load_particles(0, -W.Q_E, W.M_E, x, y, ztop, zero, zero, np.full(n, 5.0 * C_LIGHT), np.ones(n))
    g2.step(1)
    assert g2.num_particles(0) == 0 and g2.counters()["deleted"] == n


@pytest.mark.parametrize("absorb_first", [True, False])
def test_absorbing_face_stays_open_whatever_order_the_masks_are_set_in(Sim, absorb_first):
    """pic.h: absorb_mask implies the same bits of open_mask.  Setting open_mask afterwards (BrickStepper always does)
    used to drop them: particles were wrapped through a face whose guards are zeroed."""
    nx, ny, nz, d = 8, 8, 8, 0.5e-6
    g = Sim(nx, ny, nz, d, d, d, 0.0, 0.0, 0.0, W.courant_dt(d, d, d), 1, [4])
    if absorb_first:
        g.set_option("absorb_mask", 4)
        g.set_option("open_mask", 0)
    else:
        g.set_option("open_mask", 0)
        g.set_option("absorb_mask", 4)
    one = np.ones(1)
    # one particle a thousandth of a cell below the top z face, moving up at 0.98 c: it must leave, not wrap
    g.load_particles(0, -W.Q_E, W.M_E, 4.2 * d * one, 3.3 * d * one, (nz - 1e-3) * d * one, 0 * one, 0 * one,
                     5.0 * C_LIGHT * one, one)
    g.step(1)
    assert g.num_particles(0) == 0 and g.counters()["deleted"] == 1
