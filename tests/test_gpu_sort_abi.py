"""GPU tests of the sort (integer work: bit-exact), of the invariants measured
on the GPU result itself (continuity, Gauss), of the rho diagnostic, and of the
error behaviour include/pic.h states.  ``-m gpu``."""
import numpy as np
import pytest

from paper_2303_12873_b200 import workloads as W

from parity_util import by_id, make_pair

pytestmark = pytest.mark.gpu

EPS0 = 8.8541878128e-12


@pytest.fixture(scope="module")
def B():
    from paper_2303_12873_b200 import binding
    return binding


def test_sort_is_a_cell_ordered_permutation_and_offsets_match_oracle(ora, B):
    wl = W.uniform_plasma(9, 7, 5, ppc=11, u_th=0.1, order=3, seed=31, shuffle=True)
    o, g = make_pair(ora, B.Sim, wl)
    before = g.get_particles(0)
    g.sort()
    after = g.get_particles(0)
    # keys non-decreasing (keys computed by the oracle from the GPU's output positions)
    key = ora.cell_keys(o.g, after["x"], after["y"], after["z"])
    assert (np.diff(key) >= 0).all()
    # id multiset unchanged, and every attribute travelled with its id (bit-exact: payload is only moved)
    a, b = by_id(after), by_id(before)
    for k in ("x", "y", "z", "ux", "uy", "uz", "w"):
        assert np.array_equal(a[k], b[k]), k
    # cell offsets = exclusive prefix of the brute-force histogram = the oracle's
    o.sort()
    off = g.get_cell_offsets(0)
    assert np.array_equal(off.astype(np.int64), o.cell_offset[0])
    assert np.array_equal(off.astype(np.int64),
                          np.concatenate([[0], np.cumsum(np.bincount(key, minlength=wl.ncell))]))
    # sorting twice changes nothing but (possibly) the order inside a cell
    g.sort()
    again = g.get_particles(0)
    assert np.array_equal(ora.cell_keys(o.g, again["x"], again["y"], again["z"]), key)
    assert g.counters()["sorts"] == 2


def test_sort_large_spans_many_scan_chunks(ora, B):
    wl = W.uniform_plasma(40, 40, 40, ppc=4, u_th=0.05, order=1, seed=37, shuffle=True)   # 64,000 cells > 31 chunks
    o, g = make_pair(ora, B.Sim, wl)
    g.sort()
    p = g.get_particles(0)
    key = ora.cell_keys(o.g, p["x"], p["y"], p["z"])
    assert (np.diff(key) >= 0).all()
    assert np.array_equal(np.sort(p["id"]), np.arange(wl.nparticles, dtype=np.uint64))
    off = g.get_cell_offsets(0).astype(np.int64)
    assert np.array_equal(off, np.concatenate([[0], np.cumsum(np.bincount(key, minlength=wl.ncell))]))


def _div_back(F, wl):
    """Backward-difference divergence at nodes of a staggered vector field (periodic)."""
    sh = (wl.nz, wl.ny, wl.nx)
    fx, fy, fz = (F[0].reshape(sh), F[1].reshape(sh), F[2].reshape(sh))
    return ((fx - np.roll(fx, 1, 2)) / wl.dx + (fy - np.roll(fy, 1, 1)) / wl.dy + (fz - np.roll(fz, 1, 0)) / wl.dz)


@pytest.mark.parametrize("order", [1, 2, 3])
def test_gpu_continuity_and_rho_parity(ora, B, order):
    """(rho^{n+1} - rho^n)/dt + div J = 0 to roundoff on the GPU's own arrays (R20), every order, both paths."""
    wl = W.uniform_plasma(10, 9, 8, ppc=6, u_th=0.4, order=order, seed=41 + order, dx=0.5e-6, dy=0.4e-6, dz=0.6e-6)
    for path in (1, 2):
        o, g = make_pair(ora, B.Sim, wl, sort_first=(path == 2), force_path=path)
        rho0 = g.deposit_rho(0)
        assert np.abs(rho0 - o.deposit_rho(0)).max() <= 1e-12 * np.abs(rho0).max()
        g.step(1)
        rho1 = g.deposit_rho(0)
        f = g.get_fields(("Jx", "Jy", "Jz"))
        res = (rho1 - rho0).reshape(wl.nz, wl.ny, wl.nx) / wl.dt + _div_back((f["Jx"], f["Jy"], f["Jz"]), wl)
        assert np.abs(res).max() <= 1e-13 * np.abs(rho1).max() / wl.dt, (order, path)


def test_gpu_gauss_law_constant_over_100_steps(ora, B):
    """G = div E - rho/eps0 stays constant in time (R19) -- couples push, wrap, deposit, E update, sort."""
    wl = W.uniform_plasma(8, 8, 8, ppc=8, u_th=0.05, order=3, seed=43, protons=True)
    _, g = make_pair(ora, B.Sim, wl, sort_first=True)

    def gauss():
        f = g.get_fields(("Ex", "Ey", "Ez"))
        return _div_back((f["Ex"], f["Ey"], f["Ez"]), wl) - g.deposit_rho(-1).reshape(wl.nz, wl.ny, wl.nx) / EPS0

    rho_e = np.abs(g.deposit_rho(0)).max()
    G0 = gauss()
    assert np.abs(G0).max() <= 1e-12 * rho_e / EPS0          # co-located pairs: G = 0 at t = 0
    for it in range(100):
        if it % 4 == 0:
            g.sort()
        g.step(1)
    assert np.abs(gauss() - G0).max() <= 1e-11 * rho_e / EPS0


def test_roundtrip_fields_and_particles_bit_exact(B):
    wl = W.uniform_plasma(7, 6, 5, ppc=3, u_th=0.1, order=2, seed=47)
    rng = np.random.default_rng(1)
    wl.fields = {n: rng.standard_normal(wl.ncell) for n in ("Ex", "Ey", "Ez", "Bx", "By", "Bz")}
    g = B.Sim.from_workload(wl)
    f = g.get_fields()
    for n, a in wl.fields.items():
        assert np.array_equal(f[n], a), n
    assert not f["Jx"].any() and not f["Jy"].any() and not f["Jz"].any()
    p = g.get_particles(0)
    for k, a in zip(("x", "y", "z", "ux", "uy", "uz", "w"), wl.species[0].arrays()):
        assert np.array_equal(p[k], a), k
    assert np.array_equal(p["id"], np.arange(wl.nparticles, dtype=np.uint64))
    # device-resident round trip
    fd = g.get_fields(device=True)
    for n, a in wl.fields.items():
        assert np.array_equal(fd[n].cpu().numpy(), a), n
    pd = g.get_particles(0, device=True)
    assert np.array_equal(pd["uz"].cpu().numpy(), wl.species[0].uz)


def test_error_codes(B):
    d = 0.5e-6
    dt = W.courant_dt(d, d, d)
    with pytest.raises(B.PicError) as e:                       # dt above the Courant limit
        B.Sim(4, 4, 4, d, d, d, 0, 0, 0, dt * 1.02, 1, [8])
    assert e.value.code == B.PIC_EINVAL
    with pytest.raises(B.PicError) as e:                       # order 4
        B.Sim(4, 4, 4, d, d, d, 0, 0, 0, dt, 4, [8])
    assert e.value.code == B.PIC_EINVAL
    g = B.Sim(4, 4, 4, d, d, d, 0, 0, 0, dt, 1, [8])
    with pytest.raises(B.PicError) as e:                       # step before load
        g.step(1)
    assert e.value.code == B.PIC_ESTATE
    with pytest.raises(B.PicError) as e:                       # sort before load
        g.sort()
    assert e.value.code == B.PIC_ESTATE
    one = np.array([1e-6]); zero = np.zeros(1)
    with pytest.raises(B.PicError) as e:                       # outside the box (x = L exactly)
        g.load_particles(0, -W.Q_E, W.M_E, np.array([4 * d]), one, one, zero, zero, zero, np.ones(1))
    assert e.value.code == B.PIC_EINVAL and "outside" in str(e.value)
    with pytest.raises(B.PicError) as e:                       # NaN
        g.load_particles(0, -W.Q_E, W.M_E, np.array([np.nan]), one, one, zero, zero, zero, np.ones(1))
    assert e.value.code == B.PIC_EINVAL
    with pytest.raises(B.PicError) as e:                       # more than np_max
        z9 = np.full(9, 1e-6)
        g.load_particles(0, -W.Q_E, W.M_E, z9, z9, z9, z9 * 0, z9 * 0, z9 * 0, z9)
    assert e.value.code == B.PIC_ENOMEM
    with pytest.raises(B.PicError) as e:
        g.load_particles(3, -W.Q_E, W.M_E, one, one, one, zero, zero, zero, np.ones(1))
    assert e.value.code == B.PIC_EINVAL
    with pytest.raises(B.PicError) as e:
        g.set_option("no_such_option", 1)
    assert e.value.code == B.PIC_EINVAL
    g.load_particles(0, -W.Q_E, W.M_E, one, one, one, zero, zero, zero, np.ones(1))
    with pytest.raises(B.PicError) as e:                       # fused path forced without a sort
        g.set_option("force_path", 2)
        g.step(1)
    assert e.value.code == B.PIC_ESTATE
    g.set_option("force_path", 0)
    g.step(1)
    g.sync()
    assert g.counters()["steps"] == 1
    # an infinite field makes the new position non-finite during the step -> PIC_EPHYS at the next sync
    g.set_fields(Ex=np.full(64, np.inf))
    g.step(1)
    with pytest.raises(B.PicError) as e:
        g.sync()
    assert e.value.code == B.PIC_EPHYS


@pytest.mark.parametrize("fuse", [0, 1])
@pytest.mark.parametrize("deferred", [0, 1])
def test_deferred_and_immediate_sort_give_the_same_state(ora, B, deferred, fuse):
    """sort_deferred = 1 (default): pic_sort writes only the permutation and the next fused per-tile kernel (or
    pic_get_particles, or the global-atomic kernel) moves the data; 0: pic_sort moves it.  Every reader must
    see the sorted container either way: sort -> get, sort -> step -> get, sort -> sort -> step, sort ->
    rho -> step on the global path, and the physics stays within the 1-step bounds of the oracle."""
    from parity_util import check_step_parity
    wl = W.uniform_plasma(13, 9, 6, ppc=7, u_th=0.2, order=3, seed=71, shuffle=True, protons=True)
    o, g = make_pair(ora, B.Sim, wl)
    g.set_option("sort_deferred", deferred)
    g.set_option("fuse_keys", fuse)      # 1: the per-tile kernel writes the keys the next pic_sort uses
    before = [g.get_particles(s) for s in range(2)]
    g.sort()
    rho = g.deposit_rho(0)                        # reads the (possibly not yet moved) container: order-free
    assert np.abs(rho - o.deposit_rho(0)).max() <= 1e-12 * np.abs(rho).max()
    g.sort()                                       # supersedes a pending permutation
    for s in range(2):
        after = g.get_particles(s)                 # forces the move
        key = ora.cell_keys(o.g, after["x"], after["y"], after["z"])
        assert (np.diff(key) >= 0).all()
        a, b = by_id(after), by_id(before[s])
        for k in ("x", "y", "z", "ux", "uy", "uz", "w"):
            assert np.array_equal(a[k], b[k]), k
    g.sort()
    o.step(1); g.step(1)                           # tile kernel consumes the permutation
    check_step_parity(o, g, wl, "deferred=%d step 1" % deferred)
    for s in range(2):                             # outputs were written in sorted order of the OLD positions
        off = g.get_cell_offsets(s).astype(np.int64)
        assert off[-1] == wl.species[s].n
    g.sort()
    g.set_option("force_path", 1)                  # global-atomic kernel: materialises the pending permutation
    o.step(1); g.step(1)
    check_step_parity(o, g, wl, "deferred=%d step 2 (global path)" % deferred)
    g.set_option("force_path", 0)
    g.sort()
    o.step(2); g.step(2)                           # one permuted step, one in-place (drift variant) step
    check_step_parity(o, g, wl, "deferred=%d steps 3-4" % deferred)
    g.sort()                                       # keys written by the last step (fuse = 1) or recomputed
    o.sort()
    for s in range(2):
        after = g.get_particles(s)
        key = ora.cell_keys(o.g, after["x"], after["y"], after["z"])
        assert (np.diff(key) >= 0).all()
        assert np.array_equal(g.get_cell_offsets(s).astype(np.int64), o.cell_offset[s])


def test_drift_watch_moves_a_stale_species_to_the_global_kernel(ora, B):
    """ADVICE r1 / include/pic.h "drift_watch": a species sorted once and then stepped at 0.3 c leaves its
    listed cells; once more than 20 % of a launch left the fast deposit path the next steps run the
    global-atomic kernel (counter [7]) until the next pic_sort.  The values do not depend on the path."""
    from parity_util import TOL_FIELD_L2_10STEP, field_l2_error
    wl = W.uniform_plasma(16, 12, 12, ppc=6, u_th=0.3, order=3, seed=91)
    o, g = make_pair(ora, B.Sim, wl)
    g.sort()
    for _ in range(8):
        g.step(1)
        g.sync()                     # lets the asynchronous counter snapshot of this step arrive
    o.step(8)
    c = g.counters()
    assert c["fallbacks"] >= 1 and c["global"] == c["fallbacks"] * wl.nparticles, c
    assert c["fast"] + c["slow"] + c["global"] == 8 * wl.nparticles
    assert field_l2_error(o.get_fields(), g.get_fields()) <= TOL_FIELD_L2_10STEP
    g.sort()                         # sorted again: back on the fused kernel
    g.step(1)
    c2 = g.counters()
    assert c2["fallbacks"] == c["fallbacks"] and c2["global"] == c["global"]
    # with the watch off a sorted species stays on the fused kernel whatever its drift
    g2 = B.Sim.from_workload(wl)
    g2.set_option("drift_watch", 0)
    g2.sort()
    for _ in range(6):
        g2.step(1)
        g2.sync()
    assert g2.counters()["fallbacks"] == 0 and g2.counters()["global"] < 0.2 * 6 * wl.nparticles


def test_counters_report_the_yee_path_and_init_rejects_oversized_y(B):
    d = 0.5e-6
    g = B.Sim(8, 8, 8, d, d, d, 0, 0, 0, W.courant_dt(d, d, d), 1, [8])
    assert g.counters()["yee_tma"] == 1, g.last_error()     # a B200 with a current driver builds the tensor maps
    with pytest.raises(B.PicError) as e:                     # gridDim.y = ny + 2 NG must fit 65535
        B.query_arena(4, 65530, 4, 1, [8])
    assert e.value.code == B.PIC_EINVAL


def test_machine_rate_probes_return_sane_numbers():
    """pic_probe_* (SURVEY 8(d) "Builder must measure first"): DFMA issues at about 0.5 clk per warp
    instruction per SM; a conflict-free full-warp LDS.64 returns 256 B = 2 clk; REDs make progress."""
    from paper_2303_12873_b200 import peaks
    clk = peaks.probe_dfma(16, iters=2000)
    assert 0.45 <= clk <= 0.7, clk
    words = [64 + l for l in range(32)]
    clk = peaks.probe_lds(8, words, 0xFFFFFFFF, 16, iters=2000)
    assert 1.8 <= clk <= 2.6, clk
    assert peaks.probe_red(0, 5 << 20, n=16) > 1e9


def test_selfcheck_module_passes():
    from paper_2303_12873_b200 import selfcheck
    selfcheck.run_case(12, 3, "drift", verbose=False)
    selfcheck.run_case(12, 1, "global", verbose=False)


def test_auto_sort_keeps_the_fast_path_without_the_caller_sorting(ora):
    """Option "auto_sort" = 1: pic_step sorts by itself before every step, so a caller that never calls pic_sort still
    runs the fused per-tile kernel; the physics is the oracle's (which never sorts) within the step tolerances."""
    from paper_2303_12873_b200 import workloads as W
    from paper_2303_12873_b200.binding import Sim
    import parity_util as P
    wl = W.uniform_plasma(16, 8, 24, ppc=6, u_th=0.05, order=3, seed=11, protons=True, shuffle=True)
    o, g = P.make_pair(ora, Sim, wl)
    g.set_option("auto_sort", 1)
    o.step(1); g.step(1)
    P.check_step_parity(o, g, wl, "auto_sort step 1")
    o.step(3); g.step(3)
    assert P.field_l2_error(o.get_fields(), g.get_fields()) <= P.TOL_FIELD_L2_10STEP
    c = g.counters()
    assert c["sorts"] == 4 and c["steps"] == 4
    assert c["global"] == 0 and c["fast"] > 0.9 * 4 * wl.nparticles      # every launch was the fused kernel
    off = g.get_cell_offsets(0)
    assert off[-1] == wl.species[0].n and np.all(np.diff(off.astype(np.int64)) >= 0)
    # k = 3: sorts before steps 1 and 4 only
    o2, g2 = P.make_pair(ora, Sim, wl)
    g2.set_option("auto_sort", 3)
    g2.step(4)
    assert g2.counters()["sorts"] == 2
    with pytest.raises(Exception):
        g2.set_option("auto_sort", -1)
