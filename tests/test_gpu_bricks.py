"""NEXT-1: a periodic box cut into bricks, every brick its own context
on the SAME GPU, exchanging E/B guard planes, J guard planes (summed) and migrating particles through the
C-ABI halo calls, must reproduce the single-domain ORACLE within the 1-step and 10-step tolerances
(BASELINE.json:north_star).  One GPU per gpurun: no scaling number is measured here."""
import numpy as np
import pytest

from paper_2303_12873_b200 import bricks as B
from paper_2303_12873_b200 import workloads as W

from parity_util import TOL_FIELD_L2_10STEP, check_step_parity, field_l2_error

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def Sim():
    from paper_2303_12873_b200.binding import Sim as S
    return S


class _Joined:
    """The bricks presented as one simulation (get_fields / get_particles of the whole box, ids = load index)."""

    def __init__(self, layout, sims, owners, wl):
        self.layout, self.sims, self.wl = layout, sims, wl
        self.inv = []
        for o in owners:                        # brick id -> index in the whole-box arrays
            gid = B.global_ids(layout, o)
            inv = np.empty(gid.size, dtype=np.int64)
            inv[gid] = np.arange(gid.size)
            self.inv.append(inv)

    def get_fields(self):
        parts = {r: s.get_fields() for r, s in self.sims.items()}
        return {n: self.layout.join_field({r: p[n] for r, p in parts.items()}) for n in parts[0]}

    def get_particles(self, s):
        ps = [sim.get_particles(s) for sim in self.sims.values()]
        out = {k: np.concatenate([p[k] for p in ps]) for k in ps[0]}
        out["id"] = self.inv[s][out["id"].astype(np.int64)].astype(np.uint64)
        assert out["x"].size == self.wl.species[s].n, "particles were lost or duplicated in migration"
        return out


def _rand_fields(wl, seed, e_amp=3e8):
    rng = np.random.default_rng(seed)
    f = {}
    for n in ("Ex", "Ey", "Ez"):
        f[n] = e_amp * rng.standard_normal(wl.ncell)
    for n in ("Bx", "By", "Bz"):
        f[n] = (e_amp / W.C_LIGHT) * rng.standard_normal(wl.ncell)
    return f


@pytest.mark.parametrize("procs,dims", [((2, 1, 1), (32, 16, 16)), ((1, 1, 2), (16, 8, 24)), ((2, 2, 1), (16, 16, 8)),
                                         ((2, 1, 3), (8, 8, 12))])
def test_bricks_on_one_gpu_match_the_single_domain_oracle(ora, Sim, procs, dims):
    wl = W.uniform_plasma(*dims, ppc=4, u_th=0.2, order=3, seed=500 + sum(procs), protons=True)
    wl.fields = _rand_fields(wl, 51)
    layout = B.BrickLayout(wl.nx, wl.ny, wl.nz, wl.dx, wl.dy, wl.dz, 0.0, 0.0, 0.0, procs)
    sims, owners = B.make_local_bricks(Sim, layout, wl)
    st = B.BrickStepper(layout, sims, B.LocalTransport(range(layout.size)), len(wl.species), leaver_capacity=1 << 15)
    st.start()
    for s in sims.values():
        s.sort()
    o = ora.OracleSim(*wl.grid_args(), wl.dt, wl.order, len(wl.species))
    o.set_fields(**wl.fields)
    for s, sp in enumerate(wl.species):
        o.load_particles(s, sp.q, sp.m, *sp.arrays())
    J = _Joined(layout, sims, owners, wl)
    o.step(1)
    st.step()
    check_step_parity(o, J, wl, "bricks %r step 1" % (procs,))
    moved = sum(s.counters()["steps"] for s in sims.values())
    assert moved == layout.size
    for it in range(9):
        o.step(1)
        st.step(sort=(it % 2 == 0))              # unsorted bricks take the global-atomic kernel: same values
    e = field_l2_error(o.get_fields(), J.get_fields())
    assert e <= TOL_FIELD_L2_10STEP, "bricks %r: 10-step field L2 error %.3e" % (procs, e)
    # hot electrons (0.2 c) do cross brick faces in 10 steps: the brick populations changed
    n_now = [sims[r].get_particles(0)["x"].size for r in sims]
    n0 = [int((owners[0] == r).sum()) for r in sims]
    assert sum(n_now) == sum(n0) and n_now != n0
    for r, s in sims.items():                    # and every particle sits inside its brick
        p = s.get_particles(0)
        lm = layout.local_min(r)
        for d, nm in enumerate("xyz"):
            if layout.procs[d] > 1:
                assert p[nm].min() >= lm[d] and p[nm].max() < lm[d] + layout.nl[d] * layout.d[d]
    for s in sims.values():
        s.close()


def test_brick_calls_reject_bad_arguments(Sim):
    from paper_2303_12873_b200.binding import PicError
    import torch
    wl = W.uniform_plasma(8, 8, 2, ppc=1, u_th=0.0, order=1, seed=3)
    g = Sim.from_workload(wl)
    buf = torch.empty(g.halo_doubles(2), dtype=torch.float64, device="cuda")
    with pytest.raises(PicError):
        g.export_halo(0, 2, 0, buf)              # fewer than NG cells along z
    with pytest.raises(PicError):
        g.step_stage(4)
    g.set_option("open_mask", 1)
    with pytest.raises(PicError):
        g.step(1)                                 # a brick is stepped in stages
    g.set_option("open_mask", 0)
    small = torch.empty(8, dtype=torch.float64, device="cuda")
    g.step(1)
    assert g.export_leavers(0, 0, 1, small) == 0  # periodic grid: nobody is outside
    g.close()
