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


# ---------------------------------------------------------------- two processes, one brick each, one GPU
_WORKER = '''
import os, sys
sys.path.insert(0, %r)
sys.path.insert(0, os.path.join(%r, "tests"))
import numpy as np, torch, torch.distributed as dist
from paper_2303_12873_b200 import bricks as B, workloads as W
from paper_2303_12873_b200.binding import Sim
rank, world = int(os.environ["RANK"]), int(os.environ["WORLD_SIZE"])
dist.init_process_group("gloo", rank=rank, world_size=world)
torch.cuda.set_device(0)
wl = W.uniform_plasma(16, 8, 24, ppc=4, u_th=0.2, order=3, seed=611, protons=True)
rng = np.random.default_rng(61)
wl.fields = {n: (3e8 if n[0] == "E" else 1.0) * rng.standard_normal(wl.ncell) for n in ("Ex", "Ey", "Ez", "Bx", "By", "Bz")}
lay = B.BrickLayout(wl.nx, wl.ny, wl.nz, wl.dx, wl.dy, wl.dz, 0.0, 0.0, 0.0, (1, 1, 2))
owners = [lay.owner_of(sp.x, sp.y, sp.z) for sp in wl.species]
sel = [np.nonzero(o == rank)[0] for o in owners]
lm = lay.local_min(rank)
sim = Sim(*lay.nl, wl.dx, wl.dy, wl.dz, *lm, wl.dt, wl.order, [2 * len(ix) + 1024 for ix in sel])
sim.set_fields(**{k: lay.split_field(v, rank) for k, v in wl.fields.items()})
for s, (sp, ix) in enumerate(zip(wl.species, sel)):
    sim.set_option("id_base", int(sum((owners[s] == q).sum() for q in range(rank))))
    sim.load_particles(s, sp.q, sp.m, *(np.ascontiguousarray(a[ix]) for a in sp.arrays()))
st = B.BrickStepper(lay, {rank: sim}, B.DistTransport(dist, rank, "cuda:0"), len(wl.species), leaver_capacity=1 << 14)
st.start()
sim.sort()
for it in range(6):
    st.step()
f = sim.get_fields()
n_mine = torch.tensor([sim.get_particles(0)["x"].size], dtype=torch.int64)
if rank == 1:
    for n in Sim.FIELD_NAMES:
        dist.send(torch.from_numpy(f[n]), 0)
    dist.send(n_mine, 0)
else:
    from oracle import ora
    from parity_util import TOL_FIELD_L2_10STEP, field_l2_error
    other = {}
    for n in Sim.FIELD_NAMES:
        t = torch.empty(f[n].size, dtype=torch.float64)
        dist.recv(t, 1)
        other[n] = t.numpy()
    n_other = torch.zeros(1, dtype=torch.int64)
    dist.recv(n_other, 1)
    joined = {n: lay.join_field({0: f[n], 1: other[n]}) for n in Sim.FIELD_NAMES}
    o = ora.OracleSim(*wl.grid_args(), wl.dt, wl.order, 2)
    o.set_fields(**wl.fields)
    for s, sp in enumerate(wl.species):
        o.load_particles(s, sp.q, sp.m, *sp.arrays())
    o.step(6)
    e = field_l2_error(o.get_fields(), joined)
    assert e <= TOL_FIELD_L2_10STEP, e
    jmax = max(np.abs(o.get_fields()[c]).max() for c in ("Jx", "Jy", "Jz"))
    assert max(np.abs(o.get_fields()[c] - joined[c]).max() for c in ("Jx", "Jy", "Jz")) <= 1e-9 * jmax
    assert int(n_mine) + int(n_other) == wl.species[0].n and int(n_mine) != len(sel[0])
    print("RESULT ok %%.3e" %% e)
dist.barrier()
sim.close()
dist.destroy_process_group()
'''


def test_two_processes_one_brick_each_exchange_through_torch_distributed():
    """The distributed schedule for real: two processes, each one brick of a 16 x 8 x 24 box on THIS GPU, exchanging halos,
    J and particles through BrickStepper + DistTransport (gloo, staged through host memory; on several GPUs the same code
    runs over NCCL).  Rank 0 joins the fields and checks them against the single-domain oracle after 6 steps.  No kernel
    waits on another process: the ranks meet only in host-side send / recv between launches."""
    import os
    import socket
    import subprocess
    import sys
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        port = s.getsockname()[1]
    procs = []
    for rank in range(2):
        env = dict(os.environ, RANK=str(rank), LOCAL_RANK=str(rank), WORLD_SIZE="2", MASTER_ADDR="127.0.0.1",
                   MASTER_PORT=str(port))
        procs.append(subprocess.Popen([sys.executable, "-c", _WORKER % (root, root)], env=env, stdout=subprocess.PIPE,
                                      stderr=subprocess.PIPE, text=True))
    outs = []
    for p in procs:
        out, err = p.communicate(timeout=600)
        assert p.returncode == 0, err[-3000:]
        outs.append(out)
    assert "RESULT ok" in outs[0]
