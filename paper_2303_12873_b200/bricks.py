"""Brick decomposition of one PIC box over several contexts (
PAPER.md:65,69,81: the paper's weak scaling rests on a spatial decomposition with neighbour
exchange).  Host-side schedule only: every brick is an ordinary ``binding.Sim`` whose
``open_mask`` names the decomposed dimensions; what crosses a face is packed, unpacked and
partitioned by the library's kernels (``pic_export_halo`` / ``pic_import_halo`` /
``pic_export_leavers`` / ``pic_import_arrivals``, csrc/bricks.cu) and travels as device
buffers through a *transport*:

* ``LocalTransport``  every brick lives in this process (one GPU): buffers are handed over
  as they are.  This is what the single-GPU parity test drives.
* ``DistTransport``   one brick per rank of a ``torch.distributed`` group: ``isend`` /
  ``irecv`` between neighbours (NCCL over NVLink on GPUs; gloo in the CPU test).  There is
  no collective: every message has exactly one sender and one receiver.

One step of the decomposed box (``BrickStepper.step``), identical on every brick:
  stage 0 (J := 0, particles, fold)  ->  J halos (sum)  ->  leavers / arrivals, dimension
  by dimension  ->  sort  ->  B half push, B halos  ->  E push, E halos  ->  B half push,
  B halos.  Unmeasured on more than one GPU (the build box has one).
"""
from __future__ import annotations

import numpy as np

GROUP_E, GROUP_B, GROUP_J = 0, 1, 2


class BrickLayout:
    """A periodic box of (nx, ny, nz) cells cut into procs = (px, py, pz) equal bricks; rank = cx + px (cy + py cz)."""

    def __init__(self, nx, ny, nz, dx, dy, dz, xmin, ymin, zmin, procs):
        self.n = (int(nx), int(ny), int(nz))
        self.d = (float(dx), float(dy), float(dz))
        self.min = (float(xmin), float(ymin), float(zmin))
        self.procs = tuple(int(p) for p in procs)
        for n, p in zip(self.n, self.procs):
            if p < 1 or n % p:
                raise ValueError("every dimension must split into equal bricks: %r cells over %r bricks" % (self.n, self.procs))
        self.nl = tuple(n // p for n, p in zip(self.n, self.procs))
        self.size = self.procs[0] * self.procs[1] * self.procs[2]
        self.L = tuple(n * d for n, d in zip(self.n, self.d))
        # a dimension with a single brick stays periodic inside that brick
        self.open_mask = sum(1 << k for k in range(3) if self.procs[k] > 1)
        self.open_dims = [k for k in range(3) if self.procs[k] > 1]

    def coords(self, rank):
        px, py, _ = self.procs
        return (rank % px, (rank // px) % py, rank // (px * py))

    def rank_of(self, c):
        px, py, pz = self.procs
        return (c[0] % px) + px * ((c[1] % py) + py * (c[2] % pz))

    def origin(self, rank):
        """First global cell index of the brick, per dimension."""
        return tuple(c * nl for c, nl in zip(self.coords(rank), self.nl))

    def local_min(self, rank):
        # node i of the whole box sits at min + i * d (the same expression the single-domain grid uses)
        return tuple(m + o * d for m, o, d in zip(self.min, self.origin(rank), self.d))

    def neighbour(self, rank, dim, side):
        c = list(self.coords(rank))
        c[dim] += 1 if side else -1
        return self.rank_of(c)

    def arrival_shift(self, rank, dim, side):
        """Shift applied to the positions of particles ARRIVING at `rank` through its face (dim, side): they
        crossed the periodic seam of the whole box iff that face is an outer face."""
        c = self.coords(rank)[dim]
        s = [0.0, 0.0, 0.0]
        if side == 0 and c == 0:
            s[dim] = -self.L[dim]          # they left the last brick upwards: x >= xmax of the box
        elif side == 1 and c == self.procs[dim] - 1:
            s[dim] = +self.L[dim]          # they left the first brick downwards: x < xmin of the box
        return tuple(s)

    # ---- cutting the inputs of the whole box, joining the outputs -----------------------------------------
    def split_field(self, flat, rank):
        nx, ny, nz = self.n
        o, nl = self.origin(rank), self.nl
        a = np.asarray(flat, dtype=np.float64).reshape(nz, ny, nx)
        return np.ascontiguousarray(a[o[2]:o[2] + nl[2], o[1]:o[1] + nl[1], o[0]:o[0] + nl[0]]).reshape(-1)

    def join_field(self, parts):
        nx, ny, nz = self.n
        out = np.empty((nz, ny, nx))
        for rank, flat in parts.items():
            o, nl = self.origin(rank), self.nl
            out[o[2]:o[2] + nl[2], o[1]:o[1] + nl[1], o[0]:o[0] + nl[0]] = np.asarray(flat).reshape(nl[2], nl[1], nl[0])
        return out.reshape(-1)

    def owner_of(self, x, y, z):
        """Rank that owns each position (positions inside the box)."""
        idx = []
        for pos, m, d, nl, p in zip((x, y, z), self.min, self.d, self.nl, self.procs):
            cell = np.floor((np.asarray(pos) - m) * (1.0 / d)).astype(np.int64)
            idx.append(np.clip(cell // nl, 0, p - 1))
        return idx[0] + self.procs[0] * (idx[1] + self.procs[1] * idx[2])


class LocalTransport:
    """All bricks in this process: a message is the sender's buffer itself."""

    def __init__(self, ranks):
        self.ranks = list(ranks)

    def exchange(self, sends, recv_like=None):
        """sends: list of (src, dst, key, tensor).  Returns {(dst, key): tensor} for the local destinations."""
        return {(dst, key): t for (_, dst, key, t) in sends}

    def exchange_counts(self, sends):
        return {(dst, key): int(n) for (_, dst, key, n) in sends}


class DistTransport:
    """One brick per rank of a torch.distributed group; neighbour-to-neighbour isend / irecv only.  With the NCCL backend
    the device buffers travel as they are (NVLink / NVSwitch peer transfers); with gloo (the CPU test, and two processes
    sharing one GPU) they are staged through host memory."""

    def __init__(self, dist, rank, device, stage_through_host=None):
        self.dist, self.rank, self.device = dist, int(rank), device
        import torch
        self.torch = torch
        if stage_through_host is None:
            stage_through_host = dist.get_backend() != "nccl"
        self.host = bool(stage_through_host)

    @staticmethod
    def _face_order(key):
        dim, side = key
        return 2 * dim + side

    def exchange(self, sends, recv_like=None):
        """sends: [(src == my rank, dst, key, tensor)]; recv_like: {(src, key): empty tensor to receive into} for the
        messages this rank expects, keyed by the face they arrive at.  Returns {(my rank, key): tensor}.

        Messages are matched by ORDER, never by tag: the NCCL backend ignores P2P tags and pairs the sends and
        receives between two ranks in the order they were issued.  With two bricks along a dimension both faces of a
        brick talk to the same peer, so both sides must agree on the order without talking: every message is named by
        the face (dim, side) it ARRIVES at -- the sender's `key` and the receiver's `key` are that same face -- and both
        the sends to a peer and the receives from it are issued in increasing (peer, 2 dim + side).  All tags are 0,
        so the gloo test exercises exactly the matching NCCL does."""
        recvs, out, landed, posts = [], {}, [], []
        for (src, key), buf in (recv_like or {}).items():
            if src == self.rank:
                continue
            tmp = self.torch.empty(buf.shape, dtype=buf.dtype) if (self.host and buf.is_cuda) else buf
            recvs.append((src, self._face_order(key), tmp))
            if tmp is not buf:
                landed.append((tmp, buf))
            out[(self.rank, key)] = buf
        for (src, dst, key, t) in sends:
            assert src == self.rank
            if dst == self.rank:                     # a brick that is its own neighbour (never with procs > 1)
                out[(dst, key)] = t
                continue
            t = t.contiguous()
            if self.host and t.is_cuda:
                t = t.cpu()
            posts.append((dst, self._face_order(key), t))
        recvs.sort(key=lambda m: m[:2])
        posts.sort(key=lambda m: m[:2])
        ops = [self.dist.P2POp(self.dist.irecv, t, src, tag=0) for (src, _, t) in recvs]
        ops += [self.dist.P2POp(self.dist.isend, t, dst, tag=0) for (dst, _, t) in posts]
        if ops:
            for r in self.dist.batch_isend_irecv(ops):
                r.wait()
        for tmp, buf in landed:
            buf.copy_(tmp)
        return out

    def exchange_counts(self, sends, expect):
        """sends: [(src, dst, key, n)]; expect: [(src, key)] faces this rank receives on.  Returns {(rank, key): n}."""
        t = self.torch
        dev = "cpu" if self.host else self.device
        bufs = {(src, key): t.zeros(1, dtype=t.int64, device=dev) for (src, key) in expect}
        msgs = [(src, dst, key, t.tensor([int(n)], dtype=t.int64, device=dev)) for (src, dst, key, n) in sends]
        got = self.exchange(msgs, bufs)
        return {k: int(v.item()) for k, v in got.items()}


class BrickStepper:
    """Drives the bricks this process owns (all of them with LocalTransport, one with DistTransport)."""

    def __init__(self, layout, sims, transport, nspecies, leaver_capacity=1 << 16):
        import torch
        self.torch = torch
        self.layout, self.sims, self.tr, self.nspecies = layout, dict(sims), transport, int(nspecies)
        self.cap = int(leaver_capacity)
        self._halo, self._part = {}, {}
        for r, sim in self.sims.items():
            sim.set_option("open_mask", layout.open_mask)

    # ---- buffers -------------------------------------------------------------------------------------------
    def _hbuf(self, rank, dim, side, kind):
        key = (rank, dim, side, kind)
        if key not in self._halo:
            sim = self.sims[rank]
            self._halo[key] = self.torch.empty(sim.halo_doubles(dim), dtype=self.torch.float64, device=sim.device)
        return self._halo[key]

    def _pbuf(self, rank, side, kind):
        key = (rank, side, kind)
        if key not in self._part:
            self._part[key] = self.torch.empty(8 * self.cap, dtype=self.torch.float64, device=self.sims[rank].device)
        return self._part[key]

    # ---- exchanges -----------------------------------------------------------------------------------------
    def exchange_halo(self, group):
        lay = self.layout
        for d in lay.open_dims:
            sends, expect = [], {}
            for r, sim in self.sims.items():
                for side in (0, 1):
                    buf = self._hbuf(r, d, side, "out")
                    sim.export_halo(group, d, side, buf)
                    sends.append((r, lay.neighbour(r, d, side), (d, 1 - side), buf))    # arrives at the opposite face
                    expect[(lay.neighbour(r, d, side), (d, side))] = self._hbuf(r, d, side, "in")
            got = self.tr.exchange(sends, expect)
            for (dst, (dd, side)), buf in got.items():
                if dst in self.sims:
                    self.sims[dst].import_halo(group, dd, side, buf)

    def migrate(self):
        lay = self.layout
        for d in lay.open_dims:
            for s in range(self.nspecies):
                sends, counts, expect = [], [], []
                for r, sim in self.sims.items():
                    for side in (0, 1):
                        buf = self._pbuf(r, side, "out")
                        n = sim.export_leavers(s, d, side, buf)
                        nb = lay.neighbour(r, d, side)
                        counts.append((r, nb, (d, 1 - side), n))
                        sends.append((r, nb, (d, 1 - side), buf[:8 * n]))
                        expect.append((nb, (d, side)))
                if isinstance(self.tr, LocalTransport):
                    ncount = self.tr.exchange_counts(counts)
                    got = self.tr.exchange(sends)
                else:
                    ncount = self.tr.exchange_counts(counts, expect)
                    like = {}
                    for r in self.sims:
                        for side in (0, 1):
                            n = ncount.get((r, (d, side)), 0)
                            like[(lay.neighbour(r, d, side), (d, side))] = self._pbuf(r, side, "in")[:8 * n]
                    got = self.tr.exchange([m for m in sends if m[3].numel() > 0],
                                           {k: v for k, v in like.items() if v.numel() > 0})
                for (dst, (dd, side)), buf in got.items():
                    n = ncount.get((dst, (dd, side)), buf.numel() // 8)
                    if dst in self.sims and n > 0:
                        self.sims[dst].import_arrivals(s, buf, n, lay.arrival_shift(dst, dd, side))

    # ---- the step ------------------------------------------------------------------------------------------
    def start(self):
        """After pic_set_fields on every brick: fill the guard layers of E and B along the open dimensions."""
        self.exchange_halo(GROUP_E)
        self.exchange_halo(GROUP_B)

    def step(self, sort=True):
        for sim in self.sims.values():
            sim.step_stage(0)
        self.exchange_halo(GROUP_J)
        self.migrate()
        if sort:
            for sim in self.sims.values():
                sim.sort()
        for sim in self.sims.values():
            sim.step_stage(1)
        self.exchange_halo(GROUP_B)
        for sim in self.sims.values():
            sim.step_stage(2)
        self.exchange_halo(GROUP_E)
        for sim in self.sims.values():
            sim.step_stage(3)
        self.exchange_halo(GROUP_B)


def make_local_bricks(Sim, layout, wl, slack=1.5, device="cuda:0"):
    """Cut a whole-box workload into bricks that all live on one device: {rank: Sim}, loaded, with disjoint ids
    (brick r numbers its particles from the count of the bricks before it, in load order within the brick)."""
    sims = {}
    owners = [layout.owner_of(sp.x, sp.y, sp.z) for sp in wl.species]
    for r in range(layout.size):
        nl, lm = layout.nl, layout.local_min(r)
        sel = [np.nonzero(o == r)[0] for o in owners]
        np_max = [max(int(slack * len(ix)) + 1024, 1) for ix in sel]
        sim = Sim(nl[0], nl[1], nl[2], wl.dx, wl.dy, wl.dz, lm[0], lm[1], lm[2], wl.dt, wl.order, np_max, device=device)
        if wl.fields:
            sim.set_fields(**{k: layout.split_field(v, r) for k, v in wl.fields.items()})
        for s, (sp, ix) in enumerate(zip(wl.species, sel)):
            # ids: the particle's index in the whole-box load order is not recoverable from a per-brick iota, so the
            # caller matches by id through `global_ids`
            sim.set_option("id_base", int(sum(len(np.nonzero(owners[s] == q)[0]) for q in range(r))))
            sim.load_particles(s, sp.q, sp.m, *(np.ascontiguousarray(a[ix]) for a in sp.arrays()))
        sims[r] = sim
    return sims, owners


def global_ids(layout, owners_s):
    """ids the bricks gave at load (make_local_bricks), indexed by the particle's index in the whole-box arrays."""
    ids = np.empty(owners_s.size, dtype=np.int64)
    base = 0
    for r in range(layout.size):
        ix = np.nonzero(owners_s == r)[0]
        ids[ix] = base + np.arange(ix.size)
        base += ix.size
    return ids
