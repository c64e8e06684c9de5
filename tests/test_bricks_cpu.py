"""Host side of the brick decomposition (NEXT-1): layout arithmetic (neighbours across the
periodic seam, position shifts, cutting and joining arrays) and the neighbour-to-neighbour transport with
world-size-2 gloo on CPU.  No CUDA here."""
import os
import socket
import subprocess
import sys
import textwrap

import numpy as np

from paper_2303_12873_b200 import bricks as B

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_layout_neighbours_shifts_and_cuts():
    lay = B.BrickLayout(12, 8, 6, 0.5, 0.25, 1.0, -1.0, 2.0, 0.0, (3, 1, 2))
    assert lay.size == 6 and lay.nl == (4, 8, 3) and lay.open_mask == 0b101 and lay.open_dims == [0, 2]
    assert [lay.coords(r) for r in range(6)] == [(0, 0, 0), (1, 0, 0), (2, 0, 0), (0, 0, 1), (1, 0, 1), (2, 0, 1)]
    for r in range(6):
        assert lay.rank_of(lay.coords(r)) == r
        for d in (0, 2):
            for side in (0, 1):
                nb = lay.neighbour(r, d, side)
                assert lay.neighbour(nb, d, 1 - side) == r           # the relation is symmetric
    assert lay.neighbour(0, 0, 0) == 2 and lay.neighbour(2, 0, 1) == 0 and lay.neighbour(0, 2, 0) == 3
    assert lay.local_min(4) == (-1.0 + 4 * 0.5, 2.0, 3.0)
    # a particle arriving at brick 0 through its low x face left brick 2 upwards: it crossed the seam
    assert lay.arrival_shift(0, 0, 0) == (-6.0, 0.0, 0.0) and lay.arrival_shift(2, 0, 1) == (6.0, 0.0, 0.0)
    assert lay.arrival_shift(1, 0, 0) == (0.0, 0.0, 0.0) and lay.arrival_shift(3, 2, 1) == (0.0, 0.0, 6.0)
    rng = np.random.default_rng(0)
    f = rng.standard_normal(12 * 8 * 6)
    parts = {r: lay.split_field(f, r) for r in range(6)}
    assert all(p.size == 4 * 8 * 3 for p in parts.values())
    assert np.array_equal(lay.join_field(parts), f)
    i, j, k = 9, 3, 4
    assert parts[lay.rank_of((2, 0, 1))][(i - 8) + 4 * (j + 8 * (k - 3))] == f[i + 12 * (j + 8 * k)]
    x = -1.0 + (rng.random(100) * 12) * 0.5; y = 2.0 + rng.random(100) * 2.0; z = rng.random(100) * 6.0
    own = lay.owner_of(x, y, z)
    for r in range(6):
        lm = lay.local_min(r)
        sel = own == r
        assert np.all((x[sel] >= lm[0]) & (x[sel] < lm[0] + 4 * 0.5) & (z[sel] >= lm[2]) & (z[sel] < lm[2] + 3.0))
    ids = B.global_ids(lay, own)
    assert sorted(ids.tolist()) == list(range(100))


def test_local_transport_hands_buffers_over():
    t = B.LocalTransport(range(2))
    a, b = np.arange(3), np.arange(4)
    got = t.exchange([(0, 1, (0, 0), a), (1, 0, (0, 1), b)])
    assert got[(1, (0, 0))] is a and got[(0, (0, 1))] is b
    assert t.exchange_counts([(0, 1, (2, 1), 7)]) == {(1, (2, 1)): 7}


class _FakeDist:
    """Records the order in which DistTransport issues its point-to-point operations."""
    isend, irecv = "isend", "irecv"

    class P2POp:
        def __init__(self, op, tensor, peer, tag=0):
            self.op, self.tensor, self.peer, self.tag = op, tensor, peer, tag

    def __init__(self):
        self.issued = []

    def get_backend(self):
        return "nccl"

    def batch_isend_irecv(self, ops):
        self.issued = list(ops)
        return []


def test_dist_transport_orders_messages_by_arrival_face_not_by_tag():
    """The NCCL backend ignores tags and pairs the messages between two ranks in issue order.  With two
    bricks along a dimension both faces talk to the same peer: the k-th send of rank 0 to rank 1 must be the k-th
    receive rank 1 posts from rank 0, whatever order the schedule listed them in, and no tag may be relied on."""
    import torch
    lay = B.BrickLayout(16, 8, 8, 1.0, 1.0, 1.0, 0.0, 0.0, 0.0, (2, 2, 1))
    # ranks 0 and 1 are each other's neighbour through BOTH x faces; 0's y neighbour (both faces) is rank 2
    plans = {}
    for rank in (0, 1):
        fd = _FakeDist()
        tr = B.DistTransport(fd, rank, "cpu")
        sends, expect = [], {}
        for d in ((1, 0) if rank == 0 else (0, 1)):          # the two ranks walk dimensions and faces in different orders
            for side in ((0, 1) if rank == 0 else (1, 0)):
                nb = lay.neighbour(rank, d, side)
                arrives_at = (d, 1 - side)                     # face of the neighbour this message lands on
                # every tensor carries the name of the face it arrives at, as a number
                sends.append((rank, nb, arrives_at, torch.full((1,), 10.0 * d + (1 - side), dtype=torch.float64)))
                expect[(nb, (d, side))] = torch.full((1,), 10.0 * d + side, dtype=torch.float64)
        tr.exchange(sends, expect)
        assert all(op.tag == 0 for op in fd.issued)
        plans[rank] = fd.issued
    for a, b in ((0, 1), (1, 0)):
        sent = [float(op.tensor[0]) for op in plans[a] if op.op == "isend" and op.peer == b]
        posted = [float(op.tensor[0]) for op in plans[b] if op.op == "irecv" and op.peer == a]
        assert len(sent) == 2 and sent == posted, (a, b, sent, posted)   # k-th send meets the k-th receive: same face


_WORKER = textwrap.dedent("""
    import os, sys
    sys.path.insert(0, %r)
    import torch, torch.distributed as dist
    from paper_2303_12873_b200 import bricks as B
    rank, world = int(os.environ["RANK"]), int(os.environ["WORLD_SIZE"])
    dist.init_process_group("gloo", rank=rank, world_size=world)
    lay = B.BrickLayout(16, 8, 8, 1.0, 1.0, 1.0, 0.0, 0.0, 0.0, (2, 1, 1))
    tr = B.DistTransport(dist, rank, "cpu")
    d = 0
    # the halo schedule of BrickStepper.exchange_halo for this rank's brick: both faces go to the other rank
    sends, expect = [], {}
    for side in (0, 1):
        buf = torch.full((5,), float(100 * rank + 10 * side), dtype=torch.float64)
        nb = lay.neighbour(rank, d, side)
        sends.append((rank, nb, (d, 1 - side), buf))
        expect[(nb, (d, side))] = torch.empty(5, dtype=torch.float64)
    got = tr.exchange(sends, expect)
    # what arrives at my face `side` was sent by the neighbour through ITS face 1 - side
    for side in (0, 1):
        v = got[(rank, (d, side))]
        assert torch.all(v == float(100 * (1 - rank) + 10 * (1 - side))), (rank, side, v)
    # variable-length messages: counts first
    counts = [(rank, lay.neighbour(rank, d, side), (d, 1 - side), 3 * rank + side + 1) for side in (0, 1)]
    n = tr.exchange_counts(counts, [(lay.neighbour(rank, d, side), (d, side)) for side in (0, 1)])
    for side in (0, 1):
        assert n[(rank, (d, side))] == 3 * (1 - rank) + (1 - side) + 1, (rank, side, n)
    dist.barrier()
    print("RESULT ok %%d" %% rank)
    dist.destroy_process_group()
""") % ROOT


def test_two_ranks_gloo_neighbour_exchange():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        port = s.getsockname()[1]
    procs = []
    for rank in range(2):
        env = dict(os.environ, RANK=str(rank), LOCAL_RANK=str(rank), WORLD_SIZE="2", MASTER_ADDR="127.0.0.1",
                   MASTER_PORT=str(port))
        procs.append(subprocess.Popen([sys.executable, "-c", _WORKER], env=env, stdout=subprocess.PIPE,
                                      stderr=subprocess.PIPE, text=True))
    for p in procs:
        out, err = p.communicate(timeout=240)
        assert p.returncode == 0, err[-3000:]
        assert "RESULT ok" in out
