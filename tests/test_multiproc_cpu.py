"""The N > 1 path of bench.py is replicas only: cover its host-side plumbing
(rank environment, replica construction, max-over-ranks timing, job rate) with world-size-2 gloo on CPU."""
import os
import socket
import subprocess
import sys
import textwrap

import numpy as np

from paper_2303_12873_b200 import replicas as R
from paper_2303_12873_b200 import workloads as W

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_rank_env_and_job_rate():
    assert R.rank_env({}) == (0, 0, 1)
    assert R.rank_env({"RANK": "3", "LOCAL_RANK": "1", "WORLD_SIZE": "4"}) == (3, 1, 4)
    assert R.job_rate(1000, 5, 0.5, 2) == 2 * 1000 * 5 / 0.5
    assert R.max_over_ranks(1.25) == 1.25


def test_replicas_differ_only_in_momenta():
    a = W.uniform_plasma(4, 4, 4, ppc=2, u_th=0.05, order=1, seed=1)
    b = R.make_replica(W.uniform_plasma(4, 4, 4, ppc=2, u_th=0.05, order=1, seed=1), 1)
    sa, sb = a.species[0], b.species[0]
    assert np.array_equal(sa.x, sb.x) and np.array_equal(sa.w, sb.w)
    assert np.array_equal(np.roll(sa.ux, 8), sb.ux) and not np.array_equal(sa.ux, sb.ux)
    assert sb.ux.flags["C_CONTIGUOUS"]


_WORKER = textwrap.dedent("""
    import os, sys
    sys.path.insert(0, %r)
    import torch.distributed as dist
    from paper_2303_12873_b200 import replicas as R
    from paper_2303_12873_b200 import workloads as W
    rank, local, world = R.rank_env(os.environ)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    wl = R.make_replica(W.uniform_plasma(4, 4, 4, ppc=2, u_th=0.05, order=1, seed=1), rank)
    my_time = 1.0 + rank                      # rank 1 is the slow one
    t = R.max_over_ranks(my_time, dist)
    rate = R.job_rate(wl.nparticles, 3, t, world)
    dist.barrier()
    print("RESULT %%d %%d %%.6f %%.6f %%.17e" %% (rank, world, t, rate, float(wl.species[0].ux[0])))
    dist.destroy_process_group()
""") % ROOT


def test_two_ranks_gloo_max_time_and_whole_job_rate():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        port = s.getsockname()[1]
    procs = []
    for rank in range(2):
        env = dict(os.environ, RANK=str(rank), LOCAL_RANK=str(rank), WORLD_SIZE="2", MASTER_ADDR="127.0.0.1",
                   MASTER_PORT=str(port))
        procs.append(subprocess.Popen([sys.executable, "-c", _WORKER], env=env, stdout=subprocess.PIPE,
                                      stderr=subprocess.PIPE, text=True))
    outs = []
    for p in procs:
        out, err = p.communicate(timeout=240)
        assert p.returncode == 0, err[-2000:]
        outs.append([l for l in out.splitlines() if l.startswith("RESULT")][0].split())
    base = W.uniform_plasma(4, 4, 4, ppc=2, u_th=0.05, order=1, seed=1)
    for o in outs:
        rank, world, t, rate = int(o[1]), int(o[2]), float(o[3]), float(o[4])
        assert world == 2 and t == 2.0                           # the slower rank's time on both ranks
        assert rate == 2 * base.nparticles * 3 / 2.0             # whole-job aggregate
        assert float(o[5]) == float(np.roll(base.species[0].ux, 8 * rank)[0])
