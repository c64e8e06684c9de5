"""Multi-GPU plumbing for ``bench.py --gpus N``: REPLICAS ONLY.

BASELINE.json:north_star scopes the path to one GPU ("no domain decomposition across GPUs, no MPI or
collectives"), so N ranks run N independent replicas of the workload; there is no data-path
collective.  The only communication is the reduction of the timing (max over ranks).  This module
holds that host-side logic so that it can be tested with world-size-2 gloo on CPU
(tests/test_multiproc_cpu.py)."""
from __future__ import annotations

import numpy as np


def rank_env(env) -> tuple:
    """(rank, local_rank, world_size) from a torchrun-style environment mapping."""
    return int(env.get("RANK", "0")), int(env.get("LOCAL_RANK", "0")), int(env.get("WORLD_SIZE", "1"))


def make_replica(wl, rank: int):
    """Replica ``rank`` of a workload: the same plasma with the particle momenta cyclically shifted by
    8 * rank entries (so replicas are not bit-identical), positions, weights and fields unchanged."""
    if rank:
        for sp in wl.species:
            for nm in ("ux", "uy", "uz"):
                setattr(sp, nm, np.ascontiguousarray(np.roll(getattr(sp, nm), 8 * rank)))
    return wl


def max_over_ranks(value: float, dist=None, device="cpu") -> float:
    """The job's time is the slowest rank's: all-reduce MAX (no-op without a process group)."""
    if dist is None:
        return float(value)
    import torch
    t = torch.tensor([float(value)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def job_rate(units_per_rank: int, steps: int, seconds: float, world: int) -> float:
    """Whole-job throughput of ``world`` replicas: units all ranks processed / the slowest rank's time."""
    return world * units_per_rank * steps / seconds
