"""Multi-GPU plumbing of the QMC path: one process per GPU, no data-path collective.

Sectors (jobs) are independent problems: under ``torchrun`` every rank integrates its
own seeded batch on its own GPU and only the *timings* and *counts* meet -- the time of a run is the
maximum over the ranks, the work is the sum.  This module holds that host logic so that it can be
covered on CPU with the ``gloo`` backend (tests/test_multirank_gloo.py); it contains none of the method's
arithmetic.
"""
from __future__ import annotations

import os
from typing import Dict, Sequence, Tuple

MASTER_SEED = 2305


def env_rank() -> Tuple[int, int, int]:
    """(rank, world_size, local_rank) as torchrun exports them; (0, 1, 0) when run directly."""
    return (int(os.environ.get("RANK", "0")), int(os.environ.get("WORLD_SIZE", "1")),
            int(os.environ.get("LOCAL_RANK", "0")))


def rank_seed(rank: int, config_id: int):
    """Seed of the batch rank `rank` integrates: rank 0 takes the canonical workload of DESIGN.md
    section 4 (``None`` = the generator's own seed), every other rank an independent draw of the same
    shape, so that per-GPU work is fixed as the number of GPUs grows (weak scaling)."""
    if rank == 0:
        return None
    return MASTER_SEED * 100 + 50 + rank + 1000 * config_id


def aggregate(times_ms: Sequence[float], counts: Sequence[float], world: int, device="cpu") -> Tuple[list, list]:
    """MAX over ranks of every entry of `times_ms`, SUM over ranks of every entry of `counts`
    (float64 all-reduces on `device`; the identity for world == 1)."""
    if world <= 1:
        return [float(x) for x in times_ms], [float(x) for x in counts]
    import torch
    import torch.distributed as dist
    t = torch.tensor(list(times_ms), dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    c = torch.tensor(list(counts), dtype=torch.float64, device=device)
    dist.all_reduce(c, op=dist.ReduceOp.SUM)
    return [float(x) for x in t.cpu()], [float(x) for x in c.cpu()]


def throughput(evals_all_ranks: float, steps: int, ms_max_over_ranks: float) -> float:
    """Whole-job evaluations/s: all ranks' evaluations over the slowest rank's time."""
    return evals_all_ranks * steps / (ms_max_over_ranks * 1e-3)
