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


# ------------------------------------------------------------------------------------------------
# Sharding ONE batch over the ranks (SURVEY.md 8(e), strong scaling): the jobs are independent, so each rank
# integrates a subset chosen by longest-processing-time-first on the estimated cost n_i x ops_i; the only
# exchange is the amplitude, A = sum_i C_i I_i: partial sums add, and so do the variances of
# Eq. (4) -- one all-reduce of 4 J doubles.
def lpt_partition(costs: Sequence[float], world: int):
    """Longest-processing-time-first: jobs by decreasing cost, each to the least loaded rank (ties: lowest
    rank).  Returns one sorted index list per rank; every job appears exactly once."""
    parts = [[] for _ in range(world)]
    load = [0.0] * world
    for i in sorted(range(len(costs)), key=lambda i: (-float(costs[i]), i)):
        r = min(range(world), key=lambda r: (load[r], r))
        parts[r].append(i)
        load[r] += float(costs[i])
    return [sorted(p) for p in parts]


def combine_amplitudes(amp_local, world: int, device="cpu"):
    """amp_local: [J, 4] = (re, im, err_re, err_im) of this rank's jobs, a numpy array or a torch tensor (then
    the all-reduce runs on the tensor's device and stream and a tensor comes back).  Returns the amplitude of
    all ranks' jobs: means add, errors add in quadrature (Eq. 4).  The identity for world == 1."""
    import numpy as np
    is_tensor = hasattr(amp_local, "is_cuda")
    if world <= 1:
        return amp_local.clone() if is_tensor else np.asarray(amp_local, dtype=np.float64).copy()
    import torch
    import torch.distributed as dist
    a = amp_local if is_tensor else torch.tensor(np.asarray(amp_local, dtype=np.float64), device=device)
    t = torch.cat([a[:, :2], a[:, 2:] ** 2], dim=1).contiguous()
    dist.all_reduce(t, op=dist.ReduceOp.SUM)
    out = torch.cat([t[:, :2], torch.sqrt(t[:, 2:])], dim=1)
    return out if is_tensor else out.cpu().numpy()


# ------------------------------------------------------------------------------------------------
# Splitting single jobs: "longest-processing-time assignment of jobs by n_i x cost_i to GPUs; split
# only jobs larger than the mean load by shift, then by k-range".  The m shifts of a job are independent and the
# lattice indices of one (job, shift) split into disjoint ranges whose partial sums add, so a piece is
# (job, s0, s1, k0, k1): shifts s0 <= s < s1, indices k0 <= k < k1.  The pieces of all ranks go through
# qmc_integrate_pieces, one all-gather of the per-shift (hi, lo) sums, and qmc_finalize_pieces (include/qmc.h).
def split_partition(cost_per_eval: Sequence[float], n: Sequence[int], m: int, world: int, granularity: float = 0.5):
    """Returns one list of pieces (job, s0, s1, k0, k1) per rank, each sorted by job; every (job, shift, k) is in
    exactly one piece.  A job whose cost n_i m cost_i exceeds the mean load per rank is cut into pieces of at most
    `granularity` x the mean load: whole shifts first; if a single shift is still too large, every shift on its own
    and its index range into equal parts.  Whole jobs and pieces are then assigned longest-processing-time-first."""
    nj = len(n)
    cost = [float(cost_per_eval[i]) * float(n[i]) * m for i in range(nj)]
    mean = sum(cost) / max(1, world)
    items = []                                              # (cost, job, s0, s1, k0, k1)
    for i in range(nj):
        if world <= 1 or cost[i] <= mean or cost[i] == 0.0:
            items.append((cost[i], i, 0, m, 0, int(n[i])))
            continue
        parts = int(-(-cost[i] // (granularity * mean)))    # ceil
        if parts <= m:
            bounds = [(m * p) // parts for p in range(parts + 1)]
            for a, b in zip(bounds[:-1], bounds[1:]):
                if b > a:
                    items.append((cost[i] * (b - a) / m, i, a, b, 0, int(n[i])))
        else:
            q = min(int(n[i]), -(-parts // m))              # k-ranges per shift
            kb = [(int(n[i]) * p) // q for p in range(q + 1)]
            for s in range(m):
                for a, b in zip(kb[:-1], kb[1:]):
                    if b > a:
                        items.append((cost[i] * (b - a) / (float(n[i]) * m), i, s, s + 1, a, b))
    parts_of = [[] for _ in range(world)]
    load = [0.0] * world
    for it in sorted(items, key=lambda t: (-t[0], t[1], t[2], t[4])):
        r = min(range(world), key=lambda r: (load[r], r))
        parts_of[r].append(it[1:])
        load[r] += it[0]
    return [sorted(p) for p in parts_of]


def gather_parts(partial, world: int):
    """All ranks' per-shift partial sums, one after another (the path's one collective: an all-gather of
    n_jobs x m x J x 6 doubles per rank).  partial: torch tensor on the kernels' device; returns [world, ...]."""
    import torch
    if world <= 1:
        return partial.unsqueeze(0)
    import torch.distributed as dist
    parts = [torch.empty_like(partial) for _ in range(world)]
    dist.all_gather(parts, partial.contiguous())       # NCCL on the GPU, gloo in the CPU tests
    return torch.stack(parts)


# ------------------------------------------------------------------------------------------------
# The median rule over ranks (step a5 of a sharded batch).  Every candidate generating vector is a lattice rule of its
# own, so the candidate stage is a batch of n_jobs x K one-shift jobs that splits like any other: by candidate and, for
# long lattices, by k-range.  After one all-gather, qmc_median_select_pieces gives every rank the same selection, and
# the m-shift stage runs on the selected vectors as pieces again.  Marshalling only -- no arithmetic of the method.
def candidate_jobs(jobs, z_cand, shift_row_base: int = 0):
    """The n_jobs x K candidate jobs for qmc_integrate_pieces (m = 1): job i K + c has the sector and n of job i,
    z = z_cand[i, c] and uses shift row shift_row_base + i (the row of job i's shared shift)."""
    from .workloads import Job
    out = []
    for i, j in enumerate(jobs):
        for c in range(z_cand.shape[1]):
            out.append(Job(j.sector, j.n, z_cand[i, c].copy(), shift_row_base + i, 1.0 + 0.0j))
    return out


def selected_jobs(jobs, z_cand, selected):
    """The jobs of the m-shift stage: as `jobs`, with z = the selected candidate of each."""
    from .workloads import Job
    return [Job(j.sector, j.n, z_cand[i, int(selected[i])].copy(), j.shift_offset, j.coef) for i, j in enumerate(jobs)]
