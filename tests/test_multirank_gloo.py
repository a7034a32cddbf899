"""N > 1 host logic on CPU: two processes with the gloo backend exercise exactly what bench.py does
between ranks (paper_2305_19768_b200/ranks.py) -- per-rank workloads, MAX-over-ranks timing, SUM-over-ranks
work -- since the path itself needs no data-path collective (sectors are independent problems)."""
import os
import socket
import sys

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, q):
    sys.path.insert(0, ROOT)
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world),
                      LOCAL_RANK=str(rank))
    import torch.distributed as dist
    import bench
    from paper_2305_19768_b200 import ranks as R
    assert R.env_rank() == (rank, world, rank)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        wl = bench.make_workload("c1", 10007, rank)
        evals = wl.evaluations()
        # rank r pretends its steps took (10 + 5 r) ms on the device and 3 launches each
        times, counts = R.aggregate([10.0 + 5.0 * rank, 0.02 * (rank + 1)], [float(evals), 3.0], world)
        fingerprint = float(wl.sectors[0].F_coef.sum() + wl.shifts.sum())
        q.put((rank, times, counts, evals, fingerprint, R.throughput(counts[0], 4, times[0])))
    finally:
        dist.destroy_process_group()


def test_two_ranks_max_time_sum_work():
    import torch.multiprocessing as mp
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    got = sorted(q.get(timeout=180) for _ in procs)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    (r0, t0, c0, e0, f0, v0), (r1, t1, c1, e1, f1, v1) = got
    assert (r0, r1) == (0, 1)
    assert t0 == t1 == [15.0, 0.04]                      # MAX over ranks, identical on every rank
    assert c0 == c1 == [float(e0 + e1), 6.0]             # SUM over ranks
    assert e0 == e1 == 8 * 10007 * 32                    # weak scaling: the same work per rank ...
    assert f0 != f1                                      # ... on independently drawn batches
    assert v0 == v1 == pytest.approx((e0 + e1) * 4 / 15e-3)


def test_single_rank_is_identity_and_canonical_seed():
    sys.path.insert(0, ROOT)
    from paper_2305_19768_b200 import ranks as R, workloads as W
    assert R.aggregate([1.5, 2.5], [7.0], 1) == ([1.5, 2.5], [7.0])
    assert R.rank_seed(0, 2) is None and R.rank_seed(1, 2) != R.rank_seed(2, 2) != R.rank_seed(1, 3)
    import bench
    a, b = bench.make_workload("c2", 10007, 0), W.config_median(n=10007)
    assert np.array_equal(a.z_cand, b.z_cand) and np.array_equal(a.shifts, b.shifts)
