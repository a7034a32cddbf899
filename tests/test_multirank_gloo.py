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


def _shard_worker(rank, world, port, q):
    sys.path.insert(0, ROOT)
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world),
                      LOCAL_RANK=str(rank))
    import torch.distributed as dist
    from oracle import oracle as O
    from paper_2305_19768_b200 import ranks as R, workloads as W
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        wl = W.config_batch(n_sectors=7, scale=1.0 / 200000.0, m=4)          # C4's mix, tiny lattices
        costs = [float(j.n) * (1.0 + wl.sectors[j.sector].dim) for j in wl.jobs]
        mine = R.lpt_partition(costs, world)[rank]
        shard = wl.subset(mine)
        res = np.zeros((len(shard.jobs), 3, 4))
        for pos, job in enumerate(shard.jobs):                              # the oracle stands in for the GPU
            sec = O.OracleSector(shard.sectors[job.sector])
            _, r, _ = O.integrate(sec, job.n, job.z, shard.shifts[job.shift_offset:job.shift_offset + shard.m])
            res[pos, :sec.J] = r
        amp_local = O.amplitude(res, np.array([j.coef for j in shard.jobs]))
        q.put((rank, mine, R.combine_amplitudes(amp_local, world).tolist()))
    finally:
        dist.destroy_process_group()


def test_one_batch_sharded_over_two_ranks_gives_the_single_process_amplitude():
    """Strong scaling (bench.py --scaling strong): LPT shards cover every job once, and the all-reduced partial
    amplitudes (means add, Eq. (4) variances add) equal the amplitude of the whole batch in one process."""
    import torch.multiprocessing as mp
    sys.path.insert(0, ROOT)
    from oracle import oracle as O
    from paper_2305_19768_b200 import ranks as R, workloads as W
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_shard_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    got = sorted(q.get(timeout=300) for _ in procs)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    (_, mine0, amp0), (_, mine1, amp1) = got
    wl = W.config_batch(n_sectors=7, scale=1.0 / 200000.0, m=4)
    assert sorted(mine0 + mine1) == list(range(len(wl.jobs))) and mine0 and mine1
    res = np.zeros((len(wl.jobs), 3, 4))
    for i, job in enumerate(wl.jobs):
        sec = O.OracleSector(wl.sectors[job.sector])
        _, r, _ = O.integrate(sec, job.n, job.z, wl.shifts[job.shift_offset:job.shift_offset + wl.m])
        res[i, :sec.J] = r
    whole = O.amplitude(res, np.array([j.coef for j in wl.jobs]))
    assert amp0 == amp1                                                       # every rank holds the result
    assert np.allclose(np.array(amp0), whole, rtol=1e-12, atol=1e-300)


def test_lpt_partition_properties():
    sys.path.insert(0, ROOT)
    from paper_2305_19768_b200 import ranks as R
    rng = np.random.default_rng(3)
    costs = 10.0 ** rng.uniform(6, 9, 600) * rng.uniform(80, 1500, 600)       # C4: n x ops
    for world in (1, 2, 4, 8):
        parts = R.lpt_partition(costs, world)
        assert sorted(i for p in parts for i in p) == list(range(600))
        loads = np.array([costs[p].sum() for p in parts])
        # LPT is within 4/3 - 1/(3 world) of the optimum, which is at least max(mean load, largest job)
        assert loads.max() <= (4.0 / 3.0) * max(costs.sum() / world, costs.max())
    assert R.lpt_partition([5.0, 5.0, 1.0], 2) == [[0, 2], [1]]                 # ties go to the lowest rank


def test_single_rank_is_identity_and_canonical_seed():
    sys.path.insert(0, ROOT)
    from paper_2305_19768_b200 import ranks as R, workloads as W
    assert R.aggregate([1.5, 2.5], [7.0], 1) == ([1.5, 2.5], [7.0])
    assert R.rank_seed(0, 2) is None and R.rank_seed(1, 2) != R.rank_seed(2, 2) != R.rank_seed(1, 3)
    import bench
    a, b = bench.make_workload("c2", 10007, 0), W.config_median(n=10007)
    assert np.array_equal(a.z_cand, b.z_cand) and np.array_equal(a.shifts, b.shifts)


def test_bench_gpus_flag_never_disagrees_silently():
    """`python bench.py --gpus N` either runs N ranks or fails loudly: with no CUDA device here it must refuse
    (not measure one GPU and print n_gpus: 1), and a torchrun environment of another size is refused as well."""
    import subprocess
    env = {k: v for k, v in os.environ.items() if k not in ("RANK", "WORLD_SIZE", "LOCAL_RANK")}
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--gpus", "2"], env=env, capture_output=True, text=True,
                       timeout=300)
    assert r.returncode != 0 and "only 0 CUDA device(s) visible" in (r.stderr + r.stdout)
    env["WORLD_SIZE"] = "1"
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--gpus", "2"], env=env, capture_output=True, text=True,
                       timeout=300)
    assert r.returncode != 0 and "--gpus 2 but WORLD_SIZE is 1" in (r.stderr + r.stdout)


def test_bench_oracle_slices_are_the_fixed_ones():
    """BASELINE.md section 3's slices: evaluation counts of the uncut slices, and the cut-off accounting."""
    sys.path.insert(0, ROOT)
    import bench
    e, dt, what = bench.oracle_slice("c0", 60.0)
    assert e == 5 * 65521 * 32 and "cut off" not in what
    e, dt, what = bench.oracle_slice("c2", 0.2)
    assert 0 < e < 43 * 1_000_003 and "cut off" in what and "11 candidates + 32 shifts" in what
    e, dt, what = bench.oracle_slice("c1", 0.2, shifts_of=(3, 16))
    assert "every 16-th shift row from 3" in what
