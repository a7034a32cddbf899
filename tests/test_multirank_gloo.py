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


# ------------------------------------------------------------------------------------------------
# SURVEY.md 8(e), the rest: a job larger than the mean load is split by shift, then by k-range.
def test_split_partition_covers_every_point_exactly_once_and_balances():
    sys.path.insert(0, ROOT)
    from paper_2305_19768_b200 import ranks as R
    rng = np.random.default_rng(5)
    for world in (1, 2, 3, 4, 8):
        for trial in range(6):
            nj = int(rng.integers(1, 9))
            n = [int(10 ** rng.uniform(2, 7)) for _ in range(nj)]
            cost = list(rng.uniform(50, 1500, nj))
            m = int(rng.choice([1, 2, 4, 32]))
            parts = R.split_partition(cost, n, m, world)
            assert len(parts) == world
            seen = {}
            load = [0.0] * world
            for r, pl in enumerate(parts):
                assert pl == sorted(pl)
                for job, s0, s1, k0, k1 in pl:
                    assert 0 <= s0 < s1 <= m and 0 <= k0 < k1 <= n[job]
                    seen.setdefault(job, []).append((s0, s1, k0, k1))
                    load[r] += cost[job] * (s1 - s0) * (k1 - k0)
            for job in range(nj):                         # exact cover of the (shift, k) rectangle: areas add up, no overlap
                rects = seen[job]
                assert sum((b - a) * (d - c) for a, b, c, d in rects) == m * n[job]
                for i, (a, b, c, d) in enumerate(rects):
                    for (a2, b2, c2, d2) in rects[i + 1:]:
                        assert b <= a2 or b2 <= a or d <= c2 or d2 <= c
            total = sum(cost[j] * n[j] * m for j in range(nj))
            # no piece exceeds the mean load, so LPT keeps every rank within mean + the largest piece
            assert max(load) <= total / world * 2.0 + 1e-9
    # the case that motivates it: ONE job on 4 ranks (a single lattice of up to 7e10 points)
    parts = R.split_partition([154.0], [10_000_019], 4, 4)
    assert all(len(p) == 2 for p in parts)
    assert {(s1 - s0, k1 - k0) for p in parts for _, s0, s1, k0, k1 in p} == {(1, 5_000_009), (1, 5_000_010)}


def _piece_worker(rank, world, port, q, n, m):
    sys.path.insert(0, ROOT)
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world),
                      LOCAL_RANK=str(rank))
    import torch
    import torch.distributed as dist
    from oracle import oracle as O
    from paper_2305_19768_b200 import ranks as R, workloads as W
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        wl = W.config_toy(n=n, m=m)
        job = wl.jobs[0]
        sec = O.OracleSector(wl.sectors[0])
        pieces = R.split_partition([30.0], [n], m, world)[rank]         # the product's own partition
        part = np.zeros((1, m, 1, 3, 2))                                  # [job, shift, order, comp, (hi, lo)]
        for _, s0, s1, k0, k1 in pieces:                                  # the oracle stands in for the device leg
            sums, _ = O.shift_sums(sec, n, job.z, wl.shifts[s0:s1], k0, k1)
            part[0, s0:s1, :, :, 0] += sums
        gathered = R.gather_parts(torch.from_numpy(part), world).numpy()  # the path's one collective
        q.put((rank, pieces, gathered.sum(axis=0)[..., 0].tolist()))
    finally:
        dist.destroy_process_group()


@pytest.mark.parametrize("world", [2, 4])
def test_one_job_split_over_ranks_by_shift_and_k_range_adds_up(world):
    """A 1-sector problem (n = 10^7, m = 4) on 2 and 4 gloo ranks: ranks.split_partition cuts it by shift (2 ranks)
    and by shift and k-range (4 ranks), every rank sums its pieces, one all-gather, and the per-shift sums equal the
    single-process ones to 1e-12."""
    import torch.multiprocessing as mp
    from oracle import oracle as O
    from paper_2305_19768_b200 import workloads as W
    n, m = 9_999_991, 4
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_piece_worker, args=(r, world, port, q, n, m)) for r in range(world)]
    for p in procs:
        p.start()
    got = sorted(q.get(timeout=240) for _ in procs)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    wl = W.config_toy(n=n, m=m)
    ref, _ = O.shift_sums(O.OracleSector(wl.sectors[0]), n, wl.jobs[0].z, wl.shifts)
    if world == 4:
        assert any(k1 - k0 < n for _, pieces, _s in got for (_j, _s0, _s1, k0, k1) in pieces)    # k-ranges really split
    for rank, pieces, total in got:
        total = np.array(total)[0]
        assert np.allclose(total, ref, rtol=1e-12, atol=0), (rank, np.abs(total - ref).max())


# The median rule over ranks: the candidate stage as n_jobs x K one-shift jobs (ranks.candidate_jobs), split like any batch.
def _median_worker(rank, world, port, q, n, K):
    sys.path.insert(0, ROOT)
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world),
                      LOCAL_RANK=str(rank))
    import torch
    import torch.distributed as dist
    from oracle import oracle as O
    from paper_2305_19768_b200 import ranks as R, workloads as W
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        wl = W.config_median(n_sectors=2, dim=2, n=n, K=K, m=2, seed=5)
        cj = R.candidate_jobs(wl.jobs, wl.z_cand)
        pieces = R.split_partition([30.0] * len(cj), [j.n for j in cj], 1, world)[rank]
        part = np.zeros((len(cj), 1, 1, 3, 2))
        for j, s0, s1, k0, k1 in pieces:                                  # the oracle stands in for the device leg
            sec = O.OracleSector(wl.sectors[cj[j].sector])
            sums, _ = O.shift_sums(sec, cj[j].n, cj[j].z, wl.shift0[cj[j].shift_offset:cj[j].shift_offset + 1], k0, k1)
            part[j, 0, :, :, 0] += sums[0]
        gathered = R.gather_parts(torch.from_numpy(part), world).numpy()
        q.put((rank, [list(p) for p in pieces], gathered.sum(axis=0)[:, 0, 0, :, 0].tolist()))
    finally:
        dist.destroy_process_group()


def test_median_candidates_split_over_two_ranks_select_the_same_vector():
    """Two gloo ranks share the 2 x 5 candidate jobs of a median pass; after the all-gather every rank holds the same
    candidate sums, and estimate, component-wise median and the candidate nearest it are those of the oracle's
    single-process median rule; ranks.selected_jobs then carries the selected vectors into the m-shift stage."""
    import torch.multiprocessing as mp
    from oracle import oracle as O
    from paper_2305_19768_b200 import ranks as R, workloads as W
    n, K, world = 10007, 5, 2
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_median_worker, args=(r, world, port, q, n, K)) for r in range(world)]
    for p in procs:
        p.start()
    got = sorted(q.get(timeout=240) for _ in procs)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    assert got[0][2] == got[1][2]                                          # same gathered sums on both ranks
    covered = sorted(pc[0] for _, pieces, _s in got for pc in pieces)
    assert covered == list(range(2 * K)) and all(len(pieces) == K for _, pieces, _s in got)
    wl = W.config_median(n_sectors=2, dim=2, n=n, K=K, m=2, seed=5)
    sums = np.array(got[0][2]).reshape(2, K, 3)
    sel = []
    for i in range(2):
        est, med, s = O.median_rule(O.OracleSector(wl.sectors[i]), n, wl.z_cand[i], wl.shift0[i])
        assert np.allclose(sums[i, :, 0] / n, est[:, 0].real, rtol=1e-12, atol=0)
        assert np.median(sums[i, :, 0] / n) == pytest.approx(med[0].real, rel=1e-12)
        sel.append(s)
    sj = R.selected_jobs(wl.jobs, wl.z_cand, sel)
    for i, j in enumerate(sj):
        assert np.array_equal(j.z, wl.z_cand[i, sel[i]]) and (j.sector, j.n, j.shift_offset) == (i, n, wl.jobs[i].shift_offset)
