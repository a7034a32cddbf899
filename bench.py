"""bench.py -- throughput of the QMC hot path on B200 (BASELINE.json metric: integrand evaluations/s, FP64).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload c2|c1|c3|c4lite] [--impl reference]

A *step* is one pass of the whole hot path over one batch of synthetic
sectors: one C-ABI call (qmc_median_integrate_sectors for the median-rule config C2, else
qmc_integrate_sectors) = lattice points, transform, integrand, per-shift reduction, (median selection,)
mean / error and the amplitude sum.  The default workload is BASELINE.json configs[2] at its largest lattice,
n = 100 000 007 (64 dim-6 Euclidean sectors, K = 11 candidates + m = 32 shifts: 2.75e11 evaluations per step,
~2.9 s), the config the north_star's 50 %-of-FP64-peak target names; DESIGN.md section 7 says why not configs[1].
The same line carries configs[1], [3] and [4] (C4-lite; the full C4 with --c4-full) as first-class records under
"also", each with its own steps, clock sample and roofline fraction.

Prints ONE JSON line (rank 0).  `value` is timed with CUDA events on the launching stream around each
step (an L2 flush between steps, outside the events); `e2e` times the same call from host buffers
including the device->host read of the results; `roofline` is the evaluation kernels' algorithmic FP64
flop rate against the FP64 FMA peak measured in the same process; `cpu_baseline` is the oracle as it
stands on one host core over a bounded sample.  N > 1: one process per GPU (torchrun), every rank runs
its own independently seeded batch (sectors are independent problems: no data-path collective), time =
max over ranks, value = total evaluations / that time ("weak").  Run directly as `python bench.py --gpus N` with
N > 1 it starts its own N ranks (re-executes itself under torch.distributed.run) and fails loudly if fewer than N
devices are visible; `n_gpus` in the line is always the number of ranks that ran.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

from paper_2305_19768_b200 import ranks as R, workloads as W  # noqa: E402

METRIC = "integrand evaluations/sec (FP64)"
UNIT = "evaluations/s"
# nominal FP64 FMA peak of a B200: 148 SMs x 64 FP64 lanes x 2 flop x 1.965 GHz
NOMINAL_FP64_FLOPS = 148 * 64 * 2 * 1.965e9


def make_workload(name: str, n, rank: int):
    """The synthetic stand-in for the paper's benchmark integrals."""
    cid = {"c0": 0, "c1": 1, "c2": 2, "c3": 3, "c4lite": 4, "c4full": 4}.get(name)
    if cid is None:
        raise SystemExit("unknown workload %r" % name)
    seed = R.rank_seed(rank, cid)
    if name == "c2":
        wl = W.config_median(n=int(n or 100_000_007), seed=seed)
    elif name == "c1":
        wl = W.config_euclid(n=n, seed=seed)
    elif name == "c3":
        wl = W.config_physical(n=int(n or 9_999_991), seed=seed)
    elif name == "c4lite":
        wl = W.config_batch(scale=1.0 / 28.0, seed=seed)
    elif name == "c4full":
        wl = W.config_batch(scale=1.0, seed=seed)
    elif name == "c0":
        wl = W.config_toy()
    else:
        raise SystemExit("unknown workload %r" % name)
    return wl


def describe(name: str, wl) -> str:
    K = 0 if wl.z_cand is None else wl.z_cand.shape[1]
    ns = sorted({j.n for j in wl.jobs})
    nd = ("n=%d" % ns[0]) if len(ns) == 1 else ("n=%d..%d" % (ns[0], ns[-1]))
    dims = sorted({wl.sectors[j.sector].dim for j in wl.jobs})
    return "BASELINE.json configs[%s] %s: %d sectors, dim %s, %s, m=%d%s" % (
        {"c0": 0, "c1": 1, "c2": 2, "c3": 3, "c4lite": 4, "c4full": 4}[name], wl.name, len(wl.jobs),
        "/".join(map(str, dims)), nd, wl.m, (", K=%d" % K) if K else "")


# ------------------------------------------------------------------------------- clocks
class ClockSampler:
    """Samples nvidia-smi clocks and throttle reasons while the timed region runs."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.index, self.proc, self.lines = index, None, []

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), "--query-gpu=" + self.Q,
                                          "--format=csv,noheader,nounits", "-lms", "100"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.t = threading.Thread(target=self._read, daemon=True)
            self.t.start()
        except OSError:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.lines.append(line.strip())

    def stop(self) -> dict:
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except subprocess.TimeoutExpired:
            self.proc.kill()
        sm, mx, pw, reasons = [], [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for ln in self.lines:
            f = [x.strip() for x in ln.split(",")]
            if len(f) < 7:
                continue
            try:
                sm.append(float(f[0])); mx.append(float(f[1])); pw.append(float(f[2]))
            except ValueError:
                continue
            for nm, v in zip(names, f[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(nm)
        if not sm:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["no samples"]}
        return {"sm_mhz": float(np.median(sm)), "sm_max_mhz": float(max(mx)), "power_w_max": float(max(pw)),
                "samples": len(sm), "reasons": sorted(reasons)}


# ------------------------------------------------------------------------------- oracle legs
def _oracle_timed(items, seconds: float):
    """Runs the oracle (oracle/, as it stands, one thread) over `items` = (sector, n, z, shift rows) in turn, in
    k-ranges of 200 000 points, until the list is done or `seconds` have passed.  Returns (evaluations, seconds)."""
    from oracle import oracle as O
    O.lib()
    evals, t0 = 0, time.perf_counter()
    for sector, n, z, rows in items:
        sec = O.OracleSector(sector)
        for r in range(rows.shape[0]):
            for k0 in range(0, n, 200_000):
                k1 = min(n, k0 + 200_000)
                O.shift_sums(sec, n, z, rows[r:r + 1], k0, k1)
                evals += k1 - k0
                if time.perf_counter() - t0 >= seconds:
                    return evals, time.perf_counter() - t0
    return evals, time.perf_counter() - t0


def oracle_slice(name: str, seconds: float, shifts_of=None):
    """The fixed oracle slice of a config (BASELINE.md section 3 / SURVEY.md 8(d)), cut off after `seconds`:
      c0: the whole config, repeated 5x        c1: sector 0, all 32 shifts
      c2: sector 0 at n = 1 000 003, its 11 candidates (shared shift) + 32 shifts
      c3: sector 0, 2 shifts                   c4: the three smallest-n sectors, 2 shifts each
    `shifts_of` = (index, count) restricts the slice to every count-th shift row from index (the all-cores leg).
    Returns (evaluations, seconds, description)."""
    items = []
    if name == "c0":
        wl = W.config_toy()
        j = wl.jobs[0]
        items = [(wl.sectors[0], j.n, j.z, wl.shifts)] * 5
        what = "C0 whole config x5"
    elif name == "c1":
        wl = W.config_euclid()
        j = wl.jobs[0]
        items = [(wl.sectors[0], j.n, j.z, wl.shifts[:wl.m])]
        what = "C1 sector 0, 32 shifts, n=%d" % j.n
    elif name == "c2":
        wl = W.config_median(n_sectors=1, n=1_000_003)
        j = wl.jobs[0]
        items = [(wl.sectors[0], j.n, wl.z_cand[0, c], wl.shift0[0:1]) for c in range(wl.z_cand.shape[1])]
        items.append((wl.sectors[0], j.n, wl.z_cand[0, 0], wl.shifts[:wl.m]))
        what = "C2 sector 0 at n=1000003, 11 candidates + 32 shifts"
    elif name == "c3":
        wl = W.config_physical(n_sectors=1)
        j = wl.jobs[0]
        items = [(wl.sectors[0], j.n, j.z, wl.shifts[:2])]
        what = "C3 sector 0 (deformed, J=3), 2 shifts, n=%d" % j.n
    elif name in ("c4lite", "c4full"):
        wl = W.config_batch(scale=1.0 / 28.0 if name == "c4lite" else 1.0)
        order = sorted(range(len(wl.jobs)), key=lambda i: wl.jobs[i].n)[:3]
        items = [(wl.sectors[wl.jobs[i].sector], wl.jobs[i].n, wl.jobs[i].z,
                  wl.shifts[wl.jobs[i].shift_offset:wl.jobs[i].shift_offset + 2]) for i in order]
        what = "C4 the three smallest-n sectors (n=%s), 2 shifts each" % ",".join(str(wl.jobs[i].n) for i in order)
    else:
        raise SystemExit("no oracle slice for %r" % name)
    if shifts_of is not None:
        idx, cnt = shifts_of
        items = [(s, n, z, rows[idx::cnt]) for s, n, z, rows in items if rows[idx::cnt].shape[0]]
        what += " (every %d-th shift row from %d)" % (cnt, idx)
    planned = sum(n * rows.shape[0] for _, n, _, rows in items)
    evals, dt = _oracle_timed(items, seconds)
    if evals < planned:
        what += "; cut off after %.0f s: %d of %d evaluations" % (seconds, evals, planned)
    return evals, dt, what


def run_reference(args):
    """--impl reference: the oracle on the host cores, same metric / config; each step a bounded sample (the
    config's fixed slice, cut off after a few seconds)."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    wl = make_workload(args.workload, args.n, 0)
    per_step = max(0.5, min(5.0, 60.0 / max(1, args.steps + args.warmup)))
    for _ in range(args.warmup):
        oracle_slice(args.workload, per_step)
    evals = secs = 0.0
    sample = ""
    for _ in range(args.steps):
        e, dt, sample = oracle_slice(args.workload, per_step)
        evals += e
        secs += dt
    v = evals / secs
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": v, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": 1e3 * secs / max(1, args.steps), "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": describe(args.workload, wl), "sample_per_step": sample},
        "cpu_baseline": {"value": v, "unit": UNIT, "cores": 1, "kind": "oracle", "sample": sample},
        "e2e": {"value": v, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0}))


def oracle_all_cores(workload: str, seconds: float) -> dict:
    """the same slice as N independent single-threaded processes, N = the host's core count,
    each taking every N-th shift row; the aggregate is reported beside the single-core figure (context only)."""
    n_proc = os.cpu_count() or 1
    code = ("import sys, json; sys.path.insert(0, %r)\n"
            "import bench\n"
            "e, dt, _ = bench.oracle_slice(%r, %r, shifts_of=(int(sys.argv[1]), %d))\n"
            "print(json.dumps([e, dt]))\n" % (ROOT, workload, seconds, n_proc))
    procs = [subprocess.Popen([sys.executable, "-c", code, str(i)], stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
             for i in range(n_proc)]
    total = 0.0
    ok = 0
    for p in procs:
        out, _ = p.communicate(timeout=seconds * 6 + 120)
        try:
            e, dt = json.loads(out.strip().splitlines()[-1])
            if e > 0:
                total += e / dt
                ok += 1
        except Exception:
            pass
    return {"value": total, "unit": UNIT, "cores": ok, "kind": "oracle, one process per core, one shift row each"}


# ------------------------------------------------------------------------------- GPU leg
# DRAM traffic of ONE evaluation-kernel launch from the committed `ncu --set full` captures (static: NOT re-measured
# by this run; reported only when the run's configuration is the captured one).  dram__bytes_read.sum +
# dram__bytes_write.sum; the algorithmic bytes are ~0 (job table in, per-tile sums out).
STATIC_FROM_PROFILE = {
    ("c2", 100_000_007): {"traffic": 535808, "fp64_pipe_active": 0.784, "measured_tflops": 23.61, "measured_frac_of_peak": 0.656,
                          "launch": "one candidate-stage module launch (16 sectors x 11 vectors), 173.6 ms",
                          "profile": "profiles/r02_final.md", "captured_at_commit": "554efd1"},
    ("c3", 9_999_991): {"traffic": 409856 + 1140736, "fp64_pipe_active": 0.741, "measured_tflops": 22.13, "measured_frac_of_peak": 0.615,
                        "launch": "one module launch (7 sectors x 32 shifts), 89.1 ms",
                        "profile": "profiles/r02_final.md", "captured_at_commit": "554efd1"},
}


def measure_also(name: str, fp64_peak: float, steps: int, warmup: int, local: int) -> dict:
    """The same device-timed measurement on another BASELINE.json config (rank 0 of a 1-GPU run only): its own
    steps, clock sample and roofline fraction, reported under "also"."""
    import torch
    from paper_2305_19768_b200 import binding as B
    wl = make_workload(name, None, 0)
    t0 = time.perf_counter()
    plan = B.qmc_plan(wl.sectors)
    plan_s = time.perf_counter() - t0
    plan.bind_workspace(len(wl.jobs), wl.shifts.shape[0] + len(wl.jobs))
    out = B.alloc_outputs(plan, len(wl.jobs), wl.m)
    jobs_c = B.marshal_jobs(wl.jobs)
    stream = torch.cuda.current_stream()
    flush = torch.empty(512 << 20, dtype=torch.uint8, device="cuda")
    for _ in range(warmup):
        B.qmc_integrate_sectors(plan, jobs_c, wl.shifts, wl.m, out, stream)
    torch.cuda.synchronize()
    # a short workload (C1: 2 ms per step) gets enough steps for ~1.5 s, so that nvidia-smi (100 ms period) sees it
    t0 = time.perf_counter()
    B.qmc_integrate_sectors(plan, jobs_c, wl.shifts, wl.m, out, stream)
    torch.cuda.synchronize()
    steps = max(steps, min(2000, int(1.5 / max(time.perf_counter() - t0, 1e-4))))
    sampler = ClockSampler(local)
    sampler.start()
    dev_ms = eval_ms = 0.0
    launches = 0
    for _ in range(steps):
        flush.fill_(1)
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record(stream)
        B.qmc_integrate_sectors(plan, jobs_c, wl.shifts, wl.m, out, stream)
        b.record(stream)
        b.synchronize()
        dev_ms += a.elapsed_time(b)
        eval_ms += plan.last_eval_ms()
        launches += plan.last_stats()["kernel_launches"]
    clocks = sampler.stop()
    evals = wl.evaluations()
    flops = sum(plan.sector_emitted_flops(j.sector) * j.n * wl.m for j in wl.jobs)
    ops = sum(plan.sector_ops(j.sector) * j.n * wl.m for j in wl.jobs)
    amp = out["amplitude"].cpu().numpy()
    res = {"workload": describe(name, wl), "value": evals * steps / (dev_ms * 1e-3), "unit": UNIT, "steps": steps,
           "warmup": warmup, "ms_per_step": dev_ms / steps, "evaluations_per_step": evals,
           "kernel_ms_per_step": eval_ms / steps, "gpu_launches": launches, "plan_seconds_nvrtc": plan_s,
           "flops_per_eval": flops / evals,
           "roofline_frac": flops * steps / (eval_ms * 1e-3) / fp64_peak,
           "fp64_issue_frac": (ops * steps / (eval_ms * 1e-3)) / (fp64_peak / 2.0),
           "clocks": clocks, "check_amplitude0": [float(x) for x in amp[0]],
           "static_from_profile": STATIC_FROM_PROFILE.get((name, wl.jobs[0].n))}
    plan.destroy()
    return res


def spawn_ranks(args) -> int:
    """`python bench.py --gpus N` with N > 1 and no torchrun environment: start N ranks ourselves."""
    import socket
    import torch
    have = torch.cuda.device_count()
    if have < args.gpus:
        raise SystemExit("bench.py --gpus %d: only %d CUDA device(s) visible" % (args.gpus, have))
    with socket.socket() as sk:
        sk.bind(("127.0.0.1", 0))
        port = sk.getsockname()[1]
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", str(args.gpus),
           "--master-addr", "127.0.0.1", "--master-port", str(port), os.path.abspath(__file__)] + sys.argv[1:]
    return subprocess.call(cmd)


def run_gpu(args):
    import torch
    from paper_2305_19768_b200 import binding as B

    rank, world, local = R.env_rank()
    if world != args.gpus:
        raise SystemExit("bench.py: --gpus %d but WORLD_SIZE is %d; launch with --nproc-per-node %d or run "
                         "`python bench.py --gpus %d` directly" % (args.gpus, world, args.gpus, args.gpus))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the product has no CPU fallback")
    if torch.cuda.device_count() <= local:
        raise SystemExit("bench.py: rank %d needs device %d, only %d visible" % (rank, local, torch.cuda.device_count()))
    torch.cuda.set_device(local)
    dev = "cuda:%d" % local
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device(dev))
    B.lib()

    strong = args.scaling == "strong"
    wl = make_workload(args.workload, args.n, 0 if strong else rank)
    median = wl.z_cand is not None
    K = wl.z_cand.shape[1] if median else 0
    presampled = None
    if args.presample > 0:
        # deformation-parameter presampling (qmc_presample_lambda) BEFORE the plan: lambda is compiled in
        t0 = time.perf_counter()
        infos = [i for i in B.presample_sectors(wl.sectors, n_pre=args.presample, min_abs_f=args.min_abs_f, device=dev) if i is not None]
        presampled = {"n_pre": args.presample, "min_abs_f": args.min_abs_f, "sectors": len(infos), "seconds": time.perf_counter() - t0,
                      "all_ok": all(i["ok"] for i in infos),
                      "lambda_min_median_max": [float(x) for x in np.percentile([i["lam"] for i in infos], [0, 50, 100])] if infos else None}
    t0 = time.perf_counter()
    plan = B.qmc_plan(wl.sectors, **({"wide_lattice": 1} if args.wide else {}))
    plan_s = time.perf_counter() - t0
    pieces = None
    if strong:
        # ONE batch for the whole job: whole jobs by LPT, a job above the mean load cut by shift, then
        # by k-range (ranks.split_partition; cost = emitted FP64 ops x points).  Every rank holds the plan of all
        # sectors and the whole job table; it evaluates its pieces, the per-shift (hi, lo) sums of all ranks meet in
        # ONE all-gather (NCCL), and every rank finalizes.
        pieces = R.split_partition([plan.sector_ops(j.sector) for j in wl.jobs], [j.n for j in wl.jobs], wl.m, world)[rank]
    cand_jobs = cand_c = cand_pieces = cand_partial = None
    if strong and median:
        # the median rule shards the same way: n_jobs x K one-shift candidate jobs (shift rows = wl.shift0), their sums
        # all-gathered, qmc_median_select_pieces on every rank, then the m-shift stage on the selected vectors
        cand_jobs = R.candidate_jobs(wl.jobs, wl.z_cand)
        cand_c = B.marshal_jobs(cand_jobs)
        cand_pieces = R.split_partition([plan.sector_ops(j.sector) for j in cand_jobs], [j.n for j in cand_jobs], 1, world)[rank]
        cand_partial = torch.zeros((len(cand_jobs), 1, plan.J, 3, 2), dtype=torch.float64, device=dev)
    max_jobs = max(len(wl.jobs) * (K + 1), len(pieces or []), len(cand_pieces or [])) + 8
    plan.bind_workspace(max_jobs, wl.shifts.shape[0] + len(wl.jobs), device=dev)
    out = B.alloc_outputs(plan, len(wl.jobs), wl.m, K=K, device=dev)
    jobs_c = B.marshal_jobs(wl.jobs)
    if strong:
        my = {}
        for job, s0, s1, k0, k1 in pieces:
            my[job] = my.get(job, 0) + (s1 - s0) * (k1 - k0)
        for cj, s0, s1, k0, k1 in (cand_pieces or []):
            my[cj // K] = my.get(cj // K, 0) + (k1 - k0)
        evals_step = sum(my.values())
        flops_step = sum(plan.sector_emitted_flops(wl.jobs[j].sector) * e for j, e in my.items())
        model_flops_step = sum(plan.sector_flops(wl.jobs[j].sector) * e for j, e in my.items())
        ops_step = sum(plan.sector_ops(wl.jobs[j].sector) * e for j, e in my.items())
        partial = torch.zeros((len(wl.jobs), wl.m, plan.J, 3, 2), dtype=torch.float64, device=dev)
    else:
        evals_step = wl.evaluations()
        flops_step = sum(plan.sector_emitted_flops(j.sector) * j.n * (wl.m + K) for j in wl.jobs)
        model_flops_step = sum(plan.sector_flops(j.sector) * j.n * (wl.m + K) for j in wl.jobs)
        ops_step = sum(plan.sector_ops(j.sector) * j.n * (wl.m + K) for j in wl.jobs)
    stream = torch.cuda.current_stream()

    def step():
        """One pass; returns the evaluation-kernel time of calls whose events a later call of the step overwrites."""
        extra_ms, extra_launches = 0.0, 0
        if strong and median:
            B.qmc_integrate_pieces(plan, cand_c, cand_pieces, wl.shift0, 1, cand_partial, None, stream)
            B.qmc_median_select_pieces(plan, cand_c, K, R.gather_parts(cand_partial, world), world, out, stream)
            sel = out["selected"].cpu().numpy()          # the selected vectors enter the next job table on the host
            extra_ms, extra_launches = plan.last_eval_ms(), plan.last_stats()["kernel_launches"] + 2
            sel_jobs = B.marshal_jobs(R.selected_jobs(wl.jobs, wl.z_cand, sel))
            B.qmc_integrate_pieces(plan, sel_jobs, pieces, wl.shifts, wl.m, partial, out["diag"], stream)
            B.qmc_finalize_pieces(plan, sel_jobs, wl.m, R.gather_parts(partial, world), world, out, stream)
        elif strong:
            B.qmc_integrate_pieces(plan, jobs_c, pieces, wl.shifts, wl.m, partial, out["diag"], stream)
            parts = R.gather_parts(partial, world)       # the path's one exchange step
            B.qmc_finalize_pieces(plan, jobs_c, wl.m, parts, world, out, stream)
        elif median:
            B.qmc_median_integrate_sectors(plan, jobs_c, wl.z_cand, wl.shift0, wl.shifts, wl.m, out, stream)
        else:
            B.qmc_integrate_sectors(plan, jobs_c, wl.shifts, wl.m, out, stream)
        return extra_ms, extra_launches

    # host buffers the e2e leg reads the results into (pinned)
    res_names = ["job_results", "amplitude", "shift_sums"] + (["cand_est", "median", "selected"] if median else [])
    host = {k: torch.empty(out[k].shape, dtype=out[k].dtype, pin_memory=True) for k in res_names}
    d2h_bytes = sum(h.numel() * h.element_size() for h in host.values())
    h2d_bytes = (len(wl.jobs) * (80 + 16 + 16 + 8 * 4 * max(1, K)) + (wl.shifts.shape[0] + len(wl.jobs)) * 64)

    flush = torch.empty(512 << 20, dtype=torch.uint8, device=dev)   # > 126 MB L2

    def barrier():
        if world > 1:
            import torch.distributed as dist
            dist.barrier()
        torch.cuda.synchronize()

    fp64_peak = B.qmc_measure_fp64_peak(300.0)    # also warms the clocks up
    fp64_peak_mixed = B.qmc_measure_fp64_peak_mixed(200.0)

    for _ in range(args.warmup):
        step()
    torch.cuda.synchronize()

    # ---- device-timed steps ---------------------------------------------------------------
    sampler = ClockSampler(local)
    if rank == 0:
        sampler.start()
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(args.steps)]
    eval_ms, launches = 0.0, 0
    barrier()
    for a, b in ev:
        flush.fill_(1)
        a.record(stream)
        extra_ms, extra_launches = step()
        b.record(stream)
        b.synchronize()
        eval_ms += plan.last_eval_ms() + extra_ms    # the library's own events around its evaluation kernels
        st = plan.last_stats()
        launches += st["kernel_launches"] + (2 if strong else 0) + extra_launches   # + finalize_parts and amplitude of the strong path
    barrier()
    dev_ms = sum(a.elapsed_time(b) for a, b in ev)

    # ---- end to end: host buffers in, results back on the host, every step -------------------
    e2e_steps = max(1, min(args.steps, args.e2e_steps))
    barrier()
    t0 = time.perf_counter()
    for _ in range(e2e_steps):
        step()
        for k in res_names:
            host[k].copy_(out[k], non_blocking=True)
        torch.cuda.synchronize()
    e2e_s = time.perf_counter() - t0
    barrier()
    clocks = sampler.stop() if rank == 0 else None

    (dev_ms, e2e_s, eval_ms), (evals_all, launches_all) = R.aggregate(
        [dev_ms, e2e_s, eval_ms], [float(evals_step), float(launches)], world, device=dev)
    launches_all = int(launches_all)

    if rank == 0:
        value = R.throughput(evals_all, args.steps, dev_ms)
        achieved = flops_step * args.steps / (eval_ms * 1e-3)
        mean0 = host["job_results"][0, 0].tolist()
        n0 = wl.jobs[0].n
        static = STATIC_FROM_PROFILE.get((args.workload, n0)) if not args.wide and world == 1 else None
        line = {
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
            "ms_per_step": dev_ms / args.steps, "higher_is_better": True, "scaling": "strong" if strong else "weak",
            "vs_baseline": None,
            "dtype": "f64", "data": "synthetic",
            "config": {"workload": describe(args.workload, wl), "evaluations_per_step_per_gpu": evals_step,
                       "timing": "CUDA events per step on the launching stream; 512 MiB L2 flush between steps; "
                                 "the call's own job-table upload (%d B) is inside the events" % h2d_bytes,
                       "plan_seconds_nvrtc": plan_s, "modules": plan.modules(), "wide_lattice": bool(args.wide),
                       "check_job0": mean0, "check_amplitude": host["amplitude"].tolist(),
                       "sign_check_failures": int(out["diag"][:, 1].sum().item()), "presampled": presampled},
            "e2e": {"value": evals_all * e2e_steps / e2e_s, "unit": UNIT, "h2d_bytes_per_step": h2d_bytes,
                    "d2h_bytes_per_step": d2h_bytes, "steps": e2e_steps},
            "gpu_launches": launches_all,
            "clocks": clocks,
            "roofline": {"bound": "alu", "achieved": achieved / 1e12, "peak": fp64_peak / 1e12, "unit": "TFLOP/s",
                         "frac": achieved / fp64_peak,
                         "traffic": static["traffic"] if static else None,
                         "peak_kind": "FP64 FMA rate measured in this process (qmc_measure_fp64_peak); nominal %.1f"
                                      % (NOMINAL_FP64_FLOPS / 1e12),
                         # the FMA rate with one integer instruction interleaved per FMA (measured here too; within
                         # 1 % of the pure rate: integer work beside the FP64 pipe is free in a regular stream)
                         "peak_mixed": fp64_peak_mixed / 1e12, "frac_of_peak_mixed": achieved / fp64_peak_mixed,
                         "kernel": "qmc_eval_kernel (all module launches of a step)",
                         "kernel_ms_per_step": eval_ms / args.steps,
                         "flops_per_eval": flops_step / evals_step,
                         "flops_kind": "FP64 flops of the generated code per evaluation (fma = 2): the quantity ncu measures "
                                       "as 2 DFMA + DMUL + DADD; SURVEY.md 8(d)'s monomial-by-monomial model is given beside it",
                         "survey_model_flops_per_eval": model_flops_step / evals_step,
                         "survey_model_frac": model_flops_step * args.steps / (eval_ms * 1e-3) / fp64_peak,
                         "emitted_fp64_ops_per_eval": ops_step / evals_step,
                         "fp64_issue_frac": (ops_step * args.steps / (eval_ms * 1e-3)) / (fp64_peak / 2.0),
                         # figures of the committed ncu capture of this kernel: static, not re-measured by this run
                         "static_from_profile": static},
        }
        if world == 1 and args.workload == "c2" and args.n is None and not args.no_also:
            k = max(1, args.steps)
            line["also"] = {"c1": measure_also("c1", fp64_peak, max(10, k), 3, local),
                            "c3": measure_also("c3", fp64_peak, max(10, min(k, 20)), 3, local),
                            "c4lite": measure_also("c4lite", fp64_peak, max(3, min(k, 5)), 2, local)}
            if args.c4_full:
                line["also"]["c4full"] = measure_also("c4full", fp64_peak, 1, 0, local)
        if world == 1 and not args.no_cpu_baseline:
            slice_name = args.workload
            e, dt, sample = oracle_slice(slice_name, args.cpu_seconds)
            line["cpu_baseline"] = {"value": e / dt, "unit": UNIT, "cores": 1, "kind": "oracle", "sample": sample}
            if not args.no_also:
                line["cpu_baseline"]["all_cores"] = oracle_all_cores(slice_name, min(8.0, args.cpu_seconds))
                line["cpu_baseline"]["other_slices"] = {}
                for w in ("c0", "c1", "c3", "c4lite"):
                    if w != slice_name:
                        e, dt, sample = oracle_slice(w, 4.0)
                        line["cpu_baseline"]["other_slices"][w] = {"value": e / dt, "unit": UNIT, "cores": 1, "sample": sample}
        print(json.dumps(line))
    plan.destroy()
    if world > 1:
        import torch.distributed as dist
        dist.destroy_process_group()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="c2", choices=["c0", "c1", "c2", "c3", "c4lite", "c4full"])
    ap.add_argument("--n", type=int, default=None, help="lattice size override (c1, c2, c3)")
    ap.add_argument("--cpu-seconds", type=float, default=16.0)
    ap.add_argument("--e2e-steps", type=int, default=5, help="steps of the end-to-end leg (at most --steps)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-also", action="store_true", help="skip the extra C1 / C3 / C4-lite measurements of the default run")
    ap.add_argument("--c4-full", action="store_true",
                    help="also time ONE step of the full C4 batch (2.9e12 evaluations, ~90 s + ~20 s of NVRTC)")
    ap.add_argument("--presample", type=int, default=0, metavar="N_PRE",
                    help="presample the deformation parameter of every deformed sector on N_PRE points before planning")
    ap.add_argument("--min-abs-f", type=float, default=0.0, help="with --presample: smallest |F(z)| a lambda may reach on the presamples")
    ap.add_argument("--scaling", default="weak", choices=["weak", "strong"],
                    help="N > 1: weak = one batch per rank (default); strong = one batch LPT-sharded over the ranks")
    ap.add_argument("--wide", action="store_true", help="compile the plan with 64-bit lattice indices (n up to 2^53)")
    args = ap.parse_args()
    if args.gpus < 1:
        raise SystemExit("--gpus must be >= 1")
    if args.impl == "reference":
        run_reference(args)
    elif args.gpus > 1 and "WORLD_SIZE" not in os.environ:
        sys.exit(spawn_ranks(args))
    else:
        run_gpu(args)


if __name__ == "__main__":
    main()
