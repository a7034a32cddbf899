"""bench.py -- throughput of the QMC hot path on B200 (BASELINE.json metric: integrand evaluations/s, FP64).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload c2|c1|c3|c4lite] [--impl reference]

A *step* is one pass of the whole hot path over one batch of synthetic
sectors: one C-ABI call (qmc_median_integrate_sectors for the median-rule config C2, else
qmc_integrate_sectors) = lattice points, transform, integrand, per-shift reduction, (median selection,)
mean / error and the amplitude sum.  The default workload is BASELINE.json configs[2] at n = 9 999 991
(64 dim-6 Euclidean sectors, K = 11 candidates + m = 32 shifts: 2.75e10 evaluations per step), the config
the north_star's 50 %-of-FP64-peak target names; DESIGN.md section 7 says why not configs[1].

Prints ONE JSON line (rank 0).  `value` is timed with CUDA events on the launching stream around each
step (an L2 flush between steps, outside the events); `e2e` times the same call from host buffers
including the device->host read of the results; `roofline` is the evaluation kernels' algorithmic FP64
flop rate against the FP64 FMA peak measured in the same process; `cpu_baseline` is the oracle as it
stands on one host core over a bounded sample.  N > 1: one process per GPU (torchrun), every rank runs
its own independently seeded batch (sectors are independent problems: no data-path collective), time =
max over ranks, value = total evaluations / that time ("weak").
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
    cid = {"c0": 0, "c1": 1, "c2": 2, "c3": 3, "c4lite": 4}.get(name)
    if cid is None:
        raise SystemExit("unknown workload %r" % name)
    seed = R.rank_seed(rank, cid)
    if name == "c2":
        wl = W.config_median(n=int(n or 9_999_991), seed=seed)
    elif name == "c1":
        wl = W.config_euclid(n=n, seed=seed)
    elif name == "c3":
        wl = W.config_physical(n=int(n or 9_999_991), seed=seed)
    elif name == "c4lite":
        wl = W.config_batch(scale=1.0 / 28.0, seed=seed)
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
        {"c0": 0, "c1": 1, "c2": 2, "c3": 3, "c4lite": 4}[name], wl.name, len(wl.jobs),
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
def oracle_sample(wl, seconds: float):
    """Times the CPU oracle (oracle/, as it stands, one thread) on a bounded sample of the workload:
    job 0, shift 0, consecutive k-ranges of the full lattice until `seconds` have passed."""
    from oracle import oracle as O
    O.lib()
    job = wl.jobs[0]
    sec = O.OracleSector(wl.sectors[job.sector])
    z = job.z if wl.z_cand is None else wl.z_cand[0, 0]
    sh = wl.shifts[job.shift_offset:job.shift_offset + 1]
    chunk, k0, evals = 200_000, 0, 0
    t0 = time.perf_counter()
    while True:
        k1 = min(job.n, k0 + chunk)
        O.shift_sums(sec, job.n, z, sh, k0, k1)
        evals += k1 - k0
        k0 = 0 if k1 >= job.n else k1
        dt = time.perf_counter() - t0
        if dt >= seconds:
            break
    return evals, dt, "job 0 (dim %d, %s), shift 0, %d lattice points of n=%d in k order" % (
        sec.dim, "deformed J=%d" % sec.J if wl.sectors[job.sector].deformed else "real", evals, job.n)


def run_reference(args):
    """--impl reference: the oracle on the host cores, same metric / config; each step a bounded sample."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    wl = make_workload(args.workload, args.n, 0)
    per_step = max(0.5, min(5.0, 60.0 / max(1, args.steps + args.warmup)))
    for _ in range(args.warmup):
        oracle_sample(wl, per_step)
    evals = secs = 0.0
    sample = ""
    for _ in range(args.steps):
        e, dt, sample = oracle_sample(wl, per_step)
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


def oracle_all_cores(workload: str, n, seconds: float) -> dict:
    """the same oracle sample run as N independent single-threaded processes, N = the host's
    core count; the aggregate is reported beside the single-core figure (context only)."""
    n_proc = os.cpu_count() or 1
    code = ("import sys, json; sys.path.insert(0, %r)\n"
            "import bench\n"
            "wl = bench.make_workload(%r, %r, 0)\n"
            "e, dt, _ = bench.oracle_sample(wl, %r)\n"
            "print(json.dumps([e, dt]))\n" % (ROOT, workload, n, seconds))
    procs = [subprocess.Popen([sys.executable, "-c", code], stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
             for _ in range(n_proc)]
    total = 0.0
    ok = 0
    for p in procs:
        out, _ = p.communicate(timeout=seconds * 6 + 120)
        try:
            e, dt = json.loads(out.strip().splitlines()[-1])
            total += e / dt
            ok += 1
        except Exception:
            pass
    return {"value": total, "unit": UNIT, "cores": ok, "kind": "oracle, one process per core"}


# ------------------------------------------------------------------------------- GPU leg
def measure_also(name: str, fp64_peak: float, steps: int = 3, warmup: int = 3) -> dict:
    """The same device-timed measurement on another BASELINE.json config (rank 0 of a 1-GPU run only), reported
    under "also" so that one bench line carries configs[1], [2] and [3]."""
    import torch
    from paper_2305_19768_b200 import binding as B
    wl = make_workload(name, None, 0)
    plan = B.qmc_plan(wl.sectors)
    plan.bind_workspace(len(wl.jobs), wl.shifts.shape[0] + len(wl.jobs))
    out = B.alloc_outputs(plan, len(wl.jobs), wl.m)
    jobs_c = B.marshal_jobs(wl.jobs)
    stream = torch.cuda.current_stream()
    flush = torch.empty(512 << 20, dtype=torch.uint8, device="cuda")
    for _ in range(warmup):
        B.qmc_integrate_sectors(plan, jobs_c, wl.shifts, wl.m, out, stream)
    torch.cuda.synchronize()
    dev_ms = eval_ms = 0.0
    for _ in range(steps):
        flush.fill_(1)
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record(stream)
        B.qmc_integrate_sectors(plan, jobs_c, wl.shifts, wl.m, out, stream)
        b.record(stream)
        b.synchronize()
        dev_ms += a.elapsed_time(b)
        eval_ms += plan.last_eval_ms()
    evals = wl.evaluations()
    flops = sum(plan.sector_emitted_flops(j.sector) * j.n * wl.m for j in wl.jobs)
    ops = sum(plan.sector_ops(j.sector) * j.n * wl.m for j in wl.jobs)
    res = {"workload": describe(name, wl), "value": evals * steps / (dev_ms * 1e-3), "unit": UNIT, "steps": steps,
           "ms_per_step": dev_ms / steps,
           "roofline_frac": flops * steps / (eval_ms * 1e-3) / fp64_peak,
           "fp64_issue_frac": (ops * steps / (eval_ms * 1e-3)) / (fp64_peak / 2.0)}
    plan.destroy()
    return res


def run_gpu(args):
    import torch
    from paper_2305_19768_b200 import binding as B

    rank, world, local = R.env_rank()
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the product has no CPU fallback")
    torch.cuda.set_device(local)
    dev = "cuda:%d" % local
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device(dev))
    B.lib()

    strong = args.scaling == "strong" and world > 1
    wl = make_workload(args.workload, args.n, 0 if strong else rank)
    median = wl.z_cand is not None
    K = wl.z_cand.shape[1] if median else 0
    t0 = time.perf_counter()
    plan = B.qmc_plan(wl.sectors, **({"wide_lattice": 1} if args.wide else {}))
    plan_s = time.perf_counter() - t0
    if strong:
        # ONE batch for the whole job: this rank takes its LPT share of the jobs (cost = points x emitted ops);
        # the plan holds all sectors on every rank, unused ones are never launched
        costs = [plan.sector_ops(j.sector) * j.n * (wl.m + K) for j in wl.jobs]
        wl = wl.subset(R.lpt_partition(costs, world)[rank])
    plan.bind_workspace(len(wl.jobs) * (K + 1), wl.shifts.shape[0] + len(wl.jobs), device=dev)
    out = B.alloc_outputs(plan, len(wl.jobs), wl.m, K=K, device=dev)
    jobs_c = B.marshal_jobs(wl.jobs)
    evals_step = wl.evaluations()
    flops_step = sum(plan.sector_emitted_flops(j.sector) * j.n * (wl.m + K) for j in wl.jobs)
    model_flops_step = sum(plan.sector_flops(j.sector) * j.n * (wl.m + K) for j in wl.jobs)
    ops_step = sum(plan.sector_ops(j.sector) * j.n * (wl.m + K) for j in wl.jobs)
    stream = torch.cuda.current_stream()

    def step():
        if median:
            B.qmc_median_integrate_sectors(plan, jobs_c, wl.z_cand, wl.shift0, wl.shifts, wl.m, out, stream)
        else:
            B.qmc_integrate_sectors(plan, jobs_c, wl.shifts, wl.m, out, stream)
        if strong:   # the one exchange step of a sharded batch: partial amplitudes add (4 J doubles, NCCL)
            out["amplitude"].copy_(R.combine_amplitudes(out["amplitude"], world))

    # host buffers the e2e leg reads the results into (pinned)
    res_names = ["job_results", "amplitude", "shift_sums"] + (["cand_est", "median", "selected"] if median else [])
    host = {k: torch.empty(out[k].shape, dtype=out[k].dtype, pin_memory=True) for k in res_names}
    d2h_bytes = sum(h.numel() * h.element_size() for h in host.values())
    h2d_bytes = (len(wl.jobs) * (64 + 16 + 16 + 8 * 4 * max(1, K)) + (wl.shifts.shape[0] + len(wl.jobs)) * 64)

    flush = torch.empty(512 << 20, dtype=torch.uint8, device=dev)   # > 126 MB L2

    def barrier():
        if world > 1:
            import torch.distributed as dist
            dist.barrier()
        torch.cuda.synchronize()

    fp64_peak = B.qmc_measure_fp64_peak(300.0)    # also warms the clocks up

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
        step()
        b.record(stream)
        b.synchronize()
        eval_ms += plan.last_eval_ms()           # the library's own events around its evaluation kernels
        st = plan.last_stats()
        launches += st["kernel_launches"]
    barrier()
    dev_ms = sum(a.elapsed_time(b) for a, b in ev)

    # ---- end to end: host buffers in, results back on the host, every step -------------------
    barrier()
    t0 = time.perf_counter()
    for _ in range(args.steps):
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
        line = {
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
            "ms_per_step": dev_ms / args.steps, "higher_is_better": True, "scaling": "strong" if strong else "weak",
            "vs_baseline": None,
            "dtype": "f64", "data": "synthetic",
            "config": {"workload": describe(args.workload, wl), "evaluations_per_step_per_gpu": evals_step,
                       "timing": "CUDA events per step on the launching stream; 512 MiB L2 flush between steps; "
                                 "the call's own job-table upload (%d B) is inside the events" % h2d_bytes,
                       "plan_seconds_nvrtc": plan_s, "modules": plan.modules(), "wide_lattice": bool(args.wide),
                       "check_job0": mean0},
            "e2e": {"value": evals_all * args.steps / e2e_s, "unit": UNIT, "h2d_bytes_per_step": h2d_bytes,
                    "d2h_bytes_per_step": d2h_bytes},
            "gpu_launches": launches_all,
            "clocks": clocks,
            "roofline": {"bound": "alu", "achieved": achieved / 1e12, "peak": fp64_peak / 1e12, "unit": "TFLOP/s",
                         "frac": achieved / fp64_peak,
                         # dram__bytes_read + write of ONE evaluation launch (16-sector C2 module, n = 1 000 003) from
                         # the ncu --set full capture in profiles/r01g_final.md; algorithmic bytes ~ 0
                         "traffic": 466176 if args.workload == "c2" else (2022144 if args.workload == "c3" else None),
                         "peak_kind": "FP64 FMA rate measured in this process (qmc_measure_fp64_peak); nominal %.1f"
                                      % (NOMINAL_FP64_FLOPS / 1e12),
                         "kernel": "qmc_eval_kernel (all module launches of a step)",
                         "kernel_ms_per_step": eval_ms / args.steps,
                         "flops_per_eval": flops_step / evals_step,
                         "flops_kind": "FP64 flops of the generated code per evaluation (fma = 2): the quantity ncu measures "
                                       "as 2 DFMA + DMUL + DADD; SURVEY.md 8(d)'s monomial-by-monomial model is given beside it",
                         "survey_model_flops_per_eval": model_flops_step / evals_step,
                         "survey_model_frac": model_flops_step * args.steps / (eval_ms * 1e-3) / fp64_peak,
                         "emitted_fp64_ops_per_eval": ops_step / evals_step,
                         "fp64_issue_frac": (ops_step * args.steps / (eval_ms * 1e-3)) / (fp64_peak / 2.0),
                         # static figures of the committed ncu capture of this kernel (not re-measured here)
                         "ncu": {"c2": {"fp64_pipe_active": 0.769, "measured_tflops": 22.55, "measured_frac_of_peak": 0.628,
                                        "profile": "profiles/r01g_final.md"},
                                 "c3": {"fp64_pipe_active": 0.736, "measured_tflops": 21.45, "measured_frac_of_peak": 0.597,
                                        "profile": "profiles/r01g_final.md"}}.get(args.workload)},
        }
        if world == 1 and args.workload == "c2" and args.n is None and not args.no_also:
            line["also"] = {w: measure_also(w, fp64_peak) for w in ("c1", "c3")}
        if world == 1 and not args.no_cpu_baseline:
            e, dt, sample = oracle_sample(wl, args.cpu_seconds)
            line["cpu_baseline"] = {"value": e / dt, "unit": UNIT, "cores": 1, "kind": "oracle", "sample": sample}
            if not args.no_also:
                line["cpu_baseline"]["all_cores"] = oracle_all_cores(args.workload, args.n, min(6.0, args.cpu_seconds))
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
    ap.add_argument("--workload", default="c2", choices=["c0", "c1", "c2", "c3", "c4lite"])
    ap.add_argument("--n", type=int, default=None, help="lattice size override (c1, c2, c3)")
    ap.add_argument("--cpu-seconds", type=float, default=12.0)
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-also", action="store_true", help="skip the extra C1 / C3 measurements of the default run")
    ap.add_argument("--scaling", default="weak", choices=["weak", "strong"],
                    help="N > 1: weak = one batch per rank (default); strong = one batch LPT-sharded over the ranks")
    ap.add_argument("--wide", action="store_true", help="compile the plan with 64-bit lattice indices (n up to 2^53)")
    args = ap.parse_args()
    if args.impl == "reference":
        run_reference(args)
    else:
        run_gpu(args)


if __name__ == "__main__":
    main()
