"""Helpers shared by the GPU parity tests: run a workload through the C ABI (binding) and
through the oracle, and compare with the tolerances BASELINE.json's north_star states.

Tolerances (written out here, used by every parity test):
  * lattice integer coordinates: bit-exact;
  * per-shift sums S_{s,j} (re, im) and A_{s,j}: |gpu - cpu| <= 1e-11 * A_{s,j}  (A = sum |W g| over the points);
  * mean and error: |gpu - cpu| <= 1e-10 * max(|mean_cpu|, mean_s A_s / n)  (reading Q9);
  * diagnostics counters (zero-weight points, Im F >= 0 points): equal.
"""
from __future__ import annotations

import numpy as np

TOL_SUM = 1e-11
TOL_MEAN = 1e-10


def oracle_jobs(wl, z_override=None, jobs=None):
    """Oracle results of every job of a workload: sums[nj, m, J, 3], results[nj, J, 4], diag[nj, 2]."""
    from oracle import oracle as O
    idx = range(len(wl.jobs)) if jobs is None else jobs
    secs = {}
    sums_all, res_all, diag_all = [], [], []
    for i in idx:
        job = wl.jobs[i]
        sec = secs.setdefault(job.sector, O.OracleSector(wl.sectors[job.sector]))
        z = job.z if z_override is None else z_override[i]
        sh = wl.shifts[job.shift_offset:job.shift_offset + wl.m]
        sums, res, diag = O.integrate(sec, job.n, z, sh)
        sums_all.append(sums)
        res_all.append(res)
        diag_all.append(diag)
    return sums_all, res_all, diag_all


def pad_orders(a, J, axis):
    """Oracle arrays have the sector's own J; the library pads to the plan's J_out with zeros."""
    a = np.asarray(a)
    if a.shape[axis] == J:
        return a
    pad = [(0, 0)] * a.ndim
    pad[axis] = (0, J - a.shape[axis])
    return np.pad(a, pad)


def assert_sums_close(gpu_sums, cpu_sums, what=""):
    """gpu/cpu: [m, J, 3] (Re S, Im S, A)."""
    gpu_sums, cpu_sums = np.asarray(gpu_sums), np.asarray(cpu_sums)
    J = cpu_sums.shape[1]
    g = gpu_sums[:, :J]
    scale = cpu_sums[:, :, 2:3]
    err = np.abs(g - cpu_sums)
    bound = TOL_SUM * scale
    bad = err > bound
    assert not bad.any(), "%s per-shift sums differ: max |d|/A = %.3e (tol %.1e)" % (
        what, float(np.max(err / np.maximum(scale, 1e-300))), TOL_SUM)
    assert np.all(gpu_sums[:, J:] == 0.0), what + " unused order slots must be zero"
    return float(np.max(err / np.maximum(scale, 1e-300)))


def assert_result_close(gpu_res, cpu_res, cpu_sums, n, what=""):
    """gpu/cpu: [J, 4] (mean_re, mean_im, err_re, err_im)."""
    gpu_res, cpu_res, cpu_sums = np.asarray(gpu_res), np.asarray(cpu_res), np.asarray(cpu_sums)
    J = cpu_res.shape[0]
    worst = 0.0
    for j in range(J):
        abar = float(np.mean(cpu_sums[:, j, 2])) / float(n)
        scale = max(abs(complex(cpu_res[j, 0], cpu_res[j, 1])), abar)
        d = np.abs(gpu_res[j] - cpu_res[j])
        assert np.all(d <= TOL_MEAN * scale), "%s order %d mean/err differ: %s vs %s (scale %.3e)" % (
            what, j, gpu_res[j], cpu_res[j], scale)
        worst = max(worst, float(np.max(d)) / max(scale, 1e-300))
    assert np.all(gpu_res[J:] == 0.0)
    return worst


def run_gpu(wl, plan=None, jobs=None, median=False, **plan_opts):
    """One qmc_integrate_sectors / qmc_median_integrate_sectors call; returns numpy outputs."""
    import torch
    from paper_2305_19768_b200 import binding as B
    own = plan is None
    if own:
        plan = B.qmc_plan(wl.sectors, **plan_opts)
    sel = list(range(len(wl.jobs))) if jobs is None else list(jobs)
    jl = [wl.jobs[i] for i in sel]
    K = wl.z_cand.shape[1] if median else 0
    plan.bind_workspace(max(1, len(jl) * max(1, K + 1)), wl.shifts.shape[0] + len(jl))
    out = B.alloc_outputs(plan, len(jl), wl.m, K=K)
    if median:
        B.qmc_median_integrate_sectors(plan, jl, wl.z_cand[sel], wl.shift0[sel], wl.shifts, wl.m, out)
    else:
        B.qmc_integrate_sectors(plan, jl, wl.shifts, wl.m, out)
    torch.cuda.synchronize()
    res = {k: (v.cpu().numpy() if v is not None else None) for k, v in out.items()}
    res["stats"] = plan.last_stats()
    res["rare"] = plan.slow_path_counts()
    res["J"] = plan.J
    if own:
        plan.destroy()
    return res


def compare_workload(wl, gpu, jobs=None, z_override=None):
    """Element-by-element comparison of every job of a GPU run with the oracle."""
    from oracle import oracle as O
    sel = list(range(len(wl.jobs))) if jobs is None else list(jobs)
    sums, res, diag = oracle_jobs(wl, z_override=z_override, jobs=sel)
    worst_s = worst_r = 0.0
    for pos, i in enumerate(sel):
        tag = "%s job %d" % (wl.name, i)
        worst_s = max(worst_s, assert_sums_close(gpu["shift_sums"][pos], sums[pos], tag))
        worst_r = max(worst_r, assert_result_close(gpu["job_results"][pos], res[pos], sums[pos], wl.jobs[i].n, tag))
        if gpu.get("diag") is not None:
            assert tuple(gpu["diag"][pos]) == tuple(diag[pos]), "%s diagnostics %s vs %s" % (tag, gpu["diag"][pos], diag[pos])
    if gpu.get("amplitude") is not None:
        J = gpu["J"]
        res_p = np.stack([pad_orders(r, J, 0) for r in res])
        coefs = np.array([wl.jobs[i].coef for i in sel])
        amp = O.amplitude(res_p, coefs)
        # tolerance: 1e-10 of the scale sum_i |C_i| max(|mean_i|, Abar_i/n)
        for j in range(J):
            scale = 0.0
            for pos, i in enumerate(sel):
                if j < res[pos].shape[0]:
                    abar = float(np.mean(sums[pos][:, j, 2])) / float(wl.jobs[i].n)
                    scale += abs(coefs[pos]) * max(abs(complex(res[pos][j, 0], res[pos][j, 1])), abar)
            d = np.abs(gpu["amplitude"][j] - amp[j])
            assert np.all(d <= TOL_MEAN * max(scale, 1e-300)), "%s amplitude order %d: %s vs %s" % (
                wl.name, j, gpu["amplitude"][j], amp[j])
    return worst_s, worst_r
