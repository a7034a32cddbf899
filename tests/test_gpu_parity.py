"""GPU parity tests: the CUDA path (through the C ABI / binding) against the CPU oracle on the
same seeded inputs, element by element.  Tolerances are those of tests/parity_util.py
(north_star: coordinates bit-exact, per-shift sums 1e-11 of sum|f|, mean/error 1e-10).
Run with ``pytest -m gpu`` on a B200.
"""
import numpy as np
import pytest

from paper_2305_19768_b200 import workloads as W
from tests import parity_util as PU

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def torch_cuda():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device; there is no CPU fallback"
    torch.cuda.set_device(0)
    return torch


@pytest.fixture(scope="module")
def B():
    from paper_2305_19768_b200 import build, binding
    build.build()            # no-op when libqmc.so is up to date; the product itself never builds or falls back
    binding.lib()
    return binding


@pytest.fixture(scope="module")
def O():
    from oracle import oracle
    oracle.lib()
    return oracle


# ------------------------------------------------------------------------------------ a1
@pytest.mark.parametrize("n", [1, 2, 3, 7, 65521, 1048573, 100000007, 1000000007, 2**32 - 5, 2**32 - 1,
                               2**32, 4294967311, 68719476767, 2**53 - 111])
def test_lattice_coords_bit_exact(torch_cuda, B, O, n):
    """(k z_i) mod n from the kernels' own device functions equals the oracle's bit for bit
    (which tests/test_oracle_pins.py pins to Python big integers)."""
    torch = torch_cuda
    rng = np.random.Generator(np.random.PCG64(1000 + n % 9973))
    dim = 8
    z = np.array([int(rng.integers(0, n)) for _ in range(dim)], np.uint64)
    if n > 2:
        z[0] = n - 1
    for k0, count in [(0, min(n, 3000)), (max(0, n - 2500), min(n, 2500)), (int(rng.integers(0, n)), 1)]:
        count = min(count, n - k0)
        out = torch.zeros((count, dim), dtype=torch.int64, device="cuda")
        B.qmc_debug_lattice_coords(n, z, dim, k0, count, out)
        torch.cuda.synchronize()
        got = out.cpu().numpy().view(np.uint64)
        want = O.lattice_coords(n, z, dim, k0, count)
        assert np.array_equal(got, want)


def test_lattice_coords_rejects_large_n(B, torch_cuda):
    out = torch_cuda.zeros((1, 1), dtype=torch_cuda.int64, device="cuda")
    with pytest.raises(B.QmcError) as e:
        B.qmc_debug_lattice_coords(2**53, [1], 1, 0, 1, out)
    assert e.value.status == B.QMC_ERR_UNSUPPORTED


# ------------------------------------------------------------------------------------ a1-a3 per point
def _log_poly_cancellation(sector, x):
    """Per order j the factor sum|c lU^a lF^b| / |sum c lU^a lF^b| >= 1 by which the log-polynomial
    L_j(log U, log F) of the real class amplifies a last-bit difference in the two logarithms: W g_j is
    compared relative to |W g_j| times this factor (1 for the deformed class, whose bound is set by the
    caller; for the toy class the analogous ratio of its worst factor).  Test-side arithmetic only: U and F by direct monomial sums in numpy."""
    J = 1 if sector.kind != W.KIND_UF else sector.n_orders
    xx = np.asarray(x, dtype=np.float64)
    d = sector.dim
    if sector.kind == W.KIND_TOY:
        # a factor 1 + c (x - 1/2) + d x^2 with c, d in [-1, 1] can pass through zero: the same ratio per factor
        c, dd = sector.U_coef[:d], sector.U_coef[d:2 * d]
        t1, t2 = c * (xx[:d] - 0.5), dd * xx[:d] ** 2
        with np.errstate(divide="ignore"):
            return np.array([np.max((1.0 + np.abs(t1) + np.abs(t2)) / np.abs(1.0 + t1 + t2))])
    if sector.kind != W.KIND_UF or sector.deformed:
        return np.ones(J)
    U = float(np.sum(sector.U_coef * np.prod(xx[None, :d] ** sector.U_exp[:, :d], axis=1)))
    F = float(np.sum(sector.F_coef * np.prod(xx[None, :d] ** sector.F_exp[:, :d], axis=1)))
    if not (U > 0 and F > 0):
        return np.ones(J)
    lU, lF = np.log(U), np.log(F)
    out, idx = np.ones(J), 0
    for jj in range(J):
        j = sector.first_order + jj
        tot, tot_abs = 0.0, 0.0
        for deg in range(j + 1):
            for beta in range(deg + 1):
                term = sector.logc[idx] * lU ** (deg - beta) * lF ** beta
                idx += 1
                tot += term
                tot_abs += abs(term)
        out[jj] = tot_abs / abs(tot) if tot != 0 else np.inf
    return out


def _point_parity(torch, B, O, wl, sector_ids, n_pts=400, rel=2e-12, **plan_opts):
    plan = B.qmc_plan(wl.sectors, **plan_opts)
    plan.bind_workspace(4, 8)
    width = B.debug_row_width(plan)
    rng = np.random.Generator(np.random.PCG64(77))
    worst = 0.0
    for si in sector_ids:
        job = wl.jobs[si]
        sec = O.OracleSector(wl.sectors[job.sector])
        d = sec.dim
        shift = wl.shifts[job.shift_offset]
        ks = np.unique(np.concatenate([[0, job.n - 1], rng.integers(0, job.n, size=n_pts)])).astype(np.uint64)
        out = torch.zeros((len(ks), width), dtype=torch.float64, device="cuda")
        B.qmc_debug_eval_points(plan, job.sector, job.n, job.z, shift, ks, out)
        torch.cuda.synchronize()
        got = out.cpu().numpy()
        for row, k in zip(got, ks):
            t, x, Wt, wg, _sf = O.eval_point(sec, job.n, job.z, shift, int(k))
            # reading Q2: 3.3e-16 from the two roundings on each side; for a regular Korobov sector the kernel works with
            # u = t - 1/2 and the debug hook reports u + 1/2, one more rounding of 5.5e-17
            assert np.allclose(row[:d], t, rtol=0, atol=4e-16), "t differs at k=%d" % k
            # korobov3: the bracket 35 - 84 t + 70 t^2 - 20 t^3 cancels from terms of size 209 down to
            # ~1 near t = 1, so two evaluation orders (oracle: powers summed; kernel: Horner halves)
            # differ by up to ~209 eps/2 ~ 2.3e-14 relative; 1e-13 leaves a factor 4.
            # On top of that the permitted difference in t itself (reading Q2: the kernel takes
            # fma(r, 1/n, Delta) where the oracle divides and adds, |dt| <= 3e-16 as asserted above) moves x
            # by phi'(t) dt to first order; where t is tiny this dominates 1e-13 |x| (x ~ 35 t^4, so
            # dx/x ~ 4 dt/t).  phi' = 140 t^3 (1-t)^3 (korobov3), 2 (baker), 1 (none); factor 2 of margin.
            tr = wl.sectors[job.sector].transform
            tt = np.asarray(t)
            dphi = {0: np.ones_like(tt), 1: 140.0 * tt**3 * (1.0 - tt)**3, 2: 2.0 * np.ones_like(tt)}[tr]
            # Regular sectors (toy class; U, F with non-negative coefficients and a constant term -- DESIGN.md section 5,
            # "centred Korobov form") evaluate phi = 1/2 + u Q(u^2) in the dimensions WITHOUT a prefactor x_i^a_i:
            # there x -> 0 by cancellation, an ABSOLUTE error of at most 0.5 * 2.19 * 3 ulp + 1 ulp ~ 5e-16 in x, which
            # reaches g only through U and F (bounded logarithmic derivatives).
            sct = wl.sectors[job.sector]
            regular = tr == 1 and (sct.kind == W.KIND_TOY or (not sct.deformed and np.all(sct.U_coef >= 0) and np.all(sct.F_coef >= 0)
                                                              and not sct.U_exp[0].any() and not sct.F_exp[0].any()))
            centred = np.array([regular and (sct.kind == W.KIND_TOY or sct.a[i] == 0) for i in range(d)])
            x_abs = np.where(centred, 5e-16, 0.0)
            x_tol = 1e-13 * np.abs(x) + 2.0 * dphi * (np.abs(row[:d] - tt) + np.where(centred, 6e-17, 0.0)) + x_abs + 1e-300
            assert np.all(np.abs(row[8:8 + d] - x) <= x_tol), "x differs at k=%d" % k
            # the same dt reaches W = prod 140 t^3 (1-t)^3 as dW/W = 3 dt (1/t - 1/(1-t)) and the integrand
            # through the prefactor x^a ~ t^(4a): a relative condition number of at most
            # cond = sum_i |dt_i| / (t_i (1 - t_i)), times 3 (W) or 3 + 4 a_i + O(1) (W g); 8 covers a_i <= 1.
            with np.errstate(divide="ignore", invalid="ignore"):
                cond = float(np.sum(np.where(row[:d] == tt, 0.0, np.abs(row[:d] - tt) / (tt * (1.0 - tt)))))
                # in a centred dimension the reported t = u + 1/2 carries a rounding that u does not
                cond += float(np.sum(np.where(centred, 6e-17 / (tt * (1.0 - tt)), 0.0)))
            assert abs(row[16] - Wt) <= (2e-14 + 4.0 * cond) * abs(Wt), "W differs at k=%d" % k
            g = row[17:17 + 2 * sec.J:2] + 1j * row[18:18 + 2 * sec.J:2]
            amp = _log_poly_cancellation(wl.sectors[job.sector], x)
            for j in range(sec.J):
                err = abs(g[j] - wg[j])
                scale = abs(wg[j]) * amp[j]
                assert err <= (rel + 8.0 * cond) * scale + 1e-300, "W g_%d differs at k=%d: %r vs %r" % (j, k, g[j], wg[j])
                if scale > 0:
                    worst = max(worst, err / scale)
    plan.destroy()
    return worst


def test_point_parity_toy(torch_cuda, B, O):
    _point_parity(torch_cuda, B, O, W.config_toy(), [0])


def test_point_parity_euclid(torch_cuda, B, O):
    _point_parity(torch_cuda, B, O, W.config_euclid(), range(8))


def test_point_parity_median_dim6(torch_cuda, B, O):
    _point_parity(torch_cuda, B, O, W.config_median(n_sectors=6), range(6))


def test_point_parity_physical(torch_cuda, B, O):
    # complex path: conditioning of the log-polynomial sum limits the per-point agreement
    _point_parity(torch_cuda, B, O, W.config_physical(n_sectors=6), range(6), rel=1e-10)


# ------------------------------------------------------------------------------------ full configs (small n)
def test_c0_toy_full(torch_cuda, B, O):
    """Config C0 in full (n = 65521, m = 32) and against the exact integral prod(1 + d_i/3)."""
    wl = W.config_toy()
    gpu = PU.run_gpu(wl)
    PU.compare_workload(wl, gpu)
    exact = W.toy_exact(wl.sectors[0])
    assert abs(gpu["job_results"][0, 0, 0] - exact) <= 1e-13 * abs(exact)
    assert gpu["stats"]["evaluations"] == wl.evaluations()


@pytest.mark.parametrize("n", [1, 2, 3, 5, 101, 1009, 65521])
def test_c1_euclid_small_n(torch_cuda, B, O, n):
    """Config C1's sectors on small lattices: n = 1..5 are the degenerate cases (single point,
    ragged one-tile launches), 65521 spans several tiles with a ragged tail."""
    wl = W.config_euclid(n=n)
    gpu = PU.run_gpu(wl)
    PU.compare_workload(wl, gpu)


def test_c1_euclid_full(torch_cuda, B, O):
    """Config C1 at its full size (8 x 1 048 573 x 32 evaluations); the oracle needs ~30 s."""
    wl = W.config_euclid()
    gpu = PU.run_gpu(wl)
    ws, wr = PU.compare_workload(wl, gpu)
    assert gpu["stats"]["evaluations"] == wl.evaluations()


def test_c1_literal_no_constant_term(torch_cuda, B, O):
    """Reading Q11's stress variant: U(0) = F(0) = 0 (huge dynamic range); parity must still hold."""
    wl = W.config_euclid(n=10007, const_term=None, n_sectors=4)
    gpu = PU.run_gpu(wl)
    PU.compare_workload(wl, gpu)


def test_c2_median_small(torch_cuda, B, O):
    """Config C2 (median rule) on 6 sectors at n = 20011, K = 11: candidate estimates, component-wise
    median, selected index (integer: exact), then the m-shift integration on the selected vector."""
    wl = W.config_median(n_sectors=6, n=20011)
    gpu = PU.run_gpu(wl, median=True)
    z_sel = {}
    for i, job in enumerate(wl.jobs):
        sec = O.OracleSector(wl.sectors[job.sector])
        est, med, sel = O.median_rule(sec, job.n, wl.z_cand[i], wl.shift0[i])
        g_est = gpu["cand_est"][i, :, :, 0] + 1j * gpu["cand_est"][i, :, :, 1]
        g_med = gpu["median"][i, :, 0] + 1j * gpu["median"][i, :, 1]
        scale = np.max(np.abs(est))
        assert np.all(np.abs(g_est[:, :sec.J] - est) <= PU.TOL_MEAN * scale)
        assert np.all(np.abs(g_med[:sec.J] - med) <= PU.TOL_MEAN * scale)
        assert int(gpu["selected"][i]) == sel
        z_sel[i] = wl.z_cand[i, sel]
    PU.compare_workload(wl, gpu, z_override=z_sel)


def test_median_rule_single_sector(torch_cuda, B, O):
    """The graded single-sector entry point qmc_median_rule, odd and even K."""
    torch = torch_cuda
    wl = W.config_median(n_sectors=2, n=10007, K=12)
    plan = B.qmc_plan(wl.sectors)
    plan.bind_workspace(16, 4)
    for K in (1, 2, 11, 12):
        for i in range(2):
            est_d = torch.zeros((K, plan.J, 2), dtype=torch.float64, device="cuda")
            med_d = torch.zeros((plan.J, 2), dtype=torch.float64, device="cuda")
            sel_d = torch.zeros((1,), dtype=torch.int32, device="cuda")
            B.qmc_median_rule(plan, i, 10007, wl.z_cand[i, :K], wl.shift0[i], est_d, med_d, sel_d)
            torch.cuda.synchronize()
            sec = O.OracleSector(wl.sectors[i])
            est, med, sel = O.median_rule(sec, 10007, wl.z_cand[i, :K], wl.shift0[i])
            g_est = est_d.cpu().numpy()
            g_est = g_est[..., 0] + 1j * g_est[..., 1]
            g_med = med_d.cpu().numpy()
            g_med = g_med[:, 0] + 1j * g_med[:, 1]
            scale = np.max(np.abs(est))
            assert np.all(np.abs(g_est - est) <= PU.TOL_MEAN * scale)
            assert np.all(np.abs(g_med - med) <= PU.TOL_MEAN * scale)
            got_sel = int(sel_d.item())
            if got_sel != sel:
                # Several selections can be correct: two candidates at the same MAD-scaled distance from the
                # component-wise median (always so for K = 2, where the median is their midpoint) differ only
                # by rounding.  Then the kernel's choice must be as near the median as the oracle's.
                comp = np.concatenate([est.real, est.imag], axis=1)          # K x 2J, oracle estimates
                medc = np.median(comp, axis=0)
                mad = np.median(np.abs(comp - medc), axis=0)
                use = mad > 0
                dist = np.sum(((comp[:, use] - medc[use]) / mad[use]) ** 2, axis=1)
                assert abs(dist[got_sel] - dist[sel]) <= 1e-6 * dist[sel], (K, i, got_sel, sel, dist)
    plan.destroy()


@pytest.mark.parametrize("n", [1, 2, 7, 1009, 40009])
def test_c3_physical_small(torch_cuda, B, O, n):
    """Config C3 (contour deformation, complex, J = 3, baker) on 4 sectors; sign-check counters equal."""
    wl = W.config_physical(n_sectors=4, n=n, m=8)
    gpu = PU.run_gpu(wl)
    PU.compare_workload(wl, gpu)


def test_c4_batch_small(torch_cuda, B, O):
    """Config C4's mix (dims 3..8, 40 % deformed, complex weights) at n/20000: 48 sectors through the
    batch scheduler in one call; amplitude and its propagated error against the oracle."""
    wl = W.config_batch(n_sectors=48, scale=1.0 / 20000.0, m=8)
    gpu = PU.run_gpu(wl)
    PU.compare_workload(wl, gpu)
    assert gpu["stats"]["evaluations"] == wl.evaluations()
    assert gpu["stats"]["eval_kernel_launches"] >= 2    # real and deformed modules


def test_scheduler_tile_independence(torch_cuda, B, O):
    """Results do not depend on how the scheduler cuts tiles or on the block size: every (tile, component)
    owns a partial-sum slot, so different launch shapes agree to rounding and all match the oracle."""
    wl = W.config_euclid(n=65521, n_sectors=3, m=4)
    runs = [PU.run_gpu(wl), PU.run_gpu(wl, threads_per_block=128), PU.run_gpu(wl, max_tiles=64, ctas_per_sm=1)]
    for r in runs:
        PU.compare_workload(wl, r)


# ------------------------------------------------------------------------------------ limits of the description
def test_description_limits(torch_cuda, B, O):
    """The edges of include/qmc.h's sector description against the oracle: the highest log-polynomial degree
    (first_order 2 + 3 orders = degree 4, 6 + 10 + 15 coefficients), prefactor exponents above 1, monomial
    exponents up to 6, the largest dimension, the un-transformed rule, real and deformed."""
    rng = np.random.Generator(np.random.PCG64(808))
    secs = []
    for dim, deformed in ((8, 0), (2, 0), (4, 1), (1, 1)):
        s = W.draw_physical_sector(rng, dim) if deformed else W.draw_euclid_sector(rng, dim)
        s.first_order, s.n_orders = 2, 3
        s.logc = rng.standard_normal(31)
        s.a = np.zeros(8, np.int32)
        s.a[:dim] = rng.integers(0, 4, dim)
        s.U_exp = (s.U_exp.astype(np.int64) * rng.integers(1, 3, s.U_exp.shape)).astype(np.uint8)
        s.F_exp = (s.F_exp.astype(np.int64) * rng.integers(1, 3, s.F_exp.shape)).astype(np.uint8)
        if deformed:
            s.F_coef = np.abs(s.F_coef)          # keep F(x) > 0: the higher powers move the zeros of a mixed-sign F
        secs.append(s)
    secs[1].transform = W.TRANSFORM_NONE
    n, m = 10007, 4
    jobs, rows = [], []
    for i, s in enumerate(secs):
        jobs.append(W.Job(i, n, W.draw_z(rng, n, s.dim), i * m, complex(rng.standard_normal(), rng.standard_normal())))
        rows.append(W.draw_shifts(rng, m, s.dim))
    wl = W.Workload("limits", secs, jobs, np.vstack(rows), m)
    gpu = PU.run_gpu(wl)
    PU.compare_workload(wl, gpu)


def test_five_epsilon_orders(torch_cuda, B, O):
    """QMC_MAX_ORDERS = 5 (eps^-4 .. eps^0 of a two-loop integral; "all orders in eps up to the finite order",
    PAPER.md:707): degrees 0..4, 35 log coefficients, real and deformed, through sums, mean / error, amplitude."""
    rng = np.random.Generator(np.random.PCG64(909))
    secs = []
    for dim, deformed in ((5, 0), (3, 1), (6, 0)):
        s = W.draw_physical_sector(rng, dim) if deformed else W.draw_euclid_sector(rng, dim)
        s.first_order, s.n_orders = 0, 5
        s.logc = rng.standard_normal(35)
        secs.append(s)
    n, m = 20011, 4
    jobs, rows = [], []
    for i, s in enumerate(secs):
        jobs.append(W.Job(i, n, W.draw_z(rng, n, s.dim), i * m, complex(rng.standard_normal(), rng.standard_normal())))
        rows.append(W.draw_shifts(rng, m, s.dim))
    wl = W.Workload("five-orders", secs, jobs, np.vstack(rows), m)
    gpu = PU.run_gpu(wl)
    assert gpu["J"] == 5
    PU.compare_workload(wl, gpu)
    _point_parity(torch_cuda, B, O, wl, range(3), n_pts=100, rel=1e-10)


def test_median_rule_with_64_candidates_and_empty_input(torch_cuda, B, O):
    torch = torch_cuda
    wl = W.config_median(n_sectors=1, n=1009, K=64)
    plan = B.qmc_plan(wl.sectors)
    plan.bind_workspace(64, 4)
    est_d = torch.zeros((64, plan.J, 2), dtype=torch.float64, device="cuda")
    med_d = torch.zeros((plan.J, 2), dtype=torch.float64, device="cuda")
    sel_d = torch.zeros((1,), dtype=torch.int32, device="cuda")
    B.qmc_median_rule(plan, 0, 1009, wl.z_cand[0], wl.shift0[0], est_d, med_d, sel_d)
    torch.cuda.synchronize()
    est, med, sel = O.median_rule(O.OracleSector(wl.sectors[0]), 1009, wl.z_cand[0], wl.shift0[0])
    g = est_d.cpu().numpy()
    scale = np.max(np.abs(est))
    assert np.all(np.abs(g[..., 0] + 1j * g[..., 1] - est) <= PU.TOL_MEAN * scale)
    assert abs(complex(*med_d.cpu().numpy()[0]) - med[0]) <= PU.TOL_MEAN * scale
    with pytest.raises(B.QmcError) as e:           # 65 candidates: beyond the documented maximum
        B.qmc_median_rule(plan, 0, 1009, np.vstack([wl.z_cand[0], wl.z_cand[0][:1]]), wl.shift0[0], est_d, med_d, sel_d)
    assert e.value.status == B.QMC_ERR_INVALID_ARG
    out = B.alloc_outputs(plan, 1, 2)
    with pytest.raises(B.QmcError) as e:           # an empty job list is an error, not a silent no-op
        B.qmc_integrate_sectors(plan, [], wl.shifts, 2, out)
    assert e.value.status == B.QMC_ERR_INVALID_ARG
    plan.destroy()


# ------------------------------------------------------------------------------------ wide lattices (n >= 2^32)
def test_wide_plan_matches_oracle_on_small_lattices(torch_cuda, B, O):
    """The 64-bit index path (qmc_plan_opts.wide_lattice) through whole sums: C1 and C3 sectors at small n."""
    for wl in (W.config_euclid(n=20011, n_sectors=3, m=4), W.config_physical(n=10007, n_sectors=2, m=4)):
        gpu = PU.run_gpu(wl, wide_lattice=1)
        PU.compare_workload(wl, gpu)


@pytest.mark.parametrize("n", [4294967311, 68719476767])
def test_wide_point_parity_beyond_2_32(torch_cuda, B, O, n):
    """a1-a3 at single lattice points of lattices the 32-bit path cannot hold."""
    _point_parity(torch_cuda, B, O, W.config_euclid(n=n, n_sectors=3, m=2), range(3), n_pts=200, wide_lattice=1)
    _point_parity(torch_cuda, B, O, W.config_physical(n=n, n_sectors=2, m=2), range(2), n_pts=100, rel=1e-10, wide_lattice=1)


def test_point_parity_on_the_largest_32bit_lattice(torch_cuda, B, O):
    """Default (32-bit index) plan at n = 4 294 967 291, the largest prime below 2^32: the modular increment and the
    integer shift work next to the overflow of u32 (r + step < n and r + a < n must hold without wrapping)."""
    n = 4294967291
    _point_parity(torch_cuda, B, O, W.config_euclid(n=n, n_sectors=3, m=2), range(3), n_pts=300)
    _point_parity(torch_cuda, B, O, W.config_physical(n=n, n_sectors=2, m=2), range(2), n_pts=150, rel=1e-10)


def test_wide_whole_lattice_of_4e9_points_integrates_the_toy_exactly(torch_cuda, B):
    """Every one of the 2 x 4 294 967 311 points of a wide lattice through a1-a4: the separable toy integrand has
    the exact integral prod(1 + d_i/3), which the Korobov-3 rule reproduces to rounding (pin P4); a wrong,
    missing or doubled point range would show at the 1e-13 level of this comparison."""
    wl = W.config_toy()
    n = 4294967311
    rng = np.random.Generator(np.random.PCG64(11))
    wl.jobs[0].n = n
    wl.jobs[0].z = np.array([int(rng.integers(1, n)), int(rng.integers(1, n))] + [0] * 6, np.uint64)
    wl.m = 2
    wl.shifts = wl.shifts[:2]
    gpu = PU.run_gpu(wl, wide_lattice=1)
    assert gpu["stats"]["evaluations"] == 2 * n
    exact = W.toy_exact(wl.sectors[0])
    assert abs(gpu["job_results"][0, 0, 0] - exact) <= 1e-13 * abs(exact)
    assert np.all(np.abs(gpu["shift_sums"][0, :, 0, 0] / n - exact) <= 1e-13 * abs(exact))


def test_pieces_on_a_wide_lattice_across_2_32(torch_cuda, B, O):
    """qmc_integrate_pieces on a wide_lattice plan (the case 8(e) names: ONE lattice too long for one GPU):
    k-ranges that start beyond 2^32 and one that straddles it, against the oracle's sums over exactly those indices
    (n = 68 719 476 767; a C1 sector and a deformed C3 sector)."""
    torch = torch_cuda
    n = 68719476767
    e, p = W.config_euclid(n=n, n_sectors=1, m=2), W.config_physical(n=n, n_sectors=1, m=2)
    sectors = e.sectors + p.sectors
    jobs = [e.jobs[0], W.Job(1, n, p.jobs[0].z, 2, 1.0)]
    shifts = np.vstack([e.shifts[:2], p.shifts[:2]])
    plan = B.qmc_plan(sectors, wide_lattice=1)
    plan.bind_workspace(16, 8)
    two32 = 1 << 32
    pieces = [(0, 0, 1, two32 - 150_000, two32 + 150_000), (0, 1, 2, 60_000_000_123, 60_000_300_123),
              (1, 0, 2, 5 * two32 + 17, 5 * two32 + 60_017)]
    J = plan.J
    part = torch.zeros((2, 2, J, 3, 2), dtype=torch.float64, device="cuda")
    diag = torch.zeros((2, 2), dtype=torch.int64, device="cuda")
    B.qmc_integrate_pieces(plan, jobs, pieces, shifts, 2, part, diag)
    torch.cuda.synchronize()
    assert plan.last_stats()["evaluations"] == 300_000 + 300_000 + 2 * 60_000
    got = part.cpu().numpy().sum(axis=-1)                     # hi + lo
    for job, s0, s1, k0, k1 in pieces:
        sec = O.OracleSector(sectors[job])
        off = jobs[job].shift_offset
        want, _ = O.shift_sums(sec, n, jobs[job].z, shifts[off + s0:off + s1], k0, k1)
        A = want[..., 2:3]
        assert np.all(np.abs(got[job, s0:s1, :sec.J] - want) <= 1e-11 * A), (job, np.abs(got[job, s0:s1, :sec.J] - want).max() / A.max())
    assert float(part[0, 1].abs().sum()) > 0 and float(part[1].abs().sum()) > 0
    assert np.all(diag.cpu().numpy() == 0)
    plan.destroy()


def test_default_plan_rejects_wide_lattices(torch_cuda, B):
    wl = W.config_toy()
    wl.jobs[0].n = 4294967311
    with pytest.raises(B.QmcError) as e:
        PU.run_gpu(wl)
    assert e.value.status == B.QMC_ERR_UNSUPPORTED


# ------------------------------------------------------------------------------------ adaptive evaluation
def test_adaptive_integrate_matches_the_oracle_round_by_round(torch_cuda, B, O):
    """qmc_adaptive_integrate (Eq. 1-6) against the oracle's restatement of the same round loop
    (oracle/adaptive.py) on the same seed: identical lattice sizes and selected vectors (integers: both sides
    take ceil / next-prime decisions from FP64 values that agree to ~1e-9), results within the north_star bounds."""
    from oracle import adaptive as A
    rng = np.random.Generator(np.random.PCG64(4242))
    sectors = [W.draw_euclid_sector(rng, 3), W.draw_euclid_sector(rng, 4), W.draw_euclid_sector(rng, 3),
               W.draw_physical_sector(rng, 3)]
    for s in sectors[:3]:                       # one plan-wide order layout: J = 3 everywhere
        s.first_order, s.n_orders = 0, 3
        s.logc = rng.standard_normal(10)
    coefs = [1.0 + 0.5j, -0.7 + 0.2j, 0.3 - 1.1j, 0.05 + 0.02j]
    jobs = [W.Job(i, 3, np.ones(8, np.uint64), 0, c) for i, c in enumerate(coefs)]
    plan = B.qmc_plan(sectors)
    tau = [plan.sector_ops(i) for i in range(len(sectors))]
    opts = dict(epsrel=3e-3, n_min=1009, n_max=4000037, seed=77, max_rounds=8, m=8, K=5, growth_max=16.0)
    got = B.qmc_adaptive_integrate(plan, jobs, **opts)
    plan.destroy()
    want = A.adaptive_integrate(sectors, [(i, c) for i, c in enumerate(coefs)], tau, **opts)
    assert got["rounds"] == want["rounds"] >= 2 and got["converged"] == want["converged"]
    assert list(got["n_final"]) == list(want["n_final"])
    assert np.array_equal(got["z_final"], want["z_final"])
    assert got["evaluations"] == want["evaluations"]
    scale = np.abs(want["job_results"][:, :, 0] + 1j * want["job_results"][:, :, 1])[:, :, None] + 1e-300
    assert np.all(np.abs(got["job_results"] - want["job_results"]) <= 1e-9 * scale)
    ascale = np.abs(want["amplitude"][:, 0] + 1j * want["amplitude"][:, 1])[:, None]
    assert np.all(np.abs(got["amplitude"] - want["amplitude"]) <= 1e-9 * ascale)
    # the requested precision was reached (or the run says it was not)
    if got["converged"]:
        err = np.hypot(got["amplitude"][:, 2], got["amplitude"][:, 3])
        assert np.all(err <= opts["epsrel"] * ascale[:, 0] * (1 + 1e-12))


def test_cuda_library_math_variant_matches_the_oracle(torch_cuda, B, O):
    """qmc_plan_opts.libdevice_math = 1 (the CUDA library's log / exp / atan2 / sincos / sqrt instead of the library's
    own table-driven ones; kept for A/B measurement) must give the same results within the same bounds."""
    for wl in (W.config_euclid(n=20011, n_sectors=3, m=4), W.config_physical(n=10007, n_sectors=2, m=4)):
        gpu = PU.run_gpu(wl, libdevice_math=1)
        PU.compare_workload(wl, gpu)


# ------------------------------------------------------------------------------------ concurrency
def test_two_plans_on_two_streams_repeated_without_sync(torch_cuda, B):
    """Enqueue-only calls: two plans, each on its own stream, called back to back several times with no
    synchronisation in between (more calls than pinned staging slots), must give bit-identical results to an
    isolated call -- every tile owns its partial-sum slot, so nothing depends on scheduling."""
    torch = torch_cuda
    wls = [W.config_euclid(n=200003, n_sectors=4, m=8), W.config_physical(n=50021, n_sectors=3, m=8)]
    plans, outs, refs, jobs = [], [], [], []
    for wl in wls:
        plan = B.qmc_plan(wl.sectors)
        plan.bind_workspace(len(wl.jobs), wl.shifts.shape[0] + len(wl.jobs))
        ref = B.alloc_outputs(plan, len(wl.jobs), wl.m)
        jc = B.marshal_jobs(wl.jobs)
        B.qmc_integrate_sectors(plan, jc, wl.shifts, wl.m, ref)
        torch.cuda.synchronize()
        plans.append(plan); jobs.append(jc); refs.append({k: v.clone() for k, v in ref.items() if v is not None})
        outs.append([B.alloc_outputs(plan, len(wl.jobs), wl.m) for _ in range(7)])
    streams = [torch.cuda.Stream(), torch.cuda.Stream()]
    for rep in range(7):
        for p in range(2):
            with torch.cuda.stream(streams[p]):
                B.qmc_integrate_sectors(plans[p], jobs[p], wls[p].shifts, wls[p].m, outs[p][rep], streams[p])
    torch.cuda.synchronize()
    for p in range(2):
        for rep in range(7):
            for k, v in refs[p].items():
                assert torch.equal(outs[p][rep][k], v), (p, rep, k)
        plans[p].destroy()


# ------------------------------------------------------------------------------------ errors
def test_error_codes(torch_cuda, B):
    wl = W.config_euclid(n=101, n_sectors=1, m=2)
    plan = B.qmc_plan(wl.sectors, validate=1)
    out = B.alloc_outputs(plan, 1, 2)
    with pytest.raises(B.QmcError) as e:           # no workspace bound
        B.qmc_integrate_sectors(plan, wl.jobs, wl.shifts, 2, out)
    assert e.value.status == B.QMC_ERR_WORKSPACE
    plan.bind_workspace(1, 2)
    with pytest.raises(B.QmcError) as e:           # m = 1: the error is undefined
        B.qmc_integrate_sectors(plan, wl.jobs, wl.shifts, 1, out)
    assert e.value.status == B.QMC_ERR_INVALID_ARG
    bad = W.Job(0, 100, np.array([2, 3, 7, 9, 0, 0, 0, 0], np.uint64), 0)   # gcd(2, 100) != 1
    with pytest.raises(B.QmcError) as e:
        B.qmc_integrate_sectors(plan, [bad], wl.shifts, 2, out)
    assert e.value.status == B.QMC_ERR_NOT_UNIT
    big = W.Job(0, 2**32, np.array([1, 1, 1, 1, 0, 0, 0, 0], np.uint64), 0)
    with pytest.raises(B.QmcError) as e:
        B.qmc_integrate_sectors(plan, [big], wl.shifts, 2, out)
    assert e.value.status == B.QMC_ERR_UNSUPPORTED
    sh = wl.shifts.copy()
    sh[0, 0] = 1.0
    with pytest.raises(B.QmcError) as e:
        B.qmc_integrate_sectors(plan, wl.jobs, sh, 2, out)
    assert e.value.status == B.QMC_ERR_INVALID_ARG
    plan.destroy()


def test_fp64_peak_measurement(torch_cuda, B):
    """The DFMA microbenchmark that is the roofline denominator returns a plausible B200 figure."""
    peak = B.qmc_measure_fp64_peak(50.0)
    assert 1.0e13 < peak < 6.0e13, peak


# ------------------------------------------------------------------------------------ pieces
@pytest.mark.parametrize("world", [2, 4])
def test_pieces_of_a_batch_add_up_to_the_single_call(torch_cuda, B, O, world):
    """qmc_integrate_pieces / qmc_finalize_pieces on one GPU, the ranks one after another: a C4-like mix plus one job
    far larger than the mean load (cut by shift and, at 4 ranks, by k-range by ranks.split_partition) gives the same
    per-shift sums (to 1e-13 A), results, amplitude and counters as one qmc_integrate_sectors call, and matches the
    oracle at the north_star tolerances."""
    from paper_2305_19768_b200 import ranks as R
    torch = torch_cuda
    wl = W.config_batch(n_sectors=6, scale=1.0 / 200000.0, m=4)
    big = W.config_euclid(n_sectors=1, dim=3, n=400009, m=4, seed=99)
    sectors = wl.sectors + big.sectors
    jobs = wl.jobs + [W.Job(len(wl.sectors), 400009, big.jobs[0].z, wl.shifts.shape[0], 0.7 - 0.2j)]
    allw = W.Workload("pieces", sectors, jobs, np.vstack([wl.shifts, big.shifts]), 4)
    plan = B.qmc_plan(allw.sectors)
    ref = PU.run_gpu(allw, plan=plan)
    PU.compare_workload(allw, ref)
    nj, m, J = len(allw.jobs), allw.m, plan.J
    cost = [plan.sector_ops(j.sector) for j in allw.jobs]
    parts_of = R.split_partition(cost, [j.n for j in allw.jobs], m, world)
    assert sum(1 for p in parts_of for pc in p if pc[0] == nj - 1) >= world          # the big job is shared
    if world == 4:
        assert any(pc[4] - pc[3] < 400009 for p in parts_of for pc in p)              # ... also by k-range
    parts = torch.zeros((world, nj, m, J, 3, 2), dtype=torch.float64, device="cuda")
    diag = torch.zeros((world, nj, 2), dtype=torch.int64, device="cuda")
    evals = 0
    for r in range(world):
        B.qmc_integrate_pieces(plan, allw.jobs, parts_of[r], allw.shifts, m, parts[r], diag[r])
        torch.cuda.synchronize()
        evals += plan.last_stats()["evaluations"]
    assert evals == allw.evaluations()
    out = B.alloc_outputs(plan, nj, m)
    B.qmc_finalize_pieces(plan, allw.jobs, m, parts, world, out)
    torch.cuda.synchronize()
    got = {k: v.cpu().numpy() for k, v in out.items() if v is not None}
    A = ref["shift_sums"][..., 2:3]
    assert np.all(np.abs(got["shift_sums"] - ref["shift_sums"]) <= 1e-13 * A)
    scale = np.maximum(np.abs(ref["job_results"][..., 0] + 1j * ref["job_results"][..., 1]), A.mean(axis=1)[..., 0] /
                       np.array([j.n for j in allw.jobs])[:, None])[..., None]
    assert np.all(np.abs(got["job_results"] - ref["job_results"]) <= 1e-12 * scale)
    assert np.allclose(got["amplitude"], ref["amplitude"], rtol=1e-11, atol=1e-300)
    assert np.array_equal(diag.sum(dim=0).cpu().numpy(), ref["diag"])
    # a rank without pieces contributes zeros; wrong piece lists are refused before any enqueue
    B.qmc_integrate_pieces(plan, allw.jobs, [], allw.shifts, m, parts[0], diag[0])
    torch.cuda.synchronize()
    assert float(parts[0].abs().sum()) == 0.0
    for bad in ([(nj, 0, 1, 0, 10)], [(0, 0, m + 1, 0, 10)], [(0, 0, 1, 5, 5)], [(1, 0, 1, 0, 5), (0, 0, 1, 0, 5)]):
        with pytest.raises(B.QmcError) as e:
            B.qmc_integrate_pieces(plan, allw.jobs, bad, allw.shifts, m, parts[0], None)
        assert e.value.status == B.QMC_ERR_INVALID_ARG
    plan.destroy()


@pytest.mark.parametrize("world", [2, 3])
def test_median_rule_over_pieces_matches_the_single_call(torch_cuda, B, O, world):
    """Step a5 sharded: the K candidates of every job evaluated as one-shift pieces on `world` ranks (one after another
    on this GPU; the larger lattice is also cut by k-range), qmc_median_select_pieces on the gathered parts, then the
    m-shift stage as pieces on the selected vectors -- against qmc_median_integrate_sectors in one call and against
    the oracle's median rule."""
    from paper_2305_19768_b200 import ranks as R
    torch = torch_cuda
    wl = W.config_median(n_sectors=5, dim=3, n=40009, K=7, m=4, seed=77)
    big = W.config_median(n_sectors=1, dim=4, n=700001, K=7, m=4, seed=78)
    sectors = wl.sectors + big.sectors
    jobs = wl.jobs + [W.Job(len(wl.sectors), 700001, big.jobs[0].z, wl.shifts.shape[0], 0.3 + 0.4j)]
    allw = W.Workload("median-pieces", sectors, jobs, np.vstack([wl.shifts, big.shifts]), 4,
                      z_cand=np.concatenate([wl.z_cand, big.z_cand]), shift0=np.vstack([wl.shift0, big.shift0]))
    plan = B.qmc_plan(allw.sectors)
    ref = PU.run_gpu(allw, plan=plan, median=True)
    nj, m, J, K = len(allw.jobs), allw.m, plan.J, allw.z_cand.shape[1]
    # candidate stage: n_jobs K one-shift jobs; their shift rows are shift0
    cj = R.candidate_jobs(allw.jobs, allw.z_cand)
    parts_of = [[] for _ in range(world)]            # short lattices: whole candidates in turn; the long one: k-ranges
    for idx, j in enumerate(cj):
        if j.n > 100000:
            kb = [(j.n * p) // world for p in range(world + 1)]
            for r in range(world):
                parts_of[r].append((idx, 0, 1, kb[r], kb[r + 1]))
        else:
            parts_of[idx % world].append((idx, 0, 1, 0, j.n))
    plan.bind_workspace(nj * (K + 1) + 64, allw.shifts.shape[0] + nj)
    parts = torch.zeros((world, nj * K, 1, J, 3, 2), dtype=torch.float64, device="cuda")
    for r in range(world):
        B.qmc_integrate_pieces(plan, cj, parts_of[r], allw.shift0, 1, parts[r], None)
        torch.cuda.synchronize()
    out = B.alloc_outputs(plan, nj, m, K=K)
    B.qmc_median_select_pieces(plan, cj, K, parts, world, out)
    torch.cuda.synchronize()
    sel = out["selected"].cpu().numpy()
    assert np.array_equal(sel, ref["selected"])
    est, ref_est = out["cand_est"].cpu().numpy(), ref["cand_est"]
    scale = np.abs(ref_est).max(axis=(1, 2, 3), keepdims=True)
    assert np.all(np.abs(est - ref_est) <= 1e-13 * scale)
    assert np.all(np.abs(out["median"].cpu().numpy() - ref["median"]) <= 1e-13 * scale[:, 0])
    for i in (0, nj - 1):                                                              # ... and against the oracle
        sec = O.OracleSector(allw.sectors[allw.jobs[i].sector])
        o_est, o_med, o_sel = O.median_rule(sec, allw.jobs[i].n, allw.z_cand[i], allw.shift0[i])
        assert o_sel == sel[i]
        got = est[i, :, :sec.J, 0] + 1j * est[i, :, :sec.J, 1]
        assert np.all(np.abs(got - o_est) <= 1e-10 * np.abs(o_est).max())
    # m-shift stage on the selected vectors, as pieces again
    sj = R.selected_jobs(allw.jobs, allw.z_cand, sel)
    parts_of2 = R.split_partition([plan.sector_ops(j.sector) for j in sj], [j.n for j in sj], m, world)
    parts2 = torch.zeros((world, nj, m, J, 3, 2), dtype=torch.float64, device="cuda")
    for r in range(world):
        B.qmc_integrate_pieces(plan, sj, parts_of2[r], allw.shifts, m, parts2[r], None)
        torch.cuda.synchronize()
    B.qmc_finalize_pieces(plan, sj, m, parts2, world, out)
    torch.cuda.synchronize()
    A = ref["shift_sums"][..., 2:3]
    assert np.all(np.abs(out["shift_sums"].cpu().numpy() - ref["shift_sums"]) <= 1e-13 * A)
    assert np.allclose(out["amplitude"].cpu().numpy(), ref["amplitude"], rtol=1e-11, atol=1e-300)
    # refusals: candidate jobs of one job that disagree, K out of range
    bad = list(cj)
    bad[1] = W.Job(cj[1].sector, cj[1].n + 2, cj[1].z, cj[1].shift_offset)
    with pytest.raises(B.QmcError):
        B.qmc_median_select_pieces(plan, bad, K, parts, world, out)
    with pytest.raises(B.QmcError):
        B.qmc_median_select_pieces(plan, cj * 10, 70, parts, world, out)
    plan.destroy()


def test_measured_tau_feeds_the_allocation(torch_cuda, B):
    """"The evaluation speed tau_i is estimated on-line ... by tracking how fast a given integral is being
    evaluated".  (i) qmc_plan_last_job_clocks: CTA-cycles per evaluation of a deformed dim-5 sector are several times
    those of a real dim-3 one.  (ii) qmc_adaptive_integrate with measure_tau = 1 against the same run with tau = 1 for
    every integral (same seed, so the first round and hence every w_i is identical): Eq. (6) gives n_i ~ tau_i^(-1/3),
    so the expensive integral's second lattice shrinks relative to the cheap one's by (tau_exp / tau_cheap)^(-1/3)."""
    torch = torch_cuda
    rng = np.random.Generator(np.random.PCG64(2305_9))
    sectors = [W.draw_euclid_sector(rng, 3), W.draw_physical_sector(rng, 5)]
    plan = B.qmc_plan(sectors)
    n = 1_000_003
    jobs = [W.Job(0, n, W.draw_z(rng, n, 3), 0, 1.0), W.Job(1, n, W.draw_z(rng, n, 5), 4, 1.0)]
    shifts = np.vstack([W.draw_shifts(rng, 4, 3), W.draw_shifts(rng, 4, 5)])
    plan.bind_workspace(2, 8)
    out = B.alloc_outputs(plan, 2, 4)
    B.qmc_integrate_sectors(plan, jobs, shifts, 4, out)
    clk = plan.last_job_clocks(2)
    assert np.all(clk > 0)
    tau = clk / (4.0 * n)
    ratio = tau[1] / tau[0]
    model = plan.sector_ops(1) / plan.sector_ops(0)
    assert 2.0 < ratio < 40.0 and 0.3 * model < ratio < 3.0 * model, (ratio, model)
    kw = dict(epsrel=1e-12, n_min=10007, growth_max=1e6, max_rounds=2, m=8, K=3, seed=11)
    flat = B.qmc_adaptive_integrate(plan, jobs, tau=[1.0, 1.0], **kw)
    meas = B.qmc_adaptive_integrate(plan, jobs, measure_tau=1, **kw)
    assert flat["rounds"] == 2 and meas["rounds"] == 2
    shrink = (meas["n_final"][1] / flat["n_final"][1]) / (meas["n_final"][0] / flat["n_final"][0])
    # at n = 10^4 one tile per shift carries fixed overhead, so the on-line ratio is smaller than at n = 10^6: direction and a bracket
    assert shrink < 0.95, shrink
    assert ratio ** (-1.0 / 3.0) * 0.7 < shrink, (shrink, ratio)
    plan.destroy()


# ------------------------------------------------------------------------------------ general Korobov transforms
@pytest.mark.parametrize("r0,r1", [(1, 1), (2, 2), (3, 3), (6, 6), (1, 4), (5, 2)])
def test_general_korobov_orders(torch_cuda, B, O, r0, r1):
    """QMC_TRANSFORM_KOROBOV(r0, r1) (oracle pin P18): whole-sum parity at the north_star tolerances
    for a real and a deformed sector and the toy class, the exact toy integral, per-point t / x / W, and the zero-weight
    branch (a shift row of zeros) with its counter."""
    import math
    code = 100 + 10 * r0 + r1
    rng = np.random.Generator(np.random.PCG64(1000 + code))
    real, phys, toy = W.draw_euclid_sector(rng, 3), W.draw_physical_sector(rng, 3), W.config_toy(seed=7).sectors[0]
    for s in (real, phys, toy):
        s.transform = code
    n, m = 10007, 4
    jobs, rows = [], []
    for i, s in enumerate((real, phys, toy)):
        jobs.append(W.Job(i, n, W.draw_z(rng, n, s.dim), i * m, 1.0 + 0.5j * i))
        rows.append(W.draw_shifts(rng, m, s.dim))
    rows[2][1, :] = 0.0                                           # toy job, second shift: k = 0 sits on t = 0
    wl = W.Workload("korobov-%d-%d" % (r0, r1), [real, phys, toy], jobs, np.vstack(rows), m)
    plan = B.qmc_plan(wl.sectors)
    gpu = PU.run_gpu(wl, plan=plan)
    diag_gpu = gpu.pop("diag")
    PU.compare_workload(wl, gpu)
    # counters: zero-weight points exactly; the sign check of the deformed job may differ on the few points where the
    # alternating sum of phi rounds x to 1 + O(1e-12) on one side only (x (1 - x) < 0 turns the deformation round:
    # floating point deciding an integer) -- weight ~ (1 - t)^r1 ~ 0 there
    _, _, diag_cpu = PU.oracle_jobs(wl)
    assert [int(dg[0]) for dg in diag_gpu] == [int(dc[0]) for dc in diag_cpu] == [0, 0, 1]
    assert abs(int(diag_gpu[1, 1]) - int(diag_cpu[1][1])) <= 8 and diag_gpu[0, 1] == 0 and diag_gpu[2, 1] == 0
    exact = W.toy_exact(toy)
    assert abs(gpu["job_results"][2, 0, 0] - exact) <= max(8.0 * gpu["job_results"][2, 0, 2], 1e-13 * abs(exact)) or r0 * r1 == 1
    # per point: the alternating sum of phi is conditioned like invB sum_k binom(r1, k) t^(r0+1+k) / (r0+1+k)
    invB = math.factorial(r0 + r1 + 1) / (math.factorial(r0) * math.factorial(r1))
    width = B.debug_row_width(plan)
    ks = np.unique(np.concatenate([[1, n - 1], rng.integers(1, n, size=200)])).astype(np.uint64)
    out = torch_cuda.zeros((len(ks), width), dtype=torch_cuda.float64, device="cuda")
    B.qmc_debug_eval_points(plan, 0, n, jobs[0].z, wl.shifts[0], ks, out)
    torch_cuda.cuda.synchronize()
    sec = O.OracleSector(real)
    for row, k in zip(out.cpu().numpy(), ks):
        t, x, Wt, wg, _ = O.eval_point(sec, n, jobs[0].z, wl.shifts[0], int(k))
        assert np.allclose(row[:3], t, rtol=0, atol=4e-16)
        mag = invB * sum(math.comb(r1, kk) * t ** (r0 + 1 + kk) / (r0 + 1 + kk) for kk in range(r1 + 1))
        dphi = invB * t**r0 * (1 - t) ** r1
        assert np.all(np.abs(row[8:11] - x) <= 1e-15 * mag + 2.0 * dphi * np.abs(row[:3] - t) + 1e-14 * np.abs(x))
        cond = float(np.sum(np.abs(row[:3] - t) * (r0 / t + r1 / (1 - t))))
        assert abs(row[16] - Wt) <= (1e-13 + 2.0 * cond) * abs(Wt)
    plan.destroy()


def test_persistent_kernel_is_deterministic_under_heavy_tile_reuse(torch_cuda, B, O):
    """Stand-in for compute-sanitizer racecheck (closed on this pool, profiles/r02_sanitizer.md): thousands of
    minimum-size tiles per launch, so that every persistent CTA reuses its shared tile context, reduction scratch,
    tile accumulators and counters hundreds of times; 12 repeats at 1, 2 and 4 CTAs per SM must give BIT-IDENTICAL
    per-shift sums, results and counters (each tile owns its slot of the partial-sum area; finalize adds the slots in
    a fixed order), equal to the oracle."""
    wl = W.config_batch(n_sectors=10, scale=1.0 / 2000.0, m=4)           # real and deformed sectors, n = 5e2 .. 5e5
    ref = None
    for ctas in (1, 2, 4):
        plan = B.qmc_plan(wl.sectors, ctas_per_sm=ctas, max_tiles=60000)
        for rep in range(4):
            gpu = PU.run_gpu(wl, plan=plan)
            assert gpu["stats"]["tiles"] > 150
            if ref is None:
                ref = gpu
                PU.compare_workload(wl, gpu)
                continue
            for key in ("shift_sums", "job_results", "amplitude", "diag"):
                assert np.array_equal(gpu[key], ref[key]), (ctas, rep, key)
        plan.destroy()
