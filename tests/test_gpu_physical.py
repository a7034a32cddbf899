"""GPU parity in the regimes pins P15 / P16 cover on the oracle side (tests/test_oracle_pins_physical.py): the
physical region -- F changing sign under the -i delta prescription -- and the zero-weight / sign-check counters
with non-zero values.  The CUDA path (through the C ABI) is compared with the oracle AND with the closed form."""
import numpy as np
import pytest

from paper_2305_19768_b200 import workloads as W
from tests import parity_util as PU
from tests import test_oracle_pins_physical as P

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
    build.build()
    binding.lib()
    return binding


def _workload(sectors, n, zs, m, seed, name):
    rng = np.random.default_rng(seed)
    jobs, rows = [], []
    for i, s in enumerate(sectors):
        z = np.zeros(8, np.uint64)
        z[:s.dim] = zs[i]
        jobs.append(W.Job(i, n, z, i * m))
        sh = np.zeros((m, 8))
        sh[:, :s.dim] = rng.random((m, s.dim))
        rows.append(sh)
    return W.Workload(name, list(sectors), jobs, np.vstack(rows), m)


def test_physical_region_matches_oracle_and_closed_form(torch_cuda, B):
    """P15's sectors through qmc_integrate_sectors: d = 1, F = a - x, q in {-1/2, -1.3, 3/4}, both transforms, and
    the mirror prescription (f_im > 0, lambda < 0)."""
    G = P._golden()
    cases = [(0.37, -0.5, 0.3, -1e-12, W.TRANSFORM_KOROBOV3), (0.37, -0.5, 1.0, -1e-12, W.TRANSFORM_KOROBOV3),
             (0.37, -1.3, 0.5, -1e-12, W.TRANSFORM_BAKER), (0.62, 0.75, 0.3, -1e-12, W.TRANSFORM_KOROBOV3),
             (0.62, -0.5, 0.5, -1e-12, W.TRANSFORM_BAKER), (0.37, -0.5, -0.5, +1e-12, W.TRANSFORM_KOROBOV3)]
    sectors = [P.physical_1d_sector(a, q, lam, f_im, tr) for a, q, lam, f_im, tr in cases]
    n = 100003
    wl = _workload(sectors, n, [[1]] * len(sectors), 8, 15, "P15-1d")
    gpu = PU.run_gpu(wl)
    PU.compare_workload(wl, gpu)                                   # vs the oracle: sums, mean / error, diag counters
    for i, (a, q, lam, f_im, tr) in enumerate(cases):
        I_pow, I_log = P._gc(G, "phys1d_a%s_q%s_pow" % (a, q)), P._gc(G, "phys1d_a%s_q%s_log" % (a, q))
        want0, want1 = I_pow, 0.5 * I_pow - 2.0 * I_log
        if f_im > 0:
            want0, want1 = want0.conjugate(), want1.conjugate()
            assert int(gpu["diag"][i, 1]) == n * wl.m               # Im F > 0 on every point: all flagged
        else:
            assert int(gpu["diag"][i, 1]) == 0
        # baker converges like n^-2 here: the closed form is met within the error bars, not to 1e-13
        assert P._within(gpu["job_results"][i, 0], want0, floor=1e-12), (cases[i], gpu["job_results"][i, 0], want0)
        assert P._within(gpu["job_results"][i, 1], want1, floor=1e-12), (cases[i], gpu["job_results"][i, 1], want1)


def test_physical_region_two_dimensional(torch_cuda, B):
    """F = a - x1 x2 (off-diagonal Hessian, sign change on a hyperbola) and the separable variant with U = 1 + b x2."""
    G = P._golden()
    s_sep = P._uf(2, U=[(1.0, (0, 0)), (0.8, (0, 1))], F=[(0.37, (0, 0)), (-1.0, (1, 0))], p=-1.7, q=-0.5, logc=[1.0],
                  first_order=0, n_orders=1, transform=W.TRANSFORM_KOROBOV3, lam=0.7, f_im=-1e-12)
    s_hyp = P._uf(2, U=[(1.0, (0, 0))], F=[(0.45, (0, 0)), (-1.0, (1, 1))], p=0.0, q=-0.5, logc=[1.0],
                  first_order=0, n_orders=1, transform=W.TRANSFORM_KOROBOV3, lam=0.8, f_im=-1e-12)
    n = 100003
    wl = _workload([s_sep, s_hyp], n, [[1, 38117], [1, 38117]], 8, 18, "P15-2d")
    gpu = PU.run_gpu(wl)
    PU.compare_workload(wl, gpu)
    exact = P._gc(G, "phys1d_a0.37_q-0.5_pow") * G["sep_u_b0.8_p-1.7"]
    assert P._within(gpu["job_results"][0, 0], exact, floor=1e-12)
    assert gpu["job_results"][1, 0, 1] > 0.5                        # Im of int (a - x1 x2 - i0)^(-1/2): positive branch


def test_zero_weight_points_and_counters_nonzero(torch_cuda, B):
    """P16 on the GPU: g = x^(-1/2) is infinite where the Korobov weight is exactly 0 (n = 12, z = 4 is not a unit:
    r = 0 at k = 0, 3, 6, 9; first shift row 0.0): the kernel must skip those points, count 4 and agree with the
    oracle on the rest.  The evaluation there goes through the guarded slow paths of qmc_log / qmc_exp (log 0, exp inf)."""
    sec = W.Sector(dim=1, kind=W.KIND_UF, transform=W.TRANSFORM_KOROBOV3, deformed=0, first_order=0, n_orders=1,
                   a=np.zeros(8, np.int32), p=0.0, q=-0.5, U_coef=np.ones(1), U_exp=np.zeros((1, 1), np.uint8),
                   F_coef=np.ones(1), F_exp=np.ones((1, 1), np.uint8), logc=np.ones(1))
    z = np.zeros(8, np.uint64)
    z[0] = 4
    shifts = np.zeros((2, 8))
    shifts[1, 0] = 0.3125
    wl = W.Workload("P16-zero-weight", [sec], [W.Job(0, 12, z, 0)], shifts, 2)
    gpu = PU.run_gpu(wl)
    assert tuple(gpu["diag"][0]) == (4, 0)
    assert np.all(np.isfinite(gpu["shift_sums"]))
    PU.compare_workload(wl, gpu)
    # W = 0 from one of two dimensions (toy class)
    toy = W.Sector(dim=2, kind=W.KIND_TOY, transform=W.TRANSFORM_KOROBOV3, U_coef=np.array([0.5, -0.25, 0.75, 0.125]),
                   U_exp=np.zeros((4, 2), np.uint8))
    z2 = np.zeros(8, np.uint64)
    z2[:2] = (3, 5)
    sh2 = np.zeros((2, 8))
    sh2[0, :2] = (0.4375, 0.0)
    sh2[1, :2] = (0.0, 0.0)
    wl2 = W.Workload("P16-toy", [toy], [W.Job(0, 7, z2, 0)], sh2, 2)
    gpu2 = PU.run_gpu(wl2)
    assert tuple(gpu2["diag"][0]) == (2, 0)
    PU.compare_workload(wl2, gpu2)


def test_sign_check_counter_partial_count(torch_cuda, B):
    """diag[1] with a non-trivial value: f_im = +0.05 against lambda = 0.5 on F = a - x flags exactly the points with
    x (1 - x) <= 0.1; lambda = 0 flags every point for f_im >= 0 and none for f_im < 0."""
    n, m = 1009, 3
    cases = [(0.5, 0.05), (0.0, 1e-12), (0.0, 0.0), (0.0, -1e-12)]
    sectors = [P.physical_1d_sector(0.37, -0.5, lam, f_im, W.TRANSFORM_BAKER) for lam, f_im in cases]
    wl = _workload(sectors, n, [[1]] * 4, m, 20, "P16-sign")
    gpu = PU.run_gpu(wl)
    PU.compare_workload(wl, gpu)                                    # includes diag == oracle's
    d = gpu["diag"][:, 1]
    assert 0 < d[0] < n * m and d[1] == n * m and d[2] == n * m and d[3] == 0


# ------------------------------------------------------------------------------------ branches no workload takes
def _count_points(wl):
    return sum(j.n for j in wl.jobs) * wl.m


def test_configs_never_take_a_rare_path(torch_cuda, B):
    """On the BASELINE.json workload shapes neither the guarded re-evaluation nor a CUDA-library fallback runs."""
    for wl, med in ((W.config_median(n_sectors=4, n=10007, m=4), True), (W.config_physical(n_sectors=4, n=10007, m=4), False),
                    (W.config_batch(n_sectors=12, scale=1e-4, m=4), False)):
        gpu = PU.run_gpu(wl, median=med)
        assert gpu["rare"] == {"checked_evals": 0, "slow_calls": 0}, (wl.name, gpu["rare"])


def test_deformed_exponent_outside_the_fast_range_is_re_evaluated(torch_cuda, B):
    """eval_checked, forced: U = 2, F = 1/2 - x, p = q = 1010, so that Re(p Log U + q Log F) = 1010 log(2 |F(z)|) runs
    from 0 (x = 0, 1: the points that carry the integral) down to -700 at x = 1/2; every point with
    1010 log(2 |F(z)|) < -690 sets the flag of the unguarded evaluator and is re-done by the guarded one (counted by
    hand below), and the per-shift sums agree with the oracle to 1e-11 A."""
    s = P._uf(1, U=[(2.0, (0,))], F=[(0.5, (0,)), (-1.0, (1,))], p=1010.0, q=1010.0, logc=[1.0, 0.5, 7.0, -2.0],
              first_order=0, n_orders=2, transform=W.TRANSFORM_BAKER, lam=1.0, f_im=-1e-12)
    n, m = 40009, 4
    wl = _workload([s], n, [[1]], m, 31, "rare-exp")
    gpu = PU.run_gpu(wl)
    PU.compare_workload(wl, gpu)
    want = 0
    for r in range(m):
        t = (np.arange(n) / n + wl.shifts[r, 0]) % 1.0
        x = 1.0 - np.abs(2.0 * t - 1.0)
        want += int(np.sum(1010.0 * (np.log(2.0) + 0.5 * np.log((0.5 - x) ** 2 + (x * (1.0 - x)) ** 2)) < -690.0))
    got = gpu["rare"]["checked_evals"]
    assert want > 100 and abs(got - want) <= 4, (got, want)        # <= 4: points within rounding of the threshold
    assert gpu["rare"]["slow_calls"] >= got                        # each re-evaluation ran exp() of the CUDA library


def test_deformed_subnormal_modulus_squared(torch_cuda, B):
    """|F|^2 subnormal: F = c (1/2 - x) with c = 1e-160 (and lambda = 0.5e160, so that the contour is the usual one).
    re^2 + im^2 underflows, the unguarded evaluator flags every point, and the guarded complex logarithm rescales
    before squaring (qmc_clog_re_scaled) -- the oracle's std::log(std::complex) does the same inside libm."""
    c = 1e-160
    s = P._uf(1, U=[(1.0, (0,))], F=[(0.5 * c, (0,)), (-c, (1,))], p=0.0, q=-0.5, logc=[1.0, 0.5, 7.0, -2.0],
              first_order=0, n_orders=2, transform=W.TRANSFORM_KOROBOV3, lam=0.5 / c, f_im=-1e-12 * c)
    n, m = 10007, 4
    wl = _workload([s], n, [[1]], m, 32, "rare-subnormal")
    gpu = PU.run_gpu(wl)
    PU.compare_workload(wl, gpu)
    assert gpu["rare"]["checked_evals"] == _count_points(wl)
    assert gpu["rare"]["slow_calls"] >= _count_points(wl)          # the scaled logarithm and atan2 of a tiny argument
    # the same integral as P15 up to the factor c^q: (F / c) = 1/2 - x
    G = P._golden()
    ref = PU.run_gpu(_workload([P._uf(1, U=[(1.0, (0,))], F=[(0.5, (0,)), (-1.0, (1,))], p=0.0, q=-0.5,
                                      logc=[1.0, 0.5, 7.0, -2.0], first_order=0, n_orders=2,
                                      transform=W.TRANSFORM_KOROBOV3, lam=0.5, f_im=-1e-12)], n, [[1]], m, 32, "ref"))
    scale = c ** -0.5
    assert np.allclose(gpu["job_results"][0, 0, :2], ref["job_results"][0, 0, :2] * scale, rtol=1e-10, atol=0)
    assert ref["rare"] == {"checked_evals": 0, "slow_calls": 0}


def test_real_class_guarded_functions_take_their_slow_paths(torch_cuda, B):
    """qmc_log / qmc_exp range guards of the real class (sectors whose range the generator cannot bound): F subnormal
    on the whole cube (log of a subnormal), and U^p below e^-690 (exp of a large negative argument; e^+690 would
    overflow the squares in the error estimate).  Results against the
    oracle; every evaluation must have gone through the CUDA-library fallback."""
    one = (np.ones(1), np.zeros((1, 1), np.uint8))
    lin = lambda c: (np.array([c, c]), np.array([[0], [1]], np.uint8))           # c (1 + x)
    mk = lambda U, F, p, q: W.Sector(dim=1, kind=W.KIND_UF, transform=W.TRANSFORM_KOROBOV3, deformed=0, first_order=1,
                                     n_orders=1, a=np.zeros(8, np.int32), p=p, q=q, U_coef=U[0], U_exp=U[1],
                                     F_coef=F[0], F_exp=F[1], logc=np.array([0.3, -0.7, 1.1]))
    s_log = mk(lin(1.0), lin(1e-310), -1.0, -0.5)          # F in [1e-310, 2e-310]: subnormal
    s_exp = mk(lin(1e-251), one, 1.2, 0.0)                 # U^p = e^(-693.5 .. -692.7): beyond the fast range of qmc_exp
    n, m = 101, 2
    wl = _workload([s_log, s_exp], n, [[1], [1]], m, 33, "rare-real")
    gpu = PU.run_gpu(wl)
    PU.compare_workload(wl, gpu)
    assert np.all(np.isfinite(gpu["shift_sums"]))
    assert gpu["rare"]["checked_evals"] == 0
    assert gpu["rare"]["slow_calls"] == 2 * n * m


# ------------------------------------------------------------------------------------ presampling of lambda (P19)
def test_presampled_lambda_matches_the_oracle_and_repairs_a_failing_sector(torch_cuda, B):
    """qmc_presample_lambda against oracle/presample.py (same candidates, same presample lattice): the selected lambda
    is the same double; a sector whose fixed lambda = 2 violates the sign check on thousands of points integrates with
    no violation at the presampled value, and the closed-form threshold of pin P19 is respected."""
    from oracle import presample as PS
    from tests.test_oracle_pins_transforms import _cubic_sector
    rng = np.random.Generator(np.random.PCG64(19))
    # (i) the cubic of pin P19: lambda* = 0.903..., candidates from 2.0
    s = _cubic_sector(0.4, -4.0)
    n_pre, z, sh = 20011, np.array([1], np.uint64), np.array([0.123])
    got = B.qmc_presample_lambda(s, n_pre, z, sh, lambda_max=2.0, decrease=0.9)
    want = PS.presample_lambda(s, n_pre, z, sh, lambda_max=2.0, decrease=0.9)
    assert got["ok"] and got["lam"] == want["lam"] and got["steps"] == want["steps"]
    assert got["max_im_f"] == pytest.approx(want["max_im_f"], rel=1e-9) and got["min_abs_f"] == pytest.approx(want["min_abs_f"], rel=1e-9)
    assert 0.8 < got["lam"] < 0.9036
    # (ii) the same sector integrated with lambda = 2 and with the presampled value
    import copy
    n, m = 100003, 4
    bad, good = copy.deepcopy(s), copy.deepcopy(s)
    bad.lam, good.lam = 2.0, got["lam"]
    wl = _workload([bad, good], n, [[1], [1]], m, 41, "presample-repair")
    gpu = PU.run_gpu(wl)
    PU.compare_workload(wl, gpu)
    assert gpu["diag"][0, 1] > 1000 and gpu["diag"][1, 1] == 0
    # (iii) BASELINE.json config 3 sectors (d = 5, 18 mixed-sign monomials): oracle and library agree on every one
    wl3 = W.config_physical(n_sectors=6)
    for s3 in wl3.sectors:
        z3, sh3 = W.draw_z(rng, 4099, 5), W.draw_shifts(rng, 1, 5)[0]
        g3 = B.qmc_presample_lambda(s3, 4099, z3, sh3, min_abs_f=0.02)
        w3 = PS.presample_lambda(s3, 4099, z3, sh3, min_abs_f=0.02)
        assert (g3["ok"], g3["lam"], g3["steps"]) == (w3["ok"], w3["lam"], w3["steps"]), (g3, w3)
    # (iv) min_abs_f and the error path
    r = B.qmc_presample_lambda(P.physical_1d_sector(0.37, -0.5, 0.5, -1e-12, W.TRANSFORM_BAKER), 1009, z, np.array([0.3]), min_abs_f=0.2)
    assert r["ok"] and r["lam"] >= 0.2 / (0.37 * 0.63) * 0.999 and r["min_abs_f"] >= 0.2
    r = B.qmc_presample_lambda(P.physical_1d_sector(0.37, -0.5, 0.5, +0.3, W.TRANSFORM_BAKER), 101, z, np.array([0.3]), lambda_min=0.05)
    assert not r["ok"] and r["lam"] == 0.05
    # an unreachable distance: the farthest sign-admissible contour is returned with ok = False (same as the oracle)
    s1 = P.physical_1d_sector(0.37, -0.5, 0.5, -1e-12, W.TRANSFORM_BAKER)
    r = B.qmc_presample_lambda(s1, 1009, z, np.array([0.3]), min_abs_f=0.5, lambda_min=0.3)
    w = PS.presample_lambda(s1, 1009, z, np.array([0.3]), min_abs_f=0.5, lambda_min=0.3)
    assert not r["ok"] and (r["lam"], r["steps"]) == (w["lam"], w["steps"]) == (1.0, 0)
    assert r["min_abs_f"] == pytest.approx(w["min_abs_f"], rel=1e-12)
    with pytest.raises(B.QmcError):
        B.qmc_presample_lambda(W.config_euclid(n_sectors=1).sectors[0], 101, np.ones(4, np.uint64), np.full(4, 0.3))


def test_presampling_lowers_the_error_of_a_c4_like_amplitude(torch_cuda, B):
    """DESIGN.md section 6 noted that the error of the C4 amplitude is dominated by a few deformed sectors whose fixed
    lambda = 0.5 puts zeros of F next to the contour.  With lambda presampled per sector under a distance condition
    (binding.presample_sectors, min_abs_f), the same batch on the same lattices has a smaller amplitude error and no
    sign-check failure."""
    import copy
    wl = W.config_batch(n_sectors=60, scale=1.0 / 300.0, m=8)
    fixed = PU.run_gpu(wl)
    wl2 = copy.deepcopy(wl)
    infos = B.presample_sectors(wl2.sectors, n_pre=20011, lambda_max=1.0, min_abs_f=0.05)
    assert all(i is None or i["max_im_f"] < 0 for i in infos)          # every sector got a sign-admissible contour
    assert any(i is not None and i["lam"] != 0.5 for i in infos)
    pres = PU.run_gpu(wl2)
    assert np.all(pres["diag"][:, 1] == 0)
    # the same through qmc_plan(presample=...): identical deformation strengths compiled in, identical results
    plan = B.qmc_plan(wl.sectors, presample=20011, presample_opts=dict(lambda_max=1.0, min_abs_f=0.05))
    again = PU.run_gpu(wl, plan=plan)
    plan.destroy()
    assert np.array_equal(again["shift_sums"], pres["shift_sums"])
    err_fixed = np.hypot(fixed["amplitude"][:, 2], fixed["amplitude"][:, 3])
    err_pres = np.hypot(pres["amplitude"][:, 2], pres["amplitude"][:, 3])
    assert np.all(err_pres < err_fixed), (err_pres, err_fixed)
    # the two contours integrate the same functions: the amplitudes agree within their errors
    d = np.abs((fixed["amplitude"][:, 0] + 1j * fixed["amplitude"][:, 1]) - (pres["amplitude"][:, 0] + 1j * pres["amplitude"][:, 1]))
    assert np.all(d <= 8.0 * (err_fixed + err_pres))
