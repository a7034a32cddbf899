"""Pins of the adaptive-allocation oracle (oracle/adaptive.py; Eq. 1-6) to things other than
itself: the Lagrange conditions of Eq. (5), the constraint Eq. (4), an independent constrained optimiser
(scipy SLSQP), brute-force perturbations on the constraint surface, and textbook special cases."""
import math

import numpy as np
import pytest

from oracle import adaptive as A


def _problem(seed, N=9):
    rng = np.random.default_rng(seed)
    w = 10.0 ** rng.uniform(-6, 2, N)
    tau = 10.0 ** rng.uniform(-9, -7, N)
    c2 = rng.uniform(0.1, 4.0, N)
    return w, tau, c2


@pytest.mark.parametrize("alpha", [1.0, 2.0, 3.0])
def test_eq6_meets_the_requested_variance_exactly(alpha):
    w, tau, c2 = _problem(1)
    V = 1e-8
    n = A.allocate_lattices(w, tau, c2, alpha, V)
    assert A.sum_variance(w, c2, n, alpha) == pytest.approx(V, rel=1e-12)        # Eq. (4)


@pytest.mark.parametrize("alpha", [1.0, 2.0, 3.0])
def test_eq6_is_a_stationary_point_of_the_lagrangian(alpha):
    """Eq. (5): dT/dn_i = -lambda dvar/dn_i for one common lambda > 0."""
    w, tau, c2 = _problem(2)
    n = np.array(A.allocate_lattices(w, tau, c2, alpha, 3e-9))
    lam = tau / (alpha * c2 * w / n ** (alpha + 1.0))
    assert np.all(lam > 0) and np.ptp(lam) <= 1e-12 * lam.mean()


def test_eq6_beats_every_feasible_perturbation_and_matches_slsqp():
    from scipy import optimize as SO
    alpha, V = 2.0, 1e-7
    w, tau, c2 = _problem(3, N=6)
    n = np.array(A.allocate_lattices(w, tau, c2, alpha, V))
    T0 = A.total_time(tau, n)
    rng = np.random.default_rng(4)
    for _ in range(200):
        m = n * np.exp(rng.normal(0, 0.2, n.size))
        m *= (A.sum_variance(w, c2, m, alpha) / V) ** (1.0 / alpha)              # back onto var = V
        assert A.sum_variance(w, c2, m, alpha) == pytest.approx(V, rel=1e-12)
        assert A.total_time(tau, m) >= T0 * (1 - 1e-12)
    # independent optimiser, in log n with scaled objective
    f = lambda u: float(np.sum(tau * np.exp(u)) / T0)
    g = {"type": "eq", "fun": lambda u: float(np.sum(c2 * w * np.exp(-alpha * u)) / V - 1.0)}
    r = SO.minimize(f, np.log(n) + rng.normal(0, 0.3, n.size), constraints=[g], method="SLSQP",
                    options={"ftol": 1e-15, "maxiter": 500})
    assert r.success and np.allclose(np.exp(r.x), n, rtol=1e-5)


def test_special_cases():
    # identical integrals: equal shares, n = (N c w / V)^(1/alpha)
    N, alpha, V = 5, 2.0, 1e-6
    n = A.allocate_lattices([0.3] * N, [1e-8] * N, [2.0] * N, alpha, V)
    assert np.allclose(n, (N * 2.0 * 0.3 / V) ** (1.0 / alpha), rtol=1e-13)
    # alpha = 1 (plain Monte Carlo scaling): the classical Neyman allocation n_i ~ sqrt(c_i w_i / tau_i)
    w, tau, c2 = _problem(5)
    n = np.array(A.allocate_lattices(w, tau, c2, 1.0, 1e-5))
    ratio = n / np.sqrt(c2 * w / tau)
    assert np.ptp(ratio) <= 1e-12 * ratio.mean()
    # an integral that does not enter the sum gets no points; the others are unaffected
    c2z = c2.copy(); c2z[2] = 0.0
    nz = A.allocate_lattices(w, tau, c2z, 2.0, 1e-5)
    assert nz[2] == 0.0
    keep = [i for i in range(len(w)) if i != 2]
    assert np.allclose([nz[i] for i in keep], A.allocate_lattices(w[keep], tau[keep], c2[keep], 2.0, 1e-5), rtol=1e-13)
    # tighter target: n scales as V^(-1/alpha)
    a = np.array(A.allocate_lattices(w, tau, c2, 2.0, 1e-6)); b = np.array(A.allocate_lattices(w, tau, c2, 2.0, 1e-8))
    assert np.allclose(b / a, 10.0, rtol=1e-12)


def test_several_sums_in_turn_never_decrease_and_meet_every_target():
    """formula for the first sum, update, then the next; afterwards every var(A_k) <= V_k."""
    rng = np.random.default_rng(6)
    N, K, alpha = 8, 3, 2.0
    tau = 10.0 ** rng.uniform(-9, -7, N)
    ws = [10.0 ** rng.uniform(-6, 0, N) for _ in range(K)]
    cs = [rng.uniform(0.1, 3.0, N) for _ in range(K)]
    Vs = [1e-8, 3e-9, 1e-7]
    n0 = [1e4] * N
    n = A.allocate_for_sums(ws, tau, cs, alpha, Vs, n0)
    assert all(x >= 1e4 for x in n)
    for w, c2, V in zip(ws, cs, Vs):
        assert A.sum_variance(w, c2, n, alpha) <= V * (1 + 1e-12)


# ------------------------------------------------------------------------------------------------
# Property pins of the ROUND LOOP (oracle/adaptive.py::adaptive_integrate, readings R2-R9 of DESIGN.md section 11).
# None of them restates the loop: they check what PAPER.md:245-253 and Eq. (4)-(6) fix about any correct loop.
def _small_problem():
    from paper_2305_19768_b200 import workloads as W
    rng = np.random.Generator(np.random.PCG64(77))
    sectors = [W.draw_euclid_sector(rng, 2), W.draw_euclid_sector(rng, 3), W.config_toy(seed=5).sectors[0],
               W.draw_physical_sector(rng, 2)]
    for s in sectors[:2]:
        s.first_order, s.n_orders = 0, 1
        s.logc = s.logc[:1]
    sectors[3].n_orders = 1
    sectors[3].logc = sectors[3].logc[:1]
    coefs = [1.5 - 0.5j, -0.7 + 2.0j, 0.3 + 0.1j, 1.0 + 1.0j]
    return sectors, [(i, coefs[i]) for i in range(4)]


def test_round_loop_invariants_on_real_integrands():
    """n_i prime, >= n_min, never decreasing, growing by at most growth_max per round; `evaluations` = the sum over
    rounds and over the integrals evaluated in that round of n_i (K + m); a converged run meets its target; the
    reported amplitude is Eq. (4) of the reported job results; n_final is the lattice each result was computed on."""
    from paper_2305_19768_b200 import workloads as W
    sectors, jobs = _small_problem()
    tau = [1.0, 2.5, 0.4, 6.0]
    K, m, n_min, gmax, epsrel = 5, 8, 101, 8.0, 2e-7
    r = A.adaptive_integrate(sectors, jobs, tau, epsrel=epsrel, n_min=n_min, growth_max=gmax, seed=3, max_rounds=8, m=m, K=K)
    hist = r["history"]
    assert len(hist) == r["rounds"] >= 2
    evals = 0
    for rnd, ns in enumerate(hist):
        for i, n in enumerate(ns):
            assert W._is_prime(n) and n >= n_min
            if rnd == 0:
                assert n == 101                                  # the first prime >= n_min (101 is prime)
                evals += n * (K + m)
                continue
            prev = hist[rnd - 1][i]
            assert n >= prev
            if n > prev:
                # at most growth_max x, rounded up to the next prime (Bertrand: a prime below twice the bound)
                assert n <= 2 * math.ceil(gmax * prev)
                lo = math.ceil(gmax * prev)
                assert n <= lo or all(not W._is_prime(c) for c in range(lo, n))
                evals += n * (K + m)
    assert r["evaluations"] == evals
    assert list(r["n_final"]) == [max(ns[i] for ns in hist) for i in range(len(jobs))]
    # Eq. (4), component-wise, recomputed with numpy from the reported job results
    res, amp = r["job_results"], r["amplitude"]
    C = np.array([c for _, c in jobs])
    mean = res[:, 0, 0] + 1j * res[:, 0, 1]
    assert amp[0, 0] + 1j * amp[0, 1] == pytest.approx(np.sum(C * mean), rel=1e-13)
    var = np.sum(np.abs(C) ** 2 * (res[:, 0, 2] ** 2 + res[:, 0, 3] ** 2))
    assert amp[0, 2] ** 2 + amp[0, 3] ** 2 == pytest.approx(var, rel=1e-12)
    assert r["converged"] == 1
    assert math.sqrt(var) <= epsrel * abs(np.sum(C * mean))
    # a looser target never costs more evaluations; an unreachable one stops at max_rounds without the flag
    r2 = A.adaptive_integrate(sectors, jobs, tau, epsrel=1e-3, n_min=n_min, growth_max=gmax, seed=3, max_rounds=8, m=m, K=K)
    assert r2["converged"] == 1 and r2["evaluations"] <= r["evaluations"]
    r3 = A.adaptive_integrate(sectors, jobs, tau, epsrel=1e-30, n_min=n_min, growth_max=2.0, seed=3, max_rounds=3, m=m, K=K)
    assert r3["converged"] == 0 and r3["rounds"] == 3


def _synthetic_integrator(monkeypatch, w_true, a_true, values):
    """Replaces the oracle's integrator by a model integral with var(I_i) = w_i / n^a exactly (Eq. 2)."""
    from oracle import oracle as O
    index = {}

    class Sec:
        J = 1

        def __init__(self, s):
            self.i = index.setdefault(id(s), len(index))

    def median_rule(sec, n, zc, sh0):
        return None, None, 0

    def integrate(sec, n, z, sh):
        i = sec.i
        err = math.sqrt(w_true[i] / float(n) ** a_true[i])
        return None, np.array([[values[i].real, values[i].imag, err * 0.6, err * 0.8]]), None

    monkeypatch.setattr(O, "OracleSector", Sec)
    monkeypatch.setattr(O, "median_rule", median_rule)
    monkeypatch.setattr(O, "integrate", integrate)


def test_round_loop_reaches_the_eq6_allocation_on_exact_power_laws(monkeypatch):
    """If var(I_i) = w_i / n_i^alpha holds exactly (Eq. 2), the second round's lattices must be Eq. (6)'s: the ratios
    n_i / n_j = ((w_i |C_i|^2 / tau_i) / (w_j |C_j|^2 / tau_j))^(1/(alpha+1)) (the multiplier cancels), and
    var(A) lands on safety x V (up to the rounding of n_i to primes), so the run converges in exactly two rounds."""
    N, alpha = 6, 2.0
    rng = np.random.default_rng(8)
    w_true = 10.0 ** rng.uniform(-2, 2, N)
    tau = 10.0 ** rng.uniform(-1, 1, N)
    C = rng.standard_normal(N) + 1j * rng.standard_normal(N)
    vals = rng.standard_normal(N) + 1j * rng.standard_normal(N)
    _synthetic_integrator(monkeypatch, w_true, [alpha] * N, vals)
    sectors = [object() for _ in range(N)]
    jobs = [(i, C[i]) for i in range(N)]
    Aabs = abs(np.sum(C * vals))
    epsrel, safety = 1e-7, 0.5
    r = A.adaptive_integrate(sectors, jobs, list(tau), epsrel=epsrel, alpha=alpha, safety=safety, growth_max=1e9,
                             n_min=10007, seed=1, max_rounds=6, m=4, K=3)
    assert r["rounds"] == 2 and r["converged"] == 1
    n = np.array(r["n_final"], float)
    key = (w_true * np.abs(C) ** 2 / tau) ** (1.0 / (alpha + 1.0))
    ratio = n / key
    assert np.ptp(ratio) <= 2e-4 * ratio.mean()                         # primes are ~ln n apart: relative 1e-5
    var = np.sum(np.abs(C) ** 2 * w_true / n ** alpha)
    assert var == pytest.approx(safety * (epsrel * Aabs) ** 2, rel=2e-4) and var <= safety * (epsrel * Aabs) ** 2
    # and it is cheaper than the equal-lattice allocation that meets the same variance
    n_eq = (np.sum(np.abs(C) ** 2 * w_true) / var) ** (1.0 / alpha)
    assert np.sum(tau * n) < np.sum(tau) * n_eq


def test_round_loop_with_a_faster_true_convergence_still_converges_and_never_shrinks(monkeypatch):
    """alpha = 2 is 'chosen conservatively': when the true variance falls like n^-3 the Eq. (6) step
    overshoots, the run converges after the second round with var(A) below the target, and no n_i ever decreases."""
    N = 5
    rng = np.random.default_rng(9)
    w_true = 10.0 ** rng.uniform(0, 3, N)
    tau = np.ones(N)
    C = np.ones(N, complex)
    vals = np.ones(N, complex)
    _synthetic_integrator(monkeypatch, w_true, [3.0] * N, vals)
    r = A.adaptive_integrate([object() for _ in range(N)], [(i, C[i]) for i in range(N)], list(tau), epsrel=1e-8,
                             growth_max=1e9, n_min=10007, seed=2, max_rounds=6, m=4, K=3)
    assert r["converged"] == 1 and r["rounds"] == 2
    for a, b in zip(r["history"][:-1], r["history"][1:]):
        assert all(y >= x for x, y in zip(a, b))
    var = np.sum(w_true / np.array(r["n_final"], float) ** 3.0)
    assert var < 0.5 * (1e-8 * N) ** 2


def test_measured_tau_moves_the_allocation_in_the_direction_of_eq6(monkeypatch):
    """Eq. (6): n_i ~ tau_i^(-1/(alpha+1)) at fixed multiplier -- an integral that is 8x more expensive per evaluation
    gets a lattice 8^(1/3) = 2x smaller relative to the others (alpha = 2), and the total time goes down compared
    with ignoring the cost."""
    N, alpha = 4, 2.0
    w_true, C, vals = np.full(N, 5.0), np.ones(N, complex), np.ones(N, complex)
    _synthetic_integrator(monkeypatch, w_true, [alpha] * N, vals)
    run = lambda tau: np.array(A.adaptive_integrate([object() for _ in range(N)], [(i, C[i]) for i in range(N)], tau,
                                                    epsrel=1e-7, growth_max=1e9, n_min=10007, seed=4, max_rounds=4,
                                                    m=4, K=3)["n_final"], float)
    n_flat = run([1.0, 1.0, 1.0, 1.0])
    n_cost = run([1.0, 1.0, 1.0, 8.0])
    assert np.ptp(n_flat) <= 1e-4 * n_flat.mean()
    assert n_cost[3] / n_cost[0] == pytest.approx(0.5, rel=1e-3)
    assert n_cost[3] < n_flat[3] and n_cost[0] > n_flat[0]
    tau = np.array([1.0, 1.0, 1.0, 8.0])
    # both allocations meet the same variance target; the cost-aware one is cheaper
    assert np.sum(w_true / n_cost ** 2) == pytest.approx(np.sum(w_true / n_flat ** 2), rel=1e-3)
    assert np.sum(tau * n_cost) < np.sum(tau * n_flat)
