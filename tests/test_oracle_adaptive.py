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
