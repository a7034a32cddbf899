"""TEST INFRASTRUCTURE, NOT THE PRODUCT -- oracle of the adaptive lattice-size choice.

Plain Python restatement of arXiv:2305.19768 section 2.1.3 ("Adaptive weighted sum evaluation"),
in the paper's notation:

  Eq. (2)  var(I_i) = w_i / n_i^alpha
  Eq. (3)  T = sum_i tau_i n_i
  Eq. (4)  var(A_k) = sum_i |C_ki|^2 w_i / n_i^alpha = V_k
  Eq. (6)  lambda_k = (1/alpha) ( (1/V_k) sum_i (|C_ki|^2 w_i tau_i^alpha)^(1/(alpha+1)) )^((alpha+1)/alpha)
           n_i      = ( alpha w_i lambda_k |C_ki|^2 / tau_i )^(1/(alpha+1))
  "If multiple sums are requested, Disteval uses this formula first for the first sum, then updates n_i and
   applies it to the next sum, and so on."

Eq. (4) and (6) are printed with index typos (C_ji, and k reused as the summation index inside lambda_k); the
reading -- the sum runs over the integrals i of the one sum k -- is the only one under which Eq. (6) solves
Eq. (5), which tests/test_oracle_adaptive.py checks (stationarity, the constraint, an independent optimiser).
Shares no code with the CUDA library; only tests may import it.
"""
from __future__ import annotations

import math
from typing import Sequence


def allocate_lattices(w: Sequence[float], tau: Sequence[float], c_abs2: Sequence[float], alpha: float, V: float):
    """Eq. (6): real-valued lattice sizes n_i minimising T = sum tau_i n_i subject to
    sum_i c_abs2_i w_i / n_i^alpha = V.  Items with w_i c_abs2_i = 0 need no points (n_i = 0)."""
    s = 0.0
    for wi, ti, ci in zip(w, tau, c_abs2):
        s += (ci * wi * ti ** alpha) ** (1.0 / (alpha + 1.0))
    lam = (1.0 / alpha) * (s / V) ** ((alpha + 1.0) / alpha)
    return [(alpha * wi * lam * ci / ti) ** (1.0 / (alpha + 1.0)) for wi, ti, ci in zip(w, tau, c_abs2)]


def allocate_for_sums(w_per_sum, tau, c_abs2_per_sum, alpha, V_per_sum, n_start):
    """the formula for the first sum, then n_i updated (never decreased) with the next sum's."""
    n = [float(x) for x in n_start]
    for w, c2, V in zip(w_per_sum, c_abs2_per_sum, V_per_sum):
        cand = allocate_lattices(w, tau, c2, alpha, V)
        n = [max(a, b) for a, b in zip(n, cand)]
    return n


def total_time(tau, n):
    """Eq. (3)."""
    return math.fsum(t * x for t, x in zip(tau, n))


def sum_variance(w, c_abs2, n, alpha):
    """Eq. (4), left-hand side."""
    return math.fsum(c * wi / x ** alpha for wi, c, x in zip(w, c_abs2, n) if wi * c != 0.0)


# ------------------------------------------------------------------------------------------------
# The round loop of the adaptive evaluation (DESIGN.md section 11 lists the readings R1-R8), step by step
# with the oracle's own integrator.  The random draws come from a counter-based generator that this file
# restates on its own (the CUDA library has its own copy): splitmix64 nested over (seed, round, job, stream,
# counter).
_M64 = (1 << 64) - 1


def splitmix64(x: int) -> int:
    x = (x + 0x9E3779B97F4A7C15) & _M64
    z = x
    z = ((z ^ (z >> 30)) * 0xBF58476D1CE4E5B9) & _M64
    z = ((z ^ (z >> 27)) * 0x94D049BB133111EB) & _M64
    return z ^ (z >> 31)


def draw(seed: int, rnd: int, job: int, stream: int, counter: int) -> int:
    """streams: 0 candidate generating vectors, 1 the candidates' shared shift, 2 the m shifts."""
    return splitmix64(splitmix64(splitmix64(splitmix64(seed ^ rnd) ^ job) ^ stream) ^ counter)


def draw_shift(u: int) -> float:
    v = u >> 11
    return float(v if v else 1) * 2.0 ** -53


def is_prime(n: int) -> bool:
    if n < 2:
        return False
    for p in (2, 3, 5, 7, 11, 13, 17, 19, 23, 29, 31, 37):
        if n % p == 0:
            return n == p
    i = 41
    while i * i <= n:           # trial division: slow and obviously correct (n < 2^32 here)
        if n % i == 0:
            return False
        i += 2
    return True


def next_prime(n: int) -> int:
    n = max(n, 2)
    while not is_prime(n):
        n += 1
    return n


def prev_prime(n: int) -> int:
    while n > 2 and not is_prime(n):
        n -= 1
    return n


def adaptive_integrate(sectors, jobs, tau, *, epsrel=0.0, epsabs=0.0, alpha=2.0, growth_max=64.0, safety=0.5,
                       n_min=10000, n_max=4294967291, seed=0, max_rounds=12, m=32, K=11):
    """jobs: list of (sector_index, complex coefficient).  Returns a dict with job_results [nj, J, 4],
    amplitude [J, 4], n_final, z_final, rounds, converged, evaluations, history (n per round)."""
    import numpy as np
    from oracle import oracle as O
    nj = len(jobs)
    secs = [O.OracleSector(sectors[s]) for s, _ in jobs]
    J = max(s.J for s in secs)
    coef = [complex(c) for _, c in jobs]
    c2 = [abs(c) ** 2 for c in coef]
    n_hi = prev_prime(n_max)
    n = [min(next_prime(n_min), n_hi)] * nj
    n_done = [0] * nj
    need = [True] * nj
    res = np.zeros((nj, J, 4))
    zsel = np.zeros((nj, 8), np.uint64)
    amp = np.zeros((J, 4))
    evals, rounds, converged, history = 0, 0, 0, []
    for rnd in range(max_rounds):
        batch = [i for i in range(nj) if need[i]]
        if not batch:
            break
        history.append(list(n))
        for i in batch:
            zc = np.zeros((K, 8), np.uint64)
            for c in range(K):
                for k in range(8):
                    zc[c, k] = 1 + draw(seed, rnd, i, 0, c * 8 + k) % (n[i] - 1)
            sh0 = np.array([draw_shift(draw(seed, rnd, i, 1, k)) for k in range(8)])
            sh = np.array([[draw_shift(draw(seed, rnd, i, 2, s * 8 + k)) for k in range(8)] for s in range(m)])
            _est, _med, sel = O.median_rule(secs[i], n[i], zc, sh0)                 # A8
            _sums, r, _diag = O.integrate(secs[i], n[i], zc[sel], sh)               # A1-A7
            res[i] = 0.0
            res[i, :secs[i].J] = r
            zsel[i] = zc[sel]
            n_done[i] = n[i]
            evals += n[i] * (K + m)
        rounds += 1
        # Eq. (4) with the measured variances; targets
        Vt, met = [], True
        for j in range(J):
            are = sum(coef[i].real * res[i, j, 0] - coef[i].imag * res[i, j, 1] for i in range(nj))
            aim = sum(coef[i].real * res[i, j, 1] + coef[i].imag * res[i, j, 0] for i in range(nj))
            vre = sum(coef[i].real ** 2 * res[i, j, 2] ** 2 + coef[i].imag ** 2 * res[i, j, 3] ** 2 for i in range(nj))
            vim = sum(coef[i].imag ** 2 * res[i, j, 2] ** 2 + coef[i].real ** 2 * res[i, j, 3] ** 2 for i in range(nj))
            amp[j] = (are, aim, math.sqrt(vre), math.sqrt(vim))
            target = max(epsabs, epsrel * math.hypot(are, aim))
            Vt.append(target * target)
            if not (vre + vim <= Vt[j]):
                met = False
        if met:
            converged = 1
            break
        # Eq. (2) -> w; Eq. (6) order by order, never decreasing
        want = [float(x) for x in n]
        for j in range(J):
            w = [(res[i, j, 2] ** 2 + res[i, j, 3] ** 2) * float(n_done[i]) ** alpha for i in range(nj)]
            if not sum(wi * ci for wi, ci in zip(w, c2)) > 0:
                continue
            cand = allocate_lattices(w, tau, c2, alpha, safety * Vt[j])
            want = [max(a, b) for a, b in zip(want, cand)]
        grow = False
        for i in range(nj):
            cap = min(float(n_hi), growth_max * float(n[i]))
            t = int(math.ceil(min(want[i], cap)))
            need[i] = False
            if t > n[i]:
                p = min(next_prime(t), n_hi)
                if p > n[i]:
                    n[i], need[i], grow = p, True, True
        if not grow:
            break
    return {"job_results": res, "amplitude": amp, "n_final": n_done, "z_final": zsel, "rounds": rounds,
            "converged": converged, "evaluations": evals, "history": history}
