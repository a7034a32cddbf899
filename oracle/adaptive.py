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
