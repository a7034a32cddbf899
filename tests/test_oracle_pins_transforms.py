"""Pin P18 of the CPU oracle: the general Korobov transform (r0, r1), transform code 100 + 10 r0 + r1
("higher Korobov orders / asymmetric weights"; the paper names `korobov3` as the default of that
family).  None of these tests touches the CUDA path.

  omega(t) = t^r0 (1 - t)^r1 / B(r0 + 1, r1 + 1),   phi(t) = int_0^t omega.

What fixes it independently of the oracle: for a polynomial g and theta in [0, 1) the shifted rectangle rule is EXACTLY
    (1/n) sum_{k=0}^{n-1} g((k + theta)/n) = int_0^1 g + sum_{j=1}^{deg g + 1} B_j(theta)/j! (g^(j-1)(1) - g^(j-1)(0)) / n^j
(Euler-Maclaurin terminates for polynomials; B_j are the Bernoulli polynomials), evaluated here in exact rationals.
For r0 = r1 = 3 this is pin P3's 1 - 70 B4/n^4 - 140 B6/n^6 (checked below).  Wrong normalisation, a wrong power, a
swapped (r0, r1) or a wrong sign in the alternating sum of phi each fail.
"""
import math
from fractions import Fraction

import numpy as np
import pytest

from oracle import oracle as O
from paper_2305_19768_b200 import workloads as W


def _bernoulli_numbers(n):
    B = [Fraction(0)] * (n + 1)
    B[0] = Fraction(1)
    for m in range(1, n + 1):
        B[m] = -sum(Fraction(math.comb(m + 1, k)) * B[k] for k in range(m)) / (m + 1)
    return B                                    # B_1 = -1/2 convention


def _bernoulli_poly(j, theta, Bn):
    return sum(Fraction(math.comb(j, k)) * Bn[j - k] * theta ** k for k in range(j + 1))


def _omega_coeffs(r0, r1):
    """Coefficients (ascending powers of t) of t^r0 (1 - t)^r1 / B(r0+1, r1+1), exact."""
    invB = Fraction(math.factorial(r0 + r1 + 1), math.factorial(r0) * math.factorial(r1))
    c = [Fraction(0)] * (r0 + r1 + 1)
    for k in range(r1 + 1):
        c[r0 + k] = invB * (-1) ** k * math.comb(r1, k)
    return c


def _deriv_at(c, order, t):
    """order-th derivative of sum c_i t^i at t (exact)."""
    return sum(ci * Fraction(math.perm(i, order)) * Fraction(t) ** (i - order) for i, ci in enumerate(c) if i >= order)


def rule_of_constant_exact(r0, r1, n, delta):
    c = _omega_coeffs(r0, r1)
    deg = len(c) - 1
    Bn = _bernoulli_numbers(deg + 2)
    theta = (n * Fraction(delta)) % 1
    total = sum(ci / (i + 1) for i, ci in enumerate(c))                       # int_0^1 omega = 1
    assert total == 1
    for j in range(1, deg + 2):
        jump = _deriv_at(c, j - 1, 1) - _deriv_at(c, j - 1, 0)
        total += _bernoulli_poly(j, theta, Bn) / math.factorial(j) * jump / Fraction(n) ** j
    return total


def _const_sector(code):
    return W.Sector(dim=1, kind=W.KIND_TOY, transform=code, U_coef=np.zeros(2), U_exp=np.zeros((2, 1), np.uint8))


def test_p18_formula_reduces_to_pin_p3_for_r3():
    for n in (1, 2, 5, 13):
        for delta in ("1/10", "37/100", "93/100"):
            th = (n * Fraction(delta)) % 1
            B4 = th**4 - 2 * th**3 + th**2 - Fraction(1, 30)
            B6 = th**6 - 3 * th**5 + Fraction(5, 2) * th**4 - Fraction(1, 2) * th**2 + Fraction(1, 42)
            assert rule_of_constant_exact(3, 3, n, delta) == 1 - 70 * B4 / Fraction(n)**4 - 140 * B6 / Fraction(n)**6


@pytest.mark.parametrize("r0,r1", [(1, 1), (2, 2), (3, 3), (4, 4), (6, 6), (1, 3), (3, 1), (2, 5), (6, 1)])
def test_p18_general_korobov_rule_of_constant(r0, r1):
    sec = O.OracleSector(_const_sector(100 + 10 * r0 + r1))
    for n in (1, 2, 3, 7, 13):
        for delta in ("1/10", "37/100", "1/2", "93/100"):
            sums, _ = O.shift_sums(sec, n, np.array([1], np.uint64), np.array([[float(Fraction(delta))]]))
            want = float(rule_of_constant_exact(r0, r1, n, delta))
            assert sums[0, 0, 0] / n == pytest.approx(want, abs=4e-15 * max(1.0, abs(want))), (n, delta)


@pytest.mark.parametrize("r0,r1", [(1, 1), (3, 3), (5, 5), (2, 4), (4, 2), (6, 3)])
def test_p18_map_is_the_integral_of_the_weight(r0, r1):
    """phi(0) = 0, phi(1) = 1, phi_{r0,r1}(t) = 1 - phi_{r1,r0}(1 - t), and phi = the exact rational antiderivative."""
    sec, swp = O.OracleSector(_const_sector(100 + 10 * r0 + r1)), O.OracleSector(_const_sector(100 + 10 * r1 + r0))
    c = _omega_coeffs(r0, r1)
    one = np.array([1], np.uint64)
    for t in (Fraction(1, 16), Fraction(3, 8), Fraction(1, 2), Fraction(13, 16), Fraction(63, 64)):
        _, x, Wt, _, _ = O.eval_point(sec, 1, one, np.array([float(t)]), 0)
        _, xs, Ws, _, _ = O.eval_point(swp, 1, one, np.array([float(1 - t)]), 0)
        phi = sum(ci * t ** (i + 1) / (i + 1) for i, ci in enumerate(c))
        om = sum(ci * t ** i for i, ci in enumerate(c))
        assert x[0] == pytest.approx(float(phi), rel=2e-13, abs=1e-300)     # alternating sum: a few hundred ulp at r1 = 6
        assert Wt == pytest.approx(float(om), rel=1e-14)
        assert x[0] + xs[0] == pytest.approx(1.0, abs=3e-13) and Wt == pytest.approx(Ws, rel=1e-13)
    _, x1, W1, _, _ = O.eval_point(sec, 2, one, np.array([0.5]), 1)        # t = frac(1/2 + 1/2) = 0
    assert x1[0] == 0.0 and W1 == 0.0


def test_p18_code_133_is_korobov3():
    a, b = O.OracleSector(_const_sector(133)), O.OracleSector(_const_sector(W.TRANSFORM_KOROBOV3))
    for t in np.random.default_rng(0).random(50):
        ra = O.eval_point(a, 1, np.array([1], np.uint64), np.array([t]), 0)
        rb = O.eval_point(b, 1, np.array([1], np.uint64), np.array([t]), 0)
        assert ra[1][0] == pytest.approx(rb[1][0], rel=1e-13, abs=1e-300) and ra[2] == pytest.approx(rb[2], rel=1e-14)   # 35 - 84 t + .. cancels ~200x near t = 1


@pytest.mark.parametrize("code", [111, 155, 124])
def test_p18_toy_integral_converges_under_every_order(code):
    """BASELINE.json config 0's exact integral prod (1 + d_i/3) is reproduced under other orders too: higher order,
    faster convergence (the smoothing these transforms exist for)."""
    w = W.config_toy(n=4099, seed=21)
    s = w.sectors[0]
    s.transform = code
    _, res, _ = O.integrate(O.OracleSector(s), 4099, w.jobs[0].z, w.shifts)
    exact = W.toy_exact(s)
    tol = {111: 3e-6, 124: 3e-8, 155: 1e-10}[code]
    assert abs(res[0, 0] - exact) <= max(6.0 * res[0, 2], 1e-14) and res[0, 2] < tol * abs(exact)


# ------------------------------------------------------------------------------- P19: presampling of lambda
def _cubic_sector(a, c, transform=W.TRANSFORM_BAKER):
    """d = 1, F = a - x + c x^3 (deformed; U = 1)."""
    from tests.test_oracle_pins_physical import _uf
    return _uf(1, U=[(1.0, (0,))], F=[(a, (0,)), (-1.0, (1,)), (c, (3,))], p=0.0, q=-0.5, logc=[1.0], first_order=0,
               n_orders=1, transform=transform, lam=0.5, f_im=-1e-12)


def test_p19_presampled_lambda_against_the_closed_form_threshold():
    """F = a - x + c x^3 with c < 0: with v = Im z = lambda x (1 - x) (1 - 3 c x^2),
        Im F(z) = -lambda x (1 - x) (1 - 3 c x^2)^2 - c v^3 - delta,
    which is >= 0 (up to delta) exactly where |c| lambda^2 x^2 (1 - x)^2 (1 - 3 c x^2) > 1: the largest admissible
    lambda is lambda* = (max_x |c| x^2 (1 - x)^2 (1 + 3 |c| x^2))^(-1/2).  The presampler, on a fine lattice, must return
    the largest candidate below lambda* -- worked out here with numpy on a dense grid, not with the oracle."""
    from oracle import presample as PS
    a, c = 0.4, -4.0
    xg = np.linspace(0.0, 1.0, 2_000_001)
    h = abs(c) * xg**2 * (1 - xg) ** 2 * (1 + 3 * abs(c) * xg**2)
    lam_star = 1.0 / np.sqrt(h.max())
    assert 0.85 < lam_star < 0.95
    cands = PS.candidates(2.0, 0.9, 1e-5)
    want = max(l for l in cands if l < lam_star)
    n_pre, z = 20011, np.array([1], np.uint64)
    r = PS.presample_lambda(_cubic_sector(a, c), n_pre, z, np.array([0.123]), lambda_max=2.0, decrease=0.9)
    assert r["ok"] and r["lam"] == want and r["steps"] == cands.index(want)
    assert r["max_im_f"] < 0.0
    # the candidate before it really fails the sign check on the presample set, the returned one passes on a denser set
    from oracle import oracle as O
    sec = O.OracleSector(_cubic_sector(a, c))
    fails = sum(O.deformed_f(sec, np.array([x]), want / 0.9).imag >= 0 for x in xg[::200])
    assert fails > 0
    assert all(O.deformed_f(sec, np.array([x]), want).imag < 0 for x in xg[1:-1:97])


def test_p19_special_cases():
    from oracle import presample as PS
    from tests.test_oracle_pins_physical import physical_1d_sector
    z = np.array([1], np.uint64)
    # F = a - x: Im F = -lambda x (1 - x) - delta < 0 for every lambda > 0: the maximum is kept
    r = PS.presample_lambda(physical_1d_sector(0.37, -0.5, 0.5, -1e-12, W.TRANSFORM_BAKER), 1009, z, np.array([0.3]), lambda_max=1.0)
    assert r["ok"] and r["lam"] == 1.0 and r["steps"] == 0
    # ... but asking for a distance |F| >= 0.2 from the zero at x = a forces |Im F| = lambda a (1 - a) >= 0.2 there: lambda >= 0.858
    r2 = PS.presample_lambda(physical_1d_sector(0.37, -0.5, 0.5, -1e-12, W.TRANSFORM_BAKER), 1009, z, np.array([0.3]),
                             lambda_max=1.0, min_abs_f=0.2)
    assert r2["ok"] and r2["lam"] >= 0.2 / (0.37 * 0.63) * 0.999 and r2["min_abs_f"] >= 0.2
    # the wrong prescription (f_im > 0 with lambda > 0 small) is never admissible: ok = False, lambda_min returned
    r3 = PS.presample_lambda(physical_1d_sector(0.37, -0.5, 0.5, +0.3, W.TRANSFORM_BAKER), 101, z, np.array([0.3]),
                             lambda_max=1.0, lambda_min=0.05)
    assert not r3["ok"] and r3["lam"] == 0.05
    # candidates: one multiplication per step, all >= lambda_min
    cs = PS.candidates(1.0, 0.9, 1e-5)
    assert cs[0] == 1.0 and cs[1] == 0.9 and cs[2] == 0.9 * 0.9 and len(cs) == 110 and cs[-1] >= 1e-5 > cs[-1] * 0.9


def test_p19_unreachable_distance_falls_back_to_the_farthest_sign_admissible_contour():
    """F = a - x: |F(z)|^2 = (a - x)^2 + lambda^2 x^2 (1 - x)^2, so over the contour min |F| is close to lambda a (1 - a)
    (at x = a) for lambda <= 1.  Asking for |F| >= 0.5 is impossible for lambda <= 1 (0.22 at most): no candidate is
    admissible, every candidate passes the sign check, and the rule returns the one farthest from the zero -- the largest
    lambda -- with ok = False, instead of collapsing the contour to lambda_min."""
    from oracle import presample as PS
    from tests.test_oracle_pins_physical import physical_1d_sector
    r = PS.presample_lambda(physical_1d_sector(0.37, -0.5, 0.5, -1e-12, W.TRANSFORM_BAKER), 1009, np.array([1], np.uint64),
                            np.array([0.3]), lambda_max=1.0, min_abs_f=0.5, lambda_min=0.3)
    assert not r["ok"] and r["lam"] == 1.0 and r["steps"] == 0
    xg = np.linspace(0.0, 1.0, 1_000_001)
    least = np.sqrt((0.37 - xg) ** 2 + (xg * (1 - xg)) ** 2).min()           # lambda = 1: a little below a (1 - a) = 0.233
    assert 0.21 < least < 0.2331 and r["min_abs_f"] == pytest.approx(least, rel=1e-4) and r["max_im_f"] < 0
