"""Pins of the CPU oracle against what the mathematics fixes.

None of these tests touches the CUDA path.  Each pin is chosen so that a plausible mistake
in oracle/qmc_oracle.cpp (dropped term, wrong sign or index, transposed operand, wrong
constant) fails at least one of them:

  P1  brute force over the points of tiny lattices (exact rational arithmetic)   A1-A6
  P2  integer coordinates vs Python big-int                                      A1
  P3  Euler-Maclaurin closed form of the Korobov-3 rule for f = 1               A2, A3
  P4  separable exact integral prod (1 + d_i/3)  (BASELINE.json config 0)       A4'
  P5  trigonometric-polynomial exactness / aliasing formula                     A1, A2, A6
  P6  shift-order invariance; A7 against numpy's sample standard deviation      A7
  P7  one-loop Euclidean bubble closed form                                     A4 (logs)
  P8  one-loop Euclidean triangle closed form                                   A4 (powers)
  P9  variance identity of Eq. (4)                               A9
  P10 lambda -> 0 limit and lambda-independence of the deformed class           A5
  P11 det M against a finite-difference Jacobian and the cofactor expansion     A5
  P12 median = middle order statistic, selection equivariant under permutation  A8
"""
import math
import os
from fractions import Fraction

import numpy as np
import pytest

from oracle import oracle as O
from paper_2305_19768_b200 import workloads as W


def _toy(dim, c, d, transform=W.TRANSFORM_KOROBOV3):
    return W.Sector(dim=dim, kind=W.KIND_TOY, transform=transform,
                    U_coef=np.array(list(c) + list(d), float), U_exp=np.zeros((2 * dim, dim), np.uint8))


def _uf(dim, U, F, p, q, logc, first_order, n_orders=1, a=None, transform=W.TRANSFORM_KOROBOV3,
        deformed=0, lam=0.0, f_im=0.0):
    """U, F: lists of (coef, exponent tuple)."""
    aa = np.zeros(8, np.int32)
    if a is not None:
        aa[:dim] = a
    return W.Sector(dim=dim, kind=W.KIND_UF, transform=transform, deformed=deformed,
                    first_order=first_order, n_orders=n_orders, a=aa, p=p, q=q,
                    U_coef=np.array([t[0] for t in U], float), U_exp=np.array([t[1] for t in U], np.uint8).reshape(len(U), dim),
                    F_coef=np.array([t[0] for t in F], float), F_exp=np.array([t[1] for t in F], np.uint8).reshape(len(F), dim),
                    lam=lam, f_im=f_im, logc=np.array(logc, float))


# ------------------------------------------------------------------------------- P1
def _brute_toy(n, z, delta, c, d, transform):
    """Exact rational evaluation of (1/n) sum_k W f(phi(frac(k z/n + Delta))) for the toy class."""
    total = Fraction(0)
    for k in range(n):
        W_, f = Fraction(1), Fraction(1)
        for i in range(len(z)):
            t = Fraction((k * z[i]) % n, n) + Fraction(delta[i])
            if t >= 1:
                t -= 1
            if transform == W.TRANSFORM_KOROBOV3:
                x = t**4 * (35 - 84 * t + 70 * t**2 - 20 * t**3)
                W_ *= 140 * t**3 * (1 - t)**3
            elif transform == W.TRANSFORM_BAKER:
                x = 1 - abs(2 * t - 1)
            else:
                x = t
            f *= 1 + Fraction(c[i]) * (x - Fraction(1, 2)) + Fraction(d[i]) * x * x
        total += W_ * f
    return float(total / n)


@pytest.mark.parametrize("transform", [W.TRANSFORM_NONE, W.TRANSFORM_KOROBOV3, W.TRANSFORM_BAKER])
@pytest.mark.parametrize("n,z", [(1, (0, 0)), (2, (1, 1)), (3, (1, 2)), (5, (2, 3)), (7, (3, 5))])
def test_p1_brute_force_tiny_lattices(n, z, transform):
    c, d = (0.75, -0.5), (0.25, -0.875)          # dyadic: exactly representable
    delta = np.array([[0.3125, 0.84375], [0.5625, 0.09375]])
    sec = O.OracleSector(_toy(2, c, d, transform))
    zz = np.array([max(v, 0) for v in z], np.uint64)
    sums, _ = O.shift_sums(sec, n, zz, delta)
    for s in range(2):
        want = _brute_toy(n, z, delta[s], c, d, transform)
        assert sums[s, 0, 0] / n == pytest.approx(want, rel=2e-15, abs=1e-300)
        assert sums[s, 0, 1] == 0.0


def test_p1_single_point_is_weight_times_integrand():
    """n = 1: Q = W(Delta) f(phi(Delta)) for the U/F class, against the point-wise entry point."""
    w = W.config_euclid(n_sectors=1, n=11)
    sec = O.OracleSector(w.sectors[0])
    delta = w.shifts[:1]
    z = np.ones(8, np.uint64)
    sums, _ = O.shift_sums(sec, 1, z, delta)
    t, x, Wt, wg, _ = O.eval_point(sec, 1, z, delta[0], 0)
    assert np.allclose(t, delta[0, :4], rtol=0, atol=0)
    g, _ = O.integrand(sec, x)
    assert sums[0, 0, 0] == pytest.approx((Wt * g[0]).real, rel=1e-15)
    assert sums[0, 0, 2] == pytest.approx(abs(Wt * g[0]), rel=1e-15)


# ------------------------------------------------------------------------------- P2
def test_p2_integer_coordinates_match_bigint():
    rng = np.random.default_rng(7)
    # beyond 2^32 the product k z no longer fits 64 bits (wide lattices: PAPER.md:279 n = 4.3e9, PAPER.md:300 ~7e10)
    for n in [2, 3, 65521, 1048573, 1000000007, 2**32 - 5, 2**31 - 1, 4294967311, 68719476767, 2**53 - 111]:
        z = np.zeros(8, np.uint64)
        zl = [int(rng.integers(1, n)) for _ in range(5)] if n > 2 else [1] * 5
        z[:5] = zl
        for k0 in [0, max(0, n - 40), int(rng.integers(0, n))]:
            cnt = min(40, n - k0)
            got = O.lattice_coords(n, z, 5, k0, cnt)
            want = np.array([[((k0 + k) * zi) % n for zi in zl] for k in range(cnt)], np.uint64)
            assert np.array_equal(got, want)


# ------------------------------------------------------------------------------- P3
def _korobov3_closed_form(n, delta):
    """1 - 70 B4(theta)/n^4 - 140 B6(theta)/n^6, theta = frac(n Delta), in exact rationals
    (the three terms cancel to a few per cent at n = 1, so floats would lose digits)."""
    th = (n * Fraction(delta)) % 1
    B4 = th**4 - 2 * th**3 + th**2 - Fraction(1, 30)
    B6 = th**6 - 3 * th**5 + Fraction(5, 2) * th**4 - Fraction(1, 2) * th**2 + Fraction(1, 42)
    return float(1 - 70 * B4 / Fraction(n)**4 - 140 * B6 / Fraction(n)**6)


@pytest.mark.parametrize("n", [1, 2, 5, 7, 13])
def test_p3_korobov3_rule_of_constant_has_euler_maclaurin_closed_form(n):
    sec = O.OracleSector(_toy(1, [0.0], [0.0]))
    deltas = np.array([[0.1], [0.37], [0.5], [0.93]])
    sums, _ = O.shift_sums(sec, n, np.array([1], np.uint64), deltas)
    for s in range(len(deltas)):
        assert sums[s, 0, 0] / n == pytest.approx(_korobov3_closed_form(n, deltas[s, 0]), abs=2e-15)


def test_p3_korobov3_map_fixed_points():
    """phi(1/2) = 1/2 with weight 140/64; phi(t) + phi(1-t) = 1 and the weight is symmetric."""
    sec = O.OracleSector(_toy(1, [0.0], [0.0]))
    _, x, Wt, _, _ = O.eval_point(sec, 1, np.array([1], np.uint64), np.array([0.5]), 0)
    assert x[0] == pytest.approx(0.5, abs=1e-16) and Wt == pytest.approx(140.0 / 64.0, rel=1e-15)
    for t in [0.05, 0.2, 0.41]:
        _, xa, Wa, _, _ = O.eval_point(sec, 1, np.array([1], np.uint64), np.array([t]), 0)
        _, xb, Wb, _, _ = O.eval_point(sec, 1, np.array([1], np.uint64), np.array([1.0 - t]), 0)
        assert xa[0] + xb[0] == pytest.approx(1.0, abs=1e-14) and Wa == pytest.approx(Wb, rel=1e-14)


def test_p3_baker_is_the_tent_map():
    sec = O.OracleSector(_toy(1, [0.0], [0.0], W.TRANSFORM_BAKER))
    for t, want in [(0.125, 0.25), (0.5, 1.0), (0.75, 0.5), (0.9375, 0.125)]:
        _, x, Wt, _, _ = O.eval_point(sec, 1, np.array([1], np.uint64), np.array([t]), 0)
        assert x[0] == want and Wt == 1.0


# ------------------------------------------------------------------------------- P4
def test_p4_config0_matches_exact_integral():
    w = W.config_toy()
    sec = O.OracleSector(w.sectors[0])
    _, res, diag = O.integrate(sec, w.jobs[0].n, w.jobs[0].z, w.shifts)
    exact = W.toy_exact(w.sectors[0])
    assert abs(res[0, 0] - exact) <= 1e-13 * abs(exact)
    assert res[0, 1] == 0.0 and res[0, 3] == 0.0 and diag[0] == 0


@pytest.mark.parametrize("transform,tol", [(W.TRANSFORM_KOROBOV3, 5e-9), (W.TRANSFORM_BAKER, 2e-5)])
def test_p4_small_lattices_converge_within_error(transform, tol):
    w = W.config_toy(n=1009, seed=11)
    s = w.sectors[0]
    s.transform = transform
    sec = O.OracleSector(s)
    exact = W.toy_exact(s)
    errs = []
    for n in (101, 1009):
        wl = W.config_toy(n=n, seed=11)
        _, res, _ = O.integrate(sec, n, wl.jobs[0].z, wl.shifts)
        assert abs(res[0, 0] - exact) <= 6.0 * res[0, 2] + 1e-15
        errs.append(res[0, 2])
    assert errs[1] < errs[0] / 20.0 and errs[1] < tol


# ------------------------------------------------------------------------------- P5
def _trig(dim, c0, hs, amps, phases):
    return W.Sector(dim=dim, kind=W.KIND_TRIG, transform=W.TRANSFORM_NONE, logc=np.array([c0]),
                    trig_h=np.array(hs, np.int32).reshape(len(hs), dim), trig_amp=np.array(amps, float),
                    trig_phase=np.array(phases, float))


def test_p5_trig_polynomials_resolved_by_the_lattice_are_integrated_exactly():
    n, z = 101, np.array([1, 40, 0, 0, 0, 0, 0, 0], np.uint64)
    hs = [(1, 0), (0, 3), (2, -1), (-3, 2), (5, 4)]
    assert all((h[0] * 1 + h[1] * 40) % n != 0 for h in hs)
    sec = O.OracleSector(_trig(2, 0.625, hs, [1.0, -0.5, 0.3, 0.7, 0.2], [0.1, 0.2, 0.3, 1.0, 2.0]))
    rng = np.random.default_rng(3)
    shifts = rng.random((8, 2))
    sums, res, _ = O.integrate(sec, n, z, shifts)
    assert np.allclose(sums[:, 0, 0] / n, 0.625, rtol=0, atol=5e-15)
    assert res[0, 2] < 1e-15


def test_p5_aliased_frequency_survives_with_the_shift_phase():
    n, z = 101, np.array([1, 40, 0, 0, 0, 0, 0, 0], np.uint64)
    h_alias = (40, -1)                      # 40*1 - 1*40 = 0 mod n
    hs = [(1, 0), h_alias, (2, 3)]
    amps, ph = [0.4, 0.9, -0.3], [0.3, 0.7, 1.1]
    sec = O.OracleSector(_trig(2, -0.25, hs, amps, ph))
    rng = np.random.default_rng(4)
    shifts = rng.random((6, 2))
    sums, _ = O.shift_sums(sec, n, z, shifts)
    want = -0.25 + 0.9 * np.cos(2 * np.pi * (40 * shifts[:, 0] - shifts[:, 1]) + 0.7)
    assert np.allclose(sums[:, 0, 0] / n, want, rtol=0, atol=2e-13), np.abs(sums[:, 0, 0] / n - want).max()


# ------------------------------------------------------------------------------- P6 / A7
def test_p6_shift_order_invariance_and_sample_std():
    w = W.config_euclid(n_sectors=1, n=1009)
    sec = O.OracleSector(w.sectors[0])
    sums, res, _ = O.integrate(sec, 1009, w.jobs[0].z, w.shifts)
    perm = np.random.default_rng(0).permutation(w.m)
    sums_p, res_p, _ = O.integrate(sec, 1009, w.jobs[0].z, w.shifts[perm])
    assert np.array_equal(sums_p, sums[perm])
    assert np.allclose(res_p, res, rtol=1e-14, atol=0)
    Q = sums[:, 0, 0] / 1009
    assert res[0, 0] == pytest.approx(np.mean(Q), rel=1e-15)
    assert res[0, 2] == pytest.approx(np.std(Q, ddof=1) / math.sqrt(w.m), rel=1e-12)


def _golden():
    """tests/golden/closed_forms.txt: name -> value (written by tests/golden/make_closed_forms.py)."""
    out = {}
    path = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden", "closed_forms.txt")
    for ln in open(path):
        if ln.strip() and not ln.startswith("#"):
            k, v = ln.split()
            out[k] = float(v)
    return out


def test_p3_korobov3_rule_against_stored_values():
    """The same closed form as above, from the stored fixture (deltas as exact decimal fractions)."""
    G = _golden()
    sec = O.OracleSector(_toy(1, [0.0], [0.0]))
    for n in (1, 2, 5, 7, 13):
        for name, delta in (("1/10", 0.1), ("37/100", 0.37), ("1/2", 0.5), ("93/100", 0.93)):
            sums, _ = O.shift_sums(sec, n, np.array([1], np.uint64), np.array([[delta]]))
            assert sums[0, 0, 0] / n == pytest.approx(G["korobov3_const_n%d_d%s" % (n, name)], abs=2e-15)


# ------------------------------------------------------------------------------- P7
def _beta(m2, P2):
    return math.sqrt(1.0 + 4.0 * m2 / P2)


def test_p7_one_loop_euclidean_bubble_finite_part():
    """eps^0 coefficient of the massive bubble: two identical 1-D sectors with U = 1 + t,
    F = m^2 (1+t)^2 + P^2 t, integrand U^-2 (2 log U - log F); closed form
    -[log m^2 - 2 + beta log((beta+1)/(beta-1))]."""
    m2, P2 = 1.3, 2.7
    b = _beta(m2, P2)
    exact = -(math.log(m2) - 2.0 + b * math.log((b + 1.0) / (b - 1.0)))
    assert exact == pytest.approx(-0.552571193868, abs=1e-11)   # value recorded in SURVEY.md P7
    assert exact == pytest.approx(_golden()["bubble_eps0_m2_1.3_P2_2.7"], abs=1e-15)
    sec = O.OracleSector(_uf(1, U=[(1.0, (0,)), (1.0, (1,))],
                             F=[(m2, (0,)), (2 * m2 + P2, (1,)), (m2, (2,))],
                             p=-2.0, q=0.0, logc=[0.0, 2.0, -1.0], first_order=1))
    n = 10007
    shifts = np.random.default_rng(5).random((8, 1))
    _, res, _ = O.integrate(sec, n, np.array([1], np.uint64), shifts)
    assert 2.0 * res[0, 0] == pytest.approx(exact, abs=5e-11)


def test_p8_one_loop_euclidean_triangle():
    """Three 2-D sectors, U = 1 + t1 + t2, p = q = -1, no logs; F = m^2 U^2 + P^2 t1 t2 once and
    m^2 U^2 + P^2 t1 twice; total = log^2((beta+1)/(beta-1)) / (2 P^2)."""
    m2, P2 = 1.3, 2.7
    b = _beta(m2, P2)
    exact = math.log((b + 1.0) / (b - 1.0)) ** 2 / (2.0 * P2)
    assert exact == pytest.approx(0.33196505, abs=1e-8)          # value recorded in SURVEY.md P8
    assert exact == pytest.approx(_golden()["triangle_m2_1.3_P2_2.7"], abs=1e-15)
    U = [(1.0, (0, 0)), (1.0, (1, 0)), (1.0, (0, 1))]
    U2 = {(0, 0): 1.0, (1, 0): 2.0, (0, 1): 2.0, (2, 0): 1.0, (0, 2): 1.0, (1, 1): 2.0}

    def F_with(extra):
        f = {e: m2 * c for e, c in U2.items()}
        f[extra] = f.get(extra, 0.0) + P2
        return [(c, e) for e, c in f.items()]

    n, z = 100003, np.array([1, 38117], np.uint64)
    shifts = np.random.default_rng(6).random((8, 2))
    total, err2 = 0.0, 0.0
    for extra, mult in [((1, 1), 1.0), ((1, 0), 2.0)]:
        sec = O.OracleSector(_uf(2, U=U, F=F_with(extra), p=-1.0, q=-1.0, logc=[1.0], first_order=0))
        _, res, _ = O.integrate(sec, n, z, shifts)
        total += mult * res[0, 0]
        err2 += (mult * res[0, 2]) ** 2
    assert total == pytest.approx(exact, abs=max(6.0 * math.sqrt(err2), 1e-9))
    assert math.sqrt(err2) < 1e-7


# ------------------------------------------------------------------------------- P9
def test_p9_amplitude_and_variance_identity():
    rng = np.random.default_rng(9)
    nj, J = 7, 3
    results = rng.standard_normal((nj, J, 4))
    results[:, :, 2:] = np.abs(results[:, :, 2:])
    coefs = rng.standard_normal(nj) + 1j * rng.standard_normal(nj)
    amp = O.amplitude(results, coefs)
    mean = results[:, :, 0] + 1j * results[:, :, 1]
    want = (coefs[:, None] * mean).sum(axis=0)
    assert np.allclose(amp[:, 0] + 1j * amp[:, 1], want, rtol=1e-14)
    lhs = amp[:, 2] ** 2 + amp[:, 3] ** 2
    rhs = (np.abs(coefs[:, None]) ** 2 * (results[:, :, 2] ** 2 + results[:, :, 3] ** 2)).sum(axis=0)
    assert np.allclose(lhs, rhs, rtol=1e-13)
    # a purely real weight must not mix the real and imaginary errors
    amp_r = O.amplitude(results[:1], np.array([2.0 + 0.0j]))
    assert np.allclose(amp_r[:, 2], 2.0 * results[0, :, 2]) and np.allclose(amp_r[:, 3], 2.0 * results[0, :, 3])
    amp_i = O.amplitude(results[:1], np.array([0.0 + 2.0j]))
    assert np.allclose(amp_i[:, 2], 2.0 * results[0, :, 3]) and np.allclose(amp_i[:, 3], 2.0 * results[0, :, 2])


# ------------------------------------------------------------------------------- P10
def test_p10_lambda_zero_reproduces_the_real_class_per_point():
    rng = np.random.Generator(np.random.PCG64(10))
    real = W.draw_euclid_sector(rng, 4, first_order=0, n_orders=3)
    real.transform = W.TRANSFORM_BAKER
    import copy
    defo = copy.deepcopy(real)
    defo.deformed, defo.lam, defo.f_im = 1, 0.0, 0.0
    so, sd = O.OracleSector(real), O.OracleSector(defo)
    for x in rng.random((20, 4)):
        gr, _ = O.integrand(so, x)
        gd, _ = O.integrand(sd, x)
        assert np.all(gd.imag == 0.0)
        assert np.allclose(gd.real, gr.real, rtol=1e-14, atol=0)


def test_p10_integral_is_independent_of_lambda_on_a_positive_sector():
    rng = np.random.Generator(np.random.PCG64(12))
    base = W.draw_euclid_sector(rng, 3, first_order=0, n_orders=3)
    base.transform = W.TRANSFORM_KOROBOV3
    n, z = 10007, W.draw_z(rng, 10007, 3)
    shifts = W.draw_shifts(rng, 8, 3)
    import copy
    ref = None
    for lam in (0.0, 0.1, 0.5):
        s = copy.deepcopy(base)
        s.deformed, s.lam, s.f_im = 1, lam, 0.0
        _, res, diag = O.integrate(O.OracleSector(s), n, z, shifts)
        assert diag[1] == 0 or lam == 0.0     # Im F < 0 whenever the contour is actually deformed
        if ref is None:
            ref = res
            continue
        scale = np.abs(ref[:, 0]) + 1e-300
        assert np.all(np.abs(res[:, 0] - ref[:, 0]) <= 8.0 * np.hypot(res[:, 2], ref[:, 2]) + 1e-9 * scale)
        assert np.all(np.abs(res[:, 1]) <= 8.0 * res[:, 3] + 1e-9 * scale)


# ------------------------------------------------------------------------------- P14
@pytest.mark.parametrize("dim", [1, 2])
def test_p14_complex_log_polynomial_orders_against_real_axis_quadrature(dim):
    """Pins the complex orders j = 0 .. 4 (d = 1) and 0 .. 2 (d = 2) of the deformed class (A5 with complex Log U,
    Log F, every coefficient non-zero) to something other than the oracle: the integrand is analytic between the real cube and
    the deformed contour, and the deformation vanishes on the boundary, so by Cauchy's theorem the contour integral
    equals the integral of the REAL function x^a U^p F^q L_j(log U, log F) over [0,1]^d, which scipy's adaptive
    quadrature (QUADPACK) computes here directly from the polynomial description.  A wrong branch, a wrong sign in
    z(x) or in the Jacobian, or a transposed log coefficient moves the result away from it; Im must vanish."""
    from scipy import integrate as SI
    rng = np.random.default_rng(14 + dim)
    if dim == 1:
        U = [(1.0, (0,)), (0.7, (1,))]
        F = [(1.0, (0,)), (2.0, (1,)), (0.5, (2,))]
        a = [1]
    else:
        U = [(1.0, (0, 0)), (0.6, (1, 0)), (0.9, (0, 1)), (0.3, (1, 1))]
        F = [(1.0, (0, 0)), (0.8, (2, 0)), (0.5, (1, 1)), (0.7, (0, 3)), (0.4, (1, 0))]
        a = [1, 0]
    p_, q_ = -1.3, -2.1
    J = 5 if dim == 1 else 3                     # d = 1 also pins the highest degrees the description allows (0..4)
    nc = sum((j + 1) * (j + 2) // 2 for j in range(J))
    logc = rng.uniform(0.5, 1.5, size=nc) * rng.choice([-1.0, 1.0], size=nc)
    sec = _uf(dim, U=U, F=F, p=p_, q=q_, logc=list(logc), first_order=0, n_orders=J, a=a,
              transform=W.TRANSFORM_KOROBOV3, deformed=1, lam=0.5, f_im=-1e-30)   # -i0: x = 1 exactly has Im F = 0

    def poly(P, x):
        return sum(c * np.prod([xi ** e for xi, e in zip(x, ex)]) for c, ex in P)

    def real_integrand(j, *x):
        u, f = poly(U, x), poly(F, x)
        lu, lf = math.log(u), math.log(f)
        off = [0, 1, 4, 10, 20][j]
        L, idx = 0.0, off
        for deg in range(j + 1):
            for beta in range(deg + 1):
                L += logc[idx] * lu ** (deg - beta) * lf ** beta
                idx += 1
        return np.prod([xi ** ai for xi, ai in zip(x, a)]) * u ** p_ * f ** q_ * L

    n = 100003
    z = np.array([1, 38117][:dim], np.uint64)
    shifts = np.random.default_rng(15).random((8, dim))
    _, res, diag = O.integrate(O.OracleSector(sec), n, z, shifts)
    # Im F(z) < 0 (admissible contour) except where phi(t) rounds to 1 + 1 ulp for t -> 1: there x (1 - x) ~ -1e-16,
    # the deformation is off by that much and the weight is < 1e-9
    assert diag[1] <= 1e-4 * n * len(shifts)
    for j in range(J):
        if dim == 1:
            exact, qerr = SI.quad(lambda x: real_integrand(j, x), 0.0, 1.0, epsabs=1e-13, epsrel=1e-13)
        else:
            exact, qerr = SI.dblquad(lambda y, x: real_integrand(j, x, y), 0.0, 1.0, 0.0, 1.0, epsabs=1e-11, epsrel=1e-11)
        tol = max(8.0 * math.hypot(res[j, 2], res[j, 3]), 10.0 * qerr, 1e-10)
        assert abs(res[j, 0] - exact) <= tol, (j, res[j], exact)
        assert abs(res[j, 1]) <= tol, (j, res[j])
        assert tol < 1e-6 * abs(exact)                    # the comparison is sharp, not vacuous


# ------------------------------------------------------------------------------- P11
def test_p11_jacobian_determinant_vs_finite_differences():
    rng = np.random.Generator(np.random.PCG64(13))
    for dim in (2, 3, 5):
        s = W.draw_physical_sector(rng, dim, lam=0.5)
        sec = O.OracleSector(s)
        for x in 0.1 + 0.8 * rng.random((4, dim)):
            _, jac = O.deformation(sec, x)
            Jfd = np.zeros((dim, dim), complex)
            h = 1e-6
            for k in range(dim):
                xp, xm = x.copy(), x.copy()
                xp[k] += h
                xm[k] -= h
                zp, _ = O.deformation(sec, xp)
                zm, _ = O.deformation(sec, xm)
                Jfd[:, k] = (zp - zm) / (2 * h)
            assert jac == pytest.approx(np.linalg.det(Jfd), rel=2e-7)


def test_p11_determinant_vs_cofactor_expansion():
    """d = 2, F = 1 + a x0 x1 + b x0^2: gradient, Hessian and det M written out by hand."""
    a, b, lam = 0.7, -0.4, 0.5
    sec = O.OracleSector(_uf(2, U=[(1.0, (0, 0))], F=[(1.0, (0, 0)), (a, (1, 1)), (b, (2, 0))], p=-1.0, q=-1.0,
                             logc=[1.0], first_order=0, deformed=1, lam=lam, transform=W.TRANSFORM_BAKER))
    x0, x1 = 0.3, 0.6
    G0, G1 = a * x1 + 2 * b * x0, a * x0
    H00, H01, H11 = 2 * b, a, 0.0
    M00 = 1 - 1j * lam * ((1 - 2 * x0) * G0 + x0 * (1 - x0) * H00)
    M01 = -1j * lam * x0 * (1 - x0) * H01
    M10 = -1j * lam * x1 * (1 - x1) * H01
    M11 = 1 - 1j * lam * ((1 - 2 * x1) * G1 + x1 * (1 - x1) * H11)
    z, jac = O.deformation(sec, np.array([x0, x1]))
    assert jac == pytest.approx(M00 * M11 - M01 * M10, rel=1e-14)
    assert z[0] == pytest.approx(x0 - 1j * lam * x0 * (1 - x0) * G0, rel=1e-15)
    assert z[1] == pytest.approx(x1 - 1j * lam * x1 * (1 - x1) * G1, rel=1e-15)
    g, _ = O.integrand(sec, np.array([x0, x1]))
    Fz = 1 + a * z[0] * z[1] + b * z[0] ** 2
    assert g[0] == pytest.approx(jac / Fz, rel=1e-14)


# ------------------------------------------------------------------------------- P12
def test_p12_median_is_the_middle_order_statistic_and_selection_is_equivariant():
    w = W.config_median(n_sectors=1, dim=3, n=1009, K=11)
    sec = O.OracleSector(w.sectors[0])
    est, med, sel = O.median_rule(sec, 1009, w.z_cand[0], w.shift0[0])
    vals = est[:, 0].real
    order = np.argsort(vals)
    assert med[0].real == vals[order[5]] and sel == order[5] and med[0].imag == 0.0
    # each candidate estimate is the one-shift rule of that z
    s5, _ = O.shift_sums(sec, 1009, w.z_cand[0, 5], w.shift0[:1])
    assert est[5, 0].real == s5[0, 0, 0] / 1009
    perm = np.random.default_rng(1).permutation(11)
    est_p, med_p, sel_p = O.median_rule(sec, 1009, w.z_cand[0][perm], w.shift0[0])
    assert med_p[0] == med[0] and perm[sel_p] == sel
    # even K: mean of the two middle values
    est_e, med_e, _ = O.median_rule(sec, 1009, w.z_cand[0][:10], w.shift0[0])
    v = np.sort(est_e[:, 0].real)
    assert med_e[0].real == pytest.approx(0.5 * (v[4] + v[5]), rel=1e-15)


def test_p12_componentwise_median_for_complex_orders():
    w = W.config_physical(n_sectors=1, dim=3, n=211)
    sec = O.OracleSector(w.sectors[0])
    rng = np.random.Generator(np.random.PCG64(5))
    zc = np.stack([W.draw_z(rng, 211, 3) for _ in range(7)])
    est, med, sel = O.median_rule(sec, 211, zc, w.shifts[0])
    assert np.allclose(med.real, np.median(est.real, axis=0), rtol=0, atol=0)
    assert np.allclose(med.imag, np.median(est.imag, axis=0), rtol=0, atol=0)
    comp = np.concatenate([est.real, est.imag], axis=1)
    mad = np.median(np.abs(comp - np.median(comp, axis=0)), axis=0)
    dist = (((comp - np.median(comp, axis=0)) / mad) ** 2).sum(axis=1)
    assert sel == int(np.argmin(dist))
